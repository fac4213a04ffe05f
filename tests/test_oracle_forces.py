"""Pins for C7-C8 (ANN, forces, virial; Eqs. 1-3): finite differences of E,
strain derivative, sum rules, symmetry cases, ANN special cases."""
import copy

import numpy as np
import pytest

from oracle import nep_oracle as O
from oracle.problem import make_problem
from paper_2606_19557_b200 import workloads as wl


@pytest.fixture(scope="module")
def prob():
    return make_problem(wl.tiny_workload(0))


def _energy(w, th, sc, pos, box=None):
    st = copy.deepcopy(w.structures)
    st.pos = pos
    if box is not None:
        st.box = box
    return O.forward(O.OracleData(w.model, st), th, sc)[0]


def test_forces_equal_central_fd_of_energy(prob):
    w = prob.workload
    E, F, W = O.forward(prob.data, prob.theta, prob.scaler)
    h = 1e-5
    Ffd = np.zeros_like(F)
    for i in range(len(F)):
        for a in range(3):
            p = w.structures.pos.copy(); p[i, a] += h
            Ep = _energy(w, prob.theta, prob.scaler, p).sum()
            p[i, a] -= 2 * h
            Em = _energy(w, prob.theta, prob.scaler, p).sum()
            Ffd[i, a] = -(Ep - Em) / (2 * h)
    assert np.linalg.norm(F - Ffd) / np.linalg.norm(F) < 1e-8
    ao = w.structures.atom_off
    for s in range(w.structures.n_struct):
        assert np.abs(F[ao[s]:ao[s + 1]].sum(0)).max() < 1e-12     # sum F = 0 per structure


def test_virial_equals_minus_strain_derivative_and_is_symmetric(prob):
    w = prob.workload
    _, _, W = O.forward(prob.data, prob.theta, prob.scaler)
    ao = w.structures.atom_off
    h = 1e-5
    for s in range(w.structures.n_struct):
        Wfd = np.zeros((3, 3))
        for a in range(3):
            for b in range(3):
                Es = []
                for sg in (1, -1):
                    eps = np.eye(3); eps[a, b] += sg * h           # r -> (I + eps) r for positions and cell
                    p = w.structures.pos.copy(); bx = w.structures.box.copy()
                    p[ao[s]:ao[s + 1]] = p[ao[s]:ao[s + 1]] @ eps.T
                    bx[s] = (bx[s].reshape(3, 3) @ eps.T).reshape(9)
                    Es.append(_energy(w, prob.theta, prob.scaler, p, bx)[s])
                Wfd[a, b] = -(Es[0] - Es[1]) / (2 * h)
        Ws = W[s].reshape(3, 3)
        assert np.linalg.norm(Ws - Wfd) / np.linalg.norm(Wfd) < 1e-8
        assert np.abs(Ws - Ws.T).max() < 1e-12


def test_virial_is_minus_sum_d_outer_p_for_a_dimer():
    # two atoms, big box: F_0 = p, F_1 = -p, W = -(d (x) p) summed over both directed pairs = -2 d(x)p_01
    model = wl.ModelSpec(1, 4.0, 3.5, 2, 2, 4, 4, 4, 2, 1, 3)
    w = wl.tiny_workload(1, n_species=1, sizes=(2,), box=(20.0,), model=model)
    st = w.structures
    st.pos[:] = [[5, 5, 5], [5.9, 6.3, 4.2]]
    pr = make_problem(w)
    E, F, W = O.forward(pr.data, pr.theta, pr.scaler)
    d = st.pos[1] - st.pos[0]
    assert np.allclose(F[0], -F[1], atol=1e-14)
    # directed pair 0->1 has p_01 with F_0 = p_01 - p_10 and by symmetry p_10 = -p_01
    assert np.allclose(W[0].reshape(3, 3), -np.outer(d, F[0]), atol=1e-13)
    assert np.allclose(np.cross(d, F[0]), 0, atol=1e-13)           # central force


def test_perfect_lattices_zero_force_isotropic_virial():
    for lat, a, model in (("fcc", 3.6, wl.ModelSpec(1, 5.0, 4.0, 2, 2, 4, 4, 4, 2, 1, 5)),
                          ("bcc", 3.16, wl.ModelSpec(1, 5.0, 4.0, 2, 2, 4, 4, 4, 2, 1, 5))):
        pos, cell = wl._lattice(lat, a, (2, 2, 2))
        st = wl.StructureSet(np.array([len(pos)], np.int32), wl._wrap(pos, cell), cell.reshape(1, 9),
                             np.zeros(len(pos), np.int32), [lat])
        w = wl.Workload(0, lat, model, st, 1, (1, 1, 1), dict(zip(("teacher", "student", "batch"), np.random.SeedSequence(5).spawn(3))))
        data = O.OracleData(model, st)
        rng = np.random.default_rng(0)
        th = rng.uniform(-1, 1, model.n_par)
        sc = np.ones(model.D)
        E, F, W = O.forward(data, th, sc)
        assert np.abs(F).max() < 1e-11
        Wm = W[0].reshape(3, 3)
        assert np.abs(Wm - np.eye(3) * np.trace(Wm) / 3).max() < 1e-10 * max(1.0, abs(np.trace(Wm)))


def test_ann_special_cases(prob):
    w = prob.workload; m = w.model; sl = m.block_slices()
    th = prob.theta.copy()
    for t in range(m.n_species):
        th[sl["w0"][t]] = 0.0
    E, F, W = O.forward(prob.data, th, prob.scaler)
    ao = w.structures.atom_off
    for s in range(w.structures.n_struct):
        ref = 0.0
        for i in range(ao[s], ao[s + 1]):
            t = w.structures.type[i]
            ref += th[sl["w1"][t]] @ np.tanh(-th[sl["b0"][t]]) - th[sl["b1"]][0]   # Eq. 3 with w0 = 0
        assert abs(E[s] - ref) < 1e-13
    assert np.abs(F).max() == 0.0 and np.abs(W).max() == 0.0
    # linear regime: tiny w0, b0 = 0 -> E_i ~ sum_mu w1 (w0 . q~) - b1
    th = prob.theta.copy()
    for t in range(m.n_species):
        th[sl["w0"][t]] *= 1e-6
        th[sl["b0"][t]] = 0.0
    q = O.descriptors(prob.data, th) * prob.scaler
    E, _, _ = O.forward(prob.data, th, prob.scaler)
    for s in range(w.structures.n_struct):
        ref = 0.0
        for i in range(ao[s], ao[s + 1]):
            t = w.structures.type[i]
            ref += th[sl["w1"][t]] @ (th[sl["w0"][t]].reshape(m.neurons, m.D) @ q[i]) - th[sl["b1"]][0]
        assert abs(E[s] - ref) < 1e-12


def test_energy_invariances(prob):
    w = prob.workload; st = w.structures
    E0, F0, W0 = O.forward(prob.data, prob.theta, prob.scaler)
    rng = np.random.default_rng(4)
    A = rng.normal(size=(3, 3)); Q, _ = np.linalg.qr(A)
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1
    rot = copy.deepcopy(st)
    rot.pos = st.pos @ Q.T
    rot.box = np.array([(b.reshape(3, 3) @ Q.T).reshape(9) for b in st.box])
    E1, F1, W1 = O.forward(O.OracleData(w.model, rot), prob.theta, prob.scaler)
    assert np.allclose(E1, E0, atol=1e-11)
    assert np.allclose(F1, F0 @ Q.T, atol=1e-11)                   # forces rotate covariantly
    for s in range(st.n_struct):
        assert np.allclose(W1[s].reshape(3, 3), Q @ W0[s].reshape(3, 3) @ Q.T, atol=1e-10)
    sh = copy.deepcopy(st)
    ao = st.atom_off
    for s in range(st.n_struct):
        sh.pos[ao[s]:ao[s + 1]] = wl._wrap(st.pos[ao[s]:ao[s + 1]] + rng.uniform(-3, 3, 3), st.box[s].reshape(3, 3))
    E2, F2, W2 = O.forward(O.OracleData(w.model, sh), prob.theta, prob.scaler)
    assert np.allclose(E2, E0, atol=1e-11) and np.allclose(F2, F0, atol=1e-10) and np.allclose(W2, W0, atol=1e-10)


def test_batch_subset_and_order(prob):
    E0, F0, W0 = O.forward(prob.data, prob.theta, prob.scaler)
    E1, F1, W1 = O.forward(prob.data, prob.theta, prob.scaler, batch=[1, 0])
    ao = prob.workload.structures.atom_off
    assert np.array_equal(E1, E0[[1, 0]]) and np.array_equal(W1, W0[[1, 0]])
    assert np.array_equal(F1, np.concatenate([F0[ao[1]:ao[2]], F0[ao[0]:ao[1]]]))
