"""Pins for C3-C5 (descriptors; Eqs. 15-20) against routes that share nothing with the oracle:
Legendre addition theorem, scipy's complex spherical harmonics, Wigner-3j contraction, cosine triple sums,
dimer closed forms, and the invariances the paper states."""
import math

import numpy as np
import pytest
from scipy.special import eval_legendre, sph_harm_y

from oracle import nep_oracle as O
from paper_2606_19557_b200 import workloads as wl
from tests._ref_np import np_fk, np_neighbors

K4 = -45.0 / (8.0 * math.sqrt(14.0) * math.pi ** 1.5)
K5 = 21.0 / (80.0 * math.pi ** 2)


def _theta_with_coeffs(model, seed):
    rng = np.random.default_rng(seed)
    th = np.zeros(model.n_par)
    sl = model.block_slices()
    th[sl["cR"]] = rng.uniform(-1, 1, sl["cR"].stop - sl["cR"].start)
    th[sl["cA"]] = rng.uniform(-1, 1, sl["cA"].stop - sl["cA"].start)
    return th


def _coeffs(model, th):
    sl = model.block_slices()
    T = model.n_species
    return (th[sl["cR"]].reshape(T, T, model.n_R, model.K_R), th[sl["cA"]].reshape(T, T, model.n_A, model.K_A))


def _set(pos, cell, types):
    pos = np.asarray(pos, float)
    return wl.StructureSet(np.array([len(pos)], np.int32), pos, np.asarray(cell, float).reshape(1, 9),
                           np.asarray(types, np.int32), ["x"])


@pytest.fixture(scope="module")
def small():
    model = wl.ModelSpec(2, 3.4, 2.9, 2, 3, 4, 5, 4, 2, 1, 3)
    w = wl.tiny_workload(7, sizes=(6,), box=(3.3,), model=model)
    th = _theta_with_coeffs(model, 11)
    data = O.OracleData(model, w.structures)
    return model, w.structures, th, O.descriptors(data, th)


def _per_atom_neighbors(st, rc):
    out = [[] for _ in range(len(st.pos))]
    for i, j, s, d in np_neighbors(st.pos, st.box[0], rc, wide=5):
        out[i].append((j, d))
    return out


def test_radial_descriptor_plain_sum(small):
    model, st, th, q = small
    cR, _ = _coeffs(model, th)
    for i, lst in enumerate(_per_atom_neighbors(st, model.rc_R)):
        ref = np.zeros(model.n_R)
        for j, d in lst:
            ref += cR[st.type[i], st.type[j]] @ np_fk(np.linalg.norm(d), model.rc_R, model.basis_R)
        assert np.allclose(q[i, :model.n_R], ref, atol=1e-12)


def test_three_body_addition_theorem_and_scipy_harmonics(small):
    model, st, th, q = small
    _, cA = _coeffs(model, th)
    nR, nA = model.n_R, model.n_A
    for i, lst in enumerate(_per_atom_neighbors(st, model.rc_A)):
        if not lst:
            continue
        dv = np.array([d for _, d in lst]); r = np.linalg.norm(dv, axis=1); u = dv / r[:, None]
        g = np.array([cA[st.type[i], st.type[j]] @ np_fk(rr, model.rc_A, model.basis_A) for (j, _), rr in zip(lst, r)])  # [nb, nA]
        cos = np.clip(u @ u.T, -1, 1)
        theta = np.arccos(np.clip(u[:, 2], -1, 1)); phi = np.arctan2(u[:, 1], u[:, 0])
        for l in range(1, 5):
            for n in range(nA):
                ref1 = (2 * l + 1) / (4 * np.pi) * g[:, n] @ eval_legendre(l, cos) @ g[:, n]   # addition theorem
                A = np.array([np.sum(g[:, n] * sph_harm_y(l, m, theta, phi)) for m in range(-l, l + 1)])
                ref2 = np.sum(np.abs(A) ** 2)                                                # Eq. 20 literally
                got = q[i, nR + (l - 1) * nA + n]
                assert abs(got - ref1) < 1e-11 * max(1, abs(ref1))
                assert abs(got - ref2) < 1e-11 * max(1, abs(ref2))


def test_four_and_five_body_closed_forms(small):
    model, st, th, q = small
    _, cA = _coeffs(model, th)
    nR, nA = model.n_R, model.n_A
    from sympy.physics.wigner import wigner_3j
    w3 = {(a, b, c): float(wigner_3j(2, 2, 2, a, b, c)) for a in range(-2, 3) for b in range(-2, 3) for c in range(-2, 3) if a + b + c == 0}
    for i, lst in enumerate(_per_atom_neighbors(st, model.rc_A)):
        if not lst:
            continue
        dv = np.array([d for _, d in lst]); r = np.linalg.norm(dv, axis=1); u = dv / r[:, None]
        g = np.array([cA[st.type[i], st.type[j]] @ np_fk(rr, model.rc_A, model.basis_A) for (j, _), rr in zip(lst, r)])
        c = u @ u.T
        theta = np.arccos(np.clip(u[:, 2], -1, 1)); phi = np.arctan2(u[:, 1], u[:, 0])
        for n in range(nA):
            gn = g[:, n]
            # cosine triple sum: tr T^3 = sum_jkl g g g [c_jk c_kl c_lj - (c_jk^2 + c_kl^2 + c_lj^2)/3 + 2/9]
            t3 = (np.einsum("j,k,l,jk,kl,lj->", gn, gn, gn, c, c, c)
                  - np.einsum("j,k,l,jk->", gn, gn, gn, c ** 2) + 2.0 / 9.0 * gn.sum() ** 3)
            got4 = q[i, nR + 4 * nA + n]
            assert abs(got4 - K4 * t3) < 1e-11 * max(1, abs(got4))
            # Wigner-3j contraction of the orthonormal l = 2 moments (what "higher-order contraction", means)
            A2 = {m: np.sum(gn * sph_harm_y(2, m, theta, phi)) for m in range(-2, 3)}
            w = sum(v * A2[a] * A2[b] * A2[cc] for (a, b, cc), v in w3.items())
            assert abs(w.imag) < 1e-12 and abs(got4 - w.real) < 1e-10 * max(1, abs(got4))
            # 5-body: kappa5 |s|^4 with s = sum g r^ ; also (7/15) (sum_m |A_1m|^2)^2
            s = gn @ u
            got5 = q[i, nR + 5 * nA + n]
            assert abs(got5 - K5 * (s @ s) ** 2) < 1e-12 * max(1, abs(got5))
            assert abs(got5 - 7.0 / 15.0 * q[i, nR + 0 * nA + n] ** 2) < 1e-12 * max(1, abs(got5))


def test_dimer_closed_forms():
    model = wl.ModelSpec(1, 4.0, 3.5, 2, 2, 4, 4, 4, 2, 1, 3)
    th = _theta_with_coeffs(model, 3)
    cR, cA = _coeffs(model, th)
    rvec = np.array([0.7, -1.1, 1.9]); r = np.linalg.norm(rvec)
    st = _set([[5, 5, 5], np.array([5, 5, 5]) + rvec], np.eye(3) * 20.0, [0, 0])
    q = O.descriptors(O.OracleData(model, st), th)
    gR = cR[0, 0] @ np_fk(r, model.rc_R, model.basis_R); gA = cA[0, 0] @ np_fk(r, model.rc_A, model.basis_A)
    for i in range(2):
        assert np.allclose(q[i, :3], gR, atol=1e-13)
        for l in range(1, 5):
            assert np.allclose(q[i, 3 + (l - 1) * 3: 3 + l * 3], (2 * l + 1) / (4 * np.pi) * gA ** 2, atol=1e-13)
        assert np.allclose(q[i, 3 + 12: 3 + 15], 2.0 / 9.0 * K4 * gA ** 3, atol=1e-13)
        assert np.allclose(q[i, 3 + 15: 3 + 18], K5 * gA ** 4, atol=1e-13)


def test_invariances(small):
    model, st, th, q = small
    # translation (then re-wrap), rigid rotation of positions and cell, same-species relabelling
    cell = st.box[0].reshape(3, 3)
    shifted = _set(wl._wrap(st.pos + np.array([0.37, -1.2, 2.2]), cell), cell, st.type)
    assert np.allclose(O.descriptors(O.OracleData(model, shifted), th), q, atol=1e-11)
    A = np.random.default_rng(2).normal(size=(3, 3)); Q, _ = np.linalg.qr(A)
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1
    rot = _set(st.pos @ Q.T, cell @ Q.T, st.type)
    assert np.allclose(O.descriptors(O.OracleData(model, rot), th), q, atol=1e-11)
    perm = np.array([3, 1, 2, 0, 5, 4])
    pq = O.descriptors(O.OracleData(model, _set(st.pos[perm], cell, st.type[perm])), th)
    assert np.allclose(pq, q[perm], atol=1e-12)


def test_descriptor_vanishes_smoothly_at_cutoff():
    model = wl.ModelSpec(1, 4.0, 3.5, 2, 2, 4, 4, 4, 2, 1, 3)
    th = _theta_with_coeffs(model, 3)
    vals = []
    for eps in (1e-2, 1e-3, 1e-4):
        st = _set([[5, 5, 5], [5, 5, 5 + model.rc_A - eps]], np.eye(3) * 20.0, [0, 0])
        q = O.descriptors(O.OracleData(model, st), th)
        vals.append(np.abs(q[0, 3:]).max())
    assert vals[0] > vals[1] > vals[2] and vals[2] < 1e-12     # angular part ~ eps^4 (g ~ eps^2, squared)
    st = _set([[5, 5, 5], [5, 5, 5 + model.rc_R + 1e-9]], np.eye(3) * 20.0, [0, 0])
    assert np.abs(O.descriptors(O.OracleData(model, st), th)).max() == 0.0


def test_harmonic_table_against_scipy_and_gradient_fd():
    # real functions b_L with weights w_L reproduce sum_m |Y_lm|^2 pairwise: sum_L w_L b_L(u) b_L(v) = (2l+1)/(4pi) P_l(u.v)
    rng = np.random.default_rng(8)
    w = O.harmonic_weights(4)
    u = rng.normal(size=3); v = rng.normal(size=3)
    bu, dbu = O.angular_functions(u); bv, _ = O.angular_functions(v)
    cosg = u @ v / np.linalg.norm(u) / np.linalg.norm(v)
    L = 0
    for l in range(1, 5):
        s = sum(w[L + k] * bu[L + k] * bv[L + k] for k in range(2 * l + 1))
        assert abs(s - (2 * l + 1) / (4 * np.pi) * eval_legendre(l, cosg)) < 1e-13
        L += 2 * l + 1
    h = 1e-6
    for a in range(3):
        e = np.zeros(3); e[a] = h
        fd = (O.angular_functions(u + e)[0] - O.angular_functions(u - e)[0]) / (2 * h)
        assert np.allclose(dbu[:, a], fd, atol=1e-8)
    assert np.allclose(dbu @ u, 0.0, atol=1e-12)             # tangential: functions of the direction only


# ---- C6: the descriptor scaler of Eq. 2, reading G10 ----
def test_scaler_closed_form_on_hand_built_columns():
    """q_nu~ = q_nu / (q_nu^max - q_nu^min) (Eq. 2): the range is over every atom, all species together (Eq. 2 has
    no species index), not the maximum alone; a constant column has no range and gets s = 1 (reading G10)."""
    q = np.array([
        # positive range | straddles zero | constant | two "species" mixed in one column | negative only
        [2.0, -1.5, 0.75, 10.0, -4.0],
        [5.0, 0.25, 0.75, 11.0, -1.0],
        [3.5, 2.5, 0.75, -3.0, -2.5],
        [4.0, 0.0, 0.75, -2.0, -3.0],
    ])
    s = O.scaler(q)
    expect = np.array([1.0 / (5.0 - 2.0), 1.0 / (2.5 + 1.5), 1.0, 1.0 / (11.0 + 3.0), 1.0 / (-1.0 + 4.0)])
    assert np.allclose(s, expect, rtol=1e-15, atol=0)
    # the mutations a plausible slip would make all differ from the closed form on these columns
    assert not np.allclose(expect, 1.0 / q.max(0))                                  # 1 / max
    assert not np.allclose(expect, 1.0 / np.abs(q).max(0))                          # 1 / max |q|
    per_species = 1.0 / np.minimum(np.ptp(q[:2], axis=0) + 1e-300, np.ptp(q[2:], axis=0) + 1e-300)
    assert not np.allclose(expect[3], per_species[3])                               # per-species ranges (rows 0-1 / 2-3)
    # scale covariance and shift invariance of a range
    assert np.allclose(O.scaler(3.0 * q + 7.0)[[0, 1, 3, 4]], expect[[0, 1, 3, 4]] / 3.0, rtol=1e-14)
    # one atom: every range is degenerate
    assert np.array_equal(O.scaler(q[:1]), np.ones(5))


def test_scaler_degenerate_threshold():
    """Reading G10: range <= 1e-12 max(1, max|q|) counts as constant (s = 1); anything wider is inverted."""
    q = np.array([[1.0, 1.0, 1e6, 1e6], [1.0 + 5e-13, 1.0 + 4e-12, 1e6 + 5e-7, 1e6 + 4e-6]])
    s = O.scaler(q)
    assert s[0] == 1.0 and s[2] == 1.0
    assert np.isclose(s[1], 1.0 / (q[1, 1] - q[0, 1]), rtol=1e-12) and np.isclose(s[3], 1.0 / (q[1, 3] - q[0, 3]), rtol=1e-12)


def test_scaler_of_descriptors_is_inverse_range(small):
    """On a real descriptor matrix: s = 1 / ptp(q) over all atoms of all species (the set has 2 species)."""
    model, st, th, q = small
    assert len(np.unique(st.type)) == 2
    s = O.scaler(q)
    assert s.shape == (model.D,)
    assert np.allclose(s, 1.0 / np.ptp(q, axis=0), rtol=1e-13)
    assert np.allclose((q * s).max(0) - (q * s).min(0), 1.0, rtol=1e-12)            # q~ spans exactly one unit (Eq. 2)


@pytest.mark.parametrize("l3,l4,l5", [(1, 0, 1), (2, 2, 0), (3, 2, 1), (2, 0, 0)])
def test_other_three_body_orders_are_row_subsets(small, l3, l4, l5):
    """l_max = (l3, l4, l5) with l3 < 4 (Table I): the descriptor coefficients do not depend on l_max, so with the
    same cR, cA every component the smaller model keeps must equal the same component of the (4, 2, 1) model, which the tests above pin
    (addition theorem, scipy harmonics, Wigner-3j, cosine sums), in the row order of DESIGN C0:
    radial n | 3-body (l, n), l = 1..l3 | 4-body n | 5-body n."""
    model, st, th, q = small
    sub = wl.ModelSpec(model.n_species, model.rc_R, model.rc_A, model.n_max_R, model.n_max_A, model.basis_R, model.basis_A, l3, l4, l5, model.neurons)
    ths = np.zeros(sub.n_par)
    a, b = model.block_slices(), sub.block_slices()
    ths[b["cR"]] = th[a["cR"]]; ths[b["cA"]] = th[a["cA"]]
    qs = O.descriptors(O.OracleData(sub, st), ths)
    nR, nA = model.n_R, model.n_A
    assert sub.D == nR + nA * (l3 + (l4 > 0) + (l5 > 0)) and qs.shape[1] == sub.D
    rows = list(range(nR + l3 * nA))                                  # radial and l = 1..l3 sit at the same indices
    if l4:
        rows += list(range(nR + 4 * nA, nR + 5 * nA))                 # 4-body block of the (4, 2, 1) model
    if l5:
        rows += list(range(nR + 5 * nA, nR + 6 * nA))                 # 5-body block
    assert np.allclose(qs, q[:, rows], rtol=0, atol=1e-13)
    assert np.abs(qs).max() > 1e-3
