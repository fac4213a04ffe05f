"""Host logic: the seeded workload generators (DESIGN.md input recipe; stand-ins for the paper's DFT sets)."""
import numpy as np

from paper_2606_19557_b200 import workloads as wl


def _frac_ok(st):
    ao = st.atom_off
    for s in range(st.n_struct):
        f = st.pos[ao[s]:ao[s + 1]] @ np.linalg.inv(st.box[s].reshape(3, 3))
        assert (f >= 0).all() and (f < 1).all()
        assert np.linalg.det(st.box[s].reshape(3, 3)) > 0


def test_config_shapes_and_prefix_determinism():
    w1 = wl.make_config(1)
    assert w1.structures.n_struct == 8 and (w1.structures.n_atoms == 64).all() and w1.model.D == 25 and w1.model.n_par == 901
    assert wl.make_config(1, variant="1b").structures.n_atoms[0] == 256
    w2 = wl.make_config(2, n_struct=3)
    assert (w2.structures.n_atoms == 128).all() and w2.model.D == 35 and w2.model.n_par == 1201
    w2b = wl.make_config(2, n_struct=5)
    assert np.array_equal(w2b.structures.pos[:384], w2.structures.pos)         # prefix property
    w3 = wl.make_config(3, n_struct=30)
    assert set(np.unique(w3.structures.n_atoms)) <= {107, 108, 143, 144, 191, 192, 255, 256}
    assert w3.model.D == 37 and w3.model.n_par == 4389 and set(np.unique(w3.structures.type)) == {0, 1}
    w4 = wl.make_config(4, n_struct=30)
    assert w4.structures.n_atoms.min() >= 128 and w4.structures.n_atoms.max() <= 512 and w4.model.n_par == 7801
    w5 = wl.make_config(5, n_struct=30)
    assert w5.structures.n_atoms.min() >= 32 and w5.structures.n_atoms.max() <= 512 and w5.model.n_par == 5881
    for w in (w1, w2, w3, w4, w5):
        _frac_ok(w.structures)
    assert sorted(m.n_par for m in wl.config5_sweep())[0] == 5881 and sorted(m.n_par for m in wl.config5_sweep())[-1] == 29745


def test_liquid_min_separation():
    rng = np.random.default_rng(0)
    pos, cell = wl._liquid(rng, 150)
    L = cell[0, 0]
    d = pos[:, None, :] - pos[None, :, :]
    d -= L * np.round(d / L)
    r = np.sqrt((d ** 2).sum(-1)) + np.eye(150) * 10
    assert r.min() >= 1.8 and abs(150 / L ** 3 - 0.08) < 1e-12


def test_batches_partition():
    w = wl.make_config(3, n_struct=23)
    w.batch_size = 5
    bs = wl.batches(w)
    assert sorted(np.concatenate(bs).tolist()) == list(range(23)) and [len(b) for b in bs] == [5, 5, 5, 5, 3]


def test_param_draw_is_seeded_and_two_phase():
    w = wl.tiny_workload(0)
    a = wl.ParamDraw(w.model, w.seeds["student"]); a.coefficients(); ta = a.network(np.zeros(w.model.D)).copy()
    b = wl.ParamDraw(w.model, w.seeds["student"]); b.coefficients(); tb = b.network(np.zeros(w.model.D)).copy()
    assert np.array_equal(ta, tb) and np.abs(ta).max() <= 1.5
