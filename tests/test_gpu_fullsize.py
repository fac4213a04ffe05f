"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times: the whole structure set of the config
is loaded into the library, the batch is the first full batch of the seeded permutation (bench.py's), and the oracle
computes that batch (it is fast enough to do all of it: no sampling needed): neighbour lists of the batch's structures
bit-exact, E <= 1e-5 eV/atom, F and W <= 1e-4 relative in norm, gradient <= 1e-3 relative in norm, sum of forces zero."""
import numpy as np
import pytest

from oracle import nep_oracle as O
from paper_2606_19557_b200 import workloads as wl
from tests import _gpu_harness as H

pytestmark = pytest.mark.gpu


def _draw(model, data, seed):
    pd = wl.ParamDraw(model, seed)
    th = pd.coefficients()
    q = O.descriptors(data, th)
    s = O.scaler(q)
    return pd.network((q * s).mean(axis=0)).copy(), s


@pytest.mark.parametrize("cfg", [2, 3, 4, "5 smallest model", "5 largest model", "5 model 6"])
def test_full_size_batch_against_oracle(cfg):
    from paper_2606_19557_b200.binding import Nep
    if isinstance(cfg, str):          # config 5: the two ends of the model-complexity sweep (n_max 4 / 8, basis 8 / 12, 30 / 100 neurons)
        # ... and model 6 (n_max 8, basis 12, 30 neurons: D = 63, 13 radial functions), the widest tile the tensor-core kernels run
        w = wl.make_config(5, model=wl.config5_sweep()[0 if "smallest" in cfg else 6 if "model 6" in cfg else -1])
    else:
        w = wl.make_config(cfg)
    st = w.structures
    batch = wl.batches(w)[0]
    assert len(batch) == w.batch_size
    sub = st.subset(batch)                                   # the oracle sees the batch's structures, in batch order
    data = O.OracleData(w.model, sub)
    th_t, s_t = _draw(w.model, data, w.seeds["teacher"])
    E, F, W = O.forward(data, th_t, s_t)                     # teacher labels of the batch (oracle, fp64)
    th, s = _draw(w.model, data, w.seeds["student"])
    th = th.astype(np.float32).astype(np.float64)
    data.set_labels(E, F, W)
    # the library holds the WHOLE set; labels outside the batch are never read by this step
    off = st.atom_off
    E_all = np.zeros(st.n_struct); F_all = np.zeros((int(off[-1]), 3)); W_all = np.zeros((st.n_struct, 9))
    E_all[batch] = E; W_all[batch] = W
    rows = np.concatenate([np.arange(off[sid], off[sid + 1]) for sid in batch])
    F_all[rows] = F
    with Nep.from_model(w.model) as nep:
        nep.load_structure_set(st, E_all, F_all, W_all)
        nep.build_neighbors()
        nep.set_params(th.astype(np.float32)); nep.set_scaler(s)
        nep.set_batch(batch)
        assert nep.batch_shape() == (len(batch), int(sub.n_atoms.sum()))
        # neighbour lists of the batch's structures (the accessor returns the whole set: compare structure by structure)
        for which, (ooff, oj, osh) in enumerate(((data.offR, data.jR, data.shR), (data.offA, data.jA, data.shA))):
            goff, gj, gsh = nep.get_neighbors(which)
            for k, sid in enumerate(batch[:: max(1, len(batch) // 40)]):        # every ~25th structure of the batch, whole lists
                kk = int(np.nonzero(batch == sid)[0][0])
                b0 = int(sub.atom_off[kk]); n = int(st.n_atoms[sid]); g0 = int(off[sid])
                assert np.array_equal(goff[g0:g0 + n + 1] - goff[g0], ooff[b0:b0 + n + 1] - ooff[b0])
                sl_g = slice(int(goff[g0]), int(goff[g0 + n])); sl_o = slice(int(ooff[b0]), int(ooff[b0 + n]))
                assert np.array_equal(gj[sl_g], oj[sl_o]) and np.array_equal(gsh[sl_g], osh[sl_o])
        Eg, Fg, Wg = nep.forward()
        Eo, Fo, Wo = O.forward(data, th, s)
        eE = float(np.max(np.abs(Eg - Eo) / sub.n_atoms))
        assert eE <= H.TOL_E_PER_ATOM, eE
        assert H.relnorm(Fg, Fo) <= H.TOL_FW_REL and H.relnorm(Wg, Wo) <= H.TOL_FW_REL
        # Newton's third law per structure, at any size: |sum F| is round-off of the terms added
        so = sub.atom_off
        for k in range(0, len(batch), max(1, len(batch) // 50)):
            f = Fg[so[k]:so[k + 1]]
            assert np.abs(f.sum(axis=0)).max() <= 1e-4 * max(1.0, np.abs(f).sum(axis=0).max())
        l4 = nep.loss_grad(*w.lambdas)
        g = nep.get_grad()
        l4o, go = O.loss_grad(data, th, s, w.lambdas)
        assert np.allclose(l4, l4o, rtol=2e-4), (l4, l4o)
        assert H.relnorm(g, go) <= H.TOL_G_REL, H.relnorm(g, go)
