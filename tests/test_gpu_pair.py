"""Short-range pair correction on the GPU against the oracle (oracle/pair_correction.py): the term adds to
E, F, W; the loss and its gradient see the corrected predictions; it has no parameter, so with labels shifted by the correction
the oracle's loss_grad is the reference (L(E_nep + E_c - E_lab) = L(E_nep - (E_lab - E_c))).  The constants are seeded numbers, not
those of Ref. [24]: the library stores none (DESIGN G29).  Tolerances: north_star's."""
import numpy as np
import pytest

from oracle import nep_oracle as O
from oracle import pair_correction as PC
from paper_2606_19557_b200 import workloads as wl
from tests import _gpu_harness as H

pytestmark = pytest.mark.gpu


def _params(T, seed, r_inner, r_outer):
    rng = np.random.default_rng(seed)
    coef = rng.uniform(0.1, 1.0, size=4); coef /= coef.sum()
    return dict(Z=rng.integers(3, 30, size=T).astype(np.float64), r_inner=r_inner, r_outer=r_outer, coef=coef,
                expo=np.sort(rng.uniform(0.2, 3.5, size=4)), a_prefac=0.47, a_pow=0.23, coulomb_k=14.4)


CASES = {
    # tiny triclinic boxes (self-images, ragged slices), the switch region covers most close pairs
    "tiny_T3_ragged": (lambda: wl.tiny_workload(2, n_species=3, sizes=(33, 2, 40), box=(7.5, 3.1, 8.0)), 1.4, 3.0),
    "tiny_thin_boxes": (lambda: wl.tiny_workload(7, n_species=2, sizes=(1, 2, 3), box=(1.6, 2.2, 2.0)), 1.2, 2.6),
    # config 4 (5 species, bcc + liquid-like snapshots with 1.8 A minimum separation): a realistic short range
    "cfg4": (lambda: wl.make_config(4, n_struct=12), 1.6, 2.4),
    # r_outer = rc_R: every radial pair is inside
    "cfg3_all_pairs": (lambda: wl.make_config(3, n_struct=4), 2.0, 6.0),
}


@pytest.mark.parametrize("name", list(CASES))
def test_pair_correction_forward_loss_and_gradient(name):
    make, ri, ro = CASES[name]
    prob = H.make_problem(make())
    par = _params(prob.workload.model.n_species, 11, ri, ro)
    Ec, Fc, Wc = PC.pair_correction(prob.data, **par)
    assert np.abs(Ec).max() > 0
    nat = prob.workload.structures.n_atoms
    lam = (1.0, 2.0, 3.0)
    with H.make_gpu(prob) as nep:
        E0, F0, W0 = nep.forward()
        nep.set_pair_correction(**par)
        E, F, W = nep.forward()
        Eo, Fo, Wo = O.forward(prob.data, prob.theta, prob.scaler)
        # the correction alone, and the corrected predictions, against the oracle
        assert np.max(np.abs((E - E0) - Ec) / nat) <= H.TOL_E_PER_ATOM
        assert H.relnorm(F - F0, Fc) <= 5 * H.TOL_FW_REL and H.relnorm(W - W0, Wc) <= 5 * H.TOL_FW_REL      # difference of two fp32 results
        assert np.max(np.abs(E - (Eo + Ec)) / nat) <= H.TOL_E_PER_ATOM
        assert H.relnorm(F, Fo + Fc) <= H.TOL_FW_REL and H.relnorm(W, Wo + Wc) <= H.TOL_FW_REL
        # loss and gradient: the oracle with labels shifted by the correction
        l4 = nep.loss_grad(*lam)
        g = nep.get_grad()
        prob.data.set_labels(prob.E - Ec, prob.F - Fc, prob.W - Wc)
        try:
            l4o, go = O.loss_grad(prob.data, prob.theta, prob.scaler, lam)
        finally:
            prob.data.set_labels(prob.E, prob.F, prob.W)
        assert np.allclose(l4, l4o, rtol=2e-4), (l4, l4o)
        assert H.relnorm(g, go) <= H.TOL_G_REL, H.relnorm(g, go)
        # the step graph carries the constants: graph and three calls agree, and switching the term off restores the plain model
        th0 = nep.get_params()
        for _ in range(3):
            nep.train_step(*lam, 1e-3, use_graph=True)
        th_a = nep.get_params()
        nep.set_params(th0); nep.set_adam_state(np.zeros_like(th0), np.zeros_like(th0), np.zeros_like(th0), 0)
        for _ in range(3):
            nep.train_step(*lam, 1e-3, use_graph=False)
        assert np.linalg.norm(th_a - nep.get_params()) <= 1e-3 * np.linalg.norm(th_a - th0)
        nep.set_params(th0)
        nep.set_pair_correction(None)
        E1, F1, W1 = nep.forward()
        assert np.allclose(E1, E0, rtol=0, atol=1e-5 * nat.max()) and H.relnorm(F1, F0) < 1e-5 and H.relnorm(W1, W0) < 1e-5


def test_pair_correction_argument_checks():
    from paper_2606_19557_b200.binding import NepError, NEP_EINVAL, NEP_ECAPACITY
    prob = H.make_problem(wl.tiny_workload(0))
    par = _params(2, 3, 1.0, 2.0)
    with H.make_gpu(prob) as nep:
        for bad, code in ((dict(r_outer=prob.workload.model.rc_R + 0.1), NEP_EINVAL), (dict(r_inner=2.5), NEP_EINVAL),
                          (dict(Z=np.array([4.0, 0.0])), NEP_EINVAL), (dict(coef=np.ones(9), expo=np.ones(9)), NEP_ECAPACITY),
                          (dict(a_prefac=0.0), NEP_EINVAL), (dict(expo=np.array([0.1, -1.0, 1.0, 2.0])), NEP_EINVAL)):
            with pytest.raises(NepError) as e:
                nep.set_pair_correction(**dict(par, **bad))
            assert e.value.code == code
        nep.set_pair_correction(**par)          # still usable
        nep.forward()
