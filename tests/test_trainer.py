"""Epoch driver (paper P:99-103, Eq. 14, Table I): schedule logic on CPU, trajectory parity and convergence on the GPU."""
import numpy as np
import pytest

from oracle import nep_oracle as O
from paper_2606_19557_b200 import trainer as T
from paper_2606_19557_b200 import workloads as wl
from tests import _gpu_harness as H


def test_plateau_schedule_matches_torch_reduce_lr_on_plateau():
    """Eq. 14 with the scheduler the paper names (ReduceLROnPlateau): same learning-rate sequence as torch's."""
    import torch
    rng = np.random.default_rng(1)
    losses = np.concatenate([np.linspace(1.0, 0.5, 12), 0.5 + 0.01 * rng.random(40), np.linspace(0.5, 0.2, 10), 0.2 + 0.0 * rng.random(60)])
    for patience, factor in ((3, 0.5), (15, 0.5), (0, 0.1)):
        p = torch.nn.Parameter(torch.zeros(1))
        opt = torch.optim.SGD([p], lr=5e-3)
        ref = torch.optim.lr_scheduler.ReduceLROnPlateau(opt, mode="min", factor=factor, patience=patience, threshold=1e-4,
                                                         threshold_mode="rel", min_lr=1e-6)
        mine = T.PlateauSchedule(5e-3, factor, patience, 1e-6, 1e-4)
        for x in losses:
            ref.step(float(x))
            assert mine.step(float(x)) == pytest.approx(opt.param_groups[0]["lr"], rel=1e-12)
        assert mine.lr < 5e-3          # the sequence has plateaus: the rate did decay
    m = T.PlateauSchedule(1e-5, 0.5, 0, 4e-6)
    for _ in range(5):
        m.step(1.0)
    assert m.lr == 4e-6                # eta_min of Eq. 14


def test_epoch_batches_are_seeded_permutations():
    b0 = T.epoch_batches(103, 16, seed=7, epoch=0)
    assert [len(b) for b in b0] == [16] * 6 + [7]
    assert np.array_equal(np.sort(np.concatenate(b0)), np.arange(103))
    assert all(np.array_equal(x, y) for x, y in zip(b0, T.epoch_batches(103, 16, seed=7, epoch=0)))
    assert not np.array_equal(np.concatenate(b0), np.concatenate(T.epoch_batches(103, 16, seed=7, epoch=1)))
    assert not np.array_equal(np.concatenate(b0), np.concatenate(T.epoch_batches(103, 16, seed=8, epoch=0)))


class _FakeNep:
    """Records what the driver asks for; the loss sequence is scripted."""
    n_struct = 10

    def __init__(self, losses):
        self.losses, self.calls, self.i = list(losses), [], 0

    def set_batch(self, ids): self.ids = ids
    def forward_device(self): pass

    def loss_grad(self, le, lf, lv, fetch_loss=True):
        self.lam = (le, lf, lv)
        x = self.losses[min(self.i, len(self.losses) - 1)]
        return np.array([x, 0.0, 0.0, 0.0])

    def adam_step(self, lr, variant=0):
        self.calls.append((self.i, self.lam, lr)); self.i += 1


def test_two_stage_switch_and_rate_constant_within_epoch():
    cfg = T.TrainConfig(epoch=8, batch=5, stage1=T.StageSpec(1e-2, 1.0, 100.0, 1.0), stage2=T.StageSpec(1e-3, 100.0, 5.0, 30.0),
                        start_stage2=4, scheduler_patience=0, scheduler_factor=0.5, min_lr=1e-6)
    nep = _FakeNep([1.0] * 100)                      # never improves after the first epoch: decay every epoch
    hist = T.Trainer(nep, cfg).fit()
    assert [r.stage for r in hist] == [1] * 4 + [2] * 4
    assert [r.lr for r in hist[:4]] == pytest.approx([1e-2, 1e-2, 5e-3, 2.5e-3])     # first epoch sets the best, then Eq. 14
    assert [r.lr for r in hist[4:]] == pytest.approx([1e-3, 1e-3, 5e-4, 2.5e-4])     # stage 2 restarts at stage2_lr
    per_epoch = {}
    for step, lam, lr in nep.calls:
        per_epoch.setdefault(step // 2, set()).add((lam, lr))
    assert all(len(v) == 1 for v in per_epoch.values())                               # constant inside an epoch
    assert per_epoch[0] == {((1.0, 100.0, 1.0), 1e-2)} and per_epoch[4] == {((100.0, 5.0, 30.0), 1e-3)}


def test_rmse_recombines_chunks_with_their_counts():
    """Trainer.rmse over unequal chunks and a virial mask = sqrt of Eqs. 5-7 over the whole set (oracle-backed stand-in context:
    the chunk bookkeeping is host logic)."""
    from tests._oracle_nep import OracleNep
    w = wl.tiny_workload(11, n_species=2, sizes=(5, 9, 3, 7, 6, 4), box=(3.4, 4.3, 3.1, 3.9, 3.6, 4.0))
    prob = H.make_problem(w)
    st = w.structures
    hv = np.array([1, 0, 1, 1, 1, 0], np.uint8)
    nep = OracleNep(w.model)
    nep.load_structure_set(st, prob.E, prob.F, prob.W, hv)
    nep.build_neighbors()
    th = prob.theta + 0.05 * np.random.default_rng(0).normal(size=prob.theta.size)      # away from the teacher: non-zero errors
    nep.set_params(th); nep.set_scaler(prob.scaler)
    r = T.Trainer(nep, T.TrainConfig()).rmse(st.n_atoms, has_virial=hv, chunk=4)            # chunks of 4 and 2 structures
    prob.data.set_labels(prob.E, prob.F, prob.W, hv)
    l4, _ = O.loss_grad(prob.data, nep.theta, prob.scaler, (1.0, 1.0, 1.0), want_grad=False)
    assert r["energy_per_atom"] == pytest.approx(np.sqrt(l4[1]), rel=1e-12)
    assert r["force"] == pytest.approx(np.sqrt(l4[2]), rel=1e-12)
    assert r["virial_per_atom"] == pytest.approx(np.sqrt(l4[3]), rel=1e-12)
    assert min(r.values()) > 0
    # the counts come from the context: leaving the mask out gives the same report (the labels carry it) ...
    r2 = T.Trainer(nep, T.TrainConfig()).rmse(chunk=4)
    assert r2 == r
    # ... a mask that contradicts the loaded one is refused, and a context without batch_counts() still works from the arguments
    with pytest.raises(ValueError):
        T.Trainer(nep, T.TrainConfig()).rmse(st.n_atoms, has_virial=np.ones(6, np.uint8), chunk=4)

    class NoCounts:
        def __init__(self, inner):
            self._i = inner
            self.n_struct = inner.n_struct

        def __getattr__(self, name):
            if name == "batch_counts":
                raise AttributeError(name)
            return getattr(self._i, name)
    r3 = T.Trainer(NoCounts(nep), T.TrainConfig()).rmse(st.n_atoms, has_virial=hv, chunk=4)
    assert r3 == r


@pytest.mark.gpu
def test_trajectory_matches_oracle_and_loss_decreases():
    w = wl.make_config(1)
    prob = H.make_problem(w)
    st = w.structures
    cfg = T.TrainConfig(epoch=3, batch=3, stage1=T.StageSpec(2e-3, 1.0, 2.0, 0.5), stage2=T.StageSpec(1e-3, 2.0, 1.0, 1.0),
                        start_stage2=2, scheduler_patience=0, scheduler_factor=0.5, seed=5)
    with H.make_gpu(prob) as nep:
        tr = T.Trainer(nep, cfg)
        hist = tr.fit()
        theta_gpu = nep.get_params().astype(np.float64)
        # the same trajectory with the oracle: same batches, same weights, same rates
        th = prob.theta.copy(); n = th.size
        m, v, vmax, t = np.zeros(n), np.zeros(n), np.zeros(n), 0
        k = 0
        for e in range(3):
            _, spec = cfg.stage_of(e)
            for ids in T.epoch_batches(st.n_struct, cfg.batch, cfg.seed, e):
                l4, g = O.loss_grad(prob.data, th, prob.scaler, (spec.lambda_e, spec.lambda_f, spec.lambda_v), batch=list(ids))
                t = O.adam_step(th, g, m, v, vmax, t, hist[e].lr)
                k += 1
        assert k == 9
        # 9 Adam steps of size <= 2e-3 each: the fp32 trajectory stays within a small fraction of the distance travelled
        moved = np.linalg.norm(th - prob.theta)
        assert np.linalg.norm(theta_gpu - th) < 2e-3 * moved, (np.linalg.norm(theta_gpu - th), moved)
        # a longer teacher-student run converges: loss falls by a large factor, RMSEs are reported
        nep.set_params(prob.theta.astype(np.float32))
        nep.set_adam_state(np.zeros(n, np.float32), np.zeros(n, np.float32), np.zeros(n, np.float32), 0)
        cfg2 = T.TrainConfig(epoch=60, batch=4, stage1=T.StageSpec(5e-3, 1.0, 1.0, 1.0), stage2=None, scheduler_patience=5, seed=1)
        tr2 = T.Trainer(nep, cfg2)
        h2 = tr2.fit()
        assert h2[-1].loss < 0.2 * h2[0].loss, (h2[0].loss, h2[-1].loss)
        # RMSE report = sqrt of the mean squares of Eqs. 5-7 over the whole set, against the oracle at the trained parameters
        hv = (np.arange(st.n_struct) % 3 != 1).astype(np.uint8)
        nep.set_labels(prob.E, prob.F, prob.W, hv)
        r = tr2.rmse(chunk=3)                 # three chunks of unequal size (3, 3, 2); the mask is the one given to set_labels
        prob.data.set_labels(prob.E, prob.F, prob.W, hv)
        try:
            l4o, _ = O.loss_grad(prob.data, nep.get_params().astype(np.float64), prob.scaler, (1.0, 1.0, 1.0), want_grad=False)
        finally:
            prob.data.set_labels(prob.E, prob.F, prob.W)
        assert r["energy_per_atom"] == pytest.approx(np.sqrt(l4o[1]), rel=2e-3)
        assert r["force"] == pytest.approx(np.sqrt(l4o[2]), rel=1e-3)
        assert r["virial_per_atom"] == pytest.approx(np.sqrt(l4o[3]), rel=1e-3)
        assert r["force"] > 0 and r["virial_per_atom"] > 0
