"""Epoch driver around the training step (paper P:99-103, Fig. 1, Table I).

Host logic only -- every number is produced by the kernels behind include/nep.h:

  * mini-batches : a seeded permutation of the structure ids per epoch, cut into batches of `batch` structures;
  * two stages   : (lambda_E, lambda_F, lambda_V, lr) switch at epoch `start_stage2` (Table I "Stage II"); the plateau
                   counter and the best loss restart with the stage, the learning rate restarts at `stage2_lr`;
  * plateau decay: ReduceLROnPlateau on the epoch-mean training loss, Eq. 14: eta_{e+1} = max(gamma eta_e, eta_min)
                   whenever the loss has not improved for `patience` consecutive epochs; the rate is constant inside an
                   epoch.  "Improved" = below best * (1 - threshold) (the relative mode of the scheduler the paper names,
                   reading: the paper gives gamma and p only; threshold 1e-4 is that scheduler's default);
  * reporting    : epoch-mean loss terms and, on request, RMSEs of energy per atom, force components and virial per atom.
"""
from __future__ import annotations

import dataclasses
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np


@dataclasses.dataclass
class StageSpec:
    lr: float
    lambda_e: float
    lambda_f: float
    lambda_v: float


@dataclasses.dataclass
class TrainConfig:
    """Names follow Table I of the paper."""
    epoch: int = 600
    batch: int = 16
    stage1: StageSpec = dataclasses.field(default_factory=lambda: StageSpec(5e-3, 1.0, 100.0, 1.0))
    stage2: Optional[StageSpec] = dataclasses.field(default_factory=lambda: StageSpec(5e-4, 100.0, 5.0, 30.0))
    start_stage2: int = 300
    scheduler_patience: int = 15
    scheduler_factor: float = 0.5
    scheduler_threshold: float = 1e-4
    min_lr: float = 1e-6
    seed: int = 0
    adam_variant: int = 0          # 0: Eqs. 9-13 literally; 1: torch.optim.Adam(amsgrad=True)

    def stage_of(self, epoch: int) -> Tuple[int, StageSpec]:
        if self.stage2 is not None and epoch >= self.start_stage2:
            return 2, self.stage2
        return 1, self.stage1


class PlateauSchedule:
    """Eq. 14: the learning rate of the next epoch from the epoch-mean losses seen so far."""

    def __init__(self, lr: float, factor: float, patience: int, min_lr: float, threshold: float = 1e-4):
        if not (0.0 < factor < 1.0):
            raise ValueError("gamma must lie in (0, 1)")
        self.lr, self.factor, self.patience, self.min_lr, self.threshold = float(lr), factor, int(patience), float(min_lr), threshold
        self.best = float("inf")
        self.bad = 0

    def step(self, loss: float) -> float:
        if loss < self.best * (1.0 - self.threshold):
            self.best = loss
            self.bad = 0
        else:
            self.bad += 1
        if self.bad > self.patience:
            self.lr = max(self.factor * self.lr, self.min_lr)
            self.bad = 0
        return self.lr


def epoch_batches(n_struct: int, batch: int, seed: int, epoch: int) -> List[np.ndarray]:
    """Seeded permutation of the structure ids of one epoch, cut into consecutive batches (the last may be smaller)."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([int(seed), int(epoch)])))
    perm = rng.permutation(n_struct).astype(np.int32)
    return [perm[i:i + batch] for i in range(0, n_struct, batch)]


@dataclasses.dataclass
class EpochRecord:
    epoch: int
    stage: int
    lr: float
    loss: float
    dE: float
    dF: float
    dV: float


class Trainer:
    """Drives a loaded `Nep` context (structures, labels, neighbour lists, parameters and scaler already set)."""

    def __init__(self, nep, cfg: TrainConfig):
        self.nep, self.cfg = nep, cfg
        self.history: List[EpochRecord] = []
        self._sched: Optional[PlateauSchedule] = None
        self._stage = 0

    def _enter(self, stage: int, spec: StageSpec):
        self._stage = stage
        self._sched = PlateauSchedule(spec.lr, self.cfg.scheduler_factor, self.cfg.scheduler_patience, self.cfg.min_lr,
                                      self.cfg.scheduler_threshold)

    def run_epoch(self, epoch: int) -> EpochRecord:
        cfg, nep = self.cfg, self.nep
        stage, spec = cfg.stage_of(epoch)
        if stage != self._stage:
            self._enter(stage, spec)
        lr = self._sched.lr
        sums = np.zeros(4)
        nb = 0
        for ids in epoch_batches(nep.n_struct, cfg.batch, cfg.seed, epoch):
            nep.set_batch(ids)
            if hasattr(nep, "train_step"):     # one call per step (a CUDA graph launch when a batch repeats)
                nep.train_step(spec.lambda_e, spec.lambda_f, spec.lambda_v, lr, variant=cfg.adam_variant)
                sums += nep.get_loss()
            else:
                nep.forward_device()
                sums += nep.loss_grad(spec.lambda_e, spec.lambda_f, spec.lambda_v, fetch_loss=True)
                nep.adam_step(lr, variant=cfg.adam_variant)
            nb += 1
        mean = sums / max(nb, 1)
        self._sched.step(float(mean[0]))          # takes effect from the next epoch (Eq. 14)
        rec = EpochRecord(epoch, stage, lr, float(mean[0]), float(mean[1]), float(mean[2]), float(mean[3]))
        self.history.append(rec)
        return rec

    def fit(self, epochs: Optional[int] = None, callback: Optional[Callable[[EpochRecord], None]] = None) -> List[EpochRecord]:
        for e in range(len(self.history), epochs if epochs is not None else self.cfg.epoch):
            rec = self.run_epoch(e)
            if callback:
                callback(rec)
        return self.history

    def rmse(self, n_atoms: Optional[Sequence[int]] = None, has_virial: Optional[Sequence[int]] = None, chunk: int = 1024) -> dict:
        """Root-mean-square errors over the whole loaded set: energy and virial per atom, force per component.

        RMSE = sqrt(Delta) with the mean squares Delta_E, Delta_F, Delta_V of Eqs. 5-7, which nep_loss_grad returns;
        the set is evaluated in chunks of structures whose Deltas are recombined with the counts they were divided by (S_b, N_b
        and S_v, the number of structures with virial labels).  The counts come from the context (`batch_counts`), which knows
        the virial mask its labels were loaded with; n_atoms / has_virial are only consulted for a context without
        `batch_counts`, and a has_virial that contradicts the context's mask is an error rather than a silently wrong weight.
        No arithmetic of Eqs. 5-7 is repeated here."""
        nep = self.nep
        own = hasattr(nep, "batch_counts")
        if not own:
            if n_atoms is None:
                raise ValueError("this context has no batch_counts(): pass n_atoms (and has_virial if the labels carry a mask)")
            n_atoms = np.asarray(n_atoms, dtype=np.int64)
            hv = np.ones(len(n_atoms), dtype=np.int64) if has_virial is None else np.asarray(has_virial, dtype=np.int64)
        wE = wF = wV = 0.0
        S = N = Sv = 0
        for i in range(0, nep.n_struct, chunk):
            ids = np.arange(i, min(i + chunk, nep.n_struct), dtype=np.int32)
            nep.set_batch(ids)
            if own:
                sb, nb, sv = nep.batch_counts()
                if has_virial is not None and sv != int(np.asarray(has_virial, dtype=np.int64)[ids].sum()):
                    raise ValueError("has_virial differs from the mask the context's labels were loaded with")
            else:
                sb, nb, sv = len(ids), int(n_atoms[ids].sum()), int(hv[ids].sum())
            nep.forward_device()
            _, dE, dF, dV = nep.loss_grad(1.0, 1.0, 1.0, fetch_loss=True)
            wE += dE * sb; wF += dF * nb; wV += dV * sv
            S += sb; N += nb; Sv += sv
        return {"energy_per_atom": (wE / max(S, 1)) ** 0.5, "force": (wF / max(N, 1)) ** 0.5,
                "virial_per_atom": (wV / Sv) ** 0.5 if Sv else 0.0}
