"""Data-parallel NEP training over several GPUs, one process (rank) per GPU.

Structures interact only with themselves (Eq. 1; the sums of Eqs. 15-20 run over the neighbours inside one
periodic structure), so the units that shard are STRUCTURES:

  * set-up   : every rank loads its own share of the data set (`shard_structures`: longest-processing-time partition
               by pair-work estimate) and builds its own neighbour lists and pair cache; nothing is exchanged;
  * per step : the batch (global structure ids) is cut by owner (`local_batch`); every rank runs nep_forward and
               nep_loss_grad on its share with the batch counts of Eqs. 5-7 taken over the WHOLE batch
               (nep_set_batch_normalisers), which makes its loss terms and its gradient additive shares;
               ONE exchange: all-reduce (sum) of g [N_par fp32] and of {L, dE, dF, dV} [4 fp64]
               (`allreduce_grad_loss`: NCCL on the GPU, gloo in the CPU tests); then every rank applies the same Adam update.

The descriptor scaler (Eq. 2) is a range over every atom of the WHOLE set: every rank asks its context for the minimum and
maximum of each component over its own atoms (nep_compute_descriptor_range), `allreduce_range` exchanges them (MIN / MAX),
and every context forms the identical s = 1 / (max - min) itself (nep_set_scaler_from_range).
No arithmetic of the method lives here: the kernels and the rule of Eq. 2 are behind include/nep.h.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional, Sequence

import numpy as np


def shard_structures(n_atoms: Sequence[int], world: int, work: Optional[Sequence[float]] = None) -> np.ndarray:
    """owner[s] in 0..world-1 for every structure.  Longest-processing-time greedy on `work` (default: atoms per structure,
    a proxy for its pair count), ties broken by structure id, so every rank computes the same table without communication."""
    n_atoms = np.asarray(n_atoms, dtype=np.int64)
    w = np.asarray(work if work is not None else n_atoms, dtype=np.float64)
    if w.shape != n_atoms.shape:
        raise ValueError("work must have one entry per structure")
    if world < 1:
        raise ValueError("world must be >= 1")
    owner = np.zeros(len(n_atoms), dtype=np.int32)
    load = np.zeros(world, dtype=np.float64)
    order = np.lexsort((np.arange(len(w)), -w))          # heaviest first, then by id
    for s in order:
        r = int(np.argmin(load))                         # first minimum: deterministic
        owner[s] = r
        load[r] += w[s]
    return owner


@dataclass
class Shard:
    rank: int
    world: int
    owner: np.ndarray        # [S] owner of every structure
    global_ids: np.ndarray   # [S_local] global ids of this rank's structures, ascending
    local_of: np.ndarray     # [S] local id on its owner

    @classmethod
    def make(cls, n_atoms: Sequence[int], rank: int, world: int, work: Optional[Sequence[float]] = None) -> "Shard":
        owner = shard_structures(n_atoms, world, work)
        local_of = np.zeros(len(owner), dtype=np.int32)
        for r in range(world):
            ids = np.nonzero(owner == r)[0]
            local_of[ids] = np.arange(len(ids), dtype=np.int32)
        return cls(rank, world, owner, np.nonzero(owner == rank)[0].astype(np.int32), local_of)

    def local_batch(self, batch_ids: Sequence[int]) -> np.ndarray:
        """Local structure ids (order of the batch kept) of the part of a global batch that this rank owns."""
        b = np.asarray(batch_ids, dtype=np.int64)
        mine = b[self.owner[b] == self.rank]
        return self.local_of[mine].astype(np.int32)


def batch_normalisers(batch_ids: Sequence[int], n_atoms: Sequence[int], has_virial: Optional[Sequence[int]] = None):
    """(S_b, N_b, S_v) of the whole batch: the counts Eqs. 5-7 divide by.  Every rank knows n_atoms and has_virial of the
    whole data set (metadata), so no communication is needed."""
    b = np.asarray(batch_ids, dtype=np.int64)
    n = np.asarray(n_atoms, dtype=np.int64)
    hv = np.ones(len(n), dtype=np.int64) if has_virial is None else np.asarray(has_virial, dtype=np.int64)
    return int(len(b)), int(n[b].sum()), int(hv[b].sum())


def _on_stream(stream):
    import contextlib
    if stream is None:
        return contextlib.nullcontext()
    import torch
    return torch.cuda.stream(stream)


def allreduce_grad_loss(g, loss4, group=None, stream=None):
    """The step's one exchange: in-place sum over the ranks of the gradient and of the four loss terms.
    stream: the CUDA stream the context launches on (the collective is ordered after its kernels and before the Adam kernel)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        with _on_stream(stream):
            dist.all_reduce(g, op=dist.ReduceOp.SUM, group=group)
            dist.all_reduce(loss4, op=dist.ReduceOp.SUM, group=group)
    return g, loss4


def allreduce_range(qmin, qmax, group=None):
    """Element-wise MIN of qmin and MAX of qmax over the ranks, in place (torch tensors on the backend's device).
    +inf / -inf of a rank without atoms are the neutral elements."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(qmin, op=dist.ReduceOp.MIN, group=group)
        dist.all_reduce(qmax, op=dist.ReduceOp.MAX, group=group)
    return qmin, qmax


class DataParallelNep:
    """A `Nep` context holding this rank's share of a structure set, driven with GLOBAL structure ids.

    nep_factory(model, **kw) builds the context (default: binding.Nep.from_model); the CPU tests pass a stand-in."""

    def __init__(self, model, structures, rank: int, world: int, group=None, work=None, nep_factory=None, **kw):
        self.group = group
        self.n_atoms = np.asarray(structures.n_atoms, dtype=np.int64)
        self.shard = Shard.make(self.n_atoms, rank, world, work)
        self.has_virial = np.ones(len(self.n_atoms), dtype=np.int64)
        if nep_factory is None:
            from .binding import Nep
            nep_factory = Nep.from_model
        self.nep = nep_factory(model, **kw)
        self.structures = structures
        self._whole = (0, 0, 0)

    def _local_rows(self):
        off = np.concatenate([[0], np.cumsum(self.n_atoms)])
        ids = self.shard.global_ids
        return np.concatenate([np.arange(off[s], off[s + 1]) for s in ids]) if len(ids) else np.zeros(0, np.int64)

    def load(self, E=None, F=None, W=None, has_virial=None):
        """Loads this rank's structures (labels optional, global arrays in the caller's order) and builds its lists."""
        sub = self.structures.subset(self.shard.global_ids)
        if has_virial is not None:
            self.has_virial = np.asarray(has_virial, dtype=np.int64)
        if E is None:
            self.nep.load_structure_set(sub)
        else:
            ids = self.shard.global_ids
            hv = None if has_virial is None else np.asarray(has_virial, dtype=np.uint8)[ids]
            self.nep.load_structure_set(sub, np.asarray(E)[ids], np.asarray(F)[self._local_rows()], np.asarray(W)[ids], hv)
        self.nep.build_neighbors()

    def set_labels(self, E, F, W, has_virial=None):
        """Attaches labels given for the WHOLE set (caller's order) to this rank's structures."""
        ids = self.shard.global_ids
        if has_virial is not None:
            self.has_virial = np.asarray(has_virial, dtype=np.int64)
        hv = None if has_virial is None else np.asarray(has_virial, dtype=np.uint8)[ids]
        self.nep.set_labels(np.asarray(E)[ids], np.asarray(F)[self._local_rows()], np.asarray(W)[ids], hv)

    def compute_scaler(self):
        """Eq. 2 over the atoms of every rank: local ranges -> MIN / MAX all-reduce -> the same scaler in every context."""
        import torch
        import torch.distributed as dist
        lo, hi = self.nep.compute_descriptor_range()
        dev = "cpu"
        if dist.is_available() and dist.is_initialized() and dist.get_backend(self.group) == "nccl":
            dev = "cuda"
        tlo, thi = torch.from_numpy(np.array(lo)).to(dev), torch.from_numpy(np.array(hi)).to(dev)
        allreduce_range(tlo, thi, self.group)
        self.nep.set_scaler_from_range(tlo.cpu().numpy(), thi.cpu().numpy())

    def set_batch(self, batch_ids: Sequence[int]):
        self.nep.set_batch(self.shard.local_batch(batch_ids))
        self._whole = batch_normalisers(batch_ids, self.n_atoms, self.has_virial)
        self.nep.set_batch_normalisers(*self._whole)

    def local_batch_shape(self):
        return self.nep.batch_shape()

    def step(self, lam, lr: float, fetch_loss: bool = False, variant: int = 0):
        """One training step on the current batch: forward, loss + gradient, the all-reduce, Adam."""
        self.nep.forward_device()
        self.nep.loss_grad(lam[0], lam[1], lam[2], fetch_loss=False)
        g, l4 = self.nep.grad_loss_tensors()
        allreduce_grad_loss(g, l4, self.group, getattr(self.nep, "stream", None))
        self.nep.adam_step(lr, variant=variant)
        return l4.cpu().numpy() if fetch_loss else None

    # ---- the surface trainer.Trainer drives (mini-batches, two-stage schedule, plateau decay), with GLOBAL ids: every
    #      rank runs the same Trainer with the same seed, so all of them select the same batches and see the same whole-batch loss
    #      terms, hence the same learning-rate decisions -- no broadcast is needed ----
    @property
    def n_struct(self) -> int:
        return len(self.n_atoms)

    def train_step(self, lambda_E: float, lambda_F: float, lambda_V: float, lr: float, variant: int = 0):
        self.step((lambda_E, lambda_F, lambda_V), lr, fetch_loss=False, variant=variant)

    def get_loss(self) -> np.ndarray:
        """{L, dE, dF, dV} of the WHOLE batch of the last step (summed over the ranks), on the host."""
        return self.nep.grad_loss_tensors()[1].cpu().numpy().copy()

    def batch_counts(self):
        """(S_b, N_b, S_v) of the whole current batch (the counts Eqs. 5-7 were divided by)."""
        return self._whole

    def forward_device(self):
        self.nep.forward_device()

    def loss_grad(self, lambda_E: float, lambda_F: float, lambda_V: float, fetch_loss: bool = True):
        """Loss terms and gradient of the whole batch (all-reduced); the RMSE report of Trainer.rmse goes through here."""
        self.nep.loss_grad(lambda_E, lambda_F, lambda_V, fetch_loss=False)
        g, l4 = self.nep.grad_loss_tensors()
        allreduce_grad_loss(g, l4, self.group, getattr(self.nep, "stream", None))
        return l4.cpu().numpy().copy() if fetch_loss else None
