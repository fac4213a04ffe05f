"""Data-parallel path: structure sharding, whole-batch normalisers, the one all-reduce.

CPU tests (gloo, world_size 2): the host logic of paper_2606_19557_b200/dataparallel.py and the claim the C call
nep_set_batch_normalisers rests on -- with the counts of Eqs. 5-7 taken over the whole batch, the loss terms and the
gradient of the ranks' shares ADD UP to those of the whole batch -- checked with the oracle on each rank.
GPU test: two contexts on one device, each holding half of the structures, summed on the device, against one context
holding everything and against the oracle."""
import os
import socket

import numpy as np
import pytest

from oracle import nep_oracle as O
from paper_2606_19557_b200 import dataparallel as dp
from paper_2606_19557_b200 import workloads as wl
from tests import _gpu_harness as H


def test_shard_structures_covers_and_balances():
    rng = np.random.default_rng(5)
    n_atoms = rng.integers(32, 513, size=400)
    for world in (1, 2, 3, 8):
        owner = dp.shard_structures(n_atoms, world)
        assert owner.shape == n_atoms.shape and owner.min() >= 0 and owner.max() < world
        load = np.bincount(owner, weights=n_atoms, minlength=world)
        assert load.max() - load.min() <= n_atoms.max()                 # LPT bound
        assert np.array_equal(owner, dp.shard_structures(n_atoms, world))   # deterministic: no communication needed
    sh = [dp.Shard.make(n_atoms, r, 3) for r in range(3)]
    batch = rng.permutation(400)[:100]
    parts = [s.local_batch(batch) for s in sh]
    assert sum(len(p) for p in parts) == 100
    back = np.sort(np.concatenate([s.global_ids[p] for s, p in zip(sh, parts)]))
    assert np.array_equal(back, np.sort(batch))                             # disjoint cover of the batch
    S, N, Sv = dp.batch_normalisers(batch, n_atoms, None)
    assert (S, N, Sv) == (100, int(n_atoms[batch].sum()), 100)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        O.set_num_threads(1)
        w = wl.tiny_workload(11, n_species=2, sizes=(5, 9, 3, 7, 6, 4), box=(3.4, 4.3, 3.1, 3.9, 3.6, 4.0))
        prob = H.make_problem(w)                                   # same seeds on every rank: same data, same theta
        st = w.structures
        hv = np.array([1, 0, 1, 1, 1, 0], np.uint8)
        prob.data.set_labels(prob.E, prob.F, prob.W, hv)
        batch = np.array([4, 0, 5, 2, 1], np.int32)                # structure 3 is not in the batch
        lam = (1.0, 2.0, 3.0)
        shard = dp.Shard.make(st.n_atoms, rank, world)
        mine = shard.global_ids[shard.local_batch(batch)]
        S, N, Sv = dp.batch_normalisers(batch, st.n_atoms, hv)
        g = np.zeros(len(prob.theta)); l4 = np.zeros(4)
        if len(mine):
            Sr, Nr, Svr = dp.batch_normalisers(mine, st.n_atoms, hv)
            # the oracle divides by the counts of the batch it is given; re-weight every term to the whole batch's counts
            for k, (cr, cw) in enumerate(((Sr, S), (Nr, N), (Svr, Sv))):
                one = [0.0, 0.0, 0.0]; one[k] = lam[k]
                if cr == 0:
                    continue
                l4k, gk = O.loss_grad(prob.data, prob.theta, prob.scaler, tuple(one), batch=list(mine))
                g += gk * (cr / cw); l4[0] += l4k[0] * (cr / cw); l4[1 + k] += l4k[1 + k] * (cr / cw)
        gt, lt = torch.from_numpy(g.astype(np.float32)), torch.from_numpy(l4)
        dp.allreduce_grad_loss(gt, lt)                             # gloo here, NCCL on the GPUs
        if rank == 0:
            l4w, gw = O.loss_grad(prob.data, prob.theta, prob.scaler, lam, batch=list(batch))
            out.put((H.relnorm(gt.numpy(), gw), float(np.max(np.abs(lt.numpy() - l4w) / np.abs(l4w))), [int(x) for x in shard.owner]))
    finally:
        dist.destroy_process_group()


def _rank_dp_nep(rank, world, port, out):
    """DataParallelNep end to end on the CPU (oracle-backed stand-in context): the two ranks hold DIFFERENT structures."""
    import torch.distributed as dist
    from tests._oracle_nep import OracleNep
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        O.set_num_threads(1)
        w = wl.tiny_workload(11, n_species=2, sizes=(5, 9, 3, 7, 6, 4), box=(3.4, 4.3, 3.1, 3.9, 3.6, 4.0))
        prob = H.make_problem(w)
        st = w.structures
        hv = np.array([1, 0, 1, 1, 1, 0], np.uint8)
        d = dp.DataParallelNep(w.model, st, rank, world, nep_factory=OracleNep.from_model)
        d.load(prob.E, prob.F, prob.W, hv)
        d.nep.set_params(prob.theta)
        lo, hi = d.nep.compute_descriptor_range()              # this rank's own atoms only
        d.compute_scaler()                                     # Eq. 2 over the union
        s = d.nep.get_scaler()
        batch = np.array([4, 0, 5, 2, 1], np.int32)
        lam = (1.0, 2.0, 3.0)
        d.set_batch(batch)
        l4 = d.step(lam, 1e-2, fetch_loss=True)
        out.put((rank, s, lo, hi, l4, d.nep.get_params(), [int(x) for x in d.shard.global_ids], d.local_batch_shape()))
    finally:
        dist.destroy_process_group()


def _rank_trainer(rank, world, port, out):
    import torch.distributed as dist
    from paper_2606_19557_b200 import trainer as T
    from tests._oracle_nep import OracleNep
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        O.set_num_threads(1)
        w, prob, hv, cfg = _trainer_problem()
        d = dp.DataParallelNep(w.model, w.structures, rank, world, nep_factory=OracleNep.from_model)
        d.load(prob.E, prob.F, prob.W, hv)
        d.nep.set_params(prob.theta); d.nep.set_scaler(prob.scaler)
        tr = T.Trainer(d, cfg)
        hist = tr.fit()
        r = tr.rmse(chunk=4)
        out.put((rank, d.nep.get_params(), [(h.lr, h.loss, h.dE, h.dF, h.dV) for h in hist], r))
    finally:
        dist.destroy_process_group()


def _trainer_problem():
    from paper_2606_19557_b200 import trainer as T
    w = wl.tiny_workload(11, n_species=2, sizes=(5, 9, 3, 7, 6, 4), box=(3.4, 4.3, 3.1, 3.9, 3.6, 4.0))
    prob = H.make_problem(w)
    hv = np.array([1, 0, 1, 1, 1, 0], np.uint8)
    cfg = T.TrainConfig(epoch=3, batch=4, stage1=T.StageSpec(5e-3, 1.0, 2.0, 0.5), stage2=T.StageSpec(2e-3, 2.0, 1.0, 1.0),
                        start_stage2=2, scheduler_patience=0, scheduler_factor=0.5, seed=3)
    return w, prob, hv, cfg


def test_trainer_over_two_ranks_follows_the_one_rank_trajectory_gloo_world2():
    """P:99-103 data-parallel: the same Trainer (same seed) on two ranks, each holding its share of the structures, selects the same
    global mini-batches, sees the whole batch's loss terms after the all-reduce, takes the same learning-rate decisions, and lands on
    the parameters, the epoch records and the RMSE report of one context holding everything."""
    import torch.multiprocessing as mp
    from paper_2606_19557_b200 import trainer as T
    from tests._oracle_nep import OracleNep
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_trainer, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=300) for _ in range(2)), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w, prob, hv, cfg = _trainer_problem()
    one = OracleNep(w.model)
    one.load_structure_set(w.structures, prob.E, prob.F, prob.W, hv)
    one.build_neighbors()
    one.set_params(prob.theta); one.set_scaler(prob.scaler)
    tr = T.Trainer(one, cfg)
    hist = tr.fit()
    r_one = tr.rmse(chunk=4)
    ref = [(h.lr, h.loss, h.dE, h.dF, h.dV) for h in hist]
    assert len(ref) == 3 and len({h[0] for h in ref}) > 1                      # the rate changed along the way (stage 2 / decay)
    moved = np.linalg.norm(one.get_params().astype(np.float64) - prob.theta)
    for _, th, h, r in res:
        assert np.linalg.norm(th.astype(np.float64) - one.get_params()) <= 1e-4 * moved
        assert [x[0] for x in h] == [x[0] for x in ref]                        # identical learning-rate sequence
        assert np.allclose(np.array(h)[:, 1:], np.array(ref)[:, 1:], rtol=1e-5)
        for k in r_one:
            assert r[k] == pytest.approx(r_one[k], rel=1e-5)


def test_dataparallel_nep_scaler_and_step_gloo_world2():
    """Eq. 2 is over every atom of the set: two ranks with different structures (and different local ranges) must end with
    the identical scaler, equal to the oracle's over the union; one DataParallelNep.step then lands both on the parameters
    of the oracle's whole-batch step."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_dp_nep, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((out.get(timeout=240) for _ in range(2)), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, s0, lo0, hi0, l40, th0, ids0, shp0), (_, s1, lo1, hi1, l41, th1, ids1, shp1) = res
    assert sorted(ids0 + ids1) == list(range(6)) and ids0 and ids1 and not set(ids0) & set(ids1)
    assert not np.allclose(lo0, lo1) and not np.allclose(hi0, hi1)            # the local ranges differ ...
    assert np.array_equal(s0, s1)                                             # ... the scaler does not
    w = wl.tiny_workload(11, n_species=2, sizes=(5, 9, 3, 7, 6, 4), box=(3.4, 4.3, 3.1, 3.9, 3.6, 4.0))
    prob = H.make_problem(w)
    s_union = O.scaler(O.descriptors(prob.data, prob.theta))                   # Eq. 2 over the union, at the same theta
    assert np.allclose(s0, s_union, rtol=1e-12)
    assert not np.allclose(1.0 / (hi0 - lo0), s_union, rtol=1e-3)             # a rank-local scaler would have been wrong
    hv = np.array([1, 0, 1, 1, 1, 0], np.uint8)
    prob.data.set_labels(prob.E, prob.F, prob.W, hv)
    batch = [4, 0, 5, 2, 1]
    l4w, gw = O.loss_grad(prob.data, prob.theta, s_union, (1.0, 2.0, 3.0), batch=batch)
    assert np.allclose(l40, l4w, rtol=1e-10) and np.array_equal(l40, l41)
    th = prob.theta.copy(); n = th.size
    O.adam_step(th, gw.astype(np.float32).astype(np.float64), np.zeros(n), np.zeros(n), np.zeros(n), 0, 1e-2)
    assert np.array_equal(th0, th1)                                           # identical updates, no parameter broadcast
    assert np.max(np.abs(th0 - th)) < 2e-6
    assert shp0[0] + shp1[0] == 5


def test_shares_add_up_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    eg, el, owner = out.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(set(owner)) == [0, 1]
    assert eg < 1e-6, eg          # fp32 all-reduce of an fp64 gradient
    assert el < 1e-12, el


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["tiny", "cfg3"])
def test_two_contexts_sum_to_one(name):
    import torch
    from paper_2606_19557_b200.binding import Nep
    w = wl.tiny_workload(11, n_species=2, sizes=(5, 9, 3, 7, 6, 4), box=(3.4, 4.3, 3.1, 3.9, 3.6, 4.0)) if name == "tiny" \
        else wl.make_config(3, n_struct=10)
    prob = H.make_problem(w)
    st = w.structures
    S = st.n_struct
    hv = (np.arange(S) % 3 != 1).astype(np.uint8)
    prob.data.set_labels(prob.E, prob.F, prob.W, hv)
    batch = np.array([s for s in np.random.default_rng(3).permutation(S) if s != 3], np.int32)
    lam = (1.0, 2.0, 3.0)
    off = st.atom_off
    gsum = None; lsum = None
    for rank in range(2):
        shard = dp.Shard.make(st.n_atoms, rank, 2)
        ids = shard.global_ids
        rows = np.concatenate([np.arange(off[s], off[s + 1]) for s in ids])
        with Nep.from_model(w.model) as nep:
            nep.load_structure_set(st.subset(ids), prob.E[ids], prob.F[rows], prob.W[ids], hv[ids])
            nep.build_neighbors()
            nep.set_params(prob.theta.astype(np.float32)); nep.set_scaler(prob.scaler)
            nep.set_batch(shard.local_batch(batch))
            nep.set_batch_normalisers(*dp.batch_normalisers(batch, st.n_atoms, hv))
            nep.forward_device()
            nep.loss_grad(*lam, fetch_loss=False)
            g, l4 = nep.grad_loss_tensors()
            torch.cuda.synchronize()
            gsum = g.clone() if gsum is None else gsum + g
            lsum = l4.clone() if lsum is None else lsum + l4
    l4o, go = O.loss_grad(prob.data, prob.theta, prob.scaler, lam, batch=list(batch))
    assert H.relnorm(gsum.cpu().numpy(), go) <= H.TOL_G_REL
    assert np.allclose(lsum.cpu().numpy(), l4o, rtol=2e-4)
    with H.make_gpu(prob) as nep:
        nep.set_labels(prob.E, prob.F, prob.W, hv)
        nep.set_batch(batch)
        nep.forward_device(); l4 = nep.loss_grad(*lam)
        assert H.relnorm(gsum.cpu().numpy(), nep.get_grad()) < 2e-5
        assert np.allclose(lsum.cpu().numpy(), l4, rtol=1e-6)
        # a whole batch smaller than the local one is refused
        with pytest.raises(Exception):
            nep.set_batch_normalisers(1, 1, 0)
