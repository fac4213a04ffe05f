#!/usr/bin/env python
"""bench.py -- NEP training-step throughput (atoms/s) on B200, BASELINE.json's metric.

A "step" is one pass of the whole hot path over one batch of synthetic input:
nep_forward (descriptors, network, E, F, virial) + nep_loss_grad (loss, every gradient) + nep_adam_step.
N = 1 workload: BASELINE.json configs[1] (1000 bcc structures x 128 atoms, full NEP4 descriptor, batch 1000).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C] [--n-struct S]

Prints ONE JSON line (rank 0).  See DESIGN.md section 9 for the keys and the flop / byte models of `roofline`.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "NEP training-step throughput (atoms/s, E+F+virial loss+grads+Adam)"
UNIT = "atoms/s"
LR = 1e-3
FP32_LANES_PER_SM = 128          # B300_MICROARCH / blackwell guide: 4 SMSPs x 32 FP32 lanes


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config id (1..5); 2 is the headline workload")
    ap.add_argument("--n-struct", type=int, default=None, help="use only the first S structures (debugging; not a bench line)")
    ap.add_argument("--flush", default="auto", choices=["auto", "always", "never"],
                    help="L2 flush between timed steps; auto: only when one step streams less than twice the L2 capacity")
    ap.add_argument("--no-flush", action="store_true", help="same as --flush never")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--model-index", type=int, default=0, help="config 5: which of the 8 sweep models")
    ap.add_argument("--sustain", type=float, default=0.0, help="also run steps back to back for this many seconds with the clocks sampled")
    return ap.parse_args()


def make_workload(args, world: int = 1):
    """The config's workload; data-parallel runs (weak scaling) take a `world` times longer prefix of the same seeded stream of
    structures and a `world` times larger batch: every rank ends up with about one config's worth of DIFFERENT structures."""
    import dataclasses
    from paper_2606_19557_b200 import workloads as wl
    model = wl.config5_sweep()[args.model_index] if args.config == 5 else None
    if world == 1:
        return wl.make_config(args.config, n_struct=args.n_struct, model=model)
    base = wl.make_config(args.config, n_struct=1, model=model)
    S = args.n_struct if args.n_struct is not None else wl._CONFIGS[args.config]["n_struct"]
    w = wl.make_config(args.config, n_struct=world * S, model=model)
    B = min(wl._CONFIGS[args.config]["batch"], S)
    del base
    return dataclasses.replace(w, batch_size=world * B)


def workload_name(w, args):
    m = w.model
    return (f"config{w.config_id}: {w.name}; {w.structures.n_struct} structures, batch {w.batch_size}; "
            f"T={m.n_species} rc={m.rc_R}/{m.rc_A} n_max={m.n_max_R}/{m.n_max_A} basis={m.basis_R}/{m.basis_A} "
            f"l_max=({m.l_max_3b},{m.l_max_4b},{m.l_max_5b}) neurons={m.neurons} D={m.D} N_par={m.n_par}")


# ----------------------------------------------------------------------------------------------------------------
# clocks
# ----------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int = 0, period_ms: int = 100):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", str(period_ms)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for r in self.rows if t0 - 0.05 <= r[0] <= t1 + 0.25] or self.rows
        for _, line in rows:
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------------------------------
# problem set-up on the GPU (input recipe of DESIGN.md section 5; everything computed by the library itself)
# ----------------------------------------------------------------------------------------------------------------
def draw_theta(nep, model, seed):
    """ParamDraw two-phase recipe with the descriptors / scaler computed by the CUDA library (the implementation under test)."""
    from paper_2606_19557_b200.workloads import ParamDraw
    pd = ParamDraw(model, seed)
    nep.set_params(pd.coefficients().astype(np.float32))
    nep.compute_scaler()                       # Eq. 2 at these coefficients, over every loaded atom
    s = nep.get_scaler()
    nep.forward(want=())
    q = nep.get_descriptors().astype(np.float64)
    theta = pd.network((q * s).mean(axis=0)).astype(np.float32)
    return theta, s


def setup_ours(w, stream=None):
    from paper_2606_19557_b200.binding import Nep
    import torch
    t0 = time.time()
    nep = Nep.from_model(w.model, stream=stream)
    st = w.structures
    nep.load_structure_set(st)
    t1 = time.time()
    nep.build_neighbors()
    nep.synchronize()
    t2 = time.time()
    th_t, s_t = draw_theta(nep, w.model, w.seeds["teacher"])
    nep.set_params(th_t); nep.set_scaler(s_t)
    E, F, W = nep.forward()                    # teacher labels (they set the values being fitted, not the work)
    nep.set_labels(E.astype(np.float64), F.astype(np.float64), W.astype(np.float64))
    th_s, s_s = draw_theta(nep, w.model, w.seeds["student"])
    nep.set_params(th_s); nep.set_scaler(s_s)
    nep.set_batch(None)
    torch.cuda.synchronize()
    return nep, dict(load_s=t1 - t0, neighbors_cache_s=t2 - t1, params_labels_s=time.time() - t2)


DP = {"world": 1, "views": None, "dpn": None}   # data-parallel state of this process: dpn = dataparallel.DataParallelNep holding
                                                 # this rank's shard of the structures (sharded by structure, LPT on atoms)


def draw_theta_dp(dpn, model, seed):
    """draw_theta over a sharded set: Eq. 2's ranges and the mean of the scaled descriptors are taken over every rank's atoms."""
    import torch
    import torch.distributed as dist
    from paper_2606_19557_b200.workloads import ParamDraw
    nep = dpn.nep
    pd = ParamDraw(model, seed)
    nep.set_params(pd.coefficients().astype(np.float32))
    dpn.compute_scaler()                       # local ranges -> MIN / MAX all-reduce -> the same scaler on every rank
    s = nep.get_scaler()
    nep.forward(want=())
    q = nep.get_descriptors().astype(np.float64)
    acc = torch.tensor(np.concatenate([(q * s).sum(axis=0), [float(len(q))]]), device="cuda", dtype=torch.float64)
    dist.all_reduce(acc)
    acc = acc.cpu().numpy()
    theta = pd.network(acc[:-1] / max(acc[-1], 1.0)).astype(np.float32)
    return theta, s


def setup_dp(w, rank, world):
    """Every rank loads ITS shard of the `world` x larger set, builds its own lists and computes its own teacher labels."""
    import torch
    from paper_2606_19557_b200.dataparallel import DataParallelNep
    t0 = time.time()
    dpn = DataParallelNep(w.model, w.structures, rank, world)
    st_local = w.structures.subset(dpn.shard.global_ids)
    dpn.nep.load_structure_set(st_local)
    t1 = time.time()
    dpn.nep.build_neighbors()
    dpn.nep.synchronize()
    t2 = time.time()
    nep = dpn.nep
    th_t, s_t = draw_theta_dp(dpn, w.model, w.seeds["teacher"])
    nep.set_params(th_t); nep.set_scaler(s_t)
    nep.set_batch(None)
    E, F, W = nep.forward()
    nep.set_labels(E.astype(np.float64), F.astype(np.float64), W.astype(np.float64))
    th_s, s_s = draw_theta_dp(dpn, w.model, w.seeds["student"])
    nep.set_params(th_s); nep.set_scaler(s_s)
    torch.cuda.synchronize()
    return dpn, dict(load_s=t1 - t0, neighbors_cache_s=t2 - t1, params_labels_s=time.time() - t2)


def set_batch_ids(nep, ids):
    """Selects a batch given by GLOBAL structure ids (None = every structure): through the shard table when data-parallel."""
    dpn = DP["dpn"]
    if dpn is None:
        nep.set_batch(ids)
    else:
        dpn.set_batch(np.arange(len(dpn.n_atoms), dtype=np.int32) if ids is None else ids)   # local part + whole-batch normalisers


def dp_exchange(nep):
    """The step's one exchange (paper_2606_19557_b200/dataparallel.py): NCCL all-reduce of g and of the 4 loss terms."""
    if DP["views"] is not None:
        from paper_2606_19557_b200.dataparallel import allreduce_grad_loss
        allreduce_grad_loss(*DP["views"])


def one_step(nep, lam, graph=False):
    """One training step.  graph: nep_train_step, the step's kernels replayed as one CUDA graph launch (single GPU only: the
    data-parallel step has the all-reduce between nep_loss_grad and nep_adam_step)."""
    if graph and DP["views"] is None:
        nep.train_step(lam[0], lam[1], lam[2], LR, use_graph=True)
        return
    nep.forward_device()
    nep.loss_grad(lam[0], lam[1], lam[2], fetch_loss=False)
    dp_exchange(nep)
    nep.adam_step(LR)


def e2e_step(nep, lam, ids):
    """The call sequence a user makes per training step, HOST buffers in and out: the batch's structure ids go in
    (nep_set_batch copies them and the slice tables to the device), the loss comes back (nep_loss_grad -> host)."""
    set_batch_ids(nep, ids)
    if DP["views"] is None:
        nep.train_step(lam[0], lam[1], lam[2], LR, use_graph=True)   # one graph launch (captured again when the batch's shape changes)
        return nep.get_loss()                      # the step's loss terms -> host
    nep.forward_device()
    nep.loss_grad(lam[0], lam[1], lam[2], fetch_loss=False)
    dp_exchange(nep)
    nep.adam_step(LR)                              # queued before the read-back below synchronises
    return DP["views"][1].cpu().numpy()            # the whole batch's loss terms -> host


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the NEP step has no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    use_dist = world > 1 or os.environ.get("NEP_BENCH_DIST") == "1"    # NEP_BENCH_DIST=1: run the NCCL path on one rank too
    saved_stdout = None
    if use_dist:
        # NCCL prints its version banner on stdout; the contract is ONE JSON line there: park stdout on stderr until the end
        sys.stdout.flush()
        saved_stdout = os.dup(1)
        os.dup2(2, 1)
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29531")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
    from paper_2606_19557_b200 import workloads as wl, roofline as rf
    from paper_2606_19557_b200 import build as nbuild
    if rank == 0:
        nbuild.build()
    if use_dist:
        dist.barrier()
    w = make_workload(args, world)
    lam = w.lambdas
    DP["world"] = world
    if use_dist:
        DP["dpn"], setup = setup_dp(w, rank, world)
        nep = DP["dpn"].nep
        DP["views"] = nep.grad_loss_tensors()
    else:
        nep, setup = setup_ours(w)
    blist = wl.batches(w)
    full_batches = [b for b in blist if len(b) == w.batch_size] or blist
    single = len(blist) == 1
    peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else None
    hbm_peak = peaks["hbm_gbs"] if peaks else 6650.0
    peak_src = "measured (MEASURED_PEAKS.json)" if peaks else "fallback (B200_PROFILING.md)"

    # Timing rule: flush L2 between timed steps, or use inputs larger than L2.  One step streams every pair record and per-atom
    # row of the batch (rf.step_totals: the algorithmic byte model); where that is more than twice the L2 the steps are timed
    # back to back as a training run issues them, otherwise (config 1) a 256 MB write flushes L2 before every timed step.
    L2_BYTES = torch.cuda.get_device_properties(local).L2_cache_size
    set_batch_ids(nep, None if single else full_batches[0])
    step_bytes = rf.step_totals(rf.kernel_models(w.model, nep.get_sizes()))["bytes"]
    mode = "never" if args.no_flush else args.flush
    do_flush = mode == "always" or (mode == "auto" and step_bytes < 2 * L2_BYTES)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda") if do_flush else None   # 2x the 126 MB L2

    def set_b(i):
        if not single:
            set_batch_ids(nep, full_batches[i % len(full_batches)])

    # ---- warm-up ----
    if single:
        set_batch_ids(nep, None)
    for i in range(max(args.warmup, 3)):
        set_b(i); one_step(nep, lam, graph=i % 2 == 1)
    torch.cuda.synchronize()

    # ---- timed region: K steps, CUDA events per step on the launching stream, L2 flushed between steps ----
    K = args.steps
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    # one event pair per step where something that is not part of the step sits between steps (the flush; the selection of the next
    # batch, whose table upload belongs to the e2e number); one pair around all K steps where the same batch is stepped back to back
    per_step = flush is not None or not single
    atoms = structs = 0
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = ClockSampler(local) if rank == 0 else None
    for i in range(3):                 # starting the sampler leaves the GPU idle for a moment: more untimed steps, then the timed region
        set_b(i); one_step(nep, lam, graph=True)
    torch.cuda.synchronize()
    l0 = nep.launch_count()
    t0 = time.time()
    for i in range(K):
        set_b(i)
        if flush is not None:
            flush.fill_(i & 0xFF)
        sz = nep.batch_shape()
        structs += sz[0]; atoms += sz[1]
        if per_step or i == 0:
            ev[i][0].record()
        one_step(nep, lam, graph=True)
        if per_step or i == K - 1:
            ev[i][1].record()
    torch.cuda.synchronize()
    t1 = time.time()
    if world > 1:
        dist.barrier()
    launches = nep.launch_count() - l0
    clk = clocks.stop(t0, t1) if clocks else None
    # ---- per-kernel times: a separate pass of steps through the three calls with CUDA events around every kernel (the event
    #      records between kernels cost ~10 % of a step, so they stay out of the timed region) ----
    n_prof = max(4, K // 5)
    nep.profile_enable(True)
    for i in range(n_prof):
        set_b(i)
        if flush is not None:
            flush.fill_(i & 0xFF)
        one_step(nep, lam, graph=False)
    torch.cuda.synchronize()
    prof = nep.profile_read()
    nep.profile_enable(False)
    total_ms = float(sum(a.elapsed_time(b) for a, b in ev)) if per_step else float(ev[0][0].elapsed_time(ev[K - 1][1]))
    if world > 1:
        t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
        c = torch.tensor([atoms, structs], device="cuda", dtype=torch.float64)
        dist.all_reduce(c)
        atoms, structs = int(c[0].item()), int(c[1].item())
    value = atoms / (total_ms * 1e-3)

    # ---- back-to-back (no flush, no per-kernel events), for transparency ----
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    for i in range(K):
        set_b(i); one_step(nep, lam, graph=True)
    b.record(); torch.cuda.synchronize()
    ms_b2b = a.elapsed_time(b) / K
    a.record()
    for i in range(K):
        set_b(i); one_step(nep, lam, graph=False)
    b.record(); torch.cuda.synchronize()
    ms_b2b_stream = a.elapsed_time(b) / K

    # ---- prediction only: nep_forward alone (descriptors, network, E, F, virial), back to back ----
    a.record()
    for i in range(K):
        set_b(i); nep.forward_device()
    b.record(); torch.cuda.synchronize()
    ms_predict = a.elapsed_time(b) / K

    # ---- sustained: seconds of back-to-back steps under the power cap, clocks and power sampled (the timed region above is short) ----
    sustained = None
    if args.sustain > 0 and rank == 0 and world == 1:
        cs = ClockSampler(local, period_ms=200)
        n_done = 0
        ts0 = time.time()
        a.record()
        while time.time() - ts0 < args.sustain:
            for i in range(200):
                set_b(n_done + i); one_step(nep, lam, graph=True)
            n_done += 200
            torch.cuda.synchronize()
        b.record(); torch.cuda.synchronize()
        ts1 = time.time()
        sustained = {"seconds": ts1 - ts0, "steps": n_done, "ms_per_step": a.elapsed_time(b) / n_done, "clocks": cs.stop(ts0, ts1)}

    # ---- e2e: host ids in, host loss out, every step ----
    e2e_batches = full_batches if not single else [np.arange(w.structures.n_struct, dtype=np.int32)]
    for i in range(3):
        e2e_step(nep, lam, e2e_batches[i % len(e2e_batches)])
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    e_atoms = 0
    h2d = d2h = 0
    te0 = time.perf_counter()
    a.record()
    for i in range(K):
        l4 = e2e_step(nep, lam, e2e_batches[i % len(e2e_batches)])
    b.record(); torch.cuda.synchronize()
    te1 = time.perf_counter()
    for i in range(K):                                            # bookkeeping of what the K steps moved, outside the clock
        ids = e2e_batches[i % len(e2e_batches)]
        if DP["dpn"] is not None:                                 # this rank's part of the batch
            ids = DP["dpn"].shard.global_ids[DP["dpn"].shard.local_batch(ids)]
        e_atoms += int(w.structures.n_atoms[ids].sum())
        nbs = int(np.sum((w.structures.n_atoms[ids] + 31) // 32))
        h2d += nbs * 16 + len(ids) * (16 + 4 * w.model.n_species)   # slice table, structure tables (nep_set_batch)
        d2h += 32
    e2e_ms = max(a.elapsed_time(b), (te1 - te0) * 1e3)   # host-side work (tables) is part of the call
    if world > 1:
        t = torch.tensor([e2e_ms, 0.0], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_ms = float(t[0].item())
        c = torch.tensor([e_atoms], device="cuda", dtype=torch.float64)
        dist.all_reduce(c)
        e_atoms = int(c.item())
    e2e_value = e_atoms / (e2e_ms * 1e-3)

    if rank != 0:
        dist.destroy_process_group()
        return
    # ---- roofline of the dominant kernel ----
    set_batch_ids(nep, None if single else full_batches[0])
    sizes = nep.get_sizes()
    models = rf.kernel_models(w.model, sizes)
    ksum = sum(v[0] for v in prof.values())
    kern = {k: {"ms": v[0] / max(v[1], 1), "launches_per_step": v[1] / max(n_prof, 1), "share": v[0] / ksum} for k, v in prof.items()}
    top = max(kern, key=lambda k: kern[k]["share"])
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    alu_peak = rf.fp32_peak_flops(sm_count, (clk or {}).get("sm_max_mhz") or 1965.0, FP32_LANES_PER_SM)
    try:
        from paper_2606_19557_b200.binding import measure_fp32_peak
        fp32_measured = measure_fp32_peak()
    except Exception:      # noqa: BLE001  (a measurement aid must not take the bench line down)
        fp32_measured = None
    mdl = models.get(top)
    roof = None
    if mdl:
        dur = kern[top]["ms"] * kern[top]["launches_per_step"] * 1e-3     # the work model is per step
        t_alu, t_hbm = mdl["flops"] / alu_peak, mdl["bytes"] / (hbm_peak * 1e9)
        if t_alu >= t_hbm:
            roof = {"kernel": top, "bound": "alu", "achieved": mdl["flops"] / dur / 1e12, "peak": alu_peak / 1e12, "unit": "TFLOP/s",
                    "peak_source": f"derived: {sm_count} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 x clocks.max.sm (DESIGN.md section 9)"}
        else:
            roof = {"kernel": top, "bound": "hbm", "achieved": mdl["bytes"] / dur / 1e9, "peak": hbm_peak, "unit": "GB/s", "peak_source": peak_src}
        roof["frac"] = roof["achieved"] / roof["peak"]
        if roof["bound"] == "alu" and fp32_measured:
            roof["peak_measured"] = fp32_measured
            roof["frac_of_peak_measured"] = roof["achieved"] / fp32_measured
            roof["peak_measured_source"] = "nep_measure_fp32_peak in this run: register-resident FFMA loop, 2048 threads per SM, best of 4"
        # the per-kernel durations come from the event-bracketed pass (an event record between every two kernels): their sum exceeds
        # the step time of the timed region (one graph launch), so every per-kernel fraction here is a LOWER bound
        roof["kernel_sum_ms"] = ksum / max(n_prof, 1)
        roof["kernel_sum_over_step"] = (ksum / max(n_prof, 1)) / (total_ms / K)
        roof["duration_source"] = "CUDA events around each kernel in a separate pass of steps (three calls, not the graph); see kernel_sum_over_step"
        roof["traffic"] = None
        tpath = os.path.join(ROOT, "profiles", "r03_traffic.json")   # DRAM bytes per launch from the committed ncu --set full capture
        if os.path.exists(tpath):
            tj = json.load(open(tpath))
            if tj.get("csrc_sha") != rf.csrc_hash():
                roof["traffic_source"] = "none: the kernel sources changed after the capture in profiles/r03_traffic.json"
            elif tj.get("workload") == f"config{w.config_id}" and args.n_struct is None and world == 1:
                roof["traffic"] = tj["bytes_per_launch"].get(top)
                roof["traffic_source"] = tj.get("source", "profiles/r03_summary.md") + " (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum)"
        roof["share_of_step"] = kern[top]["share"]
        roof["avg_ms"] = kern[top]["ms"]
        roof["algorithmic_flops_per_launch"] = mdl["flops"]
        roof["algorithmic_bytes_per_launch"] = mdl["bytes"]
    tot = rf.step_totals(models)
    ms_step = total_ms / K
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": ("f32 (network products on tcgen05 kind::tf32: X, Fp as 3xTF32 = fp32-grade, the S8 products xdot, Qbar and the weight-gradient "
                  "sums as 1xTF32; sin/cos.approx in S7/S9)" if nep.network_on_tensor_cores() else "f32 (sin/cos.approx in S7/S9)"),
        "data": "synthetic (seeded lattices, teacher-NEP labels; stand-in for the paper's DFT sets)",
        "config": {"workload": workload_name(w, args), "structures_per_s": structs / (total_ms * 1e-3),
                   "atoms_per_step": atoms // K // world, "pairs_R_per_step": sizes["P_R_b"], "pairs_A_per_step": sizes["P_A_b"],
                   "l2": ("flushed between timed steps (256 MB write)" if flush is not None else
                          f"inputs larger than L2: one step streams {step_bytes / 1e6:.0f} MB (algorithmic bytes) through a {L2_BYTES / 1e6:.0f} MB L2; no flush"
                          + ("; the K steps between one event pair" if single else "; one event pair per step (the next batch is selected between them)")),
                   "ms_per_step_back_to_back_no_flush": ms_b2b, "ms_per_step_back_to_back_three_calls": ms_b2b_stream,
                   "predict_only": {"ms_per_batch": ms_predict, "atoms_per_s": (atoms / K) / (ms_predict * 1e-3),
                                    "what": "nep_forward alone (E, F, virial of the batch; rank-local), back to back"},
                   "step_call": ("nep_train_step: one CUDA graph launch per step" if not use_dist else "nep_forward + nep_loss_grad + all-reduce + nep_adam_step"),
                   "kernel_events": f"{n_prof} extra steps after the timed region, through the three calls with CUDA events around every kernel", "setup_s": setup,
                   "device_bytes": nep.bytes_allocated, "parallelism": (f"dp{world}: {w.structures.n_struct} structures sharded by structure over the ranks (dataparallel.DataParallelNep: "
                                    f"each rank holds different ones), whole batch = {w.batch_size} structures, scaler from a MIN / MAX all-reduce, "
                                    f"one NCCL all-reduce of g [{w.model.n_par} fp32] + 4 loss terms per step" if use_dist else "dp1 (one GPU, no collective)")},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d // K, "d2h_bytes_per_step": d2h // K,
                "what": "per step: nep_set_batch(host ids) + nep_train_step (one graph launch) + nep_get_loss(-> host); geometry cache resident (P:143)"},
        "gpu_launches": int(launches),
        "clocks": clk,
        "roofline": roof,
        "kernels": {k: dict({"avg_ms": round(v["ms"], 5), "share": round(v["share"], 4), "per_step": v["launches_per_step"]},
                            **({"frac_alu": round(models[k]["flops"] / alu_peak / (v["ms"] * v["launches_per_step"] * 1e-3), 4),
                                "frac_hbm": round(models[k]["bytes"] / (hbm_peak * 1e9) / (v["ms"] * v["launches_per_step"] * 1e-3), 4)}
                               if k in models and v["ms"] > 0 else {}))
                    for k, v in sorted(kern.items(), key=lambda kv: -kv[1]["share"])},
        "step_model": {"flops": tot["flops"], "bytes": tot["bytes"], "alu_frac_of_step": tot["flops"] / alu_peak / (ms_step * 1e-3),
                       "hbm_frac_of_step": tot["bytes"] / (hbm_peak * 1e9) / (ms_step * 1e-3)},
    }
    if sustained is not None:
        out["sustained"] = sustained
    if not args.no_cpu_baseline and world == 1:
        out["cpu_baseline"] = cpu_baseline(args, w, seconds_target=15.0)
    nep.destroy()
    if saved_stdout is not None:
        sys.stdout.flush()
        os.dup2(saved_stdout, 1)
    print(json.dumps(out), flush=True)
    if use_dist:
        dist.destroy_process_group()


# ----------------------------------------------------------------------------------------------------------------
# the oracle on the host cores: cpu_baseline leg and --impl reference arm (the only places bench.py executes oracle/)
# ----------------------------------------------------------------------------------------------------------------
def oracle_problem(w, n_sample):
    """First n_sample structures of the workload, teacher labels and student parameters, all from the oracle."""
    import dataclasses
    from oracle.problem import make_problem
    st = w.structures.subset(list(range(min(n_sample, w.structures.n_struct))))
    ws = dataclasses.replace(w, structures=st, batch_size=min(w.batch_size, st.n_struct))
    return make_problem(ws)


def oracle_step(O, prob, state, lam):
    th, m, v, vm = state["theta"], state["m"], state["v"], state["vmax"]
    l4, g = O.loss_grad(prob.data, th, prob.scaler, lam)      # forward E/F/W + loss + every gradient (C7-C12)
    state["t"] = O.adam_step(th, g, m, v, vm, state["t"], LR)  # C13
    return l4


def cpu_baseline(args, w, seconds_target=15.0):
    from oracle import nep_oracle as O
    cores = O.max_threads()
    n = min(w.structures.n_struct, 32)
    prob = oracle_problem(w, n)
    npar = w.model.n_par
    state = dict(theta=prob.theta.copy(), m=np.zeros(npar), v=np.zeros(npar), vmax=np.zeros(npar), t=0)
    oracle_step(O, prob, state, w.lambdas)
    t0 = time.perf_counter(); oracle_step(O, prob, state, w.lambdas); dt = time.perf_counter() - t0
    atoms = int(prob.workload.structures.n_atoms.sum())
    # scale the sample so that 3 timed steps take about seconds_target
    want = int(max(n, min(w.structures.n_struct, n * seconds_target / 3.0 / max(dt, 1e-4))))
    if want > n:
        prob = oracle_problem(w, want)
        state = dict(theta=prob.theta.copy(), m=np.zeros(npar), v=np.zeros(npar), vmax=np.zeros(npar), t=0)
        atoms = int(prob.workload.structures.n_atoms.sum())
        oracle_step(O, prob, state, w.lambdas)
    best = 1e30
    for _ in range(3):
        t0 = time.perf_counter(); oracle_step(O, prob, state, w.lambdas); best = min(best, time.perf_counter() - t0)
    return {"value": atoms / best, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {prob.workload.structures.n_struct} structures ({atoms} atoms) of the workload, one full step "
                      f"(fp64 forward + loss + gradient + Adam), best of 3, OpenMP over structures"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return
    from oracle import nep_oracle as O
    w = make_workload(args)
    n = min(w.structures.n_struct, 128)        # bounded sample per step: the whole run stays within a few minutes
    prob = oracle_problem(w, n)
    npar = w.model.n_par
    state = dict(theta=prob.theta.copy(), m=np.zeros(npar), v=np.zeros(npar), vmax=np.zeros(npar), t=0)
    atoms = int(prob.workload.structures.n_atoms.sum())
    W = max(args.warmup, 1)
    for _ in range(W):
        oracle_step(O, prob, state, w.lambdas)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(O, prob, state, w.lambdas)
    dt = time.perf_counter() - t0
    value = atoms * args.steps / dt
    sample = f"first {n} structures ({atoms} atoms) of the workload per step"
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
           "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic (seeded lattices, teacher-NEP labels)",
           "config": {"workload": workload_name(w, args), "sample": sample},
           "cpu_baseline": {"value": value, "unit": UNIT, "kind": "oracle", "cores": O.max_threads(), "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def relaunch_under_torchrun(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no launcher around it: start the N ranks ourselves, exactly as the driver's
    torchrun line would (one process per GPU, rendezvous on 127.0.0.1), and pass their output through (rank 0 prints the JSON line;
    NCCL's communicator lines stay on stderr)."""
    import socket
    import torch
    have = torch.cuda.device_count()
    if args.impl == "ours" and have < args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but {have} CUDA device(s) are visible")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    args = parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    world = int(os.environ.get("WORLD_SIZE", "0"))
    if world == 0 and args.gpus > 1:
        sys.exit(relaunch_under_torchrun(args))
    if world > 0 and world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} contradicts WORLD_SIZE={world}")
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
