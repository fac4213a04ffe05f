"""nep_scaler_static (include/nep.h) against the context path.

nep_scaler_static exists for programs that want Eq. 2's descriptor scaler but cannot create a context: a context takes its
device memory from allocator callbacks, and a host whose memory pool owns the whole GPU, a caller that may not stall the device
with cudaMalloc in the middle of stream-ordered work, or a plain C / Fortran caller with two device pointers has none to give.
The call therefore allocates nothing and works in one fixed array inside the library, which every call on the GPU shares and
which keeps what the last call left there.  That is what this file checks: the scaler it returns equals the one
nep_compute_scaler forms on a context (same tolerance as tests/test_gpu_parity.py::test_descriptor_range_of_two_contexts...,
rtol 1e-6; the minima and maxima themselves are exact), on calls made back to back -- a long matrix first, then a short one
that uses fewer blocks, then the long one again -- so that a result which depended on the array's earlier contents would differ.

The file is named so that pytest collects it last: under `pytest -x` a failure here cannot hide any other test.  It needs
nothing from the tests before it and leaves nothing behind (the first call on the device happens here or earlier, outside any
stream capture either way)."""
import numpy as np
import pytest

from paper_2606_19557_b200 import workloads as wl
from tests import _gpu_harness as H

pytestmark = pytest.mark.gpu


def _context_path(workload):
    """The existing path: a context, nep_compute_scaler over the loaded set; also the set's unscaled descriptors [N][D]."""
    prob = H.make_problem(workload)
    with H.make_gpu(prob, labels=False, scaler="compute") as nep:
        s = nep.get_scaler()
        nep.forward()
        q = nep.get_descriptors()
    return q, s


def test_static_scaler_equals_the_context_path_on_consecutive_calls():
    import torch
    from paper_2606_19557_b200.binding import scaler_static
    long_q, long_s = _context_path(wl.make_config(2, n_struct=6))                 # 768 atoms, D = 35: seven rows per block
    short_q, short_s = _context_path(wl.tiny_workload(2, n_species=3, sizes=(33, 2, 40), box=(7.5, 3.1, 8.0)))   # 75 atoms
    assert long_q.shape[0] > 4 * short_q.shape[0]
    dev = torch.device("cuda")
    calls = [(long_q, long_s), (short_q, short_s), (long_q, long_s), (long_q, long_s)]
    outs = []
    for q, _ in calls:                                   # back to back in stream order, no synchronisation in between
        qd = torch.from_numpy(q).to(dev)
        sd = torch.full((q.shape[1],), float("nan"), dtype=torch.float32, device=dev)
        scaler_static(qd, sd)
        outs.append((qd, sd))
    torch.cuda.synchronize()
    for (q, s_ref), (_, sd) in zip(calls, outs):
        s = sd.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(s))
        assert np.allclose(s, s_ref, rtol=1e-6, atol=0.0), np.max(np.abs(s / s_ref - 1))
        lo, hi = q.min(axis=0).astype(np.float64), q.max(axis=0).astype(np.float64)      # Eq. 2 written out on the same fp32 matrix
        assert np.allclose(s, 1.0 / (hi - lo), rtol=1e-6)


def test_static_scaler_limits_and_degenerate_inputs():
    import torch
    from paper_2606_19557_b200.binding import NEP_ECAPACITY, NEP_STATIC_MAX_DESCRIPTORS, NepError, scaler_static
    dev = torch.device("cuda")
    D = NEP_STATIC_MAX_DESCRIPTORS
    g = torch.Generator(device="cpu").manual_seed(5)
    q = torch.randn(1000, D, generator=g).to(dev)                                 # the widest matrix the array admits: two rows per block
    s = torch.empty(D, dtype=torch.float32, device=dev)
    scaler_static(q, s)
    ref = 1.0 / (q.max(dim=0).values - q.min(dim=0).values)
    assert torch.allclose(s, ref, rtol=1e-6, atol=0.0)
    wide = torch.zeros(4, D + 1, device=dev)
    with pytest.raises(NepError) as ei:                                           # one column more: refused, nothing launched
        scaler_static(wide, torch.empty(D + 1, dtype=torch.float32, device=dev))
    assert ei.value.code == NEP_ECAPACITY and "NEP_STATIC_MAX_DESCRIPTORS" in str(ei.value)
    const = torch.full((50, 7), 3.25, device=dev)                                 # no range: s = 1 (DESIGN G10), as on a context
    s7 = torch.empty(7, dtype=torch.float32, device=dev)
    scaler_static(const, s7)
    assert torch.equal(s7, torch.ones(7, device=dev))
    scaler_static(torch.empty(0, 7, device=dev), s7.zero_())                      # no atoms: every range is empty
    assert torch.equal(s7, torch.ones(7, device=dev))
    scaler_static(q, s.zero_())                                                   # and the array still serves the next call
    assert torch.allclose(s, ref, rtol=1e-6, atol=0.0)
