"""Algorithmic work model of the step kernels: flops and HBM bytes each kernel MUST do per launch,
independent of how the kernel is written.  FMA = 2 flops; one special-function evaluation (rsqrt, sin, cos, tanh) = 1.
Used by bench.py for the `roofline` object; holds no kernel code and none of the method's arithmetic.

Per-pair building blocks (counted from the equations, P:226-253 and DESIGN C2-C12):
  geo      = 10                 r^2 (5), 1/r (1), r (1), unit vector (3)
  basis(K) = 8 + 4 (K-1)        u, f_c (cos), x, Chebyshev recurrence, f_k = (T_k + 1) f_c / 2           Eqs. 17-18
  basisd(K)= 14 + 11 (K-1)      the same with d/dr of every f_k
  Y        = 65                 the 24 real harmonics l = 1..4 of r^ (14 Legendre factors, Re/Im (x+iy)^m, 20 products)
  Ytan     = 96                 directional derivative of the 24 harmonics along a tangent vector
  gradc    = 100                sum_L A_L grad b_L (reverse mode of Y)
  ptan     = 35                 d~ = u_i - u_j - G^T d, t = r^ . d~, tangent of r^
"""
from __future__ import annotations

NL = 24
GEO, Y, YTAN, GRADC, PTAN = 10, 65, 96, 100, 35


def basis(K: int) -> int:
    return 8 + 4 * (K - 1)


def basisd(K: int) -> int:
    return 14 + 11 * (K - 1)


def kernel_models(model, sizes: dict) -> dict:
    """{kernel name: {"flops": per launch, "bytes": per launch}} for the current batch.

    model: ModelSpec-like (n_R, n_A, K_R, K_A, n_ang, D, neurons, n_species); sizes: nep.get_sizes()."""
    nR, nA, KR, KA, nang, D, H, T = model.n_R, model.n_A, model.K_R, model.K_A, model.n_ang, model.D, model.neurons, model.n_species
    N, PR, PA = sizes["N_b"], sizes["P_R_b"], sizes["P_A_b"]
    KRP = (KR + 3) // 4 * 4
    f4 = 4
    m = {}
    # S1 (radial q from the aggregate B) runs inside k_ang_fwd
    m["k_ang_fwd"] = dict(flops=PA * (GEO + basis(KA) + 2 * nA * KA + Y + 2 * NL * nA) + N * 2 * nR * KR * T,
                          bytes=16 * PA + N * f4 * (NL * nA + nA * nang) + N * f4 * (T * KR + nR))
    m["k_ann_fwd"] = dict(flops=N * (4 * H * D + 6 * H + 2 * D + 2 * T * nR * KR),
                          bytes=N * f4 * (2 * D + H + T * KRP + 1))
    # half list: one record per undirected pair; both directions' sums s_ij, s_ji from one evaluation of the basis
    m["k_rad_force"] = dict(flops=(PR // 2) * (GEO + basisd(KR) + 4 * KR + 30),
                            bytes=16 * (PR // 2) + N * f4 * (T * KRP + 3))
    m["k_ang_force"] = dict(flops=PA * (GEO + basisd(KA) + 4 * nA * KA + Y + nA * (4 * NL + 2) + GRADC + 14 + 24),
                            bytes=16 * PA + N * f4 * (NL * nA + nA * nang + 3))
    m["k_rad_tangent"] = dict(flops=PR * (GEO + PTAN + basisd(KR) + 2 * KR),
                              bytes=16 * PR + N * f4 * (T * KR + 3))
    m["k_ang_tangent"] = dict(flops=PA * (GEO + PTAN + basisd(KA) + 4 * nA * KA + Y + YTAN + nA * (1 + 4 * NL)),
                              bytes=16 * PA + N * f4 * (2 * NL * nA + nA * nang + 3))
    m["k_ann_bwd"] = dict(flops=N * (8 * H * D + 12 * H + 2 * D + 6 * T * nR * KR),
                          bytes=N * f4 * (4 * D + H + 2 * T * KR))
    m["k_ang_adjoint"] = dict(flops=PA * ((GEO + Y + 2 * NL * nA + basis(KA) + 2 * nA * KA)
                                          + (GEO + PTAN + Y + YTAN + nA * (4 * NL + 1) + basisd(KA) + 4 * nA * KA)),
                              bytes=2 * 16 * PA + N * f4 * (2 * NL * nA + 2 * nA * nang + 3))
    npar = T * (D + 2) * H + 1 + T * T * (nR * KR + nA * KA)
    m["k_adam"] = dict(flops=12 * npar, bytes=7 * f4 * npar)
    m["k_loss"] = dict(flops=N * 12, bytes=N * f4 * 9)
    return m


def fp32_peak_flops(sm_count: int = 148, sm_mhz: float = 1965.0, lanes: int = 128) -> float:
    """FP32 FMA peak: SMs x 128 lanes x 2 flops x clock (B200: 148 SMs, clocks.max.sm 1965 MHz -> 74.4 TFLOP/s)."""
    return sm_count * lanes * 2 * sm_mhz * 1e6


def csrc_hash() -> str:
    """SHA-256 (first 16 hex digits) over the kernel sources: a stored ncu figure is only quoted for the kernels it measured."""
    import hashlib
    import os
    d = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc")
    h = hashlib.sha256()
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".h")):
            h.update(name.encode())
            with open(os.path.join(d, name), "rb") as f:
                h.update(f.read())
    return h.hexdigest()[:16]


def step_totals(models: dict) -> dict:
    return {"flops": sum(v["flops"] for v in models.values()), "bytes": sum(v["bytes"] for v in models.values())}
