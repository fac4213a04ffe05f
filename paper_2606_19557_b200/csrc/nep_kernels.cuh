// nep_kernels.cuh -- helpers shared by the step kernels (forward, backward).
//
// Execution model of every pair sweep: ONE THREAD PER ATOM, one warp per 32-atom slice of one structure.
// Pair records of a slice are stored slot-major ([slot][lane], 16 B each), so the 32 lanes of a warp read
// 512 contiguous bytes per slot; each lane's records are sorted by neighbour type.  Per-atom tensors
// (angular moments and their adjoints, up to 5 channels x 24 harmonics) live in registers.
#pragma once
#include "nep_internal.h"
#include "nep_math.cuh"

namespace nep {

struct StepArgs {
    ModelDev m;
    DataDev d;
    BatchDev b;
    const float* theta;
    const float* scaler;
    float* g;
    int nchunks, nAP;   // angular channel chunks (blockIdx.y) and padded channel count nchunks * NCH
};

struct Lane {
    int w, lane, ti, sb, bbase;
    int64_t ib, ip;
    int ds;
};

// false if the warp is beyond the batch (whole warp returns together)
__device__ __forceinline__ bool lane_init(const StepArgs& a, Lane& L)
{
    L.w = (int)((blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5);
    L.lane = threadIdx.x & 31;
    if (L.w >= a.b.nbs) return false;
    L.ds = a.b.bslice[L.w];
    L.sb = a.b.bsb[L.w];
    L.bbase = a.b.bbase[L.w];
    L.ib = (int64_t)L.w * WARP + L.lane;
    L.ip = (int64_t)L.ds * WARP + L.lane;
    L.ti = a.d.type_p[L.ip];
    return true;
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

struct PairGeo {
    float dx, dy, dz, r, rinv, x, y, z;
    int jl, tj;
};
__device__ __forceinline__ PairGeo pair_geo(const float4& rec)
{
    PairGeo p;
    p.dx = rec.x; p.dy = rec.y; p.dz = rec.z;
    const int bits = __float_as_int(rec.w);
    p.jl = bits & 0xffffff; p.tj = bits >> 24;
    const float r2 = fmaf(p.dx, p.dx, fmaf(p.dy, p.dy, p.dz * p.dz));
    p.rinv = rsqrtf(r2);
    p.r = r2 * p.rinv;
    p.x = p.dx * p.rinv; p.y = p.dy * p.rinv; p.z = p.dz * p.rinv;
    return p;
}

// g_n(r) = sum_k c[k][n] f_k(r) (and g_n'), n = 0..NCH-1, coefficients at cs[k * nAP + n]  (Eq. 16)
template <int NCH, bool DERIV>
__device__ __forceinline__ void radial_gn(float r, float rcinv, int K, const float* __restrict__ cs, int nAP, float* g, float* dg)
{
#pragma unroll
    for (int n = 0; n < NCH; ++n) { g[n] = 0.0f; if (DERIV) dg[n] = 0.0f; }
    cheb_foreach<17>(r, rcinv, K, [&](int k, float fk, float dfk) {
#pragma unroll
        for (int n = 0; n < NCH; ++n) {
            const float c = cs[k * nAP + n];
            g[n] = fmaf(c, fk, g[n]);
            if (DERIV) dg[n] = fmaf(c, dfk, dg[n]);
        }
    });
}

// copies the angular coefficients of theta into shared memory as [pair type][k][n padded to nAP]
__device__ __forceinline__ void load_cA_smem(const StepArgs& a, float* cs)
{
    const ModelDev& m = a.m;
    const int tot = m.T * m.T * m.KA * a.nAP;
    for (int i = threadIdx.x; i < tot; i += blockDim.x) {
        const int n = i % a.nAP, k = (i / a.nAP) % m.KA, pt = i / (a.nAP * m.KA);
        cs[i] = (n < m.nA) ? a.theta[m.o_cA + (pt * m.nA + n) * m.KA + k] : 0.0f;
    }
}

// EdS_nL = dE_i/dS_nL = sum_a Fp[q index (a, n)] dq_a/dS_nL for the NCH channels of this thread (DESIGN C8)
template <int NCH>
__device__ __forceinline__ void load_EdS(const StepArgs& a, const Lane& L, int n0, float (*EdS)[NL])
{
    const ModelDev& m = a.m;
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        if (n0 + n < m.nA && L.ti >= 0) {
            float S[NL], coef[6];
#pragma unroll
            for (int l = 0; l < NL; ++l) S[l] = a.b.S[(int64_t)((n0 + n) * NL + l) * a.b.NBP + L.ib];
#pragma unroll
            for (int aa = 0; aa < 6; ++aa) coef[aa] = (aa < m.nang) ? a.b.Fp[(int64_t)(m.nR + aa * m.nA + n0 + n) * a.b.NBP + L.ib] : 0.0f;
            inv_adjoint(S, m.has4, m.has5, coef, EdS[n]);
        } else {
#pragma unroll
            for (int l = 0; l < NL; ++l) EdS[n][l] = 0.0f;
        }
    }
}

#define NEP_LAUNCH(c, name, kernel, grid, block, smem, ...)                        \
    do {                                                                           \
        nep::prof_begin((c), name);                                                \
        kernel<<<(grid), (block), (smem), (c)->stream>>>(__VA_ARGS__);             \
        nep::prof_end((c));                                                        \
        NEP_CUDA((c), cudaGetLastError());                                         \
    } while (0)

inline StepArgs make_args(nep_ctx* c, int NCH)
{
    StepArgs a;
    a.m = c->m; a.d = c->d; a.b = c->b; a.theta = c->theta; a.scaler = c->scaler; a.g = c->g;
    a.nchunks = (c->m.nA + NCH - 1) / NCH; a.nAP = a.nchunks * NCH;
    return a;
}
// channels per thread for the angular sweeps: ceil(nA / ceil(nA / 5)), at least 2
inline int pick_nch(int nA)
{
    int chunks = (nA + MAX_NCH - 1) / MAX_NCH;
    int nch = (nA + chunks - 1) / chunks;
    return nch < 2 ? 2 : nch;
}

}  // namespace nep
