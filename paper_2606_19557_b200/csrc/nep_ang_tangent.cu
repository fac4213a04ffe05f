// nep_ang_tangent.cu -- S7 (angular part), the tangent sweep of the second-order path (DESIGN C10):
//   Sd_nL = sum_j [g_n'(r) (r^ . d~) b_L + g_n(r) (grad_d b_L . d~)],   d~_ij = u_i - u_j - G_s^T d_ij,
//   qd_ang = J_q(S) Sd.
#include "nep_kernels.cuh"

namespace nep {

// STAGED: the rows the epilogue reads (moments of the chunk) are requested into shared memory before the sweep.
template <int NCH, int K, bool STAGED>
__global__ void __launch_bounds__(PAIR_TB) k_ang_tangent(StepArgs a)
{
    extern __shared__ __align__(16) float smem[];
    const ModelDev& m = a.m;
    constexpr int CST = CoefStride<NCH, K>::value;
    float4* stage = reinterpret_cast<float4*>(smem) + threadIdx.x;
    float* cs = smem + SWEEP2_SMEM_BYTES / 4;
    const int n0 = blockIdx.y * NCH;
    const int wib = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    float* area0 = cs + ((m.T * m.T * CST + 3) & ~3);
    float* area = area0 + (size_t)wib * (NCH * NL * WARP);
    uint64_t* mbar = reinterpret_cast<uint64_t*>(area0 + (size_t)nwarp * (NCH * NL * WARP)) + wib;
    if (STAGED) {
        const size_t w = (size_t)blockIdx.x * nwarp + wib;
        if (w < (size_t)a.b.nbs) rows_request(mbar, area, a.b.S + (w * m.nA + n0) * NL * WARP, chunk_rows(m, n0, NCH), nullptr, nullptr, 0);
    }
    Lane L;
    const bool inb = lane_init(a, L);
    SweepA sw;
    if (inb) {
        sw = sweep_init(a.d.recoffA, a.d.recA, a.d.cntA, L);
        sweep2_begin<SWEEP2_TB>(sw.rec, sw.width, stage);
    }
    load_cA_chunk<NCH, K>(a, cs, n0);
    __syncthreads();
    if (!inb) return;
    float G[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) G[k] = __ldg(a.b.G + 9 * L.sb + k);
    const float* ui = sb_ptr(a.b.u, L.w, 3, L.lane);
    const float uix = ui[0], uiy = ui[WARP], uiz = ui[2 * WARP];
    float2 Sd2[NCH][NL / 2];
#pragma unroll
    for (int n = 0; n < NCH; ++n)
#pragma unroll
        for (int l = 0; l < NL / 2; ++l) Sd2[n][l] = make_float2(0.0f, 0.0f);
    const float* cbase = cs + (L.ti > 0 ? L.ti : 0) * m.T * CST;
    const float rcinv = m.rcinvA;
    const float* ub = a.b.u;
    const int bbase = L.bbase;
    // per pair: the scalar part (geometry, tangent, radial functions) ...
    struct Prep { PairGeo p; Tangent T; float g[NCH], c[NCH]; };
    auto prep = [&](const float4& rc4, float on) {
        Prep P;
        P.p = pair_geo(rc4);
        P.T = pair_tangent(ub, bbase, P.p, uix, uiy, uiz, G);
        float dg[NCH];
        radial_gn<NCH, K, true, true>(P.p.r, rcinv, cbase + P.p.tj * CST, P.g, dg, on);
#pragma unroll
        for (int n = 0; n < NCH; ++n) P.c[n] = dg[n] * P.T.t;
        return P;
    };
    // ... and the rank-1 update of the 5 x 24 tangent moments
    auto accumulate = [&](const Prep& P) {
        float b[NL], bd[NL];
        const HarmZ hz = harm_z(P.p.z);
        const HarmXY hxy = harm_xy(P.p.x, P.p.y);
        harm24(hz, hxy, b);
        harm24_tangent(hz, hxy, P.T.rx, P.T.ry, P.T.rz, bd);
        float2 b2[NL / 2], bd2[NL / 2];
        pack24(b, b2); pack24(bd, bd2);
#pragma unroll
        for (int n = 0; n < NCH; ++n) {
            const float2 cc = dup2(P.c[n]), gg = dup2(P.g[n]);
#pragma unroll
            for (int l = 0; l < NL / 2; ++l) Sd2[n][l] = __ffma2_rn(cc, b2[l], __ffma2_rn(gg, bd2[l], Sd2[n][l]));
        }
    };
    sweep2_run<SWEEP2_TB>(sw.rec, sw.width, sw.cnt, stage, [&](const float4& ra, const float4& rb, bool has2) {
        const Prep A = prep(ra, 1.0f), B = prep(rb, has2 ? 1.0f : 0.0f);
        accumulate(A);
        accumulate(B);
    });
    float Sd[NCH][NL];
#pragma unroll
    for (int n = 0; n < NCH; ++n) unpack24(Sd2[n], Sd[n]);
    if (STAGED) rows_wait(mbar);
    const float* Sp = sb_ptr(a.b.S, L.w, m.nA * NL, L.lane);
    const float* Ss = area + L.lane;
    float* Sdp = sb_ptr(a.b.Sd, L.w, m.nA * NL, L.lane);
    float* qdp = sb_ptr(a.b.qd, L.w, m.D, L.lane);
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        if (n0 + n < m.nA) {
            float S[NL], qd[6];
            const size_t o = (size_t)(n0 + n) * NL * WARP;
#pragma unroll
            for (int l = 0; l < NL; ++l) {
                S[l] = STAGED ? Ss[(n * NL + l) * WARP] : Sp[o + l * WARP];
                Sdp[o + l * WARP] = Sd[n][l];
            }
            inv_tangent(S, Sd[n], qd);
            store_inv(m, qdp, n0 + n, qd);
        }
    }
}

int launch_ang_tangent(nep_ctx* c, const StepArgs& a)
{
    const ModelDev& m = c->m;
    const int nch = pick_nch(c), kpad = pick_kpad(m.KA);
    const unsigned gx = (unsigned)((c->b.nbs * WARP + PAIR_TB - 1) / PAIR_TB);
    NEP_DISPATCH_NCH_K(nch, kpad, {
        const size_t base = SWEEP2_SMEM_BYTES + ((cA_chunk_bytes<NCH, K>(m) + 15) & ~(size_t)15);
        const size_t smem = base + 4 * (size_t)(PAIR_TB / WARP) * (NCH * NL * WARP) + STAGED_BAR_BYTES;
        if (2 * smem + 2048 <= (size_t)c->max_smem_sm) {      // two blocks per SM (the register limit) keep fitting
            auto kern = k_ang_tangent<NCH, K, true>;
            if (smem > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            NEP_LAUNCH(c, "k_ang_tangent", kern, dim3(gx, a.nchunks), PAIR_TB, smem, a);
        } else {
            auto kern = k_ang_tangent<NCH, K, false>;
            if (base > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)base));
            NEP_LAUNCH(c, "k_ang_tangent", kern, dim3(gx, a.nchunks), PAIR_TB, base, a);
        }
    });
    return NEP_OK;
}

}  // namespace nep
