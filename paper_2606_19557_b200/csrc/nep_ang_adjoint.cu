// nep_ang_adjoint.cu -- S9: the adjoint sweep giving the gradient of the angular descriptor coefficients (DESIGN C12)
//   g_cA[ti][tj][n][k] += [sum_L Sb_nL b_L + sum_L EdS_nL (grad b_L . d~)] f_k + [sum_L EdS_nL b_L] (r^.d~) f_k'
// Pass 1 holds Sb = J^T Qb + Fp H Sd in registers, pass 2 holds EdS = dE_i/dS; both add into per-thread accumulators
// acc[n][k] that belong to one (t_i, t_j) block of coefficients at a time (records are sorted by neighbour type).
//
// Reduction over atoms.  One species: every lane targets the same block, so a shuffle reduction per warp at the end.
// Several species: when a lane's run of one neighbour type ends, the warp stops (vote), the lane parks its
// accumulators in shared memory and the 32 lanes add them, element-parallel, into the warp's private table
// Gw[(t_i, t_j)][n][k] -- plain loads and stores, no atomics (shared-memory float atomics are CAS loops on sm_100).
// At the end the block adds its tables into g with one RED per non-zero entry.
#include "nep_kernels.cuh"

namespace nep {

template <int NCH, int K>
__global__ void __launch_bounds__(PAIR_TB) k_ang_adjoint(StepArgs a)
{
    extern __shared__ __align__(16) float smem[];
    const ModelDev& m = a.m;
    constexpr int CST = CoefStride<NCH, K>::value;
    constexpr int NK = NCH * K, PST = NK | 1;          // parked-accumulator row stride (odd: conflict-free)
    constexpr int NWARP = PAIR_TB / WARP;
    const int TT = m.T * m.T;
    float4* stage = reinterpret_cast<float4*>(smem) + threadIdx.x;
    float* Gall = smem + SWEEP_SMEM_BYTES / 4;           // [NWARP][TT][NK]
    float* park = Gall + NWARP * TT * NK;                // [NWARP][32][PST]   (several species only)
    const bool multi = m.T > 1;
    const int n0 = blockIdx.y * NCH;
    for (int i = threadIdx.x; i < NWARP * TT * NK; i += blockDim.x) Gall[i] = 0.0f;
    __syncthreads();
    Lane L;
    const bool inb = lane_init(a, L);
    if (inb) {
        const int wib = threadIdx.x >> 5;
        float* Gw = Gall + wib * TT * NK;
        float* pk = park + wib * WARP * PST;
        const SweepA sw = sweep_init(a.d.recoffA, a.d.recA, a.d.cntA, L);
        constexpr int KH = (K + 1) / 2;
        float2 acc2[NCH][KH];   // (acc_n,2i, acc_n,2i+1); the odd tail pairs with a zero basis value
#pragma unroll
        for (int n = 0; n < NCH; ++n)
#pragma unroll
            for (int k = 0; k < KH; ++k) acc2[n][k] = make_float2(0.0f, 0.0f);
        auto accv = [&](int n, int k) -> float& { return (k & 1) ? acc2[n][k >> 1].y : acc2[n][k >> 1].x; };
        int cur = -1;
        const int tiT = (L.ti > 0 ? L.ti : 0) * m.T;
        // parks the accumulators of the lanes whose run ended and adds them into the warp table (all lanes converged)
        auto flush = [&](bool fl) {
            const unsigned fm = __ballot_sync(0xffffffffu, fl);
            if (fm == 0) return;
            if (fl) {
#pragma unroll
                for (int n = 0; n < NCH; ++n)
#pragma unroll
                    for (int k = 0; k < K; ++k) { pk[L.lane * PST + n * K + k] = accv(n, k); accv(n, k) = 0.0f; }
            }
            __syncwarp();
            const int key = tiT + cur;
            unsigned mm = fm;
            while (mm) {
                const int f = __ffs(mm) - 1;
                mm &= mm - 1;
                const int kf = __shfl_sync(0xffffffffu, key, f);
                for (int e = L.lane; e < NK; e += WARP) Gw[kf * NK + e] += pk[f * PST + e];
            }
            __syncwarp();
        };
        auto pre = [&](bool act, const float4& rc4) {
            if (!multi) return;
            const int tj = act ? (__float_as_int(rc4.w) >> 24) : -1;
            flush(cur >= 0 && tj != cur);
            cur = tj;
        };
        const float rcinv = m.rcinvA;
        float2 X2[NCH][NL / 2];
        // ---- pass 1: Sb ----
        {
            float X[NCH][NL];
            const float* Sp = sb_ptr(a.b.S, L.w, m.nA * NL, L.lane);
            const float* Sdp = sb_ptr(a.b.Sd, L.w, m.nA * NL, L.lane);
            const float* Qbp = sb_ptr(a.b.Qb, L.w, m.D, L.lane);
            const float* Fpp = sb_ptr(a.b.Fp, L.w, m.D, L.lane);
#pragma unroll
            for (int n = 0; n < NCH; ++n) {
                if (n0 + n < m.nA && L.ti >= 0) {
                    float S[NL], Sd[NL], cq[6], cf[6];
                    const size_t o = (size_t)(n0 + n) * NL * WARP;
#pragma unroll
                    for (int l = 0; l < NL; ++l) { S[l] = Sp[o + l * WARP]; Sd[l] = Sdp[o + l * WARP]; }
                    load_inv_coef(m, Qbp, n0 + n, cq);
                    load_inv_coef(m, Fpp, n0 + n, cf);
                    inv_adjoint(S, cq, X[n]);
                    inv_hessian_action(S, Sd, cf, X[n]);
                } else {
#pragma unroll
                    for (int l = 0; l < NL; ++l) X[n][l] = 0.0f;
                }
                pack24(X[n], X2[n]);
            }
        }
        sweep_pairs(sw.rec, sw.width, sw.cnt, stage, pre, [&](const float4& rc4) {
            const PairGeo p = pair_geo(rc4);
            float b[NL], al[NCH];
            float2 b2[NL / 2];
            harm24(harm_z(p.z), harm_xy(p.x, p.y), b);
            pack24(b, b2);
#pragma unroll
            for (int n = 0; n < NCH; ++n) {
                float2 s1 = make_float2(0.0f, 0.0f);
#pragma unroll
                for (int l = 0; l < NL / 2; ++l) s1 = __ffma2_rn(X2[n][l], b2[l], s1);
                al[n] = s1.x + s1.y;
            }
            float fv[2 * KH];
            fv[2 * KH - 1] = 0.0f;
            cheb_basis<K, false>(p.r, rcinv, [&](int k, float fk, float) { fv[k] = fk; });
#pragma unroll
            for (int n = 0; n < NCH; ++n) {
                const float2 aa = dup2(al[n]);
#pragma unroll
                for (int k = 0; k < KH; ++k) acc2[n][k] = __ffma2_rn(aa, make_float2(fv[2 * k], fv[2 * k + 1]), acc2[n][k]);
            }
        });
        if (multi) { flush(cur >= 0); cur = -1; }
        // ---- pass 2: EdS ----
        {
            float X[NCH][NL];
            load_EdS<NCH>(a, L, n0, X);
#pragma unroll
            for (int n = 0; n < NCH; ++n) pack24(X[n], X2[n]);
        }
        float G[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) G[k] = __ldg(a.b.G + 9 * L.sb + k);
        const float* ui = sb_ptr(a.b.u, L.w, 3, L.lane);
        const float uix = ui[0], uiy = ui[WARP], uiz = ui[2 * WARP];
        const float* ub = a.b.u;
        const int bbase = L.bbase;
        sweep_pairs(sw.rec, sw.width, sw.cnt, stage, pre, [&](const float4& rc4) {
            const PairGeo p = pair_geo(rc4);
            const Tangent T = pair_tangent(ub, bbase, p, uix, uiy, uiz, G);
            float b[NL], bd[NL], be[NCH], de[NCH];
            float2 b2[NL / 2], bd2[NL / 2];
            const HarmZ hz = harm_z(p.z);
            const HarmXY hxy = harm_xy(p.x, p.y);
            harm24(hz, hxy, b);
            harm24_tangent(hz, hxy, T.rx, T.ry, T.rz, bd);
            pack24(b, b2); pack24(bd, bd2);
#pragma unroll
            for (int n = 0; n < NCH; ++n) {
                float2 s1 = make_float2(0.0f, 0.0f), s2 = make_float2(0.0f, 0.0f);
#pragma unroll
                for (int l = 0; l < NL / 2; ++l) { s1 = __ffma2_rn(X2[n][l], b2[l], s1); s2 = __ffma2_rn(X2[n][l], bd2[l], s2); }
                be[n] = (s1.x + s1.y) * T.t; de[n] = s2.x + s2.y;
            }
            float fv[2 * KH], dfv[2 * KH];
            fv[2 * KH - 1] = 0.0f; dfv[2 * KH - 1] = 0.0f;
            cheb_basis<K, true>(p.r, rcinv, [&](int k, float fk, float dfk) { fv[k] = fk; dfv[k] = dfk; });
#pragma unroll
            for (int n = 0; n < NCH; ++n) {
                const float2 dd = dup2(de[n]), bb = dup2(be[n]);
#pragma unroll
                for (int k = 0; k < KH; ++k)
                    acc2[n][k] = __ffma2_rn(dd, make_float2(fv[2 * k], fv[2 * k + 1]), __ffma2_rn(bb, make_float2(dfv[2 * k], dfv[2 * k + 1]), acc2[n][k]));
            }
        });
        if (multi) {
            flush(cur >= 0);
        } else {
            // single species: every lane targets the same block of coefficients -> shuffle-reduce, lane 0 stores
#pragma unroll
            for (int n = 0; n < NCH; ++n)
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    const float v = warp_sum(accv(n, k));
                    if (L.lane == 0) Gw[n * K + k] = v;
                }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < TT * NK; i += blockDim.x) {
        float v = 0.0f;
#pragma unroll
        for (int w = 0; w < NWARP; ++w) v += Gall[w * TT * NK + i];
        const int pt = i / NK, e = i - pt * NK, n = e / K, k = e - n * K;
        if (v != 0.0f && k < m.KA && n0 + n < m.nA) atomicAdd(a.g + m.o_cA + (pt * m.nA + n0 + n) * m.KA + k, v);
    }
}

int launch_ang_adjoint(nep_ctx* c, const StepArgs& a)
{
    const ModelDev& m = c->m;
    const int nch = pick_nch(m.nA), kpad = pick_kpad(m.KA);
    const unsigned gx = (unsigned)((c->b.nbs * WARP + PAIR_TB - 1) / PAIR_TB);
    NEP_DISPATCH_NCH_K(nch, kpad, {
        constexpr int NK = NCH * K, PST = NK | 1, NWARP = PAIR_TB / WARP;
        const size_t smem = SWEEP_SMEM_BYTES + 4 * (size_t)NWARP * ((size_t)m.T * m.T * NK + (m.T > 1 ? WARP * PST : 0));
        if (smem > (size_t)c->max_smem_optin) return fail(c, NEP_ECAPACITY, "angular coefficient tables do not fit in shared memory");
        auto kern = k_ang_adjoint<NCH, K>;
        if (smem > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        NEP_LAUNCH(c, "k_ang_adjoint", kern, dim3(gx, a.nchunks), PAIR_TB, smem, a);
    });
    return NEP_OK;
}

}  // namespace nep
