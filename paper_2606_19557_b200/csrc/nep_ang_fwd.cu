// nep_ang_fwd.cu -- S1 + S2 of the training step.
// S2: angular moments S_nL = sum_j g_n(r_ij) b_L(r^_ij) (Eq. 19) and the invariants built from them: 3-body
//     q_nl (Eq. 20), 4-/5-body (DESIGN C5).  grid = (slice pairs, channel chunks); thread = (atom, NCH channels).
// S1: radial descriptors q_n = sum_{T'} sum_k cR[t_i][T'][n][k] B_k[T'] (Eqs. 15-16) from the one-time
//     aggregate B, done by the threads of channel chunk 0 before their pair loop.
#include "nep_kernels.cuh"

namespace nep {

// STAGED: the rows of B that S1 reads are requested into shared memory before the pair sweep and S1 runs after it (the rows have
// long arrived); otherwise S1 runs first, from global memory.
template <int NCH, int K, bool STAGED>
__global__ void __launch_bounds__(PAIR_TB) k_ang_fwd(StepArgs a)
{
    extern __shared__ __align__(16) float smem[];
    const ModelDev& m = a.m;
    constexpr int CST = CoefStride<NCH, K>::value;
    float4* stage = reinterpret_cast<float4*>(smem) + threadIdx.x;
    float* cs = smem + SWEEP2_SMEM_BYTES / 4;
    float* cR = cs + m.T * m.T * CST;                 // chunk 0 only: radial coefficients transposed to [ti][tj][k][n], n padded to 4
    const int nRP = (m.nR + 3) & ~3;
    const int TK = m.T * m.KR;
    const int wib = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    float* barea = cR + m.T * m.T * m.KR * nRP + (size_t)wib * TK * WARP;   // STAGED: this warp's rows of B
    uint64_t* mbar = reinterpret_cast<uint64_t*>(cR + m.T * m.T * m.KR * nRP + (size_t)nwarp * TK * WARP) + wib;
    const int n0 = blockIdx.y * NCH;
    Lane L;
    const bool inb = lane_init(a, L);
    SweepA sw;
    if (inb) {
        if (STAGED && blockIdx.y == 0) rows_request(mbar, barea, a.d.B + (size_t)L.ds * TK * WARP, TK, nullptr, nullptr, 0);
        sw = sweep_init(a.d.recoffA, a.d.recA, a.d.cntA, L);
        sweep2_begin<SWEEP2_TB>(sw.rec, sw.width, stage);
    }
    load_cA_chunk<NCH, K>(a, cs, n0);
    if (blockIdx.y == 0)
#pragma unroll 8
        for (int i = threadIdx.x; i < m.T * m.T * m.KR * nRP; i += blockDim.x) {
            const int pt = i / (m.KR * nRP), rem = i - pt * m.KR * nRP, k = rem / nRP, n = rem - k * nRP;
            cR[i] = n < m.nR ? __ldg(a.theta + m.o_cR + (pt * m.nR + n) * m.KR + k) : 0.0f;
        }
    __syncthreads();
    if (!inb) return;
    float* qp = sb_ptr(a.b.q, L.w, m.D, L.lane);

    // ---- S1 ----  q_n = sum_{T', k} cR[t_i][T'][n][k] B_k[T']: every B value is loaded once and meets 8 channels in registers
    auto radial_descriptors = [&](const float* Bp) {   // Bp: row 0 of B for this lane, rows WARP apart (global or staged)
        for (int n0 = 0; n0 < m.nR; n0 += 8) {
            float acc[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[j] = 0.0f;
            if (L.ti >= 0) {
                const bool two = n0 + 4 < nRP;
                const float* cc = cR + (size_t)L.ti * m.T * m.KR * nRP + n0;   // rows r = T' * KR + k are nRP apart
                for (int r0 = 0; r0 < TK; r0 += 8) {
                    float b[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) b[j] = r0 + j < TK ? Bp[(size_t)(r0 + j) * WARP] : 0.0f;   // eight loads in flight
#pragma unroll
                    for (int j = 0; j < 8; ++j)
                        if (r0 + j < TK) {
                            const float4 c0 = *reinterpret_cast<const float4*>(cc + (r0 + j) * nRP);
                            acc[0] = fmaf(c0.x, b[j], acc[0]); acc[1] = fmaf(c0.y, b[j], acc[1]); acc[2] = fmaf(c0.z, b[j], acc[2]); acc[3] = fmaf(c0.w, b[j], acc[3]);
                            if (two) {
                                const float4 c1 = *reinterpret_cast<const float4*>(cc + (r0 + j) * nRP + 4);
                                acc[4] = fmaf(c1.x, b[j], acc[4]); acc[5] = fmaf(c1.y, b[j], acc[5]); acc[6] = fmaf(c1.z, b[j], acc[6]); acc[7] = fmaf(c1.w, b[j], acc[7]);
                            }
                        }
                }
            }
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (n0 + j < m.nR) qp[(size_t)(n0 + j) * WARP] = acc[j];
        }
    };
    if (blockIdx.y == 0) {
        // the structure accumulators that the force sweeps add into start from zero (benign duplicate stores)
        if (L.lane < 9) a.b.Ws[9 * L.sb + L.lane] = 0.0f;
        else if (L.lane == 9) a.b.Es[L.sb] = 0.0;
        reinterpret_cast<float4*>(a.b.F)[L.ib] = make_float4(0.f, 0.f, 0.f, 0.f);   // both force sweeps add into F
        if (!STAGED) radial_descriptors(sb_ptr(a.d.B, L.ds, TK, L.lane));
    }

    // ---- S2 ----
    float2 S2[NCH][NL / 2];   // (S_n,2i, S_n,2i+1): accumulated with packed FFMA2 (one issue slot per two lanes' FMAs)
#pragma unroll
    for (int n = 0; n < NCH; ++n)
#pragma unroll
        for (int l = 0; l < NL / 2; ++l) S2[n][l] = make_float2(0.0f, 0.0f);
    const float* cbase = cs + (L.ti > 0 ? L.ti : 0) * m.T * CST;
    const float rcinv = m.rcinvA;
    // two pairs per iteration (sweep_pairs2): the scalar chains of both are issued together, then the two rank-1 updates
    struct Prep { PairGeo p; float g[NCH]; };
    auto prep = [&](const float4& rc4, float on) {
        Prep P;
        P.p = pair_geo(rc4);
        radial_gn<NCH, K, false>(P.p.r, rcinv, cbase + P.p.tj * CST, P.g, nullptr, on);
        return P;
    };
    auto accumulate = [&](const Prep& P) {
        float b[NL];
        harm24(harm_z(P.p.z), harm_xy(P.p.x, P.p.y), b);
#pragma unroll
        for (int n = 0; n < NCH; ++n) {
            const float2 gg = make_float2(P.g[n], P.g[n]);
#pragma unroll
            for (int l = 0; l < NL / 2; ++l) S2[n][l] = __ffma2_rn(gg, make_float2(b[2 * l], b[2 * l + 1]), S2[n][l]);
        }
    };
    sweep2_run<SWEEP2_TB>(sw.rec, sw.width, sw.cnt, stage, [&](const float4& ra, const float4& rb, bool has2) {
        const Prep A = prep(ra, 1.0f), B = prep(rb, has2 ? 1.0f : 0.0f);
        accumulate(A);
        accumulate(B);
    });
    if (STAGED && blockIdx.y == 0) {
        rows_wait(mbar);
        radial_descriptors(barea + L.lane);
    }
    float S[NCH][NL];
#pragma unroll
    for (int n = 0; n < NCH; ++n)
#pragma unroll
        for (int l = 0; l < NL / 2; ++l) { S[n][2 * l] = S2[n][l].x; S[n][2 * l + 1] = S2[n][l].y; }
    float* Sp = sb_ptr(a.b.S, L.w, m.nA * NL, L.lane);
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        if (n0 + n < m.nA) {
            float qv[6];
            inv_values(S[n], qv);
            store_inv(m, qp, n0 + n, qv);
            float* sp = Sp + (size_t)(n0 + n) * NL * WARP;
#pragma unroll
            for (int l = 0; l < NL; ++l) sp[l * WARP] = S[n][l];
        }
    }
}

int launch_ang_fwd(nep_ctx* c, const StepArgs& a)
{
    const ModelDev& m = c->m;
    const int nch = pick_nch(c), kpad = pick_kpad(m.KA);
    const unsigned gx = (unsigned)((c->b.nbs * WARP + PAIR_TB - 1) / PAIR_TB);
    NEP_DISPATCH_NCH_K(nch, kpad, {
        const size_t base = SWEEP2_SMEM_BYTES + cA_chunk_bytes<NCH, K>(m) + 4 * (size_t)(m.T * m.T * m.KR * ((m.nR + 3) & ~3));
        const size_t smem = base + 4 * (size_t)(PAIR_TB / WARP) * m.T * m.KR * WARP + STAGED_BAR_BYTES;
        if (3 * smem + 3072 <= (size_t)c->max_smem_sm) {      // three blocks per SM (the register limit) keep fitting
            auto kern = k_ang_fwd<NCH, K, true>;
            if (smem > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            NEP_LAUNCH(c, "k_ang_fwd", kern, dim3(gx, a.nchunks), PAIR_TB, smem, a);
        } else {
            auto kern = k_ang_fwd<NCH, K, false>;
            if (base > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)base));
            NEP_LAUNCH(c, "k_ang_fwd", kern, dim3(gx, a.nchunks), PAIR_TB, base, a);
        }
    });
    return NEP_OK;
}

}  // namespace nep
