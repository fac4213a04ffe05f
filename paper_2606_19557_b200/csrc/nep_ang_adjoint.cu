// nep_ang_adjoint.cu -- S9: the adjoint sweep giving the gradient of the angular descriptor coefficients (DESIGN C12)
//   g_cA[ti][tj][n][k] += [sum_L Sb_nL b_L + sum_L EdS_nL (grad b_L . d~)] f_k + [sum_L EdS_nL b_L] (r^.d~) f_k'
// The two terms need different per-atom tensors in registers (Sb = J^T Qb + HS, and EdS = dE_i/dS), so they are two PASSES over
// the pair records.  A thread accumulates acc[n][k] over its pairs.
// One species (k_ang_adjoint): a block runs both passes and shuffle-reduces the accumulators; the per-atom rows come through the
// warp's shared-memory area (rows_request): those of the first pass are requested at kernel entry, those of the second pass as soon
// as the first pass has formed its tensor, so that they arrive while the first pass runs.
// Several species (k_ang_adjoint_ms): one warp per block and pass, snapshot table (below).
#include <algorithm>

#include "nep_kernels.cuh"

namespace nep {

template <int NCH, int K, bool STAGED>
__global__ void __launch_bounds__(PAIR_TB) k_ang_adjoint(StepArgs a)
{
    extern __shared__ __align__(16) float smem[];
    const ModelDev& m = a.m;
    constexpr int NK = NCH * K, NKP = (NK + 3) & ~3;
    const int nwarp = blockDim.x >> 5;
    float4* stage = reinterpret_cast<float4*>(smem) + threadIdx.x;
    float* tab_all = smem + PAIR_TB * 16;                                           // [NK] sums of the block, then the ticket of its warps
    const int n0 = blockIdx.y * NCH;
    const int wib = threadIdx.x >> 5;
    float* area = tab_all + (size_t)nwarp * NKP + (size_t)wib * staged_warp_floats(m, NCH);
    uint64_t* mbar = reinterpret_cast<uint64_t*>(tab_all + (size_t)nwarp * NKP + (size_t)nwarp * staged_warp_floats(m, NCH)) + wib;
    const size_t wg = (size_t)blockIdx.x * nwarp + wib;
    if (STAGED && wg < (size_t)a.b.nbs)   // pass 0: tangent moments of the chunk and the angular rows of Qb
        rows_request(mbar, area, a.b.Sd + (wg * m.nA + n0) * NL * WARP, chunk_rows(m, n0, NCH),
                     area + NCH * NL * WARP, a.b.Qb + (wg * m.D + m.nR) * WARP, m.D - m.nR);
    for (int i = threadIdx.x; i <= NKP; i += blockDim.x) tab_all[i] = 0.0f;           // (the ticket at [NKP] is an unsigned zero)
    __syncthreads();
    Lane L;
    const bool inb = lane_init(a, L);
    constexpr int KH = (K + 1) / 2;
    float2 acc2[NCH][KH];   // (acc_n,2i, acc_n,2i+1); the odd tail pairs with a zero basis value
#pragma unroll
    for (int n = 0; n < NCH; ++n)
#pragma unroll
        for (int k = 0; k < KH; ++k) acc2[n][k] = make_float2(0.0f, 0.0f);
    auto accv = [&](int n, int k) -> float& { return (k & 1) ? acc2[n][k >> 1].y : acc2[n][k >> 1].x; };
    if (inb) {
        const SweepA sw = sweep_init(a.d.recoffA, a.d.recA, a.d.cntA, L);
        sweep2_begin<PAIR_TB>(sw.rec, sw.width, stage);
        const float rcinv = m.rcinvA;
        float2 X2[NCH][NL / 2];
        {
            // ---- pass 0: Sb ----
            {
                float X[NCH][NL];
                if (STAGED) {
                    load_Sbar_staged<NCH>(a, L, n0, area + L.lane, area + NCH * NL * WARP + L.lane, mbar, X);
                    // the area is free again: rows of pass 1 (moments, angular rows of Fp), on their way while pass 0 runs
                    rows_request(mbar, area, a.b.S + (wg * m.nA + n0) * NL * WARP, chunk_rows(m, n0, NCH),
                                 area + NCH * NL * WARP, a.b.Fp + (wg * m.D + m.nR) * WARP, m.D - m.nR, true);
                } else {
                    load_Sbar<NCH>(a, L, n0, X);
                }
#pragma unroll
                for (int n = 0; n < NCH; ++n) pack24(X[n], X2[n]);
            }
            struct Prep { PairGeo p; float fv[2 * KH]; };
            auto prep = [&](const float4& rc4, float on) {
                Prep P;
                P.p = pair_geo(rc4);
                P.fv[2 * KH - 1] = 0.0f;
                cheb_basis<K, false, true>(P.p.r, rcinv, [&](int k, float fk, float) { P.fv[k] = fk; }, on);
                return P;
            };
            auto contract = [&](const Prep& P) {
                float b[NL], al[NCH];
                float2 b2[NL / 2];
                harm24(harm_z(P.p.z), harm_xy(P.p.x, P.p.y), b);
                pack24(b, b2);
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    float2 s1 = make_float2(0.0f, 0.0f);
#pragma unroll
                    for (int l = 0; l < NL / 2; ++l) s1 = __ffma2_rn(X2[n][l], b2[l], s1);
                    al[n] = s1.x + s1.y;
                }
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    const float2 aa = dup2(al[n]);
#pragma unroll
                    for (int k = 0; k < KH; ++k) acc2[n][k] = __ffma2_rn(aa, make_float2(P.fv[2 * k], P.fv[2 * k + 1]), acc2[n][k]);
                }
            };
            sweep2_run<PAIR_TB>(sw.rec, sw.width, sw.cnt, stage, [&](const float4& ra, const float4& rb, bool has2) {
                const Prep A = prep(ra, 1.0f), B = prep(rb, has2 ? 1.0f : 0.0f);
                contract(A);
                contract(B);
            });
        }
        {
            // ---- pass 1: EdS ----
            sweep2_begin<PAIR_TB>(sw.rec, sw.width, stage);
            {
                float X[NCH][NL];
                if (STAGED) {
                    rows_wait(mbar, 1);
                    load_EdS_staged<NCH>(m, L.ti, n0, area + L.lane, area + NCH * NL * WARP + L.lane, X);
                } else {
                    load_EdS<NCH>(a, L, n0, X);
                }
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
            struct Prep { PairGeo p; Tangent T; float fv[2 * KH], dfv[2 * KH]; };
            auto prep = [&](const float4& rc4, float on) {
                Prep P;
                P.p = pair_geo(rc4);
                P.T = pair_tangent(ub, bbase, P.p, uix, uiy, uiz, G);
                P.fv[2 * KH - 1] = 0.0f; P.dfv[2 * KH - 1] = 0.0f;
                cheb_basis<K, true, true>(P.p.r, rcinv, [&](int k, float fk, float dfk) { P.fv[k] = fk; P.dfv[k] = dfk; }, on);
                return P;
            };
            auto contract = [&](const Prep& P) {
                float b[NL], bd[NL], be[NCH], de[NCH];
                float2 b2[NL / 2], bd2[NL / 2];
                const HarmZ hz = harm_z(P.p.z);
                const HarmXY hxy = harm_xy(P.p.x, P.p.y);
                harm24(hz, hxy, b);
                harm24_tangent(hz, hxy, P.T.rx, P.T.ry, P.T.rz, bd);
                pack24(b, b2); pack24(bd, bd2);
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    float2 s1 = make_float2(0.0f, 0.0f), s2 = make_float2(0.0f, 0.0f);
#pragma unroll
                    for (int l = 0; l < NL / 2; ++l) { s1 = __ffma2_rn(X2[n][l], b2[l], s1); s2 = __ffma2_rn(X2[n][l], bd2[l], s2); }
                    be[n] = (s1.x + s1.y) * P.T.t; de[n] = s2.x + s2.y;
                }
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    const float2 dd = dup2(de[n]), bb = dup2(be[n]);
#pragma unroll
                    for (int k = 0; k < KH; ++k)
                        acc2[n][k] = __ffma2_rn(dd, make_float2(P.fv[2 * k], P.fv[2 * k + 1]),
                                                __ffma2_rn(bb, make_float2(P.dfv[2 * k], P.dfv[2 * k + 1]), acc2[n][k]));
                }
            };
            sweep2_run<PAIR_TB>(sw.rec, sw.width, sw.cnt, stage, [&](const float4& ra, const float4& rb, bool has2) {
                const Prep A = prep(ra, 1.0f), B = prep(rb, has2 ? 1.0f : 0.0f);
                contract(A);
                contract(B);
            });
        }
        // every lane targets the same block of coefficients: reduce-scatter over the lanes, then shared-memory adds into the block's table
        // (at most 64 values at a time: a larger register array would go to local memory)
        constexpr int P = NK <= 32 ? 32 : 64, PL = P / 32;
        const int lane = threadIdx.x & 31;
#pragma unroll
        for (int base = 0; base < NK; base += P) {
            float v[P];
#pragma unroll
            for (int e = 0; e < P; ++e) v[e] = base + e < NK ? accv((base + e) / K, (base + e) % K) : 0.0f;
            warp_reduce_scatter<P>(v);
#pragma unroll
            for (int j = 0; j < PL; ++j)
                if (base + PL * lane + j < NK) atomicAdd(tab_all + base + PL * lane + j, v[j]);
        }
    }
    // no block barrier: a warp leaves when it is done; the last one of the block (ticket) adds the table to g
    __syncwarp();
    bool last = false;
    if ((threadIdx.x & 31) == 0) {
        __threadfence_block();
        last = atomicAdd(reinterpret_cast<unsigned*>(tab_all + NKP), 1u) == (unsigned)nwarp - 1u;
    }
    if (!__shfl_sync(0xffffffffu, (int)last, 0)) return;
    __threadfence_block();
    for (int i = threadIdx.x & 31; i < NK; i += WARP) {
        const float v = *reinterpret_cast<volatile float*>(tab_all + i);
        const int n = i / K, k = i - n * K;
        if (v != 0.0f && k < m.KA && n0 + n < m.nA) atomicAdd(a.g + m.o_cA + (size_t)(n0 + n) * m.KA + k, v);
    }
}

// ------------------------------------------------------------------------------------------------
// Several species, second design.  One warp per block, blockIdx.z = pass.  A lane's accumulators are never cleared: when its
// run of neighbour type t ends it stores a SNAPSHOT of them (12 x 128-bit stores into its own row of a lane-major table
// snap[lane][t][n k], row stride an odd number of 16-byte units: conflict free); types the lane does not meet get the snapshot
// of the type before them, so that the sum over the pairs with neighbour type t is snap[t] - snap[t - 1] for every lane.
// The last type's snapshot is the final state of the accumulators and stays in registers.
// After the sweep the lanes of one centre type are a contiguous range (slot order of a slice): thread r sums column
// r = (t, n, k) over that range and issues one RED per (t_i, t_j, n, k).
// ------------------------------------------------------------------------------------------------
template <int NCH, int K>
__global__ void __launch_bounds__(WARP) k_ang_adjoint_ms(StepArgs a, int ahead)
{
    extern __shared__ __align__(16) float smem[];
    const ModelDev& m = a.m;
    constexpr int NK = NCH * K, NKP = (NK + 3) & ~3, KH = (K + 1) / 2;
    const int T = m.T;
    const int TR = T - 1;                                               // table rows per lane: the last type is never stored (below)
    const int LS = (TR * NKP) + (((TR * NKP) >> 2) & 1 ? 0 : 4);        // lane stride (words): LS / 4 odd
    float4* stage = reinterpret_cast<float4*>(smem) + threadIdx.x;      // SWEEP_STAGES cells per thread, WARP apart
    float* tab = smem + (WARP * 4 * SWEEP_STAGES);
    const int n0 = blockIdx.y * NCH;
    const int lane = threadIdx.x;
    // the per-atom rows that the block `ahead` launches later (about one resident wave) will load in its prologue -> L2
    if (lane == 0 && (int)blockIdx.x + ahead < a.b.nbs) {
        const size_t w2 = (size_t)blockIdx.x + ahead, srow = (size_t)m.nA * NL * WARP, drow = (size_t)m.D * WARP;
        prefetch_l2(a.b.S + w2 * srow, (unsigned)(4 * srow));
        prefetch_l2(a.b.Fp + w2 * drow, (unsigned)(4 * drow));
        if (blockIdx.z == 0) { prefetch_l2(a.b.Sd + w2 * srow, (unsigned)(4 * srow)); prefetch_l2(a.b.Qb + w2 * drow, (unsigned)(4 * drow)); }
        else prefetch_l2(a.b.u + w2 * 3 * WARP, 12 * WARP);
    }
    Lane L;
    lane_init_slice(a, L, (int)blockIdx.x);
    float2 acc2[NCH][KH];
#pragma unroll
    for (int n = 0; n < NCH; ++n)
#pragma unroll
        for (int k = 0; k < KH; ++k) acc2[n][k] = make_float2(0.0f, 0.0f);
    auto accv = [&](int e) -> float { const int n = e / K, k = e - n * K; return e < NK ? ((k & 1) ? acc2[n][k >> 1].y : acc2[n][k >> 1].x) : 0.0f; };
    float* mine = tab + (size_t)lane * LS;
    int cur = 0;
    auto snapshot_to = [&](int tj) {      // rows cur .. tj - 1 <- the accumulators as they are (row T - 1 would hold the final values: not stored)
        const int end = tj < TR ? tj : TR;
        while (cur < end) {
            float4* dst = reinterpret_cast<float4*>(mine + cur * NKP);
#pragma unroll
            for (int i = 0; i < NKP / 4; ++i) dst[i] = make_float4(accv(4 * i), accv(4 * i + 1), accv(4 * i + 2), accv(4 * i + 3));
            ++cur;
        }
    };
    if (L.ti >= 0) {
        const SweepA sw = sweep_init(a.d.recoffA, a.d.recA, a.d.cntA, L);
        const float rcinv = m.rcinvA;
        float2 X2[NCH][NL / 2];
        if (blockIdx.z == 0) {
            {
                float X[NCH][NL];
                load_Sbar<NCH>(a, L, n0, X);
#pragma unroll
                for (int n = 0; n < NCH; ++n) pack24(X[n], X2[n]);
            }
            sweep_pairs_tb<WARP>(sw.rec, sw.width, sw.cnt, stage, [&](const float4& rc4) {
                const PairGeo p = pair_geo(rc4);
                snapshot_to(p.tj);
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
                cheb_basis<K, false, true>(p.r, rcinv, [&](int k, float fk, float) { fv[k] = fk; });
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    const float2 aa = dup2(al[n]);
#pragma unroll
                    for (int k = 0; k < KH; ++k) acc2[n][k] = __ffma2_rn(aa, make_float2(fv[2 * k], fv[2 * k + 1]), acc2[n][k]);
                }
            });
        } else {
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
            sweep_pairs_tb<WARP>(sw.rec, sw.width, sw.cnt, stage, [&](const float4& rc4) {
                const PairGeo p = pair_geo(rc4);
                snapshot_to(p.tj);
                const Tangent Tg = pair_tangent(ub, bbase, p, uix, uiy, uiz, G);
                float b[NL], bd[NL], be[NCH], de[NCH];
                float2 b2[NL / 2], bd2[NL / 2];
                const HarmZ hz = harm_z(p.z);
                const HarmXY hxy = harm_xy(p.x, p.y);
                harm24(hz, hxy, b);
                harm24_tangent(hz, hxy, Tg.rx, Tg.ry, Tg.rz, bd);
                pack24(b, b2); pack24(bd, bd2);
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    float2 s1 = make_float2(0.0f, 0.0f), s2 = make_float2(0.0f, 0.0f);
#pragma unroll
                    for (int l = 0; l < NL / 2; ++l) { s1 = __ffma2_rn(X2[n][l], b2[l], s1); s2 = __ffma2_rn(X2[n][l], bd2[l], s2); }
                    be[n] = (s1.x + s1.y) * Tg.t; de[n] = s2.x + s2.y;
                }
                float fv[2 * KH], dfv[2 * KH];
                fv[2 * KH - 1] = 0.0f; dfv[2 * KH - 1] = 0.0f;
                cheb_basis<K, true, true>(p.r, rcinv, [&](int k, float fk, float dfk) { fv[k] = fk; dfv[k] = dfk; });
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    const float2 dd = dup2(de[n]), bb = dup2(be[n]);
#pragma unroll
                    for (int k = 0; k < KH; ++k)
                        acc2[n][k] = __ffma2_rn(dd, make_float2(fv[2 * k], fv[2 * k + 1]), __ffma2_rn(bb, make_float2(dfv[2 * k], dfv[2 * k + 1]), acc2[n][k]));
                }
            });
        }
    }
    snapshot_to(T);                       // the run in progress and the types after it (a lane without pairs: zeros everywhere)
    __syncwarp();
    // Column sums per centre type: the lanes of one type are a contiguous range.  A thread owns QUADS of four consecutive
    // table columns (t_j, 4 e .. 4 e + 3) and walks the lanes of the range with one 128-bit load each; the sums of neighbour
    // type t_j are snapshot differences, taken through a small array of the column sums.
    // The snapshot of the LAST neighbour type is the final state of the accumulators, which every lane still holds in registers: its
    // column sums come from a masked reduce-scatter over the lanes instead of a table row (one row per lane less: 25 instead of 31 KB of
    // shared memory per warp at five species, 8 instead of 6 warps per SM).
    const int nquad = (TR * NKP) >> 2;
    float* cs = tab + (size_t)WARP * LS;                 // [T * NKP] column sums of the current centre type
    constexpr int P = NK <= 32 ? 32 : 64, PL = P / 32;   // at most 64 values at a time (a larger register array would go to local memory)
    const size_t tstep = (size_t)T * m.nA * m.KA;
    for (int ti = 0; ti < T; ++ti) {
        const unsigned bm = __ballot_sync(0xffffffffu, L.ti == ti);
        if (bm == 0u) continue;
        const int c0 = __ffs(bm) - 1, c1 = c0 + __popc(bm);
        for (int qd = lane; qd < nquad; qd += WARP) {
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
            for (int c = c0; c < c1; ++c) {
                const float4 x = *reinterpret_cast<const float4*>(tab + (size_t)c * LS + 4 * qd);
                v.x += x.x; v.y += x.y; v.z += x.z; v.w += x.w;
            }
            *reinterpret_cast<float4*>(cs + 4 * qd) = v;
        }
        {
            const bool in = lane >= c0 && lane < c1;
#pragma unroll
            for (int base = 0; base < NKP; base += P) {
                float v[P];
#pragma unroll
                for (int e = 0; e < P; ++e) v[e] = in ? accv(base + e) : 0.0f;
                warp_reduce_scatter<P>(v);
#pragma unroll
                for (int j = 0; j < PL; ++j)
                    if (base + PL * lane + j < NKP) cs[TR * NKP + base + PL * lane + j] = v[j];
            }
        }
        __syncwarp();
        for (int r = lane; r < T * NKP; r += WARP) {
            const int tj = r / NKP, e = r - tj * NKP, n = e / K, k = e - n * K;
            if (!(e < NK && k < m.KA && n0 + n < m.nA)) continue;
            const float v = cs[r] - (tj > 0 ? cs[r - NKP] : 0.0f);
            if (v != 0.0f) atomicAdd(a.g + m.o_cA + ((size_t)tj * m.nA + n0 + n) * m.KA + k + ti * tstep, v);
        }
        __syncwarp();
    }
}

int launch_ang_adjoint(nep_ctx* c, const StepArgs& a)
{
    const ModelDev& m = c->m;
    const int nch = pick_nch(c), kpad = pick_kpad(m.KA);
    NEP_DISPATCH_NCH_K(nch, kpad, {
        constexpr int NK = NCH * K;
        // one species: both passes in one block; a batch far below one resident wave is bound by the latency of one warp, and runs the
        // two passes side by side as separate one-warp blocks (the multi-species kernel, whose table is then empty)
        if (m.T == 1 && c->b.nbs >= c->sm_count / 2) {
            const int nw = PAIR_TB / WARP;
            const size_t base = (size_t)PAIR_TB * 64 + 4 * (size_t)nw * ((NK + 3) & ~3);
            const size_t smem = base + 4 * nw * staged_warp_floats(m, NCH) + STAGED_BAR_BYTES;
            const dim3 grid((unsigned)((c->b.nbs + nw - 1) / nw), a.nchunks);
            if (2 * smem + 2048 <= (size_t)c->max_smem_sm) {
                auto kern = k_ang_adjoint<NCH, K, true>;
                if (smem > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                NEP_LAUNCH(c, "k_ang_adjoint", kern, grid, nw * WARP, smem, a);
            } else {
                NEP_LAUNCH(c, "k_ang_adjoint", (k_ang_adjoint<NCH, K, false>), grid, nw * WARP, base, a);
            }
        } else {
            constexpr int NKP = (NK + 3) & ~3;
            const int LS = ((m.T - 1) * NKP) + (((((m.T - 1) * NKP) >> 2) & 1) ? 0 : 4);
            const size_t smem = (size_t)WARP * 16 * SWEEP_STAGES + 4 * ((size_t)WARP * LS + (size_t)m.T * NKP);
            if (smem > (size_t)c->max_smem_optin) return fail(c, NEP_ECAPACITY, "angular coefficient tables do not fit in shared memory");
            auto kern = k_ang_adjoint_ms<NCH, K>;
            if (smem > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            int occ = 1;
            NEP_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, WARP, smem));
            const int ahead = std::max(1, occ * c->sm_count / (2 * a.nchunks));      // blocks of one (chunk, pass) in a resident wave
            NEP_LAUNCH(c, "k_ang_adjoint", kern, dim3((unsigned)c->b.nbs, a.nchunks, 2), WARP, smem, a, ahead);
        }
    });
    return NEP_OK;
}

}  // namespace nep
