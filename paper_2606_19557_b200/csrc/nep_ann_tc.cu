// nep_ann_tc.cu -- the per-species tanh network of Eq. 3 on the 5th-generation tensor cores (tcgen05, TMEM).
//
// The network is the one dense contraction of the training step.  A TILE is 128 atoms of one species
// (b.alist, every species padded to whole tiles); one thread = one atom = one TMEM lane.  Per tile:
//
//   S3 (k_ann_fwd_tc)   X = Q W0s^T   [128 x D] . [D x H]     A = q rows written to TMEM by their threads (split hi + lo),
//                                                             B = W0s = w0 o s (scaler folded in) from shared memory, 3xTF32
//                       h = tanh(X - b0), E_i = w1 . h - b1, e = w1 o (1 - h^2)              (threads, from TMEM)
//                       Fp = E W0s    [128 x H] . [H x D]     A = e rows in TMEM (hi + lo), 3xTF32
//                       a_k[T'] = sum_n Fp_n cR[t][T'][n][k]                                 (threads)
//   S8 (k_ann_bwd_tc)   qd_rad = cR Bd (threads);  Xd = Qd W0s^T;  gamma = eps e - 2 h e Xd;  Qb = Gamma W0s;
//                       ACC[mu][.] += sum_atoms gamma_mu [q | B | 1] + e_mu [qd | Bd | 0]    [H x 128] . [128 x (D + T K_R + 1)]
//                       ACC lives in TMEM across all tiles of one species that the block owns; when the species changes it is
//                       flushed:  g_w0[mu][v] += s_v ACC[mu][v],  g_b0[mu] -= ACC[mu][ones],
//                                 g_cR[t][T'][n][k] += sum_mu W0s[mu][n] ACC[mu][D + T' K_R + k]   (Qb_n = s_n sum_mu gamma_mu w0[mu][n])
//                       The contraction over atoms needs its operands K-major over atoms: the threads write gamma, e, q, qd, B,
//                       Bd a second time, transposed, into shared memory ([atom / 4][row][4], row stride padded to an odd
//                       number of 16-byte units: conflict-free scalar stores).
//
// Precision per product (tolerances of BASELINE.json: E 1e-5 eV/atom, F 1e-4, g 1e-3 relative):
//   X, Fp     : 3xTF32 (hi hi + lo hi + hi lo): the energy and the forces need fp32-accurate products;
//   Xd, Qb, ACC: 1xTF32 with operands rounded to nearest (unbiased 2^-12 relative per operand): they feed only the parameter
//               gradient, whose rounding errors average over the atoms of the batch.
// Models whose tiles do not fit (shared memory, 512 TMEM columns) run the FFMA kernels of nep_ann.cu.
#include <stdio.h>
#include <stdlib.h>

#include <algorithm>

#include "nep_kernels.cuh"
#include "nep_umma.cuh"

namespace nep {
using namespace umma;

constexpr int TC_TM = 128;      // atoms per tile = threads per block = TMEM lanes

struct TcLay {
    int DP8, HP8, HP16, DP16, KMAX, TK, TKRP, nR4, NC16, MA;
    int cR2, cACC, ncols;                         // TMEM columns: R1 at 0
    int oW1H, oW1L, oW2H, oW2L, ob0, ow1, osc, ocR, oQBT, oQDT, oGT, oET, ogw1, oStg, oEi, oBar, total;   // float offsets
    int ldQ, ldG;                                 // rows' of the transposed buffers (odd)
};

static inline int pow2_cols(int n) { int c = 32; while (c < n) c <<= 1; return c; }

static TcLay tc_layout(const ModelDev& m, bool bwd)
{
    TcLay l{};
    l.DP8 = rup(m.D, 8); l.HP8 = rup(m.H, 8); l.HP16 = rup(m.H, 16); l.DP16 = rup(m.D, 16);
    l.KMAX = std::max(l.DP8, l.HP8);
    l.TK = m.T * m.KR; l.TKRP = m.T * m.KRP; l.nR4 = rup(m.nR, 4);
    l.NC16 = rup(m.D + l.TK + 1, 16);
    l.MA = l.HP8 <= 64 ? 64 : 128;
    const int r1 = bwd ? l.KMAX : 2 * l.KMAX, r2 = std::max(l.HP16, l.DP16);
    l.cR2 = r1; l.cACC = r1 + r2;
    l.ncols = pow2_cols(r1 + r2 + (bwd ? l.NC16 : 0));
    int o = 0;
    auto take = [&](int n) { int r = o; o += rup(n, 32); return r; };     // 128-byte aligned pieces
    l.ldQ = l.NC16 + 1; l.ldG = l.HP8 + 1;
    if (bwd) {
        // the transposed buffers first: the tensor core reads up to MA rows of GT / ET per K chunk, i.e. a little past their end
        l.oQBT = take((TC_TM / 4) * l.ldQ * 4); l.oQDT = take((TC_TM / 4) * l.ldQ * 4);
        l.oGT = take((TC_TM / 4) * l.ldG * 4); l.oET = take((TC_TM / 4) * l.ldG * 4 + 4 * 128);
    }
    l.oW1H = take(l.DP8 * l.HP16); l.oW2H = take(l.HP8 * l.DP16);
    if (!bwd) { l.oW1L = take(l.DP8 * l.HP16); l.oW2L = take(l.HP8 * l.DP16); }
    l.ob0 = take(l.HP8); l.ow1 = take(l.HP8); l.osc = take(l.DP8);
    l.ocR = take(bwd ? l.TK * l.nR4 : m.nR * l.TKRP);
    l.ogw1 = take(l.HP8);
    l.oStg = take(m.per_type);
    l.oEi = take(bwd ? 0 : 4 * TC_TM);
    l.oBar = take(8);
    l.total = o;
    return l;
}

// ------------------------------------------------------------------------------------------------
// weights of species t into shared memory as B operands (K-major, [K / 4][rows][4]), scaler folded in, zero padded
//   W1: rows = mu (HP16), K = v (DP8)  -> X = Q W1^T ;   W2: rows = v (DP16), K = mu (HP8) -> Fp = E W2^T
// ------------------------------------------------------------------------------------------------
template <bool SPLIT>
__device__ __forceinline__ void tc_load_weights(const StepArgs& a, const TcLay& l, float* sm, int t)
{
    const ModelDev& m = a.m;
    // raw parameters of the species (w0 | b0 | w1 are contiguous in theta) and the scaler: coalesced, eight loads in flight
    const float* th = a.theta + (size_t)t * m.per_type;
    float* stg = sm + l.oStg;
#pragma unroll 8
    for (int i = threadIdx.x; i < m.per_type; i += blockDim.x) stg[i] = __ldg(th + i);
    for (int i = threadIdx.x; i < l.DP8; i += blockDim.x) sm[l.osc + i] = (i < m.D) ? __ldg(a.scaler + i) : 0.0f;
    __syncthreads();
#pragma unroll 4
    for (int i = threadIdx.x; i < l.DP8 * l.HP16; i += blockDim.x) {
        const int c = i / (4 * l.HP16), rem = i - c * 4 * l.HP16, mu = rem >> 2, v = 4 * c + (rem & 3);
        const float wv = (mu < m.H && v < m.D) ? stg[mu * m.D + v] * sm[l.osc + v] : 0.0f;
        const float hi = tf32_rn(wv);
        sm[l.oW1H + i] = hi;
        if (SPLIT) sm[l.oW1L + i] = tf32_rn(wv - hi);
    }
#pragma unroll 4
    for (int i = threadIdx.x; i < l.HP8 * l.DP16; i += blockDim.x) {
        const int c = i / (4 * l.DP16), rem = i - c * 4 * l.DP16, v = rem >> 2, mu = 4 * c + (rem & 3);
        const float wv = (mu < m.H && v < m.D) ? stg[mu * m.D + v] * sm[l.osc + v] : 0.0f;
        const float hi = tf32_rn(wv);
        sm[l.oW2H + i] = hi;
        if (SPLIT) sm[l.oW2L + i] = tf32_rn(wv - hi);
    }
    for (int i = threadIdx.x; i < l.HP8; i += blockDim.x) {
        sm[l.ob0 + i] = (i < m.H) ? stg[m.H * m.D + i] : 0.0f;
        sm[l.ow1 + i] = (i < m.H) ? stg[m.H * m.D + m.H + i] : 0.0f;
    }
}

// rows r0 .. r0 + N - 1 of this atom's column of a slice-blocked array into registers: the N loads are in flight together
template <int N>
__device__ __forceinline__ void load_rows(const float* __restrict__ p, int r0, int nrows, float* v)
{
#pragma unroll
    for (int j = 0; j < N; ++j) v[j] = (p != nullptr && r0 + j < nrows) ? __ldg(p + (size_t)(r0 + j) * WARP) : 0.0f;
}

// tanh x = sign(x) (1 - t) / (1 + t), t = exp(-2 |x|): ex2.approx and rcp.approx are good to 2^-22, so the absolute error is
// ~2e-7 everywhere (what Eq. 3 needs: E_i = sum_mu w1_mu tanh(.)), at 8 instructions instead of tanhf's ~35
__device__ __forceinline__ float tanh_fast(float x)
{
    float t, r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(t) : "f"(-2.8853900817779268f * fabsf(x)));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.0f + t));
    return copysignf((1.0f - t) * r, x);
}

// issue the K loop of one product: D (+)= A[tmem cols acol ..] B[smem, [K/4][rows][4]]
__device__ __forceinline__ void tc_gemm_ts(uint32_t d, uint32_t acol, const float* B, int rows, int K, uint32_t idesc, bool acc)
{
    // the descriptor of K step k0 + 8 is the previous one with the start-address field (16-byte units) advanced by two K chunks
    uint64_t bd = make_desc(smem_u32(B), rows * 16, 128);
    const uint64_t step = (uint64_t)(2 * rows);
#pragma unroll 1
    for (int k0 = 0; k0 < K; k0 += 8) {
        mma_ts(d, acol + k0, bd, idesc, acc);
        bd += step;
        acc = true;
    }
}

// ------------------------------------------------------------------------------------------------
// Thread layout of both kernels: NT threads per atom (NT = 2 or 4), block = 128 NT threads.  Warp w works on the TMEM lanes
// of quarter w & 3 (the hardware lets a warp touch only lanes 32 (w % 4) ..), i.e. on atom am = 32 (w & 3) + lane of the tile;
// the NT warps that share a quarter split every per-atom loop by CHUNKS of 8 columns (the unit of a TMEM load / store):
// thread part h = w >> 2 takes the chunks c with c % NT == h.
// ------------------------------------------------------------------------------------------------
struct TcThread {
    int tid, w, lane, q, h, am;
    uint32_t tb;         // TMEM address of this thread's lane, column 0 of the block's allocation
};
__device__ __forceinline__ TcThread tc_thread(uint32_t tcol0)
{
    TcThread t;
    t.tid = threadIdx.x; t.w = t.tid >> 5; t.lane = t.tid & 31; t.q = t.w & 3; t.h = t.w >> 2; t.am = 32 * t.q + t.lane;
    t.tb = tcol0 + ((uint32_t)(32 * t.q) << 16);
    return t;
}

// ------------------------------------------------------------------------------------------------
// S3
// ------------------------------------------------------------------------------------------------
template <int NT>
__global__ void __launch_bounds__(TC_TM * NT) k_ann_fwd_tc(StepArgs a, TcLay l)
{
    extern __shared__ __align__(128) float sm[];
    const ModelDev& m = a.m;
    uint64_t* mbar = reinterpret_cast<uint64_t*>(sm + l.oBar);
    uint32_t* tslot = reinterpret_cast<uint32_t*>(mbar + 1);
    if (threadIdx.x == 0) mbar_init(mbar, 1);
    if (threadIdx.x < 32) tmem_alloc(tslot, l.ncols);
    fence_before();
    __syncthreads();
    fence_after();
    const uint32_t tcol0 = *tslot;
    const TcThread T = tc_thread(tcol0);
    const int tid = T.tid, h = T.h;
    const uint32_t tb = T.tb;
    const uint32_t idesc1 = make_idesc_tf32(128, l.HP16), idesc2 = make_idesc_tf32(128, l.DP16);
    const int tbase = a.b.ntiles / (int)gridDim.x, trem = a.b.ntiles - tbase * (int)gridDim.x;
    const int tile0 = (int)blockIdx.x * tbase + min((int)blockIdx.x, trem), tile1 = tile0 + tbase + ((int)blockIdx.x < trem ? 1 : 0);
    uint32_t phase = 0;
    int cur_t = -1;
    const float b1 = a.theta[m.o_b1];
    float* eis = sm + l.oEi;                       // [NT][128] partial E_i of the thread parts
#pragma unroll 1
    for (int tile = tile0; tile < tile1; ++tile) {
        const int t = tile_type_of(a.b, tile, m.T);
        if (t != cur_t) {
            cur_t = t;
            __syncthreads();                       // every thread is done with the previous species' tables
            tc_load_weights<true>(a, l, sm, t);
#pragma unroll 4
            for (int i = tid; i < m.nR * l.TKRP; i += TC_TM * NT) {      // cRs[n][T' KRP + k]
                const int n = i / l.TKRP, o = i - n * l.TKRP, tj = o / m.KRP, k = o - tj * m.KRP;
                sm[l.ocR + i] = (k < m.KR) ? a.theta[m.o_cR + ((t * m.T + tj) * m.nR + n) * m.KR + k] : 0.0f;
            }
        }
        const int ib = a.b.alist[(size_t)tile * TC_TM + T.am];
        const float* qp = ib >= 0 ? sb_ptr(a.b.q, ib >> 5, m.D, ib & 31) : nullptr;
        // ---- A = q (hi | lo) -> TMEM columns [0, DP8) and [KMAX, KMAX + DP8): this thread's chunks, two at a time ----
#pragma unroll 1
        for (int c = h; 8 * c < l.DP8; c += 2 * NT) {
            float qa[8], qb[8];
            const int cb = c + NT;
            load_rows<8>(qp, 8 * c, m.D, qa);
            load_rows<8>(qp, 8 * cb, m.D, qb);      // rows beyond D: zeros
            float hi[8], lo[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) { hi[j] = tf32_rn(qa[j]); lo[j] = tf32_rn(qa[j] - hi[j]); }
            tmem_st8(tb + 8 * c, hi);
            tmem_st8(tb + l.KMAX + 8 * c, lo);
            if (8 * cb < l.DP8) {
#pragma unroll
                for (int j = 0; j < 8; ++j) { hi[j] = tf32_rn(qb[j]); lo[j] = tf32_rn(qb[j] - hi[j]); }
                tmem_st8(tb + 8 * cb, hi);
                tmem_st8(tb + l.KMAX + 8 * cb, lo);
            }
        }
        tmem_st_wait();
        fence_async_smem();                        // the weights written above (generic proxy) are read by the tensor core
        fence_before();
        __syncthreads();
        if (tid == 0) {
            fence_after();
            const uint32_t d = tcol0 + l.cR2;
            tc_gemm_ts(d, tcol0, sm + l.oW1H, l.HP16, l.DP8, idesc1, false);             // hi hi
            tc_gemm_ts(d, tcol0 + l.KMAX, sm + l.oW1H, l.HP16, l.DP8, idesc1, true);     // lo hi
            tc_gemm_ts(d, tcol0, sm + l.oW1L, l.HP16, l.DP8, idesc1, true);              // hi lo
            commit(mbar);
        }
        mbar_wait(mbar, phase); phase ^= 1;
        fence_after();
        // ---- h = tanh(x - b0), E_i, e -> A of the second product (hi | lo) ----
        float ei = 0.0f;
        float* hb = a.b.hbuf + (size_t)tile * l.HP8 * TC_TM + T.am;
#pragma unroll 1
        for (int c0 = 8 * h; c0 < l.HP8; c0 += 8 * NT) {
            float x[8], hi[8], lo[8];
            tmem_ld8(tb + l.cR2 + c0, x);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const float w1 = sm[l.ow1 + c0 + j];
                const float hh = tanh_fast(x[j] - sm[l.ob0 + c0 + j]);
                ei = fmaf(w1, hh, ei);
                const float e = w1 * fmaf(-hh, hh, 1.0f);
                hb[(size_t)(c0 + j) * TC_TM] = hh;
                hi[j] = tf32_rn(e); lo[j] = tf32_rn(e - hi[j]);
            }
            tmem_st8(tb + c0, hi);
            tmem_st8(tb + l.KMAX + c0, lo);
        }
        eis[h * TC_TM + T.am] = ei;
        tmem_st_wait();
        fence_before();
        __syncthreads();
        if (tid == 0) {
            fence_after();
            const uint32_t d = tcol0 + l.cR2;
            tc_gemm_ts(d, tcol0, sm + l.oW2H, l.DP16, l.HP8, idesc2, false);
            tc_gemm_ts(d, tcol0 + l.KMAX, sm + l.oW2H, l.DP16, l.HP8, idesc2, true);
            tc_gemm_ts(d, tcol0, sm + l.oW2L, l.DP16, l.HP8, idesc2, true);
            commit(mbar);
        }
        if (h == 0 && ib >= 0) {                   // E_i of Eq. 3 (the parts' sums were exchanged before the barrier above)
            float e = -b1;
#pragma unroll
            for (int p = 0; p < NT; ++p) e += eis[p * TC_TM + T.am];
            a.b.Ei[ib] = e;
        }
        mbar_wait(mbar, phase); phase ^= 1;
        fence_after();
        // ---- Fp = dE_i/dq -> global (this thread's chunks); a_k[T'] from its radial rows (every part reads them) ----
        float* fpp = ib >= 0 ? sb_ptr(a.b.Fp, ib >> 5, m.D, ib & 31) : nullptr;
#pragma unroll 1
        for (int c0 = 8 * h; c0 < l.DP8; c0 += 8 * NT) {
            float f[8];
            tmem_ld8(tb + l.cR2 + c0, f);
            tmem_ld_wait();
            if (fpp != nullptr)
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (c0 + j < m.D) fpp[(size_t)(c0 + j) * WARP] = f[j];
        }
        float fpr[24];
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) {
            if (8 * cc < m.nR) tmem_ld8(tb + l.cR2 + 8 * cc, fpr + 8 * cc);
            else {
#pragma unroll
                for (int j = 0; j < 8; ++j) fpr[8 * cc + j] = 0.0f;
            }
        }
        tmem_ld_wait();
        if (ib >= 0) {
            float* ar = a.b.arow + (size_t)ib * l.TKRP;
#pragma unroll 1
            for (int o0 = 4 * h; o0 < l.TKRP; o0 += 4 * NT) {
                float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int n = 0; n < 24; ++n)
                    if (n < m.nR) {
                        const float4 c4 = *reinterpret_cast<const float4*>(sm + l.ocR + n * l.TKRP + o0);
                        acc.x = fmaf(fpr[n], c4.x, acc.x); acc.y = fmaf(fpr[n], c4.y, acc.y);
                        acc.z = fmaf(fpr[n], c4.z, acc.z); acc.w = fmaf(fpr[n], c4.w, acc.w);
                    }
                *reinterpret_cast<float4*>(ar + o0) = acc;
            }
        }
        fence_before();                            // this tile's TMEM reads are ordered before the next tile's writes
    }
    __syncthreads();
    if (threadIdx.x < 32) tmem_dealloc(tcol0, l.ncols);
}

// sum over the 32 lanes of 8 values per lane; lane l returns the total of element 4 b4 + 2 b3 + b2 (bits of l)
__device__ __forceinline__ float warp_reduce_scatter8(const float* v, int lane)
{
    const bool u4 = lane & 16, u3 = lane & 8, u2 = lane & 4;
    float r[4], s[2];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float keep = u4 ? v[4 + i] : v[i], send = u4 ? v[i] : v[4 + i];
        r[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const float keep = u3 ? r[2 + i] : r[i], send = u3 ? r[i] : r[2 + i];
        s[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
    float u = (u2 ? s[1] : s[0]) + __shfl_xor_sync(0xffffffffu, u2 ? s[0] : s[1], 4);
    u += __shfl_xor_sync(0xffffffffu, u, 2);
    u += __shfl_xor_sync(0xffffffffu, u, 1);
    return u;
}

// ------------------------------------------------------------------------------------------------
// S8
// ------------------------------------------------------------------------------------------------
template <int NT>
__global__ void __launch_bounds__(TC_TM * NT) k_ann_bwd_tc(StepArgs a, TcLay l)
{
    extern __shared__ __align__(128) float sm[];
    const ModelDev& m = a.m;
    uint64_t* mbar = reinterpret_cast<uint64_t*>(sm + l.oBar);
    uint32_t* tslot = reinterpret_cast<uint32_t*>(mbar + 1);
    if (threadIdx.x == 0) mbar_init(mbar, 1);
    if (threadIdx.x < 32) tmem_alloc(tslot, l.ncols);
    fence_before();
    __syncthreads();
    fence_after();
    const uint32_t tcol0 = *tslot;
    const TcThread T = tc_thread(tcol0);
    const int tid = T.tid, h = T.h, lane = T.lane, am = T.am;
    const uint32_t tb = T.tb;
    constexpr int NTH = TC_TM * NT;
    const uint32_t idesc1 = make_idesc_tf32(128, l.HP16), idesc2 = make_idesc_tf32(128, l.DP16), idesc3 = make_idesc_tf32(l.MA, l.NC16);
    const int tbase = a.b.ntiles / (int)gridDim.x, trem = a.b.ntiles - tbase * (int)gridDim.x;
    const int tile0 = (int)blockIdx.x * tbase + min((int)blockIdx.x, trem), tile1 = tile0 + tbase + ((int)blockIdx.x < trem ? 1 : 0);
    uint32_t phase = 0;
    int cur_t = -1;
    bool acc_live = false;                        // ACC holds sums of the current species
    float* gw1s = sm + l.ogw1;                    // [HP8] g_w1 of the current species, summed over this block's atoms
    int ib_next = tile0 < tile1 ? a.b.alist[(size_t)tile0 * TC_TM + am] : -1;   // atom of the tile to come (loaded one tile ahead)
    float* QBT = sm + l.oQBT; float* QDT = sm + l.oQDT; float* GT = sm + l.oGT; float* ET = sm + l.oET;
    const int tq = ((am >> 2) * l.ldQ) * 4 + (am & 3), tg = ((am >> 2) * l.ldG) * 4 + (am & 3);   // this atom's cell of row 0
    const int nrc = (m.nR + 7) >> 3;              // chunks of qd that hold radial rows

    // ACC -> g (species t): called by all threads; ends with the tables free for the next species
    auto flush = [&](int t) {
        // rows of ACC: M = 64: lane < 16 of quarter q holds row 16 q + lane; M = 128: row 32 q + lane
        const int mu = l.MA == 64 ? 16 * T.q + lane : 32 * T.q + lane;
        const bool own = (l.MA == 64 ? lane < 16 : true) && mu < m.H;
        float* gt = a.g + (size_t)t * m.per_type;
        float* stage = QBT;                         // [mu][TK] columns D .. D + TK - 1 of ACC, for the g_cR product below
#pragma unroll 1
        for (int c0 = 8 * h; c0 < l.NC16; c0 += 8 * NT) {
            float v[8];
            tmem_ld8(tb + l.cACC + c0, v);
            tmem_ld_wait();
            if (own)
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int col = c0 + j;
                    if (col < m.D) atomicAdd(gt + mu * m.D + col, sm[l.osc + col] * v[j]);
                    else if (col < m.D + l.TK) stage[mu * l.TK + (col - m.D)] = v[j];
                    else if (col == m.D + l.TK) atomicAdd(gt + m.H * m.D + mu, -v[j]);             // g_b0 = -sum gamma
                }
        }
        fence_before();
        __syncthreads();
#pragma unroll 1
        for (int i = tid; i < m.H; i += NTH) atomicAdd(gt + m.H * m.D + m.H + i, gw1s[i]);
        // g_cR[t][T'][n][k] += sum_mu w0s[mu][n] ACC[mu][D + T' KR + k]
#pragma unroll 1
        for (int o = tid; o < m.nR * l.TK; o += NTH) {
            const int n = o / l.TK, r = o - n * l.TK, tj = r / m.KR, k = r - tj * m.KR;
            const float sn = sm[l.osc + n];
            float s = 0.0f;
#pragma unroll 4
            for (int mu2 = 0; mu2 < m.H; ++mu2) s = fmaf(sm[l.oStg + mu2 * m.D + n] * sn, stage[mu2 * l.TK + r], s);
            atomicAdd(a.g + m.o_cR + ((t * m.T + tj) * m.nR + n) * m.KR + k, s);
        }
        __syncthreads();
    };

#pragma unroll 1
    for (int tile = tile0; tile < tile1; ++tile) {
        const int t = tile_type_of(a.b, tile, m.T);
        if (t != cur_t) {
            if (acc_live) flush(cur_t);
            acc_live = false;
            cur_t = t;
            __syncthreads();
            tc_load_weights<false>(a, l, sm, t);
            for (int i = tid; i < l.HP8; i += NTH) gw1s[i] = 0.0f;
#pragma unroll 4
            for (int i = tid; i < l.TK * l.nR4; i += NTH) {   // cRt[(T', k)][n]
                const int r = i / l.nR4, n = i - r * l.nR4, tj = r / m.KR, k = r - tj * m.KR;
                sm[l.ocR + i] = (n < m.nR) ? a.theta[m.o_cR + ((t * m.T + tj) * m.nR + n) * m.KR + k] : 0.0f;
            }
            __syncthreads();                       // cRt is read below before the next barrier
        }
        const int ib = ib_next;
        const bool valid = ib >= 0;
        ib_next = tile + 1 < tile1 ? a.b.alist[(size_t)(tile + 1) * TC_TM + am] : -1;
        if (tile + 1 < tile1 && h == 0) {
            // the rows of the next tile -> L2 while this one is worked on: per 32-atom slice they are contiguous blocks
            const int ib2 = ib_next;
            if (ib2 >= 0 && ((ib2 & 31) == 0 || lane == 0)) {
                const size_t ws2 = (size_t)(ib2 >> 5);
                prefetch_l2(a.b.q + ws2 * m.D * WARP, 4u * m.D * WARP);
                prefetch_l2(a.b.qd + ws2 * m.D * WARP, 4u * m.D * WARP);
                prefetch_l2(a.b.Bd + ws2 * l.TK * WARP, 4u * l.TK * WARP);
            }
            if (tid == 0) prefetch_l2(a.b.hbuf + (size_t)(tile + 1) * l.HP8 * TC_TM, 4u * l.HP8 * TC_TM);
        }
        const float *qp = nullptr, *qdp = nullptr, *Bp = nullptr, *Bdp = nullptr;
        float epsi = 0.0f;
        if (valid) {
            const int ws = ib >> 5, ln = ib & 31;
            const int4 bi = __ldg(a.b.binfo + ws);
            qp = sb_ptr(a.b.q, ws, m.D, ln); qdp = sb_ptr(a.b.qd, ws, m.D, ln);
            Bp = sb_ptr(a.d.B, bi.x, l.TK, ln); Bdp = sb_ptr(a.b.Bd, ws, l.TK, ln);
            epsi = a.b.eps[bi.y];
        }
        // ---- B, Bd -> transposed operand columns D .. D + TK - 1: chunks of 8 rows, parts offset by one against the qd chunks ----
#pragma unroll 1
        for (int r0 = 8 * ((h + NT - 1) % NT); r0 < l.TK; r0 += 8 * NT) {
            float bd[8], bv[8];
            load_rows<8>(Bdp, r0, l.TK, bd);
            load_rows<8>(Bp, r0, l.TK, bv);
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (r0 + j < l.TK) {
                    QDT[tq + (m.D + r0 + j) * 4] = tf32_rn(bd[j]);
                    QBT[tq + (m.D + r0 + j) * 4] = tf32_rn(bv[j]);
                }
        }
        if (h == NT - 1) {   // ones column (pairs with gamma: g_b0) and padding columns
            QBT[tq + (m.D + l.TK) * 4] = valid ? 1.0f : 0.0f;
            QDT[tq + (m.D + l.TK) * 4] = 0.0f;
#pragma unroll 1
            for (int col = m.D + l.TK + 1; col < l.NC16; ++col) { QBT[tq + col * 4] = 0.0f; QDT[tq + col * 4] = 0.0f; }
        }
        // ---- q, qd: transposed operands; qd also as A of the first product (TMEM columns [0, DP8)).  The radial rows of qd
        //      (the first n_R) are not stored anywhere: qd_n = sum_{T', k} cR[t][T'][n][k] Bd_k[T'], formed by the chunk's owner ----
#pragma unroll 1
        for (int c = h; 8 * c < l.DP8; c += NT) {
            float qv[8], qd[8];
            load_rows<8>(qp, 8 * c, m.D, qv);
            load_rows<8>(qdp, 8 * c, m.D, qd);
            if (c < nrc) {
                float s[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) s[j] = 0.0f;
#pragma unroll 8
                for (int r = 0; r < l.TK; ++r) {
                    const float bdr = Bdp != nullptr ? __ldg(Bdp + (size_t)r * WARP) : 0.0f;
                    const float* cr = sm + l.ocR + r * l.nR4 + 8 * c;          // nR4 >= 8 c + 4: the second quad only if it exists
                    const float4 c0 = *reinterpret_cast<const float4*>(cr);
                    s[0] = fmaf(c0.x, bdr, s[0]); s[1] = fmaf(c0.y, bdr, s[1]); s[2] = fmaf(c0.z, bdr, s[2]); s[3] = fmaf(c0.w, bdr, s[3]);
                    if (8 * c + 4 < l.nR4) {
                        const float4 c1 = *reinterpret_cast<const float4*>(cr + 4);
                        s[4] = fmaf(c1.x, bdr, s[4]); s[5] = fmaf(c1.y, bdr, s[5]); s[6] = fmaf(c1.z, bdr, s[6]); s[7] = fmaf(c1.w, bdr, s[7]);
                    }
                }
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (8 * c + j < m.nR) qd[j] = s[j];
            }
            float hi[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                hi[j] = tf32_rn(qd[j]);
                if (8 * c + j < m.D) {
                    QDT[tq + (8 * c + j) * 4] = hi[j];
                    QBT[tq + (8 * c + j) * 4] = tf32_rn(qv[j]);
                }
            }
            tmem_st8(tb + 8 * c, hi);
        }
        tmem_st_wait();
        fence_async_smem();
        fence_before();
        __syncthreads();
        if (tid == 0) {
            fence_after();
            tc_gemm_ts(tcol0 + l.cR2, tcol0, sm + l.oW1H, l.HP16, l.DP8, idesc1, false);     // Xd = Qd W0s^T
            commit(mbar);
        }
        mbar_wait(mbar, phase); phase ^= 1;
        fence_after();
        // ---- gamma, e: A of the second product (TMEM [0, HP8)) and transposed operands; g_w1 ----
        const float* hb = a.b.hbuf + (size_t)tile * l.HP8 * TC_TM + am;
#pragma unroll 1
        for (int c0 = 8 * h; c0 < l.HP8; c0 += 8 * NT) {
            float hh[8], xd[8], gam[8], om[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) hh[j] = hb[(size_t)(c0 + j) * TC_TM];
            tmem_ld8(tb + l.cR2 + c0, xd);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const float hv = hh[j], w1 = sm[l.ow1 + c0 + j];
                const float omh2 = fmaf(-hv, hv, 1.0f);
                const float e = valid ? w1 * omh2 : 0.0f;
                const float g = fmaf(epsi, e, -2.0f * hv * e * xd[j]);
                om[j] = valid ? fmaf(epsi, hv, omh2 * xd[j]) : 0.0f;
                gam[j] = tf32_rn(g);
                GT[tg + (c0 + j) * 4] = gam[j];
                ET[tg + (c0 + j) * 4] = tf32_rn(e);
            }
            tmem_st8(tb + c0, gam);
            // g_w1: sum over the warp's atoms; the lanes with (lane & 3) == 0 hold one of the 8 totals each
            const float u = warp_reduce_scatter8(om, lane);
            if ((lane & 3) == 0) atomicAdd(gw1s + c0 + ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1), u);
        }
        tmem_st_wait();
        fence_async_smem();
        fence_before();
        __syncthreads();
        if (tid == 0) {
            fence_after();
            tc_gemm_ts(tcol0 + l.cR2, tcol0, sm + l.oW2H, l.DP16, l.HP8, idesc2, false);     // Qb = Gamma W0s
            // ACC (+)= products over the 128 atoms of the tile (K-major over atoms)
            const uint32_t d = tcol0 + l.cACC;
            const uint32_t gA = smem_u32(GT), eA = smem_u32(ET), qB = smem_u32(QBT), dB = smem_u32(QDT);
            bool acc = acc_live;
            const uint64_t sA = (uint64_t)(2 * l.ldG), sB = (uint64_t)(2 * l.ldQ);     // two K chunks, in 16-byte units of the address field
            uint64_t ad = make_desc(gA, l.ldG * 16, 128), bd = make_desc(qB, l.ldQ * 16, 128);
#pragma unroll 4
            for (int k0 = 0; k0 < TC_TM; k0 += 8) {
                mma_ss(d, ad, bd, idesc3, acc);
                ad += sA; bd += sB;
                acc = true;
            }
            ad = make_desc(eA, l.ldG * 16, 128); bd = make_desc(dB, l.ldQ * 16, 128);
#pragma unroll 4
            for (int k0 = 0; k0 < TC_TM; k0 += 8) {
                mma_ss(d, ad, bd, idesc3, true);
                ad += sA; bd += sB;
            }
            commit(mbar);
        }
        acc_live = true;
        mbar_wait(mbar, phase); phase ^= 1;
        fence_after();
        // ---- Qb: only the angular rows are read later (the radial ones enter g_cR through ACC) ----
        float* qbp = valid ? sb_ptr(a.b.Qb, ib >> 5, m.D, ib & 31) : nullptr;
#pragma unroll 1
        for (int c0 = 8 * ((m.nR >> 3) + h); c0 < l.DP8; c0 += 8 * NT) {
            float f[8];
            tmem_ld8(tb + l.cR2 + c0, f);
            tmem_ld_wait();
            if (qbp != nullptr)
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (c0 + j >= m.nR && c0 + j < m.D) qbp[(size_t)(c0 + j) * WARP] = f[j];
        }
        fence_before();
    }
    if (acc_live) flush(cur_t);
    __syncthreads();
    if (threadIdx.x < 32) tmem_dealloc(tcol0, l.ncols);
}

// ------------------------------------------------------------------------------------------------
// plan and launchers
// ------------------------------------------------------------------------------------------------
bool ann_tc_fits(const nep_ctx* c, bool bwd)
{
    const ModelDev& m = c->m;
    if (m.H > 128 || m.D > 128 || m.nR > 24 || m.D + m.T * m.KR + 1 > 256) return false;
    const TcLay l = tc_layout(m, bwd);
    return l.ncols <= 512 && 4 * (size_t)l.total <= (size_t)c->max_smem_optin;
}

// Persistent grid: blocks resident per SM by registers, shared memory and the 512 TMEM columns they share.  (The runtime's
// occupancy calculator answers 1 for a kernel that allocates tensor memory, so the limits are worked out here.)
static int tc_occupancy(nep_ctx* c, const void* kern, const TcLay& l, size_t smem, int threads, int* occ)
{
    NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaFuncAttributes fa;
    NEP_CUDA(c, cudaFuncGetAttributes(&fa, kern));
    int dev = 0, smem_sm = 0, regs_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
    cudaDeviceGetAttribute(&regs_sm, cudaDevAttrMaxRegistersPerMultiprocessor, dev);
    const int by_regs = regs_sm / (rup(std::max(fa.numRegs, 1), 8) * threads);
    const int by_smem = (int)((size_t)smem_sm / (smem + fa.sharedSizeBytes + 1024));
    const int by_thr = 2048 / threads;
    *occ = std::max(1, std::min(std::min(std::min(by_regs, by_smem), by_thr), 512 / l.ncols));
    return NEP_OK;
}

// two threads per atom when two blocks fit on an SM, four when only one does: sixteen warps per SM either way
template <class K2, class K4>
static int tc_launch(nep_ctx* c, const StepArgs& a, const TcLay& l, const char* name, K2 k2, K4 k4, bool prefer4)
{
    const size_t smem = 4 * (size_t)l.total;
    int occ2 = 1, occ4 = 1, rc;
    if ((rc = tc_occupancy(c, (const void*)k2, l, smem, 2 * TC_TM, &occ2))) return rc;
    if (occ2 >= 2 && !prefer4) {
        const int grid = std::min(c->b.ntiles, occ2 * c->sm_count);
        NEP_LAUNCH(c, name, k2, grid, 2 * TC_TM, smem, a, l);
    } else {
        if ((rc = tc_occupancy(c, (const void*)k4, l, smem, 4 * TC_TM, &occ4))) return rc;
        const int grid = std::min(c->b.ntiles, occ4 * c->sm_count);
        NEP_LAUNCH(c, name, k4, grid, 4 * TC_TM, smem, a, l);
    }
    return NEP_OK;
}

int launch_ann_fwd_tc(nep_ctx* c, const StepArgs& a)
{
    if (c->b.ntiles == 0) return NEP_OK;
    // larger networks: four threads per atom also in the forward kernel (config 3, 50 x 37: 39 -> 34 us; config 2, 30 x 35: 28 -> 30)
    return tc_launch(c, a, tc_layout(c->m, false), "k_ann_fwd", k_ann_fwd_tc<2>, k_ann_fwd_tc<4>, c->m.H * c->m.D > 1500);
}
int launch_ann_bwd_tc(nep_ctx* c, const StepArgs& a)
{
    if (c->b.ntiles == 0) return NEP_OK;
    return tc_launch(c, a, tc_layout(c->m, true), "k_ann_bwd", k_ann_bwd_tc<2>, k_ann_bwd_tc<4>, false);
}

}  // namespace nep
