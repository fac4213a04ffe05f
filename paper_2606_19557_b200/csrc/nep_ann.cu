// nep_ann.cu -- the per-species tanh network of Eq. 3 on TILES of same-species atoms.
//
// S3 (k_ann_fwd):  x = w0[t] (s o q) - b0[t];  h = tanh x;  E_i = w1[t] . h - b1;  e = w1 o (1 - h^2);
//                  Fp = dE_i/dq = s o (w0^T e);  a_k[T'] = sum_n Fp_n cR[t][T'][n][k] (coefficient rows of the radial force sweep).
// S8 (k_ann_bwd):  the network tangent / adjoint and every gradient that is a sum over atoms of one species (DESIGN C11-C12):
//                  qd_rad = cR Bd;  xd = w0 (s o qd);  gamma = eps e - 2 h e xd;
//                  g_w1 += eps h + (1-h^2) xd;  g_b0 -= gamma;  g_w0 += gamma (x) q~ + e (x) (s o qd);  Qb = s o (w0^T gamma);
//                  g_cR[t][T'][n][k] += sum_atoms Qb_n B_k[T'] + Fp_n Bd_k[T'].
//
// The atoms of the batch are listed sorted by species (b.alist), every species padded to whole tiles of TM atoms, so
// one tile sees ONE weight matrix and each contraction is a small dense fp32 GEMM out of shared memory:
//   tile_gemm : [TM atoms] x [K] x [N outputs]; thread = AT atoms x 4 outputs, both operands fetched with one LDS.128
//               per k (16 FFMA per 2 LDS); outputs beyond a multiple of 32 use a strided scalar tail;
//   outer_gemm: sum over the TM atoms of outer products (the weight gradients).
// The descriptor scaler (Eq. 2) is folded into the weights held in shared memory, W0s[mu][v] = w0[mu][v] s_v, so the
// per-atom inputs are copied global -> shared unchanged with cp.async (all rows of a tile in flight at once).
// fp32 FFMA on purpose: TF32/BF16 tensor-core inputs (10/7 mantissa bits) break the 1e-5 eV/atom energy tolerance and
// the network is a small part of the step's arithmetic.
#include <algorithm>
#include <type_traits>

#include "nep_kernels.cuh"

namespace nep {

struct AnnLay {
    int TM, LD, DP8, HP8, HP32, TK, TKP, nR8;
    int W0m, W0t, b0, w1, sc, cRs, cRt, Qs, QDs, Gs, Es, Bs, BDs, FPs, ibs, aux, red, total;   // float offsets
};
__host__ __device__ inline AnnLay ann_layout(const ModelDev& m, int TM, bool bwd)
{
    AnnLay l;
    l.TM = TM; l.LD = TM + 4;
    l.DP8 = rup(m.D, 8); l.HP8 = rup(m.H, 8); l.HP32 = rup(m.H, 32);   // HP32: rows of the outer-product GEMM (zero padded)
    l.TK = m.T * m.KR; l.TKP = rup(m.T * m.KRP, 8); l.nR8 = rup(m.nR, 8);
    int o = 0;
    auto take = [&](int n) { int r = o; o += rup(n, 4); return r; };
    l.W0m = take(l.HP8 * l.DP8); l.W0t = take(l.DP8 * l.HP8);
    l.b0 = take(l.HP8); l.w1 = take(l.HP8); l.sc = take(l.DP8);
    l.cRs = l.cRt = l.QDs = l.Gs = l.Bs = l.BDs = l.FPs = l.red = 0;
    l.Qs = take(l.DP8 * l.LD);
    l.Es = take(l.HP32 * l.LD);
    l.ibs = take(TM); l.aux = take(TM);
    if (!bwd) {
        l.cRs = take(m.nR * l.TKP);
    } else {
        l.cRt = take(l.TK * l.nR8);
        l.QDs = take(l.DP8 * l.LD);
        l.Gs = take(l.HP32 * l.LD);
        l.Bs = take(l.TK * l.LD); l.BDs = take(l.TK * l.LD); l.FPs = take(m.nR * l.LD);
        l.red = take(2 * l.HP8 * 8);
    }
    l.total = o;
    return l;
}

// Outputs of one thread (lane tx of 8) among n_out (a multiple of 8): rounds of 32 as quads {32c + 4tx + j}, then a
// strided tail {32C + tx + 8j}.  f(o0, ostep, integral_constant<CW>, integral_constant<QUAD>)
template <class F>
__device__ __forceinline__ void for_outputs(int n_out, int tx, F&& f)
{
    const int C = n_out >> 5, rem = (n_out & 31) >> 3;
    for (int c = 0; c < C; ++c) f(32 * c + 4 * tx, 1, std::integral_constant<int, 4>{}, std::true_type{});
    const int o0 = 32 * C + tx;
    switch (rem) {
    case 1: f(o0, 8, std::integral_constant<int, 1>{}, std::false_type{}); break;
    case 2: f(o0, 8, std::integral_constant<int, 2>{}, std::false_type{}); break;
    case 3: f(o0, 8, std::integral_constant<int, 3>{}, std::false_type{}); break;
    default: break;
    }
}

// acc[i][j] = sum_k A[k * lda + i] * W[k * ldw + j * ostep],  i < AT consecutive atoms, j < CW outputs
// (QUAD: ostep == 1 and the four weights are one 128-bit load)
template <int AT, int CW, bool QUAD>
__device__ __forceinline__ void tile_gemm(const float* __restrict__ A, int lda, const float* __restrict__ W, int ldw, int ostep, int K,
                                          float (&acc)[AT][CW])
{
#pragma unroll
    for (int i = 0; i < AT; ++i)
#pragma unroll
        for (int j = 0; j < CW; ++j) acc[i][j] = 0.0f;
#pragma unroll 4
    for (int k = 0; k < K; ++k) {
        float av[AT];
#pragma unroll
        for (int i4 = 0; i4 < AT / 4; ++i4) {
            const float4 a4 = *reinterpret_cast<const float4*>(A + k * lda + 4 * i4);
            av[4 * i4] = a4.x; av[4 * i4 + 1] = a4.y; av[4 * i4 + 2] = a4.z; av[4 * i4 + 3] = a4.w;
        }
        float w[CW];
        if (QUAD) {
            const float4 w4 = *reinterpret_cast<const float4*>(W + k * ldw);
            w[0] = w4.x; if (CW > 1) w[1] = w4.y; if (CW > 2) w[2] = w4.z; if (CW > 3) w[3] = w4.w;
        } else {
#pragma unroll
            for (int j = 0; j < CW; ++j) w[j] = W[k * ldw + j * ostep];
        }
#pragma unroll
        for (int i = 0; i < AT; ++i)
#pragma unroll
            for (int j = 0; j < CW; ++j) acc[i][j] = fmaf(av[i], w[j], acc[i][j]);
    }
}
template <int AT>
__device__ __forceinline__ void store_atoms(float* dst, const float* v)
{
#pragma unroll
    for (int i4 = 0; i4 < AT / 4; ++i4) reinterpret_cast<float4*>(dst)[i4] = make_float4(v[4 * i4], v[4 * i4 + 1], v[4 * i4 + 2], v[4 * i4 + 3]);
}
template <int AT>
__device__ __forceinline__ void load_atoms(const float* src, float* v)
{
#pragma unroll
    for (int i4 = 0; i4 < AT / 4; ++i4) {
        const float4 a4 = reinterpret_cast<const float4*>(src)[i4];
        v[4 * i4] = a4.x; v[4 * i4 + 1] = a4.y; v[4 * i4 + 2] = a4.z; v[4 * i4 + 3] = a4.w;
    }
}

// acc[r][c] = sum_m A1[r-th row][m] B1[c-th row][m] + A2[..][m] B2[..][m]  over the TM atoms of the tile (rows LD apart)
template <int RW, int CW>
__device__ __forceinline__ void outer_gemm(const float* __restrict__ A1, const float* __restrict__ A2, int rstep,
                                           const float* __restrict__ B1, const float* __restrict__ B2, int cstep, int TM,
                                           float (&acc)[RW][CW])
{
#pragma unroll
    for (int r = 0; r < RW; ++r)
#pragma unroll
        for (int c = 0; c < CW; ++c) acc[r][c] = 0.0f;
#pragma unroll 2
    for (int mm = 0; mm < TM; mm += 4) {
        float4 a1[RW], a2[RW], b1[CW], b2[CW];
#pragma unroll
        for (int r = 0; r < RW; ++r) {
            a1[r] = *reinterpret_cast<const float4*>(A1 + r * rstep + mm);
            a2[r] = *reinterpret_cast<const float4*>(A2 + r * rstep + mm);
        }
#pragma unroll
        for (int c = 0; c < CW; ++c) {
            b1[c] = *reinterpret_cast<const float4*>(B1 + c * cstep + mm);
            b2[c] = *reinterpret_cast<const float4*>(B2 + c * cstep + mm);
        }
#pragma unroll
        for (int r = 0; r < RW; ++r)
#pragma unroll
            for (int c = 0; c < CW; ++c) {
                float s = acc[r][c];
                s = fmaf(a1[r].x, b1[c].x, s); s = fmaf(a1[r].y, b1[c].y, s); s = fmaf(a1[r].z, b1[c].z, s); s = fmaf(a1[r].w, b1[c].w, s);
                s = fmaf(a2[r].x, b2[c].x, s); s = fmaf(a2[r].y, b2[c].y, s); s = fmaf(a2[r].z, b2[c].z, s); s = fmaf(a2[r].w, b2[c].w, s);
                acc[r][c] = s;
            }
    }
}
// splits N column groups into ceil(N/5) nearly equal chunks: f(first, integral_constant<width>)
template <class F>
__device__ __forceinline__ void for_chunks(int N, F&& f)
{
    const int chunks = (N + 4) / 5;
    if (chunks == 0) return;
    const int base = N / chunks, rem = N - base * chunks;
    int j0 = 0;
    for (int c = 0; c < chunks; ++c) {
        const int cw = base + (c < rem ? 1 : 0);
        switch (cw) {
        case 1: f(j0, std::integral_constant<int, 1>{}); break;
        case 2: f(j0, std::integral_constant<int, 2>{}); break;
        case 3: f(j0, std::integral_constant<int, 3>{}); break;
        case 4: f(j0, std::integral_constant<int, 4>{}); break;
        default: f(j0, std::integral_constant<int, 5>{}); break;
        }
        j0 += cw;
    }
}


// weights of species t into shared memory, zero padded and with the scaler folded in:
// W0m[mu][v] = W0t[v][mu] = w0[mu][v] s_v;  b0, w1, scaler
__device__ __forceinline__ void ann_load_weights(const StepArgs& a, const AnnLay& l, float* sm, int t, bool want_b0)
{
    const ModelDev& m = a.m;
    const float* th = a.theta + (size_t)t * m.per_type;
    for (int mu = threadIdx.x / 32; mu < l.HP8; mu += blockDim.x / 32)
        for (int v = threadIdx.x & 31; v < l.DP8; v += 32) {
            const float w = (v < m.D && mu < m.H) ? th[mu * m.D + v] * a.scaler[v] : 0.0f;
            sm[l.W0m + mu * l.DP8 + v] = w;
            sm[l.W0t + v * l.HP8 + mu] = w;
        }
    for (int i = threadIdx.x; i < l.HP8; i += blockDim.x) {
        if (want_b0) sm[l.b0 + i] = (i < m.H) ? th[m.H * m.D + i] : 0.0f;
        sm[l.w1 + i] = (i < m.H) ? th[m.H * m.D + m.H + i] : 0.0f;
    }
    for (int i = threadIdx.x; i < l.DP8; i += blockDim.x) sm[l.sc + i] = (i < m.D) ? a.scaler[i] : 0.0f;
}

__device__ __forceinline__ void cp_async4(float* smem_dst, const float* gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"(s), "l"(gsrc) : "memory");
}
// Column gather: rows r = r0 + rg, + RG, ... < nrows of a slice-blocked array (src at row 0 of this atom; nullptr for
// a padding atom: zeros) into dst[r * LD], asynchronously (cp.async; the caller commits and waits).
__device__ __forceinline__ void gather_rows(float* __restrict__ dst, int LD, const float* __restrict__ src, int r0, int nrows, int rg, int RG)
{
    if (src != nullptr) {
        for (int r = r0 + rg; r < nrows; r += RG) cp_async4(dst + r * LD, src + (size_t)r * WARP);
    } else {
        for (int r = r0 + rg; r < nrows; r += RG) dst[r * LD] = 0.0f;
    }
}
__device__ __forceinline__ void scatter_rows(float* __restrict__ dst, const float* __restrict__ srcs, int LD, int r0, int nrows, int rg, int RG)
{
    for (int rb = r0 + rg; rb < nrows; rb += 8 * RG) {
        float t[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int r = rb + j * RG;
            t[j] = (r < nrows) ? srcs[r * LD] : 0.0f;
        }
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int r = rb + j * RG;
            if (r < nrows) dst[(size_t)r * WARP] = t[j];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S3.  TM atoms per tile, AT atoms per thread: NT = 8 TM / AT threads; thread (ty, tx) = (atom group, output lane)
// ------------------------------------------------------------------------------------------------
template <int TM, int AT>
__global__ void __launch_bounds__(8 * TM / AT) k_ann_fwd(StepArgs a)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int NT = 8 * TM / AT, RG = NT / TM;
    const ModelDev& m = a.m;
    const AnnLay l = ann_layout(m, TM, false);
    const int tid = threadIdx.x;
    // persistent block: a contiguous range of tiles (tiles are sorted by species, so the weights are reloaded rarely)
    const int tbase = a.b.ntiles / (int)gridDim.x, trem = a.b.ntiles - tbase * (int)gridDim.x;
    const int tile0 = (int)blockIdx.x * tbase + min((int)blockIdx.x, trem), tile1 = tile0 + tbase + ((int)blockIdx.x < trem ? 1 : 0);
    int cur_t = -1;
    for (int tile = tile0; tile < tile1; ++tile) {
    const int LD = l.LD;
    int* ibs = reinterpret_cast<int*>(sm + l.ibs);
    const int am = tid % TM, rg = tid / TM;          // gather role: atom am, row group rg
    const int ib = a.b.alist[(size_t)tile * TM + am];
    {   // q of the tile, unscaled, straight into shared memory
        const float* qp = ib >= 0 ? sb_ptr(a.b.q, ib >> 5, m.D, ib & 31) : nullptr;
        gather_rows(sm + l.Qs + am, LD, qp, 0, m.D, rg, RG);
        cp_async_commit();
        for (int v = m.D + rg; v < l.DP8; v += RG) sm[l.Qs + v * LD + am] = 0.0f;
        if (rg == 0) ibs[am] = ib;
    }
    const int t = tile_type_of(a.b, tile, m.T);
    if (t != cur_t) {
        cur_t = t;
        ann_load_weights(a, l, sm, t, true);
        for (int i = tid; i < m.nR * l.TKP; i += NT) {
            const int n = i / l.TKP, o = i - n * l.TKP, tj = o / m.KRP, k = o - tj * m.KRP;
            sm[l.cRs + i] = (tj < m.T && k < m.KR) ? a.theta[m.o_cR + ((t * m.T + tj) * m.nR + n) * m.KR + k] : 0.0f;
        }
    }
    cp_async_wait<0>();
    __syncthreads();
    const int ty = tid >> 3, tx = tid & 7, m0 = ty * AT;
    float ei[AT];
#pragma unroll
    for (int i = 0; i < AT; ++i) ei[i] = 0.0f;
    float* hb = a.b.hbuf + (size_t)tile * l.HP8 * TM;
    for_outputs(l.HP8, tx, [&](int o0, int ostep, auto cwc, auto quadc) {
        constexpr int CW = decltype(cwc)::value;
        constexpr bool QUAD = decltype(quadc)::value;
        float acc[AT][CW];
        tile_gemm<AT, CW, QUAD>(sm + l.Qs + m0, LD, sm + l.W0t + o0, l.HP8, ostep, m.D, acc);
#pragma unroll
        for (int j = 0; j < CW; ++j) {
            const int mu = o0 + j * ostep;
            const float b0 = sm[l.b0 + mu], w1 = sm[l.w1 + mu];
            float h[AT], e[AT];
#pragma unroll
            for (int i = 0; i < AT; ++i) {
                h[i] = tanhf(acc[i][j] - b0);
                ei[i] = fmaf(w1, h[i], ei[i]);
                e[i] = w1 * fmaf(-h[i], h[i], 1.0f);
            }
            store_atoms<AT>(sm + l.Es + mu * LD + m0, e);
            store_atoms<AT>(hb + (size_t)mu * TM + m0, h);
        }
    });
    {   // E_i: sum over the 8 threads that share the atoms
        const float b1 = a.theta[m.o_b1];
#pragma unroll
        for (int i = 0; i < AT; ++i) {
            float v = ei[i];
            v += __shfl_xor_sync(0xffffffffu, v, 1); v += __shfl_xor_sync(0xffffffffu, v, 2); v += __shfl_xor_sync(0xffffffffu, v, 4);
            if (tx == 0) sm[l.aux + m0 + i] = v - b1;
        }
    }
    __syncthreads();
    // Fp = s o (w0^T e), written over q
    for_outputs(l.DP8, tx, [&](int o0, int ostep, auto cwc, auto quadc) {
        constexpr int CW = decltype(cwc)::value;
        constexpr bool QUAD = decltype(quadc)::value;
        float acc[AT][CW];
        tile_gemm<AT, CW, QUAD>(sm + l.Es + m0, LD, sm + l.W0m + o0, l.DP8, ostep, m.H, acc);
#pragma unroll
        for (int j = 0; j < CW; ++j) {
            float o[AT];
#pragma unroll
            for (int i = 0; i < AT; ++i) o[i] = acc[i][j];
            store_atoms<AT>(sm + l.Qs + (o0 + j * ostep) * LD + m0, o);
        }
    });
    __syncthreads();
    if (ib >= 0) {
        scatter_rows(sb_ptr(a.b.Fp, ib >> 5, m.D, ib & 31), sm + l.Qs + am, LD, 0, m.D, rg, RG);
        if (rg == 0) a.b.Ei[ib] = sm[l.aux + am];
    }
    // a_k[T'] = sum_n Fp_n cR[t][T'][n][k]
    const int TKRP = m.T * m.KRP;
    for_outputs(l.TKP, tx, [&](int o0, int ostep, auto cwc, auto quadc) {
        constexpr int CW = decltype(cwc)::value;
        constexpr bool QUAD = decltype(quadc)::value;
        float acc[AT][CW];
        tile_gemm<AT, CW, QUAD>(sm + l.Qs + m0, LD, sm + l.cRs + o0, l.TKP, ostep, m.nR, acc);
#pragma unroll
        for (int i = 0; i < AT; ++i) {
            const int ibi = ibs[m0 + i];
            if (ibi < 0) continue;
            float* ar = a.b.arow + (size_t)ibi * TKRP;
            if (QUAD && o0 + 3 < TKRP) {
                *reinterpret_cast<float4*>(ar + o0) = make_float4(acc[i][0], acc[i][CW > 1 ? 1 : 0], acc[i][CW > 2 ? 2 : 0], acc[i][CW > 3 ? 3 : 0]);
            } else {
#pragma unroll
                for (int j = 0; j < CW; ++j) {
                    const int o = o0 + j * ostep;
                    if (o < TKRP) ar[o] = acc[i][j];
                }
            }
        }
    });
        __syncthreads();   // the next tile's gathers overwrite this tile's shared-memory rows
    }
}

// ------------------------------------------------------------------------------------------------
// S8
// ------------------------------------------------------------------------------------------------
template <int TM, int AT>
__global__ void __launch_bounds__(8 * TM / AT) k_ann_bwd(StepArgs a)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int NT = 8 * TM / AT, RG = NT / TM, NW = NT / 32;
    const ModelDev& m = a.m;
    const AnnLay l = ann_layout(m, TM, true);
    const int tid = threadIdx.x;
    // persistent block: a contiguous range of tiles (tiles are sorted by species, so the weights are reloaded rarely)
    const int tbase = a.b.ntiles / (int)gridDim.x, trem = a.b.ntiles - tbase * (int)gridDim.x;
    const int tile0 = (int)blockIdx.x * tbase + min((int)blockIdx.x, trem), tile1 = tile0 + tbase + ((int)blockIdx.x < trem ? 1 : 0);
    int cur_t = -1;
    for (int tile = tile0; tile < tile1; ++tile) {
    const int LD = l.LD;
    int* ibs = reinterpret_cast<int*>(sm + l.ibs);
    const int am = tid % TM, rg = tid / TM;
    const int ib = a.b.alist[(size_t)tile * TM + am];
    {   // per-atom inputs of the tile, straight into shared memory
        const float *qp = nullptr, *qdp = nullptr, *fpp = nullptr, *Bp = nullptr, *Bdp = nullptr;
        float epsi = 0.0f;
        if (ib >= 0) {
            const int w = ib >> 5, ln = ib & 31;
            const int4 bi = __ldg(a.b.binfo + w);
            qp = sb_ptr(a.b.q, w, m.D, ln); qdp = sb_ptr(a.b.qd, w, m.D, ln); fpp = sb_ptr(a.b.Fp, w, m.D, ln);
            Bp = sb_ptr(a.d.B, bi.x, l.TK, ln); Bdp = sb_ptr(a.b.Bd, w, l.TK, ln);
            if (rg == 0) epsi = a.b.eps[bi.y];
        }
        gather_rows(sm + l.BDs + am, LD, Bdp, 0, l.TK, rg, RG);
        gather_rows(sm + l.QDs + am, LD, qdp, m.nR, m.D, rg, RG);
        gather_rows(sm + l.Qs + am, LD, qp, 0, m.D, rg, RG);
        gather_rows(sm + l.FPs + am, LD, fpp, 0, m.nR, rg, RG);
        gather_rows(sm + l.Bs + am, LD, Bp, 0, l.TK, rg, RG);
        cp_async_commit();
        if (rg == 0) { sm[l.aux + am] = epsi; ibs[am] = ib; }
        for (int v = m.D + rg; v < l.DP8; v += RG) { sm[l.Qs + v * LD + am] = 0.0f; sm[l.QDs + v * LD + am] = 0.0f; }
    }
    const int t = tile_type_of(a.b, tile, m.T);
    if (t != cur_t) {
        cur_t = t;
        ann_load_weights(a, l, sm, t, false);
        for (int i = tid; i < l.TK * l.nR8; i += NT) {   // cRt[(tj, k)][n]
            const int r = i / l.nR8, n = i - r * l.nR8, tj = r / m.KR, k = r - tj * m.KR;
            sm[l.cRt + i] = (n < m.nR) ? a.theta[m.o_cR + ((t * m.T + tj) * m.nR + n) * m.KR + k] : 0.0f;
        }
        for (int i = tid; i < (l.HP32 - l.HP8) * l.LD; i += NT) { sm[l.Gs + l.HP8 * l.LD + i] = 0.0f; sm[l.Es + l.HP8 * l.LD + i] = 0.0f; }
    }
    cp_async_wait<0>();
    __syncthreads();
    const int ty = tid >> 3, tx = tid & 7, m0 = ty * AT;
    // radial tangent: qd_n = sum_{T', k} cR[t][T'][n][k] Bd_k[T']
    for_outputs(l.nR8, tx, [&](int o0, int ostep, auto cwc, auto quadc) {
        constexpr int CW = decltype(cwc)::value;
        constexpr bool QUAD = decltype(quadc)::value;
        float acc[AT][CW];
        tile_gemm<AT, CW, QUAD>(sm + l.BDs + m0, LD, sm + l.cRt + o0, l.nR8, ostep, l.TK, acc);
#pragma unroll
        for (int j = 0; j < CW; ++j) {
            const int n = o0 + j * ostep;
            if (n < m.nR) {
                float o[AT];
#pragma unroll
                for (int i = 0; i < AT; ++i) o[i] = acc[i][j];
                store_atoms<AT>(sm + l.QDs + n * LD + m0, o);
            }
        }
    });
    __syncthreads();
    // xd = w0 (s o qd);  gamma, e, and the column sums for g_b0, g_w1
    const float* hb = a.b.hbuf + (size_t)tile * l.HP8 * TM;
    float epsv[AT];
    load_atoms<AT>(sm + l.aux + m0, epsv);
    bool valid[AT];
#pragma unroll
    for (int i = 0; i < AT; ++i) valid[i] = ibs[m0 + i] >= 0;
    for_outputs(l.HP8, tx, [&](int o0, int ostep, auto cwc, auto quadc) {
        constexpr int CW = decltype(cwc)::value;
        constexpr bool QUAD = decltype(quadc)::value;
        float hh[CW][AT];
#pragma unroll
        for (int j = 0; j < CW; ++j) load_atoms<AT>(hb + (size_t)(o0 + j * ostep) * TM + m0, hh[j]);   // in flight during the GEMM
        float acc[AT][CW];
        tile_gemm<AT, CW, QUAD>(sm + l.QDs + m0, LD, sm + l.W0t + o0, l.HP8, ostep, m.D, acc);
#pragma unroll
        for (int j = 0; j < CW; ++j) {
            const int mu = o0 + j * ostep;
            const float w1 = sm[l.w1 + mu];
            float gam[AT], e[AT], sg = 0.0f, sw = 0.0f;
#pragma unroll
            for (int i = 0; i < AT; ++i) {
                const float h = hh[j][i];
                const float omh2 = fmaf(-h, h, 1.0f);
                const float ee = valid[i] ? w1 * omh2 : 0.0f;
                const float xd = acc[i][j];
                e[i] = ee;
                gam[i] = fmaf(epsv[i], ee, -2.0f * h * ee * xd);
                sg += gam[i];
                sw += valid[i] ? fmaf(epsv[i], h, omh2 * xd) : 0.0f;
            }
            store_atoms<AT>(sm + l.Gs + mu * LD + m0, gam);
            store_atoms<AT>(sm + l.Es + mu * LD + m0, e);
            // sum over the 4 atom groups of this warp (lanes with equal tx), then across warps through shared memory
            sg += __shfl_xor_sync(0xffffffffu, sg, 8); sg += __shfl_xor_sync(0xffffffffu, sg, 16);
            sw += __shfl_xor_sync(0xffffffffu, sw, 8); sw += __shfl_xor_sync(0xffffffffu, sw, 16);
            if ((tid & 31) < 8) {
                sm[l.red + ((tid >> 5) * 2 + 0) * l.HP8 + mu] = sg;
                sm[l.red + ((tid >> 5) * 2 + 1) * l.HP8 + mu] = sw;
            }
        }
    });
    __syncthreads();
    {   // g_b0[t][mu] -= sum gamma ; g_w1[t][mu] += sum (eps h + (1-h^2) xd)
        float* gt = a.g + (size_t)t * m.per_type + m.H * m.D;
        for (int i = tid; i < 2 * m.H; i += NT) {
            const int which = i / m.H, mu = i - which * m.H;
            float s = 0.0f;
#pragma unroll
            for (int w = 0; w < NW; ++w) s += sm[l.red + (w * 2 + which) * l.HP8 + mu];
            atomicAdd(gt + which * m.H + mu, which ? s : -s);
        }
    }
    if (tid < 128) {
        // g_w0[t][mu][v] += s_v sum_atoms (gamma_mu q_v + e_mu qd_v): 2 rows {ra, ra + 16} x 5 columns {cb + 8 c} per thread on
        // four warps: 14 shared-memory loads per 80 FFMA (one row per thread on all eight warps: 12 per 40)
        const int ra = tid >> 3, cb = tid & 7;
        float* gt = a.g + (size_t)t * m.per_type;
        for (int rb = 0; rb < l.HP8; rb += 32) {
            const int r0 = rb + ra;
            for_chunks(l.DP8 / 8, [&](int jc0, auto cwc) {
                constexpr int CW = decltype(cwc)::value;
                const int c0 = cb + 8 * jc0;
                float acc[2][CW];
                outer_gemm<2, CW>(sm + l.Gs + r0 * LD, sm + l.Es + r0 * LD, 16 * LD, sm + l.Qs + c0 * LD, sm + l.QDs + c0 * LD, 8 * LD, TM, acc);
#pragma unroll
                for (int r = 0; r < 2; ++r)
#pragma unroll
                    for (int cc = 0; cc < CW; ++cc) {
                        const int mu = r0 + 16 * r, v = c0 + 8 * cc;
                        if (mu < m.H && v < m.D) atomicAdd(gt + mu * m.D + v, sm[l.sc + v] * acc[r][cc]);
                    }
            });
        }
    }
    __syncthreads();
    // Qb = s o (w0^T gamma), written over q
    for_outputs(l.DP8, tx, [&](int o0, int ostep, auto cwc, auto quadc) {
        constexpr int CW = decltype(cwc)::value;
        constexpr bool QUAD = decltype(quadc)::value;
        float acc[AT][CW];
        tile_gemm<AT, CW, QUAD>(sm + l.Gs + m0, LD, sm + l.W0m + o0, l.DP8, ostep, m.H, acc);
#pragma unroll
        for (int j = 0; j < CW; ++j) {
            float o[AT];
#pragma unroll
            for (int i = 0; i < AT; ++i) o[i] = acc[i][j];
            store_atoms<AT>(sm + l.Qs + (o0 + j * ostep) * LD + m0, o);
        }
    });
    __syncthreads();
    if (ib >= 0) scatter_rows(sb_ptr(a.b.Qb, ib >> 5, m.D, ib & 31), sm + l.Qs + am, LD, m.nR, m.D, rg, RG);   // only the angular rows are read later
    // g_cR[t][T'][n][k] += sum_atoms Qb_n B_k[T'] + Fp_n Bd_k[T'] : one output per thread
    for (int o = tid; o < m.nR * l.TK; o += NT) {
        const int n = o / l.TK, r = o - n * l.TK;
        float acc[1][1];
        outer_gemm<1, 1>(sm + l.Qs + n * LD, sm + l.FPs + n * LD, 0, sm + l.Bs + r * LD, sm + l.BDs + r * LD, 0, TM, acc);
        const int tj = r / m.KR, k = r - tj * m.KR;
        atomicAdd(a.g + m.o_cR + ((t * m.T + tj) * m.nR + n) * m.KR + k, acc[0][0]);
    }
        __syncthreads();   // the next tile's gathers overwrite this tile's shared-memory rows
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
constexpr int ANN_AT = 4;   // atoms per thread: 256 threads per 128-atom tile

int ann_tile_m(const nep_ctx* c)
{
    if (c->ann_tc) return 128;
    // 128-atom tiles while two blocks of the larger (backward) kernel fit in one SM's shared memory, else 64
    const size_t bytes128 = 4 * (size_t)ann_layout(c->m, 128, true).total;
    return bytes128 <= 110 * 1024 ? 128 : 64;
}

// Blocks of the persistent network kernels: one resident wave; every block takes a contiguous range of tiles and loads the
// weights once per species it meets (config 2: k_ann_bwd 105 -> 98 us; config 4: 377 -> 295 us, k_ann_fwd 136 -> 113 us).
static int ann_grid(int ntiles, int resident) { return ntiles < resident ? ntiles : resident; }

template <int TM>
static int launch_ann_t(nep_ctx* c, const StepArgs& a, bool bwd)
{
    constexpr int NT = 8 * TM / ANN_AT;
    const size_t smem = 4 * (size_t)ann_layout(c->m, TM, bwd).total;
    if (smem > (size_t)c->max_smem_optin) return fail(c, NEP_ECAPACITY, "network tile does not fit in shared memory (neurons x descriptors too large)");
    if (c->b.ntiles == 0) return NEP_OK;
    if (bwd) {
        NEP_CUDA(c, cudaFuncSetAttribute(k_ann_bwd<TM, ANN_AT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int occ = 1;
        NEP_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_ann_bwd<TM, ANN_AT>, NT, smem));
        NEP_LAUNCH(c, "k_ann_bwd", (k_ann_bwd<TM, ANN_AT>), ann_grid(c->b.ntiles, std::max(occ, 1) * c->sm_count), NT, smem, a);
    } else {
        NEP_CUDA(c, cudaFuncSetAttribute(k_ann_fwd<TM, ANN_AT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int occ = 1;
        NEP_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_ann_fwd<TM, ANN_AT>, NT, smem));
        NEP_LAUNCH(c, "k_ann_fwd", (k_ann_fwd<TM, ANN_AT>), ann_grid(c->b.ntiles, std::max(occ, 1) * c->sm_count), NT, smem, a);
    }
    return NEP_OK;
}
int launch_ann_fwd(nep_ctx* c, const StepArgs& a)
{
    if (c->ann_tc) return launch_ann_fwd_tc(c, a);
    return c->b.tile_m == 128 ? launch_ann_t<128>(c, a, false) : launch_ann_t<64>(c, a, false);
}
int launch_ann_bwd(nep_ctx* c, const StepArgs& a)
{
    if (c->ann_tc) return launch_ann_bwd_tc(c, a);
    return c->b.tile_m == 128 ? launch_ann_t<128>(c, a, true) : launch_ann_t<64>(c, a, true);
}

}  // namespace nep
