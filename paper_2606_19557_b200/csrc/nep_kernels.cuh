// nep_kernels.cuh -- helpers shared by the step kernels.
//
// Execution model of every pair sweep: ONE THREAD PER ATOM, one warp per 32-atom slice of one structure.
// Pair records of a slice are stored slot-major ([slot][lane], 16 B each), so the 32 lanes of a warp read
// 512 contiguous bytes per slot; each lane's records are sorted by neighbour type.  The record of slot s+1 is
// fetched before slot s is processed.  Per-atom tensors (angular moments and their adjoints, up to 5 channels x
// 24 harmonics) live in registers; all sizes that shape a loop (channels per thread, basis functions) are
// compile-time constants so that no register array is indexed dynamically.
#pragma once
#include "nep_internal.h"
#include "nep_math.cuh"
#include "nep_umma.cuh"

namespace nep {

struct StepArgs {
    ModelDev m;
    DataDev d;
    BatchDev b;
    const float* theta;
    const float* scaler;
    float* g;
    int nchunks;   // angular channel chunks (blockIdx.y)
};

constexpr int PAIR_TB = 128;   // threads per block of the pair sweeps (2 slices)

struct Lane {
    int w, lane, ds, sb, bbase, ti;
    unsigned ib;   // batch-padded atom index w*32 + lane
};

__host__ __device__ inline int rup(int x, int m) { return (x + m - 1) / m * m; }

// species of a network tile (tiles are sorted by species; b.tile_start[t] = first tile of species t)
__device__ __forceinline__ int tile_type_of(const BatchDev& b, int tile, int T)
{
    int t = 0;
#pragma unroll 1
    while (t + 1 < T && tile >= b.tile_start[t + 1]) ++t;
    return t;
}

// lane state for batch slice w (w < a.b.nbs)
__device__ __forceinline__ void lane_init_slice(const StepArgs& a, Lane& L, int w)
{
    L.w = w;
    L.lane = threadIdx.x & 31;
    const int4 bi = __ldg(a.b.binfo + w);
    L.ds = bi.x; L.sb = bi.y; L.bbase = bi.z;
    L.ib = (unsigned)w * WARP + L.lane;
    L.ti = __ldg(a.d.type_p + (size_t)L.ds * WARP + L.lane);
}

// requests a block of global memory into L2 (one instruction per contiguous block)
__device__ __forceinline__ void prefetch_l2(const void* p, unsigned bytes)   // bytes: a multiple of 16
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(p), "r"(bytes) : "memory");
}

// false if the warp is beyond the batch (whole warp returns together)
__device__ __forceinline__ bool lane_init(const StepArgs& a, Lane& L)
{
    L.w = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    L.lane = threadIdx.x & 31;
    if (L.w >= a.b.nbs) return false;
    const int4 bi = __ldg(a.b.binfo + L.w);
    L.ds = bi.x; L.sb = bi.y; L.bbase = bi.z;
    L.ib = (unsigned)L.w * WARP + L.lane;
    L.ti = __ldg(a.d.type_p + (size_t)L.ds * WARP + L.lane);
    return true;
}

// slice-blocked addressing: row 0 of (slice, lane) in an array with ROWS rows per slice
__device__ __forceinline__ float* sb_ptr(float* base, int slice, int rows, int lane) { return base + ((size_t)slice * rows) * WARP + lane; }
__device__ __forceinline__ const float* sb_ptr(const float* base, int slice, int rows, int lane) { return base + ((size_t)slice * rows) * WARP + lane; }

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

// Sum over the 32 lanes of P values per lane (P a power of two >= 32) in P - P/32 shuffles instead of 5 P: in each of the five steps a
// lane keeps one half of its values and sends the other half to its partner.  Afterwards lane l holds, in v[0 .. P/32 - 1], the totals
// of the elements (P/32) l .. (P/32) l + P/32 - 1.
template <int P>
__device__ __forceinline__ void warp_reduce_scatter(float* v)
{
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int step = 0; step < 5; ++step) {
        const int mask = 16 >> step, cnt = P >> (step + 1);
        const bool up = lane & mask;
#pragma unroll
        for (int i = 0; i < cnt; ++i) {
            const float keep = up ? v[i + cnt] : v[i], send = up ? v[i] : v[i + cnt];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, mask);
        }
    }
}

// Forces of the batch: F[batch-padded atom][4] = (F_x, F_y, F_z, unused), one 16-byte cell per atom, so that a scattered pair
// reaction is ONE vector reduction (red.global.add.v4.f32) instead of three scalar ones: a warp-wide scatter costs the SM's
// load/store path ~41 cycles per instruction whatever its width.
__device__ __forceinline__ void force_add(float* F, unsigned ib, float x, float y, float z)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" :: "l"(F + 4 * (size_t)ib), "f"(x), "f"(y), "f"(z), "f"(0.0f) : "memory");
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
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(p.rinv) : "f"(r2));   // r2 is never subnormal: skip rsqrtf's scaling path
    p.r = r2 * p.rinv;
    p.x = p.dx * p.rinv; p.y = p.dy * p.rinv; p.z = p.dz * p.rinv;
    return p;
}

// Streams the pair records of one lane: body(record) for slots 0..cnt-1; all lanes of the warp walk `width` slots.
// Records are staged through shared memory with cp.async (LDGSTS), SWEEP_STAGES slots ahead, so that the HBM/L2
// latency of slot s+1, s+2 is covered by the arithmetic of slot s.  Each lane reads back only what it copied
// itself, so cp.async.wait_group is the only synchronisation needed.
constexpr int SWEEP_STAGES = 2;

__device__ __forceinline__ void cp_async16(float4* smem_dst, const float4* gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }

// one record per iteration: body(record) for the slots the lane has; staging cells of successive stages are TB apart
template <int TB, class Body>
__device__ __forceinline__ void sweep_pairs_tb(const float4* __restrict__ rec, int width, int cnt, float4* stage, Body&& body)
{
#pragma unroll
    for (int st = 0; st < SWEEP_STAGES; ++st) {
        if (st < width) cp_async16(stage + st * TB, rec + (size_t)st * WARP);
        cp_async_commit();
    }
    for (int s = 0; s < width; ++s) {
        cp_async_wait<SWEEP_STAGES - 1>();
        float4* cell = stage + (s % SWEEP_STAGES) * TB;
        const float4 cur = *cell;
        if (s + SWEEP_STAGES < width) cp_async16(cell, rec + (size_t)(s + SWEEP_STAGES) * WARP);
        cp_async_commit();
        if (s < cnt) body(cur);
    }
    cp_async_wait<0>();
}

// Two slots per iteration: body2(record of slot s, record of slot s + 1, has_second) for s = 0, 2, 4, ... < cnt.
// The dependent chains of a pair (distance, cutoff polynomial, Chebyshev recurrence) are long and a sweep runs two
// warps per scheduler, so the arithmetic of two pairs is interleaved to fill the pipe.  When the lane has no second
// record the first one is passed again with has_second = false (finite values that the body multiplies by zero).
// stage: 4 staging cells per thread, SWEEP2_TB apart.
constexpr int SWEEP2_TB = 128;
constexpr int SWEEP2_SMEM_BYTES = SWEEP2_TB * 16 * 4;
// sweep2_begin requests the first four slots (two groups); sweep2_run consumes the records.  They are separate so that a kernel can
// compute its prologue while the records arrive.
template <int TB>
__device__ __forceinline__ void sweep2_begin(const float4* __restrict__ rec, int width, float4* stage)
{
#pragma unroll
    for (int g = 0; g < 2; ++g) {
#pragma unroll
        for (int h = 0; h < 2; ++h)
            if (2 * g + h < width) cp_async16(stage + (2 * g + h) * TB, rec + (size_t)(2 * g + h) * WARP);
        cp_async_commit();
    }
}
template <int TB, class Body2>
__device__ __forceinline__ void sweep2_run(const float4* __restrict__ rec, int width, int cnt, float4* stage, Body2&& body2)
{
    for (int s = 0; s < width; s += 2) {
        cp_async_wait<1>();
        float4* c0 = stage + (s & 3) * TB;
        float4* c1 = stage + ((s + 1) & 3) * TB;
        const float4 r0 = *c0;
        float4 r1 = *c1;
        if (s + 4 < width) cp_async16(c0, rec + (size_t)(s + 4) * WARP);
        if (s + 5 < width) cp_async16(c1, rec + (size_t)(s + 5) * WARP);
        cp_async_commit();
        if (s < cnt) {
            const bool has2 = s + 1 < cnt;
            if (!has2) r1 = r0;
            body2(r0, r1, has2);
        }
    }
    cp_async_wait<0>();
}
template <int TB, class Body2>
__device__ __forceinline__ void sweep_pairs2(const float4* __restrict__ rec, int width, int cnt, float4* stage, Body2&& body2)
{
    sweep2_begin<TB>(rec, width, stage);
    sweep2_run<TB>(rec, width, cnt, stage, body2);
}

// ------------------------------------------------------------------------------------------------
// Per-atom rows through shared memory.  The prologue / epilogue of an angular sweep reads 120-300 slice-blocked rows per warp;
// loaded channel after channel into registers they are 5-10 dependent DRAM round trips with little to overlap them at two
// warps per scheduler (ncu, config 2: 27-35 % of a sweep's warp time sits there).  The rows of one slice are contiguous
// (rows x 128 bytes), so lane 0 of the warp requests each block of rows with ONE bulk copy (cp.async.bulk, the TMA engine)
// into the warp's own shared-memory area, as the first thing the kernel does (the addresses depend on the block index only);
// completion is signalled on the warp's mbarrier, independent of the cp.async groups of the pair records, and awaited where the
// rows are first needed.  Every lane then reads its column area[row * 32 + lane], conflict free.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* mbar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(umma::smem_u32(dst)), "l"(src), "r"(bytes), "r"(umma::smem_u32(mbar)) : "memory");
}
// whole warp calls; two blocks of rows (either may be empty).  rows_wait afterwards, by every lane, before the first read.
// A warp may use its area a second time (again = true, after every lane has finished reading the first contents): the mbarrier then
// completes its next phase, awaited with parity 1.
__device__ __forceinline__ void rows_request(uint64_t* mbar, float* dst0, const float* src0, int rows0, float* dst1, const float* src1, int rows1,
                                             bool again = false)
{
    __syncwarp();
    if ((threadIdx.x & 31) == 0) {
        if (!again) umma::mbar_init(mbar, 1);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // barrier initialised / area read: visible to the async proxy
        const uint32_t b0 = (uint32_t)rows0 * (4 * WARP), b1 = (uint32_t)rows1 * (4 * WARP);
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(umma::smem_u32(mbar)), "r"(b0 + b1) : "memory");
        if (b0) bulk_g2s(dst0, src0, b0, mbar);
        if (b1) bulk_g2s(dst1, src1, b1, mbar);
    }
    __syncwarp();
}
__device__ __forceinline__ void rows_wait(uint64_t* mbar, uint32_t parity = 0) { umma::mbar_wait(mbar, parity); }

struct SweepA { const float4* rec; int width, cnt; };
__device__ __forceinline__ SweepA sweep_init(const int64_t* __restrict__ recoff, const float4* __restrict__ recs,
                                             const int* __restrict__ cntp, const Lane& L)
{
    SweepA s;
    const int64_t base = __ldg(recoff + L.ds);
    s.width = (int)((__ldg(recoff + L.ds + 1) - base) >> 5);
    s.rec = recs + base + L.lane;
    s.cnt = (L.ti >= 0) ? __ldg(cntp + (size_t)L.ds * WARP + L.lane) : 0;
    return s;
}

// ------------------------------------------------------------------------------------------------
// Angular coefficients of one channel chunk in shared memory: cs[pt * CSTRIDE + k * NCHP + n], n < NCHP (zero
// padded), NCHP = 4 (NCH <= 4) or 8; CSTRIDE = K * NCHP rounded up to 4 (mod 8) so that the 128-bit loads of
// lanes with different pair types fall into different bank groups.
// ------------------------------------------------------------------------------------------------
template <int NCH> struct ChunkPad { static constexpr int value = NCH <= 4 ? 4 : 8; };
template <int NCH, int K> struct CoefStride {
    static constexpr int raw = K * ChunkPad<NCH>::value;
    static constexpr int value = raw + ((12 - raw % 8) % 8);   // == 4 (mod 8)
};

template <int NCH, int K>
__device__ __forceinline__ void load_cA_chunk(const StepArgs& a, float* cs, int n0)
{
    const ModelDev& m = a.m;
    constexpr int NCHP = ChunkPad<NCH>::value, CST = CoefStride<NCH, K>::value;
    const int tot = m.T * m.T * CST;
    // unrolled: the loads of eight elements are in flight together (at 5 species the table is ~1100 values per block)
#pragma unroll 8
    for (int i = threadIdx.x; i < tot; i += blockDim.x) {
        const int pt = i / CST, rem = i - pt * CST, k = rem / NCHP, n = rem - k * NCHP;
        float v = 0.0f;
        if (k < m.KA && n < NCH && n0 + n < m.nA) v = __ldg(a.theta + m.o_cA + (pt * m.nA + n0 + n) * m.KA + k);
        cs[i] = v;
    }
}
template <int NCH, int K>
inline size_t cA_chunk_bytes(const ModelDev& m) { return 4 * (size_t)(m.T * m.T * CoefStride<NCH, K>::value); }

// coefficients of basis function k for the NCH channels of the chunk
template <int NCH>
__device__ __forceinline__ void coef_k(const float* __restrict__ cp, int k, float* c)
{
    constexpr int NCHP = ChunkPad<NCH>::value;
    const float4 v = *reinterpret_cast<const float4*>(cp + k * NCHP);
    c[0] = v.x;
    if (NCH > 1) c[1] = v.y;
    if (NCH > 2) c[2] = v.z;
    if (NCH > 3) c[3] = v.w;
    if (NCH > 4) c[4] = cp[k * NCHP + 4];
}

// g_n(r) = sum_k c_nk f_k(r) (and g_n') for the chunk's channels  (Eq. 16)
template <int NCH, int K, bool DERIV, bool FAST = false>
__device__ __forceinline__ void radial_gn(float r, float rcinv, const float* __restrict__ cp, float* g, float* dg, float scale = 1.0f)
{
#pragma unroll
    for (int n = 0; n < NCH; ++n) { g[n] = 0.0f; if (DERIV) dg[n] = 0.0f; }
    cheb_basis<K, DERIV, FAST>(r, rcinv, [&](int k, float fk, float dfk) {
        float c[NCH];
        coef_k<NCH>(cp, k, c);
#pragma unroll
        for (int n = 0; n < NCH; ++n) {
            g[n] = fmaf(c[n], fk, g[n]);
            if (DERIV) dg[n] = fmaf(c[n], dfk, dg[n]);
        }
    }, scale);
}

// descriptor rows of the angular invariants of channel n: slots 0..3 -> l = 1..4, slot 4 -> 4-body, slot 5 -> 5-body
__device__ __forceinline__ int ang_row(const ModelDev& m, int slot, int n)
{
    const int a = slot < 4 ? slot : (slot == 4 ? m.l3 : m.l3 + m.has4);   // callers use a 3-body slot only if slot < l3
    return m.nR + a * m.nA + n;
}
__device__ __forceinline__ void store_inv(const ModelDev& m, float* __restrict__ arr, int n, const float* q)
{
#pragma unroll
    for (int s = 0; s < 4; ++s)
        if (s < m.l3) arr[(size_t)ang_row(m, s, n) * WARP] = q[s];
    if (m.has4) arr[(size_t)ang_row(m, 4, n) * WARP] = q[4];
    if (m.has5) arr[(size_t)ang_row(m, 5, n) * WARP] = q[5];
}

// packed pairs: two fp32 lanes of work per issue slot (FFMA2 on sm_100)
__device__ __forceinline__ float2 dup2(float v) { return make_float2(v, v); }
__device__ __forceinline__ void pack24(const float* b, float2* b2)
{
#pragma unroll
    for (int i = 0; i < NL / 2; ++i) b2[i] = make_float2(b[2 * i], b[2 * i + 1]);
}
__device__ __forceinline__ void unpack24(const float2* b2, float* b)
{
#pragma unroll
    for (int i = 0; i < NL / 2; ++i) { b[2 * i] = b2[i].x; b[2 * i + 1] = b2[i].y; }
}

// EdS_nL = dE_i/dS_nL = sum_a Fp[q index (a, n)] dq_a/dS_nL for the NCH channels of this thread (DESIGN C8).
// Branch free (channels beyond n_A and padding lanes read a valid row and select zero), so that the loads of all channels are
// issued together: one DRAM round trip instead of one per channel.
template <int NCH>
__device__ __forceinline__ void load_EdS(const StepArgs& a, const Lane& L, int n0, float (*EdS)[NL])
{
    const ModelDev& m = a.m;
    const float* Sp = sb_ptr(a.b.S, L.w, m.nA * NL, L.lane);
    const float* Fpp = sb_ptr(a.b.Fp, L.w, m.D, L.lane);
    float S[NCH][NL], coef[NCH][6];
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        const int nn = n0 + n < m.nA ? n0 + n : m.nA - 1;
        const float* sp = Sp + (size_t)nn * NL * WARP;
#pragma unroll
        for (int l = 0; l < NL; ++l) S[n][l] = __ldg(sp + l * WARP);
#pragma unroll
        for (int s = 0; s < 4; ++s) coef[n][s] = __ldg(Fpp + (size_t)ang_row(m, s < m.l3 ? s : 0, nn) * WARP);
        coef[n][4] = __ldg(Fpp + (size_t)ang_row(m, m.has4 ? 4 : 0, nn) * WARP);
        coef[n][5] = __ldg(Fpp + (size_t)ang_row(m, m.has5 ? 5 : 0, nn) * WARP);
    }
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        const bool ok = n0 + n < m.nA && L.ti >= 0;
#pragma unroll
        for (int s = 0; s < 4; ++s) coef[n][s] = (ok && s < m.l3) ? coef[n][s] : 0.0f;
        coef[n][4] = (ok && m.has4) ? coef[n][4] : 0.0f;
        coef[n][5] = (ok && m.has5) ? coef[n][5] : 0.0f;
        inv_adjoint(S[n], coef[n], EdS[n]);
    }
}

// Sb_nL = sum_a Qb[(a, n)] dq_a/dS_nL + sum_a Fp[(a, n)] (H_{q_a} Sd)_nL: the per-atom tensor of the first pass of the adjoint sweep
// (DESIGN C12).  Branch free like load_EdS.
template <int NCH>
__device__ __forceinline__ void load_Sbar(const StepArgs& a, const Lane& L, int n0, float (*X)[NL])
{
    const ModelDev& m = a.m;
    const float* Sp = sb_ptr(a.b.S, L.w, m.nA * NL, L.lane);
    const float* Sdp = sb_ptr(a.b.Sd, L.w, m.nA * NL, L.lane);
    const float* Qbp = sb_ptr(a.b.Qb, L.w, m.D, L.lane);
    const float* Fpp = sb_ptr(a.b.Fp, L.w, m.D, L.lane);
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        const bool ok = n0 + n < m.nA && L.ti >= 0;
        const int nn = n0 + n < m.nA ? n0 + n : m.nA - 1;
        const float* sp = Sp + (size_t)nn * NL * WARP;
        const float* dp = Sdp + (size_t)nn * NL * WARP;
        float S[NL], Sd[NL], cq[6], cf[6];
#pragma unroll
        for (int l = 0; l < NL; ++l) { S[l] = __ldg(sp + l * WARP); Sd[l] = __ldg(dp + l * WARP); }
#pragma unroll
        for (int s = 0; s < 6; ++s) {
            const int slot = (s < 4 ? s < m.l3 : (s == 4 ? m.has4 : m.has5)) ? s : 0;
            cq[s] = __ldg(Qbp + (size_t)ang_row(m, slot, nn) * WARP);
            cf[s] = __ldg(Fpp + (size_t)ang_row(m, slot, nn) * WARP);
        }
#pragma unroll
        for (int s = 0; s < 6; ++s) {
            const bool on = ok && (s < 4 ? s < m.l3 : (s == 4 ? m.has4 : m.has5));
            cq[s] = on ? cq[s] : 0.0f; cf[s] = on ? cf[s] : 0.0f;
        }
        inv_adjoint_hessian(S, Sd, cq, cf, X[n]);
        if (!ok)
#pragma unroll
            for (int l = 0; l < NL; ++l) X[n][l] = 0.0f;
    }
}

// load_Sbar with Sd (chunk rows) and the angular rows of Qb staged in shared memory (Ds, Qs: this lane's column); S and the
// coefficients from Fp come straight from global memory, all loads issued before the staged rows are awaited.
template <int NCH>
__device__ __forceinline__ void load_Sbar_staged(const StepArgs& a, const Lane& L, int n0, const float* Ds, const float* Qs, uint64_t* mbar,
                                                 float (*X)[NL])
{
    const ModelDev& m = a.m;
    const float* Sp = sb_ptr(a.b.S, L.w, m.nA * NL, L.lane);
    const float* Fpp = sb_ptr(a.b.Fp, L.w, m.D, L.lane);
    float cf[NCH][6];
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        const int nn = n0 + n < m.nA ? n0 + n : m.nA - 1;
        const float* sp = Sp + (size_t)nn * NL * WARP;
#pragma unroll
        for (int l = 0; l < NL; ++l) X[n][l] = __ldg(sp + l * WARP);          // S for now
#pragma unroll
        for (int s = 0; s < 6; ++s) {
            const int slot = (s < 4 ? s < m.l3 : (s == 4 ? m.has4 : m.has5)) ? s : 0;
            cf[n][s] = __ldg(Fpp + (size_t)ang_row(m, slot, nn) * WARP);
        }
    }
    rows_wait(mbar, 0);
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        const bool ok = n0 + n < m.nA && L.ti >= 0;
        const int nn = n0 + n < m.nA ? n0 + n : m.nA - 1;
        float S[NL], Sd[NL], cq[6], out[NL];
#pragma unroll
        for (int l = 0; l < NL; ++l) { S[l] = X[n][l]; Sd[l] = ok ? Ds[(n * NL + l) * WARP] : 0.0f; }
#pragma unroll
        for (int s = 0; s < 6; ++s) {
            const bool on = ok && (s < 4 ? s < m.l3 : (s == 4 ? m.has4 : m.has5));
            const int row = s < 4 ? s : (s == 4 ? m.l3 : m.l3 + m.has4);
            cq[s] = on ? Qs[(row * m.nA + nn) * WARP] : 0.0f;
            cf[n][s] = on ? cf[n][s] : 0.0f;
        }
        inv_adjoint_hessian(S, Sd, cq, cf[n], out);
#pragma unroll
        for (int l = 0; l < NL; ++l) X[n][l] = ok ? out[l] : 0.0f;
    }
}

// The same from rows staged in shared memory: Ss = the NCH x 24 moment rows of the chunk, Fs = the angular rows nR .. D-1 of Fp
// (both [row][lane], pointers at this lane's column).
template <int NCH>
__device__ __forceinline__ void load_EdS_staged(const ModelDev& m, int ti, int n0, const float* Ss, const float* Fs, float (*EdS)[NL])
{
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        const bool ok = n0 + n < m.nA && ti >= 0;
        const int nn = n0 + n < m.nA ? n0 + n : m.nA - 1;
        float S[NL], coef[6];
#pragma unroll
        for (int l = 0; l < NL; ++l) S[l] = ok ? Ss[(n * NL + l) * WARP] : 0.0f;
#pragma unroll
        for (int s = 0; s < 4; ++s) coef[s] = (ok && s < m.l3) ? Fs[(s * m.nA + nn) * WARP] : 0.0f;
        coef[4] = (ok && m.has4) ? Fs[(m.l3 * m.nA + nn) * WARP] : 0.0f;
        coef[5] = (ok && m.has5) ? Fs[((m.l3 + m.has4) * m.nA + nn) * WARP] : 0.0f;
        inv_adjoint(S, coef, EdS[n]);
    }
}
// rows of the chunk's moments and of the angular part of a [D]-row array, and the shared-memory floats a warp needs for both
__device__ __forceinline__ int chunk_rows(const ModelDev& m, int n0, int nch) { return (m.nA - n0 < nch ? m.nA - n0 : nch) * NL; }
__host__ __device__ inline size_t staged_warp_floats(const ModelDev& m, int nch) { return (size_t)(nch * NL + (m.D - m.nR)) * WARP; }
constexpr size_t STAGED_BAR_BYTES = (PAIR_TB / WARP) * 8;   // one mbarrier per warp of a block, after the areas

// d~ = u_i - u_j - G^T d ;  returns t = r^ . d~ and the tangent rho = (d~ - t r^) / r of r^
struct Tangent { float t, rx, ry, rz; };
__device__ __forceinline__ Tangent pair_tangent(const float* __restrict__ ub, int bbase, const PairGeo& p, float uix, float uiy, float uiz,
                                                const float* G)
{
    const unsigned jb = (unsigned)(bbase + p.jl);
    const float* uj = ub + (size_t)(jb >> 5) * (3 * WARP) + (jb & 31);
    const float ujx = __ldg(uj), ujy = __ldg(uj + WARP), ujz = __ldg(uj + 2 * WARP);
    const float tx = uix - ujx - (G[0] * p.dx + G[3] * p.dy + G[6] * p.dz);
    const float ty = uiy - ujy - (G[1] * p.dx + G[4] * p.dy + G[7] * p.dz);
    const float tz = uiz - ujz - (G[2] * p.dx + G[5] * p.dy + G[8] * p.dz);
    Tangent T;
    T.t = tx * p.x + ty * p.y + tz * p.z;
    T.rx = (tx - T.t * p.x) * p.rinv; T.ry = (ty - T.t * p.y) * p.rinv; T.rz = (tz - T.t * p.z) * p.rinv;
    return T;
}

#define NEP_LAUNCH(c, name, kernel, grid, block, smem, ...)                        \
    do {                                                                           \
        nep::prof_begin((c), name);                                                \
        kernel<<<(grid), (block), (smem), (c)->stream>>>(__VA_ARGS__);             \
        nep::prof_end((c));                                                        \
        NEP_CUDA((c), cudaGetLastError());                                         \
    } while (0)

// kernel + argument blocks of the two step kernels whose scalar arguments change from step to step (loss weights, learning
// rate, Adam bias corrections): used for the direct launch and to re-parameterise their nodes in a captured step graph
struct LossArgs {
    StepArgs a; float lamE, lamF, lamV; double dlamE, dlamF, dlamV;
    const void* func; void* ptrs[7];
};
struct AdamArgs {
    int n; float *theta; const float* g; float *m, *v, *vmax; float lr, beta1, beta2, omb1, omb2, eps, inv_bc1, inv_bc2;
    const void* func; void* ptrs[14];
};
void loss_args(nep_ctx* c, const StepArgs& a, LossArgs* o);
void adam_args(nep_ctx* c, double lr, double b1, double b2, double eps, int variant, int64_t t, AdamArgs* o);

// channels per thread for the angular sweeps: 3, 4 or 5 (fewer channels run as 3 with zero coefficients)
// A batch far below one resident wave of slices (config 1: 16 slices) is bound by the latency of a single warp's pair loop, and
// blocks are free: such batches run 3 channels per thread (more channel chunks side by side, shorter contractions per pair).
inline int pick_nch(const nep_ctx* c)
{
    const int nA = c->m.nA;
    if (c->b.nbs > 0 && c->b.nbs < c->sm_count / 2) return 3;
    const int chunks = (nA + MAX_NCH - 1) / MAX_NCH;
    const int nch = (nA + chunks - 1) / chunks;
    return nch < 3 ? 3 : nch;
}
inline int pick_kpad(int K) { return K <= 9 ? 9 : (K <= 13 ? 13 : 17); }

inline StepArgs make_args(nep_ctx* c)
{
    StepArgs a;
    a.m = c->m; a.d = c->d; a.b = c->b; a.theta = c->theta; a.scaler = c->scaler; a.g = c->g;
    const int nch = pick_nch(c);
    a.nchunks = (c->m.nA + nch - 1) / nch;
    return a;
}

// instantiates `__VA_ARGS__` with constexpr int NCH, K for the model's channel count and basis size
#define NEP_DISPATCH_NCH_K(nch, kpad, ...)                                              \
    do {                                                                                \
        if ((nch) == 3) { constexpr int NCH = 3; NEP_DISPATCH_K_(kpad, __VA_ARGS__) }   \
        else if ((nch) == 4) { constexpr int NCH = 4; NEP_DISPATCH_K_(kpad, __VA_ARGS__) } \
        else { constexpr int NCH = 5; NEP_DISPATCH_K_(kpad, __VA_ARGS__) }              \
    } while (0)
#define NEP_DISPATCH_K_(kpad, ...)                          \
    if ((kpad) == 9) { constexpr int K = 9; __VA_ARGS__; }  \
    else if ((kpad) == 13) { constexpr int K = 13; __VA_ARGS__; } \
    else { constexpr int K = 17; __VA_ARGS__; }

// launchers of the individual sweeps (one .cu file each, so that they compile in parallel)
int launch_ang_fwd(nep_ctx* c, const StepArgs& a);
int launch_ang_force(nep_ctx* c, const StepArgs& a);
int launch_ang_tangent(nep_ctx* c, const StepArgs& a);
int launch_ang_adjoint(nep_ctx* c, const StepArgs& a);
int launch_rad_force(nep_ctx* c, const StepArgs& a);
int launch_rad_tangent(nep_ctx* c, const StepArgs& a);
int launch_ann_fwd(nep_ctx* c, const StepArgs& a);
int launch_ann_bwd(nep_ctx* c, const StepArgs& a);
int launch_loss(nep_ctx* c, const StepArgs& a);
// tensor-core network kernels (nep_ann_tc.cu); ann_tc_fits: the model's tiles fit in shared memory and TMEM
bool ann_tc_fits(const nep_ctx* c, bool bwd);
int launch_ann_fwd_tc(nep_ctx* c, const StepArgs& a);
int launch_ann_bwd_tc(nep_ctx* c, const StepArgs& a);

}  // namespace nep
