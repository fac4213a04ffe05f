// nep_neighbor.cu -- S0a: cell-list neighbour build for periodic (triclinic, possibly thinner than the cutoff)
// boxes, bit-exact and canonically sorted (DESIGN C1);  S0b: per-pair geometry cache in a warp-sliced layout
// and the per-atom radial basis aggregate.  One-time set-up, outside the training step.
//
// The distance predicate is evaluated in IEEE fp64 with explicitly rounded operations (__dadd_rn/__dmul_rn,
// and this file is compiled with -fmad=false):  d = (((r_j - r_i) + n_a a) + n_b b) + n_c c,
// r2 = (dx dx + dy dy) + dz dz,  neighbour iff r2 < rc^2.  The cell list only prunes candidates, conservatively.
#include <math.h>

#include <algorithm>

#include "nep_internal.h"

namespace nep {

struct CellGeom {       // per structure
    double inv[9];      // frac_k = r . inv[:,k]
    int nc[3];          // cells per axis
    int m[3];           // search range in cells per axis
    int64_t cbase;      // first cell of the structure
};

__device__ __forceinline__ int floordiv(int a, int b) { int q = a / b; return (a % b != 0 && ((a < 0) != (b < 0))) ? q - 1 : q; }

__device__ __forceinline__ void bond_rn(const double* ri, const double* rj, const double* bx, int na, int nb, int nc, double* d)
{
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double t = __dsub_rn(rj[k], ri[k]);
        t = __dadd_rn(t, __dmul_rn((double)na, bx[k]));
        t = __dadd_rn(t, __dmul_rn((double)nb, bx[3 + k]));
        t = __dadd_rn(t, __dmul_rn((double)nc, bx[6 + k]));
        d[k] = t;
    }
}
__device__ __forceinline__ double norm2_rn(const double* d)
{
    return __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
}

__global__ void k_bin_count(int64_t N, const double* __restrict__ pos, const int* __restrict__ atom_struct,
                            const CellGeom* __restrict__ cg, int* __restrict__ cell_of, int* __restrict__ cell_cnt)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const CellGeom& g = cg[atom_struct[i]];
    int c[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double f = pos[3 * i] * g.inv[k] + pos[3 * i + 1] * g.inv[3 + k] + pos[3 * i + 2] * g.inv[6 + k];
        int ck = (int)floor(f * g.nc[k]);
        c[k] = min(max(ck, 0), g.nc[k] - 1);
    }
    int cell = (c[0] * g.nc[1] + c[1]) * g.nc[2] + c[2];
    cell_of[i] = cell;
    atomicAdd(&cell_cnt[g.cbase + cell], 1);
}

__global__ void k_bin_fill(int64_t N, const int* __restrict__ atom_struct, const int64_t* __restrict__ atom_off,
                           const CellGeom* __restrict__ cg, const int* __restrict__ cell_of,
                           const int64_t* __restrict__ cell_start, int* __restrict__ cell_fill, int* __restrict__ cell_atoms)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int s = atom_struct[i];
    int64_t cell = cg[s].cbase + cell_of[i];
    int slot = atomicAdd(&cell_fill[cell], 1);
    cell_atoms[cell_start[cell] + slot] = (int)(i - atom_off[s]);
}

// exclusive scan of n ints into n+1 int64 (single block; set-up only).  mult scales every input.
__global__ void k_scan_excl(const int* __restrict__ in, int64_t* __restrict__ out, int64_t n, int mult)
{
    __shared__ int64_t part[1024];
    int t = threadIdx.x;
    int64_t chunk = (n + blockDim.x - 1) / blockDim.x;
    int64_t b = t * chunk, e = min(b + chunk, n);
    int64_t s = 0;
    for (int64_t i = b; i < e; ++i) s += (int64_t)in[i] * mult;
    part[t] = s;
    __syncthreads();
    if (t == 0) {
        int64_t run = 0;
        for (int k = 0; k < blockDim.x; ++k) { int64_t v = part[k]; part[k] = run; run += v; }
        out[n] = run;
    }
    __syncthreads();
    s = part[t];
    for (int64_t i = b; i < e; ++i) { out[i] = s; s += (int64_t)in[i] * mult; }
}

// One warp per atom.  MODE 0: count radial / angular neighbours.  MODE 1: emit unsorted 64-bit keys.
// key = j << 25 | (na+64) << 18 | (nb+64) << 11 | (nc+64) << 4 | isAngular
template <int MODE>
__global__ void k_nbr_traverse(int64_t N, const double* __restrict__ pos, const double* __restrict__ box,
                               const int* __restrict__ atom_struct, const int64_t* __restrict__ atom_off,
                               const CellGeom* __restrict__ cg, const int* __restrict__ cell_of,
                               const int64_t* __restrict__ cell_start, const int* __restrict__ cell_atoms,
                               double rcR2, double rcA2, int* __restrict__ cntR, int* __restrict__ cntA,
                               const int64_t* __restrict__ offR, unsigned long long* __restrict__ keys)
{
    int64_t ig = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) / WARP;
    int lane = threadIdx.x & 31;
    if (ig >= N) return;
    int s = atom_struct[ig];
    const CellGeom& g = cg[s];
    int64_t a0 = atom_off[s];
    int il = (int)(ig - a0);
    double bx[9], ri[3];
#pragma unroll
    for (int k = 0; k < 9; ++k) bx[k] = box[9 * (int64_t)s + k];
#pragma unroll
    for (int k = 0; k < 3; ++k) ri[k] = pos[3 * ig + k];
    int cell = cell_of[ig];
    int cz = cell % g.nc[2], cy = (cell / g.nc[2]) % g.nc[1], cx = cell / (g.nc[2] * g.nc[1]);
    int nR = 0, nA = 0;
    int64_t wbase = (MODE == 1) ? offR[ig] : 0;
    for (int ox = -g.m[0]; ox <= g.m[0]; ++ox) {
        int gx = cx + ox, na = floordiv(gx, g.nc[0]), wx = gx - na * g.nc[0];
        for (int oy = -g.m[1]; oy <= g.m[1]; ++oy) {
            int gy = cy + oy, nb = floordiv(gy, g.nc[1]), wy = gy - nb * g.nc[1];
            for (int oz = -g.m[2]; oz <= g.m[2]; ++oz) {
                int gz = cz + oz, nc = floordiv(gz, g.nc[2]), wz = gz - nc * g.nc[2];
                int64_t cj = g.cbase + (wx * g.nc[1] + wy) * g.nc[2] + wz;
                int64_t b = cell_start[cj], e = cell_start[cj + 1];
                for (int64_t p0 = b; p0 < e; p0 += WARP) {
                    int64_t p = p0 + lane;
                    bool hitR = false, hitA = false;
                    int jl = 0;
                    if (p < e) {
                        jl = cell_atoms[p];
                        double rj[3] = { pos[3 * (a0 + jl)], pos[3 * (a0 + jl) + 1], pos[3 * (a0 + jl) + 2] }, d[3];
                        bond_rn(ri, rj, bx, na, nb, nc, d);
                        double r2 = norm2_rn(d);
                        bool self = (jl == il) && na == 0 && nb == 0 && nc == 0;
                        hitR = (r2 < rcR2) && !self;
                        hitA = (r2 < rcA2) && !self;
                    }
                    unsigned mR = __ballot_sync(0xffffffffu, hitR);
                    if (MODE == 0) {
                        nR += __popc(mR);
                        nA += __popc(__ballot_sync(0xffffffffu, hitA));
                    } else {
                        if (hitR) {
                            int64_t w = wbase + __popc(mR & ((1u << lane) - 1u));
                            keys[w] = ((unsigned long long)jl << 25) | ((unsigned long long)(na + 64) << 18) |
                                      ((unsigned long long)(nb + 64) << 11) | ((unsigned long long)(nc + 64) << 4) | (hitA ? 1ull : 0ull);
                        }
                        wbase += __popc(mR);
                    }
                }
            }
        }
    }
    if (MODE == 0 && lane == 0) { cntR[ig] = nR; cntA[ig] = nA; }
}

// One warp per atom: rank sort of the atom's keys -> canonical lists (radial: all; angular: flagged subset)
__global__ void k_nbr_sort(int64_t N, const unsigned long long* __restrict__ keys, const int64_t* __restrict__ offR,
                           const int64_t* __restrict__ offA, int* __restrict__ jR, signed char* __restrict__ shR,
                           int* __restrict__ jA, signed char* __restrict__ shA)
{
    int64_t ig = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) / WARP;
    int lane = threadIdx.x & 31;
    if (ig >= N) return;
    int64_t b = offR[ig], e = offR[ig + 1], bA = offA[ig];
    for (int64_t p = b + lane; p < e; p += WARP) {
        unsigned long long k = keys[p];
        int rank = 0, rankA = 0;
        for (int64_t q = b; q < e; ++q) {
            unsigned long long kq = keys[q];
            bool less = kq < k;
            rank += less;
            rankA += less && (kq & 1ull);
        }
        int j = (int)(k >> 25);
        signed char s0 = (signed char)((int)((k >> 18) & 127) - 64), s1 = (signed char)((int)((k >> 11) & 127) - 64),
                    s2 = (signed char)((int)((k >> 4) & 127) - 64);
        int64_t w = b + rank;
        jR[w] = j; shR[3 * w] = s0; shR[3 * w + 1] = s1; shR[3 * w + 2] = s2;
        if (k & 1ull) {
            int64_t wa = bA + rankA;
            jA[wa] = j; shA[3 * wa] = s0; shA[3 * wa + 1] = s1; shA[3 * wa + 2] = s2;
        }
    }
}

// per padded atom: neighbour counts (0 for padding); per slice: width = max count
__global__ void k_slice_width(int nslices, const int64_t* __restrict__ pbase, const int64_t* __restrict__ atom_off,
                              const int* __restrict__ slice_struct, const int* __restrict__ orig_p,
                              const int64_t* __restrict__ off, int* __restrict__ cnt_p, int* __restrict__ width)
{
    int sl = (blockIdx.x * blockDim.x + threadIdx.x) / WARP, lane = threadIdx.x & 31;
    if (sl >= nslices) return;
    int64_t ip = (int64_t)sl * WARP + lane;
    int s = slice_struct[sl];
    int c = 0;
    if (orig_p[ip] >= 0) {
        int64_t ig = atom_off[s] + orig_p[ip];
        c = (int)(off[ig + 1] - off[ig]);
    }
    cnt_p[ip] = c;
    int w = c;
#pragma unroll
    for (int o = 16; o; o >>= 1) w = max(w, __shfl_xor_sync(0xffffffffu, w, o));
    if (lane == 0) width[sl] = w;
}

// fp64 radial basis for the one-time aggregate (Eqs. 17-18)
__device__ void basis_f64(double r, double rc, int K, double* f)
{
    double u = r / rc, fc = 0.5 * (cospi(u) + 1.0), x = 2.0 * (u - 1.0) * (u - 1.0) - 1.0;
    double T2 = 1.0, T1 = x;
    f[0] = fc;
    if (K > 1) f[1] = 0.5 * (x + 1.0) * fc;
    for (int k = 2; k < K; ++k) { double T = 2.0 * x * T1 - T2; T2 = T1; T1 = T; f[k] = 0.5 * (T + 1.0) * fc; }
}

// One thread per padded atom: writes the atom's pair records sorted by neighbour type (stable in canonical order),
// record = (dx, dy, dz, bits) with bits = j_local | t_j << 24.  RADIAL also accumulates B_k[T'] in fp64
// (slice-blocked: B[slice][T' * KR + k][lane]).
template <bool RADIAL>
__global__ void k_cache_fill(int nslices, ModelDev m, const double* __restrict__ pos, const double* __restrict__ box,
                             const int* __restrict__ type, const int64_t* __restrict__ pbase, const int64_t* __restrict__ atom_off,
                             const int* __restrict__ slice_struct, const int* __restrict__ orig_p, const int* __restrict__ slot_of,
                             const int64_t* __restrict__ off, const int* __restrict__ nj, const signed char* __restrict__ sh,
                             const int64_t* __restrict__ recoff, float4* __restrict__ rec, float* __restrict__ B, int64_t NP)
{
    int sl = (blockIdx.x * blockDim.x + threadIdx.x) / WARP, lane = threadIdx.x & 31;
    if (sl >= nslices) return;
    int64_t ip = (int64_t)sl * WARP + lane;
    if (orig_p[ip] < 0) {
        if (RADIAL) for (int k = 0; k < m.T * m.KR; ++k) B[((int64_t)sl * m.T * m.KR + k) * WARP + lane] = 0.0f;
        return;
    }
    int s = slice_struct[sl];
    int64_t a0 = atom_off[s];
    int il = orig_p[ip];
    int64_t ig = a0 + il;
    double bx[9], ri[3];
    for (int k = 0; k < 9; ++k) bx[k] = box[9 * (int64_t)s + k];
    for (int k = 0; k < 3; ++k) ri[k] = pos[3 * ig + k];
    int64_t b = off[ig], e = off[ig + 1];
    float4* out = rec + recoff[sl] + lane;
    int slot = 0;
    for (int t = 0; t < m.T; ++t) {
        double acc[17];
        for (int k = 0; k < 17; ++k) acc[k] = 0.0;
        for (int64_t p = b; p < e; ++p) {
            int jl = nj[p];
            if (type[a0 + jl] != t) continue;
            double rj[3] = { pos[3 * (a0 + jl)], pos[3 * (a0 + jl) + 1], pos[3 * (a0 + jl) + 2] }, d[3];
            bond_rn(ri, rj, bx, sh[3 * p], sh[3 * p + 1], sh[3 * p + 2], d);
            out[(int64_t)slot * WARP] = make_float4((float)d[0], (float)d[1], (float)d[2], __int_as_float(slot_of[a0 + jl] | (t << 24)));
            ++slot;
            if (RADIAL) {
                double f[17];
                basis_f64(sqrt(norm2_rn(d)), (double)m.rcR, m.KR, f);   // rcR as float->double: same value the step kernels use
                for (int k = 0; k < m.KR; ++k) acc[k] += f[k];
            }
        }
        if (RADIAL) for (int k = 0; k < m.KR; ++k) B[((int64_t)sl * m.T * m.KR + t * m.KR + k) * WARP + lane] = (float)acc[k];
    }
}

// ------------------------------------------------------------------------------------------------
// Half list of the radial pairs (one record per UNDIRECTED pair) for the radial force sweep: the pair (i, j, n) and its mirror
// (j, i, -n) share f_k'(r), so one thread evaluates the basis once, forms s_ij + s_ji and scatters the reaction to j.
// Owner of a pair: for i != j the atom with the smaller slot if i + j is odd, the larger one if it is even (every atom keeps about
// half of its pairs); a self-image pair (i, i, n) is kept for the image whose bond vector is lexicographically positive (its mirror
// has exactly the negated vector).  Records keep their order (sorted by neighbour type).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool owns_pair(int i, const float4& rec)
{
    const int j = __float_as_int(rec.w) & 0xffffff;
    if (j != i) return ((i + j) & 1) ? (i < j) : (i > j);
    return rec.x > 0.0f || (rec.x == 0.0f && (rec.y > 0.0f || (rec.y == 0.0f && rec.z > 0.0f)));
}
template <bool FILL>
__global__ void k_half_list(int nslices, const int64_t* __restrict__ pbase, const int* __restrict__ slice_struct, const int* __restrict__ cnt,
                            const int64_t* __restrict__ recoff, const float4* __restrict__ rec, int* __restrict__ cntH, int* __restrict__ widthH,
                            const int64_t* __restrict__ recoffH, float4* __restrict__ recH)
{
    const int sl = (int)((blockIdx.x * blockDim.x + threadIdx.x) / WARP), lane = threadIdx.x & 31;
    if (sl >= nslices) return;
    const int64_t ip = (int64_t)sl * WARP + lane;
    const int i = (int)(ip - pbase[slice_struct[sl]]);
    const int n = cnt[ip];
    const float4* r4 = rec + recoff[sl] + lane;
    float4* out = FILL ? recH + recoffH[sl] + lane : nullptr;
    int c = 0;
    for (int s = 0; s < n; ++s) {
        const float4 r = r4[(int64_t)s * WARP];
        if (owns_pair(i, r)) {
            if (FILL) out[(int64_t)c * WARP] = r;
            ++c;
        }
    }
    if (!FILL) {
        cntH[ip] = c;
        int w = c;
#pragma unroll
        for (int o = 16; o; o >>= 1) w = max(w, __shfl_xor_sync(0xffffffffu, w, o));
        if (lane == 0) widthH[sl] = w;
    }
}

static int scan_excl(nep_ctx* c, const int* in, int64_t* out, int64_t n, int mult)
{
    prof_begin(c, "k_scan_excl");
    k_scan_excl<<<1, 1024, 0, c->stream>>>(in, out, n, mult);
    prof_end(c);
    NEP_CUDA(c, cudaGetLastError());
    return NEP_OK;
}

#define DALLOC(ptr, type, count)                                                \
    type* ptr = (type*)dev_alloc(c, sizeof(type) * (size_t)std::max<int64_t>((int64_t)(count), 1)); \
    if (!ptr) return NEP_ENOMEM;

int build_neighbors_dev(nep_ctx* c)
{
    DataDev& d = c->d;
    const ModelDev& m = c->m;
    const int S = c->S;
    const int64_t N = c->N;
    // release lists of a previous build
    {
        const void* ptrs[] = { d.offR, d.jR, d.shR, d.offA, d.jA, d.shA, d.cntR, d.recoffR, d.recR, d.cntA, d.recoffA, d.recA, d.B,
                               d.cntH, d.recoffH, d.recH };
        for (const void* p : ptrs) dev_free(c, const_cast<void*>(p));
        d.offR = d.offA = nullptr; d.jR = d.jA = nullptr; d.shR = d.shA = nullptr; d.cntR = d.cntA = nullptr;
        d.recoffR = d.recoffA = nullptr; d.recR = d.recA = nullptr; d.B = nullptr;
        d.cntH = nullptr; d.recoffH = nullptr; d.recH = nullptr;
        c->have_nbrs = false;
    }
    // ---- host: cell geometry per structure ----
    std::vector<CellGeom> cg(S);
    std::vector<int> atom_struct((size_t)N);
    int64_t ncells = 0;
    for (int s = 0; s < S; ++s) {
        const double* b = &c->h_box[9 * (size_t)s];
        double det = b[0] * (b[4] * b[8] - b[5] * b[7]) - b[1] * (b[3] * b[8] - b[5] * b[6]) + b[2] * (b[3] * b[7] - b[4] * b[6]);
        CellGeom& g = cg[s];
        double inv[9] = { (b[4] * b[8] - b[5] * b[7]) / det, (b[2] * b[7] - b[1] * b[8]) / det, (b[1] * b[5] - b[2] * b[4]) / det,
                          (b[5] * b[6] - b[3] * b[8]) / det, (b[0] * b[8] - b[2] * b[6]) / det, (b[2] * b[3] - b[0] * b[5]) / det,
                          (b[3] * b[7] - b[4] * b[6]) / det, (b[1] * b[6] - b[0] * b[7]) / det, (b[0] * b[4] - b[1] * b[3]) / det };
        for (int k = 0; k < 9; ++k) g.inv[k] = inv[k];
        for (int k = 0; k < 3; ++k) {
            // perpendicular thickness h_k = 1 / |k-th column of inv|
            double nrm = sqrt(inv[k] * inv[k] + inv[3 + k] * inv[3 + k] + inv[6 + k] * inv[6 + k]);
            double h = 1.0 / nrm;
            int nc = (int)floor(h / c->rcR);
            nc = std::max(1, std::min(nc, 32));
            g.nc[k] = nc;
            // |delta cell| <= floor(rc nc / h) + 1 (S0a); tiny slack against rounding of h
            g.m[k] = (int)floor(c->rcR * nc / h * (1.0 + 1e-9) + 1e-9) + 1;
            int images = (g.m[k] + nc) / nc + 1;
            if (images > 60) return fail(c, NEP_ECAPACITY, "box of structure " + std::to_string(s) + " is thinner than rc_R/60");
        }
        g.cbase = ncells;
        ncells += (int64_t)g.nc[0] * g.nc[1] * g.nc[2];
        if (c->h_nat[s] >= (1 << 24)) return fail(c, NEP_ECAPACITY, "structure with >= 2^24 atoms");
        for (int64_t i = c->h_aoff[s]; i < c->h_aoff[s + 1]; ++i) atom_struct[i] = s;
    }
    if (N == 0) {   // empty set: empty lists
        DALLOC(o1, int64_t, 1); DALLOC(o2, int64_t, 1); DALLOC(r1, int64_t, 1); DALLOC(r2, int64_t, 1);
        NEP_CUDA(c, cudaMemsetAsync(o1, 0, 8, c->stream)); NEP_CUDA(c, cudaMemsetAsync(o2, 0, 8, c->stream));
        NEP_CUDA(c, cudaMemsetAsync(r1, 0, 8, c->stream)); NEP_CUDA(c, cudaMemsetAsync(r2, 0, 8, c->stream));
        d.offR = o1; d.offA = o2; d.recoffR = r1; d.recoffA = r2; c->PR = c->PA = 0;
        c->h_pairsR_struct.assign(S, 0); c->h_pairsA_struct.assign(S, 0);
        return NEP_OK;
    }
    DALLOC(d_cg, CellGeom, S); DALLOC(d_as, int, N); DALLOC(d_cell_of, int, N);
    DALLOC(d_cell_cnt, int, ncells); DALLOC(d_cell_fill, int, ncells); DALLOC(d_cell_start, int64_t, ncells + 1);
    DALLOC(d_cell_atoms, int, N); DALLOC(d_cR, int, N); DALLOC(d_cA, int, N);
    NEP_CUDA(c, cudaMemcpyAsync(d_cg, cg.data(), sizeof(CellGeom) * S, cudaMemcpyHostToDevice, c->stream));
    NEP_CUDA(c, cudaMemcpyAsync(d_as, atom_struct.data(), 4 * (size_t)N, cudaMemcpyHostToDevice, c->stream));
    NEP_CUDA(c, cudaMemsetAsync(d_cell_cnt, 0, 4 * (size_t)ncells, c->stream));
    NEP_CUDA(c, cudaMemsetAsync(d_cell_fill, 0, 4 * (size_t)ncells, c->stream));
    const int TB = 256;
    const unsigned gN = (unsigned)((N + TB - 1) / TB), gW = (unsigned)((N * WARP + TB - 1) / TB);
    prof_begin(c, "k_bin_count");
    k_bin_count<<<gN, TB, 0, c->stream>>>(N, d.pos, d_as, d_cg, d_cell_of, d_cell_cnt);
    prof_end(c);
    int rc;
    if ((rc = scan_excl(c, d_cell_cnt, d_cell_start, ncells, 1))) return rc;
    prof_begin(c, "k_bin_fill");
    k_bin_fill<<<gN, TB, 0, c->stream>>>(N, d_as, d.atom_off, d_cg, d_cell_of, d_cell_start, d_cell_fill, d_cell_atoms);
    prof_end(c);
    const double rcR2 = c->rcR * c->rcR, rcA2 = c->rcA * c->rcA;
    prof_begin(c, "k_nbr_count");
    k_nbr_traverse<0><<<gW, TB, 0, c->stream>>>(N, d.pos, d.box, d_as, d.atom_off, d_cg, d_cell_of, d_cell_start, d_cell_atoms,
                                               rcR2, rcA2, d_cR, d_cA, nullptr, nullptr);
    prof_end(c);
    DALLOC(offR, int64_t, N + 1); DALLOC(offA, int64_t, N + 1);
    if ((rc = scan_excl(c, d_cR, offR, N, 1))) return rc;
    if ((rc = scan_excl(c, d_cA, offA, N, 1))) return rc;
    std::vector<int64_t> hoR((size_t)N + 1), hoA((size_t)N + 1);
    NEP_CUDA(c, cudaMemcpyAsync(hoR.data(), offR, 8 * (size_t)(N + 1), cudaMemcpyDeviceToHost, c->stream));
    NEP_CUDA(c, cudaMemcpyAsync(hoA.data(), offA, 8 * (size_t)(N + 1), cudaMemcpyDeviceToHost, c->stream));
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    const int64_t PR = hoR[N], PA = hoA[N];
    c->h_pairsR_struct.resize(S); c->h_pairsA_struct.resize(S);
    for (int s = 0; s < S; ++s) {
        c->h_pairsR_struct[s] = hoR[c->h_aoff[s + 1]] - hoR[c->h_aoff[s]];
        c->h_pairsA_struct[s] = hoA[c->h_aoff[s + 1]] - hoA[c->h_aoff[s]];
    }
    // slot order inside every structure: (species, angular neighbour count descending, caller's index)
    {
        std::vector<int> order;
        for (int s = 0; s < S; ++s) {
            const int64_t a0 = c->h_aoff[s];
            const int n = c->h_nat[s];
            order.resize(n);
            for (int i = 0; i < n; ++i) order[i] = i;
            std::sort(order.begin(), order.end(), [&](int x, int y) {
                const int tx = c->h_type[a0 + x], ty = c->h_type[a0 + y];
                if (tx != ty) return tx < ty;
                const int64_t cx = hoA[a0 + x + 1] - hoA[a0 + x], cy = hoA[a0 + y + 1] - hoA[a0 + y];
                if (cx != cy) return cx > cy;
                return x < y;
            });
            for (int sl = 0; sl < n; ++sl) c->h_slot_of[a0 + order[sl]] = sl;
        }
        if ((rc = upload_slot_tables(c))) return rc;
    }
    DALLOC(keys, unsigned long long, PR);
    DALLOC(jR, int, PR); DALLOC(shR, signed char, 3 * PR); DALLOC(jA, int, PA); DALLOC(shA, signed char, 3 * PA);
    prof_begin(c, "k_nbr_fill");
    k_nbr_traverse<1><<<gW, TB, 0, c->stream>>>(N, d.pos, d.box, d_as, d.atom_off, d_cg, d_cell_of, d_cell_start, d_cell_atoms,
                                               rcR2, rcA2, nullptr, nullptr, offR, keys);
    prof_end(c);
    prof_begin(c, "k_nbr_sort");
    k_nbr_sort<<<gW, TB, 0, c->stream>>>(N, keys, offR, offA, jR, shR, jA, shA);
    prof_end(c);
    NEP_CUDA(c, cudaGetLastError());
    d.offR = offR; d.offA = offA; d.jR = jR; d.shR = shR; d.jA = jA; d.shA = shA;
    c->PR = PR; c->PA = PA;

    // ---- S0b: sliced pair cache + radial aggregate ----
    const int ns = c->nslices;
    const unsigned gS = (unsigned)(((int64_t)ns * WARP + TB - 1) / TB);
    DALLOC(cntRp, int, c->NP); DALLOC(cntAp, int, c->NP); DALLOC(wR, int, ns); DALLOC(wA, int, ns);
    DALLOC(recoffR, int64_t, ns + 1); DALLOC(recoffA, int64_t, ns + 1);
    prof_begin(c, "k_slice_width");
    k_slice_width<<<gS, TB, 0, c->stream>>>(ns, d.pbase, d.atom_off, d.slice_struct, d.orig_p, offR, cntRp, wR);
    prof_end(c);
    prof_begin(c, "k_slice_width");
    k_slice_width<<<gS, TB, 0, c->stream>>>(ns, d.pbase, d.atom_off, d.slice_struct, d.orig_p, offA, cntAp, wA);
    prof_end(c);
    if ((rc = scan_excl(c, wR, recoffR, ns, WARP))) return rc;
    if ((rc = scan_excl(c, wA, recoffA, ns, WARP))) return rc;
    int64_t totR = 0, totA = 0;
    NEP_CUDA(c, cudaMemcpyAsync(&totR, recoffR + ns, 8, cudaMemcpyDeviceToHost, c->stream));
    NEP_CUDA(c, cudaMemcpyAsync(&totA, recoffA + ns, 8, cudaMemcpyDeviceToHost, c->stream));
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    DALLOC(recR, float4, totR); DALLOC(recA, float4, totA); DALLOC(B, float, (int64_t)m.T * m.KR * c->NP);
    NEP_CUDA(c, cudaMemsetAsync(recR, 0, 16 * (size_t)std::max<int64_t>(totR, 1), c->stream));
    NEP_CUDA(c, cudaMemsetAsync(recA, 0, 16 * (size_t)std::max<int64_t>(totA, 1), c->stream));
    prof_begin(c, "k_cache_fill_R");
    k_cache_fill<true><<<gS, TB, 0, c->stream>>>(ns, m, d.pos, d.box, d.type, d.pbase, d.atom_off, d.slice_struct, d.orig_p, d.slot_of,
                                                offR, jR, shR, recoffR, recR, B, c->NP);
    prof_end(c);
    prof_begin(c, "k_cache_fill_A");
    k_cache_fill<false><<<gS, TB, 0, c->stream>>>(ns, m, d.pos, d.box, d.type, d.pbase, d.atom_off, d.slice_struct, d.orig_p, d.slot_of,
                                                 offA, jA, shA, recoffA, recA, nullptr, c->NP);
    prof_end(c);
    NEP_CUDA(c, cudaGetLastError());
    // half list of the radial pairs
    DALLOC(cntHp, int, c->NP); DALLOC(wH, int, ns); DALLOC(recoffH, int64_t, ns + 1);
    prof_begin(c, "k_half_list");
    k_half_list<false><<<gS, TB, 0, c->stream>>>(ns, d.pbase, d.slice_struct, cntRp, recoffR, recR, cntHp, wH, nullptr, nullptr);
    prof_end(c);
    if ((rc = scan_excl(c, wH, recoffH, ns, WARP))) return rc;
    int64_t totH = 0;
    NEP_CUDA(c, cudaMemcpyAsync(&totH, recoffH + ns, 8, cudaMemcpyDeviceToHost, c->stream));
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    DALLOC(recH, float4, totH);
    NEP_CUDA(c, cudaMemsetAsync(recH, 0, 16 * (size_t)std::max<int64_t>(totH, 1), c->stream));
    prof_begin(c, "k_half_list");
    k_half_list<true><<<gS, TB, 0, c->stream>>>(ns, d.pbase, d.slice_struct, cntRp, recoffR, recR, nullptr, nullptr, recoffH, recH);
    prof_end(c);
    NEP_CUDA(c, cudaGetLastError());
    NEP_CUDA(c, cudaStreamSynchronize(c->stream));
    dev_free(c, wH);
    d.cntR = cntRp; d.cntA = cntAp; d.recoffR = recoffR; d.recoffA = recoffA; d.recR = recR; d.recA = recA; d.B = B;
    d.cntH = cntHp; d.recoffH = recoffH; d.recH = recH;
    void* temps[] = { d_cg, d_as, d_cell_of, d_cell_cnt, d_cell_fill, d_cell_start, d_cell_atoms, d_cR, d_cA, keys, wR, wA };
    for (void* p : temps) dev_free(c, p);
    return NEP_OK;
}

}  // namespace nep
