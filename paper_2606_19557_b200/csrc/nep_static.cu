// nep_static.cu -- nep_scaler_static: the descriptor scaler of Eq. 2 for callers that cannot hand this library an allocator.
//
// Everything else in libnep_b200 works on a context, and a context is built from the caller's nep_alloc_fn / nep_free_fn: the
// library itself never allocates device memory.  Some programs that want the scaler have no such callbacks to offer and may not
// call cudaMalloc either:
//   - a molecular-dynamics or training host whose framework reserved (nearly) all of the GPU's memory in its own pool at start-up
//     and hands out fixed buffers only, so that a cudaMalloc from a plug-in fails or steals from the pool's head-room;
//   - a caller in the middle of stream-ordered work that must not stall: cudaMalloc / cudaFree synchronise the whole device;
//   - a plain C or Fortran caller that holds two device pointers (its descriptor matrix and a place for the result) and nothing else.
// For them this one call computes s_v = 1 / (max_i q_v^i - min_i q_v^i) from a descriptor matrix that is already on the device.
// The kernel is the two-level form of k_descriptor_range + k_scaler_from_range (nep_misc.cu): per-block minima and maxima go to
// scratch memory, the last block to finish combines them.  In the context path that scratch comes from the allocator; here it is
// the file-scope array below, which is part of the library's image: every GPU on which the library's code is loaded holds its
// NEP_STATIC_SCRATCH_BYTES until the process exits, whether this call is ever used or not.
//
// Rules that follow from the fixed array (also in include/nep.h):
//   - n_desc <= NEP_STATIC_MAX_DESCRIPTORS, otherwise NEP_ECAPACITY (nothing is launched);
//   - all calls on one device share the array: two calls whose kernels may overlap on that GPU (different streams, different
//     host threads) race on it -- serialise them;
//   - the array keeps what the previous call left.  The per-block slots are overwritten before they are read (a call reads only
//     the slots of its own blocks); the block ticket must start at zero and is cleared on the caller's stream before every launch;
//   - the first call on a device looks the array's device address up (cudaGetSymbolAddress) and caches it; make that first call
//     outside any stream capture.
// No cudaMalloc, cudaFree, cudaMallocAsync or allocating library routine is called on this path.
#include <cuda_runtime.h>
#include <math.h>

#include <mutex>
#include <string>

#include "nep_internal.h"

namespace nep {

constexpr int STATIC_MAX_D = NEP_STATIC_MAX_DESCRIPTORS;
constexpr int STATIC_MAX_BLOCKS = 296;       // two blocks per SM of a B200; the grid never exceeds this, whatever the row count
constexpr int STATIC_THREADS = 256;

struct StaticScratch {
    float lo[STATIC_MAX_BLOCKS][STATIC_MAX_D];   // minimum of column v over the rows block b walked
    float hi[STATIC_MAX_BLOCKS][STATIC_MAX_D];   // maximum
    unsigned ticket;                             // blocks that have written their slots (zero before a launch)
    unsigned pad[63];
};
static_assert(sizeof(StaticScratch) == NEP_STATIC_SCRATCH_BYTES, "include/nep.h states the size of the resident array");

// The resident scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress, not a device address.
static __device__ __align__(256) unsigned char g_static_scratch[sizeof(StaticScratch)];

// q [n][D] row-major.  The first nt = (256 / D) * D threads of a block are used, so that a thread keeps ONE column (tid % D) while
// consecutive threads read consecutive floats: coalesced without a per-element modulo.  Block b walks rows b*rpb, b*rpb + gridDim*rpb, ...
__global__ void __launch_bounds__(STATIC_THREADS) k_scaler_static(const float* __restrict__ q, long long n, int D, float* __restrict__ s,
                                                                  StaticScratch* sc)
{
    const int rpb = STATIC_THREADS / D;          // rows per block and pass
    const int nt = rpb * D;
    const int tid = threadIdx.x;
    const int col = tid % D;
    float lo = INFINITY, hi = -INFINITY;
    if (tid < nt) {
        for (long long r = (long long)blockIdx.x * rpb + tid / D; r < n; r += (long long)gridDim.x * rpb) {
            const float x = __ldg(q + r * D + col);
            lo = fminf(lo, x); hi = fmaxf(hi, x);
        }
    }
    __shared__ float slo[STATIC_THREADS], shi[STATIC_THREADS];
    __shared__ bool last;
    slo[tid] = lo; shi[tid] = hi;
    __syncthreads();
    if (tid < D) {
        for (int k = 1; k < rpb; ++k) { lo = fminf(lo, slo[tid + k * D]); hi = fmaxf(hi, shi[tid + k * D]); }
        sc->lo[blockIdx.x][tid] = lo; sc->hi[blockIdx.x][tid] = hi;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) last = (atomicAdd(&sc->ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!last) return;
    __threadfence();
    if (tid < D) {
        lo = INFINITY; hi = -INFINITY;
        for (unsigned b = 0; b < gridDim.x; ++b) { lo = fminf(lo, __ldcg(&sc->lo[b][tid])); hi = fmaxf(hi, __ldcg(&sc->hi[b][tid])); }
        // Eq. 2; a component without a range gets s = 1 -- the same rule, in the same arithmetic, as k_scaler_from_range
        const float range = hi - lo, am = fmaxf(fabsf(lo), fabsf(hi));
        s[tid] = (hi >= lo && isfinite(range) && range > 64.0f * 1.1920929e-7f * fmaxf(1e-4f, am)) ? 1.0f / range : 1.0f;
    }
    if (tid == 0) sc->ticket = 0u;
}

// Device address of g_static_scratch on the CURRENT device, looked up once per device.
static int static_scratch_ptr(StaticScratch** out)
{
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static StaticScratch* ptr[MAX_DEV] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, NEP_ECUDA, std::string("nep_scaler_static: cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= MAX_DEV) return fail(nullptr, NEP_ECAPACITY, "nep_scaler_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p)
            return fail(nullptr, NEP_ECUDA, std::string("nep_scaler_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        ptr[dev] = static_cast<StaticScratch*>(p);
    }
    *out = ptr[dev];
    return NEP_OK;
}

}  // namespace nep

extern "C" int nep_scaler_static(const float* q_dev, int64_t n_atoms, int n_desc, float* s_dev, void* cuda_stream)
{
    using namespace nep;
    if (n_desc < 1) return fail(nullptr, NEP_EINVAL, "nep_scaler_static: n_desc must be >= 1");
    if (n_desc > STATIC_MAX_D)
        return fail(nullptr, NEP_ECAPACITY, "nep_scaler_static: n_desc = " + std::to_string(n_desc) + " exceeds NEP_STATIC_MAX_DESCRIPTORS = " +
                                                std::to_string(STATIC_MAX_D) + " (the resident scratch array has a fixed size; use a context and nep_compute_scaler)");
    if (n_atoms < 0) return fail(nullptr, NEP_EINVAL, "nep_scaler_static: n_atoms must be >= 0");
    if (!s_dev || (n_atoms > 0 && !q_dev)) return fail(nullptr, NEP_EINVAL, "nep_scaler_static: NULL device pointer");
    StaticScratch* sc = nullptr;
    if (int rc = static_scratch_ptr(&sc)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int rpb = STATIC_THREADS / n_desc;
    long long blocks = (n_atoms + rpb - 1) / rpb;
    if (blocks < 1) blocks = 1;                        // no rows: every range is empty, s = 1
    if (blocks > STATIC_MAX_BLOCKS) blocks = STATIC_MAX_BLOCKS;
    cudaError_t e = cudaMemsetAsync(&sc->ticket, 0, sizeof(unsigned), st);   // a launch that died earlier may have left a count
    if (e != cudaSuccess) return fail(nullptr, NEP_ECUDA, std::string("nep_scaler_static: cudaMemsetAsync: ") + cudaGetErrorString(e));
    k_scaler_static<<<(unsigned)blocks, STATIC_THREADS, 0, st>>>(q_dev, (long long)n_atoms, n_desc, s_dev, sc);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, NEP_ECUDA, std::string("nep_scaler_static: launch: ") + cudaGetErrorString(e));
    return NEP_OK;
}
