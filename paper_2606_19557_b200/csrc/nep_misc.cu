// nep_misc.cu -- S6 (loss and its seeds, Eqs. 4-7) in one kernel, the type-sorted atom list of the batch,
// the descriptor scaler (S0c, Eq. 2) and the re-ordering of outputs from the slice-blocked layout to batch order.
#include <algorithm>

#include "nep_kernels.cuh"

namespace nep {

// ------------------------------------------------------------------------------------------------
// S6.  thread = batch-padded atom: u_i = dL/dF_i = 2 lF (F_i - F_i^lab) / (3 N_b), sum |dF|^2          (Eq. 6)
//      thread < S_b also = structure: eps_s = dL/dE_s, G_s = dL/dW_s, sums of (dE/N)^2, (dW/N)^2       (Eqs. 5, 7)
//      every thread clears its share of g (the sweeps that follow accumulate into it);
//      the last block to finish forms L (Eq. 4) and g_b1 = -sum_s eps_s N_s, and re-arms the accumulators.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_loss(StepArgs a, float lamE, float lamF, float lamV, double dlamE, double dlamF, double dlamV)
{
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    const int nthreads = gridDim.x * blockDim.x;
    for (int i = gid; i < a.m.npar; i += nthreads) a.g[i] = 0.0f;
    double sF = 0.0, sE = 0.0, sW = 0.0, sB = 0.0;
    // grid-stride: at most two blocks per SM, so that the same-address atomics below number a few hundred, not one set per 256 atoms
    for (int64_t ia = gid; ia < a.b.NBP; ia += nthreads) {
        const int w = (int)(ia >> 5), lane = (int)(ia & 31);
        const int4 bi = __ldg(a.b.binfo + w);
        const float c = (float)(2.0 * dlamF / (3.0 * a.b.nrmN));
        const float4 F4 = reinterpret_cast<const float4*>(a.b.F)[ia];
        const float Fp[3] = { F4.x, F4.y, F4.z };
        const float* Fl = sb_ptr(a.d.Flab, bi.x, 3, lane);
        float* up = sb_ptr(a.b.u, w, 3, lane);
        float s2 = 0.0f;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const float dF = Fp[k] - __ldg(Fl + k * WARP);   // padding slots hold 0 in both (no type lookup on this path)
            s2 = fmaf(dF, dF, s2);
            up[k * WARP] = c * dF;
        }
        sF += (double)s2;
    }
    // one fp64 division per structure (1 / N_s): a chain of ~40 of them per thread was the critical path of this kernel
    const double cE = a.b.nrmS > 0.0 ? 2.0 * dlamE / a.b.nrmS : 0.0, cV = a.b.nrmV > 0.0 ? 2.0 * dlamV / (9.0 * a.b.nrmV) : 0.0;
    for (int sb = gid; sb < a.b.Sb; sb += nthreads) {
        const int sid = a.b.bsid[sb];
        const double n = (double)a.b.bnat[sb];
        const double rn = 1.0 / n, rn2 = rn * rn;
        const double dE = a.b.Es[sb] - a.d.Elab[sid];
        sE += dE * dE * rn2;                                                        // Eq. 5
        const float eps = (float)(cE * dE * rn2);
        a.b.eps[sb] = eps;
        sB += (double)eps * n;
        const bool hv = a.d.hasv[sid] != 0;
#pragma unroll
        for (int k = 0; k < 9; ++k) {
            const double t = hv ? (double)a.b.Ws[9 * sb + k] - (double)a.d.Wlab[9 * (size_t)sid + k] : 0.0;
            sW += t * t * rn2;                                                      // Eq. 7
            a.b.G[9 * sb + k] = hv ? (float)(cV * t * rn2) : 0.0f;
        }
    }
    // block reduction -> the block's four partial sums go to its own slot (no same-address floating-point atomics: a few
    // hundred of those on one address cost ~10 us); the last block to finish (ticket) adds the slots in a fixed order
    __shared__ double red[4][8];
    __shared__ bool last;
    sF = warp_sum(sF); sE = warp_sum(sE); sW = warp_sum(sW); sB = warp_sum(sB);
    const int wid = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { red[0][wid] = sE; red[1][wid] = sF; red[2][wid] = sW; red[3][wid] = sB; }
    __syncthreads();
    double* part = a.b.lacc + 8;                 // [gridDim.x][4]
    if (threadIdx.x < 4) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += red[threadIdx.x][w];
        part[4 * blockIdx.x + threadIdx.x] = s;
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = (atomicAdd(a.b.counter, 1u) == gridDim.x - 1);
    __syncthreads();
    if (last) {
        __threadfence();
        if (wid < 4) {                           // warp q sums quantity q over the blocks
            double s = 0.0;
            for (unsigned b = threadIdx.x & 31; b < gridDim.x; b += 32) s += __ldcg(part + 4 * b + wid);
            s = warp_sum(s);
            if ((threadIdx.x & 31) == 0) red[wid][0] = s;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            double* l = a.b.lacc;
            const double dE = a.b.nrmS > 0.0 ? red[0][0] / a.b.nrmS : 0.0, dF = a.b.nrmN > 0.0 ? red[1][0] / (3.0 * a.b.nrmN) : 0.0,
                         dV = a.b.nrmV > 0.0 ? red[2][0] / (9.0 * a.b.nrmV) : 0.0;
            l[4] = dlamE * dE + dlamF * dF + dlamV * dV; l[5] = dE; l[6] = dF; l[7] = dV;   // Eq. 4
            a.g[a.m.o_b1] = (float)(-red[3][0]);                                             // g_b1 = -sum_i eps_s(i)
            *a.b.counter = 0u;
        }
    }
}

void loss_args(nep_ctx* c, const StepArgs& a, LossArgs* o)
{
    o->a = a;
    o->lamE = (float)c->lamE; o->lamF = (float)c->lamF; o->lamV = (float)c->lamV;
    o->dlamE = c->lamE; o->dlamF = c->lamF; o->dlamV = c->lamV;
    o->func = (const void*)k_loss;
    o->ptrs[0] = &o->a; o->ptrs[1] = &o->lamE; o->ptrs[2] = &o->lamF; o->ptrs[3] = &o->lamV;
    o->ptrs[4] = &o->dlamE; o->ptrs[5] = &o->dlamF; o->ptrs[6] = &o->dlamV;
}

int launch_loss(nep_ctx* c, const StepArgs& a)
{
    const int64_t n = std::max<int64_t>(std::max<int64_t>(c->b.NBP, c->b.Sb), 1);
    const unsigned grid = (unsigned)std::min<int64_t>((n + 255) / 256, 2 * (int64_t)c->sm_count);
    LossArgs A;
    loss_args(c, a, &A);
    prof_begin(c, "k_loss");
    cudaError_t e = cudaLaunchKernel(A.func, dim3(grid), dim3(256), A.ptrs, 0, c->stream);
    prof_end(c);
    NEP_CUDA(c, e);
    return NEP_OK;
}

// ------------------------------------------------------------------------------------------------
// Type-sorted atom list of the batch (tiles of the network kernels).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_build_alist(StepArgs a)
{
    const int ib = blockIdx.x * blockDim.x + threadIdx.x;
    if (ib >= a.b.NBP) return;
    const int w = ib >> 5, lane = ib & 31;
    const int4 bi = __ldg(a.b.binfo + w);
    const size_t ip = (size_t)bi.x * WARP + lane;
    const int t = a.d.type_p[ip];
    if (t < 0) return;
    const int pos = a.b.tile_start[t] * a.b.tile_m + a.b.bsoff[bi.y * a.m.T + t] + a.d.rank_p[ip];
    a.b.alist[pos] = ib;
}

int launch_build_alist(nep_ctx* c)
{
    if (c->b.ntiles == 0) return NEP_OK;
    NEP_CUDA(c, cudaMemsetAsync(c->b.alist, 0xFF, 4 * (size_t)c->b.ntiles * c->b.tile_m, c->stream));
    StepArgs a = make_args(c);
    NEP_LAUNCH(c, "k_build_alist", k_build_alist, (unsigned)((c->b.NBP + 255) / 256), 256, 0, a);
    return NEP_OK;
}

// ------------------------------------------------------------------------------------------------
// outputs in batch order, descriptors, scaler
// ------------------------------------------------------------------------------------------------
__global__ void k_gather_outputs(StepArgs a, float* E, float* F, float* W)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < a.b.Sb) {
        if (E) E[i] = (float)a.b.Es[i];
        if (W) for (int k = 0; k < 9; ++k) W[9 * i + k] = a.b.Ws[9 * i + k];
    }
    if (F && i < a.b.NBP) {
        const int w = (int)(i >> 5), lane = (int)(i & 31);
        const int4 bi = a.b.binfo[w];
        const int il = a.d.orig_p[(size_t)bi.x * WARP + lane];
        if (il >= 0) {
            const int64_t o = a.b.bfoff[bi.y] + il;
            const float4 F4 = reinterpret_cast<const float4*>(a.b.F)[i];
            F[3 * o] = F4.x; F[3 * o + 1] = F4.y; F[3 * o + 2] = F4.z;
        }
    }
}
__global__ void k_gather_q(StepArgs a, float* q)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= a.b.NBP) return;
    const int w = (int)(i >> 5), lane = (int)(i & 31);
    const int4 bi = a.b.binfo[w];
    const int il = a.d.orig_p[(size_t)bi.x * WARP + lane];
    if (il < 0) return;
    const int64_t o = a.b.bfoff[bi.y] + il;
    const float* qp = sb_ptr(a.b.q, w, a.m.D, lane);
    for (int v = 0; v < a.m.D; ++v) q[o * a.m.D + v] = qp[(size_t)v * WARP];
}
// S0c (Eq. 2): one block per descriptor component: minimum and maximum over the atoms of the batch -> rng[v], rng[DP + v]
// (no atoms: +inf, -inf, the neutral elements of a min / max exchange between data-parallel contexts)
__global__ void __launch_bounds__(256) k_descriptor_range(StepArgs a, float* rng)
{
    const int v = blockIdx.x;
    float lo = INFINITY, hi = -INFINITY;
    for (int64_t i = threadIdx.x; i < a.b.NBP; i += blockDim.x) {
        const int w = (int)(i >> 5), lane = (int)(i & 31);
        const int ds = a.b.binfo[w].x;
        if (a.d.type_p[(size_t)ds * WARP + lane] >= 0) {
            const float x = sb_ptr(a.b.q, w, a.m.D, lane)[(size_t)v * WARP];
            lo = fminf(lo, x); hi = fmaxf(hi, x);
        }
    }
    __shared__ float slo[256], shi[256];
    slo[threadIdx.x] = lo; shi[threadIdx.x] = hi;
    __syncthreads();
    for (int o = 128; o; o >>= 1) {
        if (threadIdx.x < o) {
            slo[threadIdx.x] = fminf(slo[threadIdx.x], slo[threadIdx.x + o]);
            shi[threadIdx.x] = fmaxf(shi[threadIdx.x], shi[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { rng[v] = slo[0]; rng[a.m.DP + v] = shi[0]; }
}
// s = 1 / (max - min) (Eq. 2).  A component without a range gets s = 1 (reading G10): "without a range" is a range below
// the resolution of the arithmetic that produced q, here fp32 sums: 64 eps_fp32 max(1e-4, max |q|).  The rule is relative to the
// component's magnitude, so that a small but well resolved component (a 5-body invariant of a sparse structure, |q| ~ 1e-6) keeps
// its 1 / range as in the fp64 oracle (whose floor is 1e-12).  It cannot be purely relative: a component that vanishes by symmetry
// (l = 1, 3 moments of a centrosymmetric lattice) is the SQUARE of fp32 round-off, ~1e-12 with a range of the same size, and
// 1 / range of that would be ~1e12; the absolute floor 64 eps 1e-4 = 7.6e-10 stays two orders above it.
__global__ void k_scaler_from_range(int D, int DP, const float* __restrict__ rng, float* __restrict__ s)
{
    const int v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= DP) return;
    float out = 0.0f;
    if (v < D) {
        const float lo = rng[v], hi = rng[DP + v];
        const float range = hi - lo, am = fmaxf(fabsf(lo), fabsf(hi));
        out = (hi >= lo && isfinite(range) && range > 64.0f * 1.1920929e-7f * fmaxf(1e-4f, am)) ? 1.0f / range : 1.0f;
    }
    s[v] = out;
}

int launch_descriptor_range(nep_ctx* c, float* d_rng)
{
    StepArgs a = make_args(c);
    NEP_LAUNCH(c, "k_descriptor_range", k_descriptor_range, c->m.D, 256, 0, a, d_rng);
    return NEP_OK;
}
int launch_scaler_from_range(nep_ctx* c, const float* d_rng, float* d_s)
{
    NEP_LAUNCH(c, "k_scaler_from_range", k_scaler_from_range, (c->m.DP + 63) / 64, 64, 0, c->m.D, c->m.DP, d_rng, d_s);
    return NEP_OK;
}

int launch_gather_outputs(nep_ctx* c, float* dE, float* dF, float* dW)
{
    StepArgs a = make_args(c);
    const int64_t n = std::max<int64_t>(c->b.NBP, c->b.Sb);
    if (n == 0) return NEP_OK;
    NEP_LAUNCH(c, "k_gather_outputs", k_gather_outputs, (unsigned)((n + 255) / 256), 256, 0, a, dE, dF, dW);
    return NEP_OK;
}

int launch_gather_q(nep_ctx* c, float* dq)
{
    StepArgs a = make_args(c);
    if (c->b.NBP == 0) return NEP_OK;
    NEP_LAUNCH(c, "k_gather_q", k_gather_q, (unsigned)((c->b.NBP + 255) / 256), 256, 0, a, dq);
    return NEP_OK;
}

// ------------------------------------------------------------------------------------------------
// the step: order of the sweeps
// ------------------------------------------------------------------------------------------------
// A batch far below one resident wave leaves most of the GPU idle and every kernel costs its launch-to-drain latency: while a step
// is being captured into its graph, the radial sweep of a radial / angular pair (they are independent: both force sweeps add into F,
// E_s, W_s with atomics; the tangent sweeps write different arrays) goes to a side stream and becomes a parallel branch of the graph.
// At full size the pair gains nothing (the kernel launched first fills the GPU: profiles/r01d_summary.md), so it is not forked there.
struct SweepFork {
    nep_ctx* c; bool on; cudaStream_t main;
    explicit SweepFork(nep_ctx* c_) : c(c_), on(false), main(c_->stream)
    {
        if (!c->capturing || c->b.nbs >= 2 * c->sm_count) return;
        if (!c->side_stream && cudaStreamCreateWithFlags(&c->side_stream, cudaStreamNonBlocking) != cudaSuccess) return;
        if (!c->ev_fork && cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess) return;
        if (!c->ev_join && cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) return;
        if (cudaEventRecord(c->ev_fork, main) != cudaSuccess || cudaStreamWaitEvent(c->side_stream, c->ev_fork, 0) != cudaSuccess) return;
        on = true;
        c->stream = c->side_stream;          // the next launcher enqueues on the side stream
    }
    void back() { c->stream = main; }        // ... the one after it on the main stream again
    int join()
    {
        c->stream = main;
        if (!on) return NEP_OK;
        NEP_CUDA(c, cudaEventRecord(c->ev_join, c->side_stream));
        NEP_CUDA(c, cudaStreamWaitEvent(main, c->ev_join, 0));
        return NEP_OK;
    }
};

int launch_forward(nep_ctx* c, bool descriptors_only)
{
    if (c->b.nbs == 0) return NEP_OK;
    const StepArgs a = make_args(c);
    int rc;
    if ((rc = launch_ang_fwd(c, a))) return rc;        // S1 + S2 (also clears E_s, W_s of the batch)
    if (descriptors_only) return NEP_OK;
    if ((rc = launch_ann_fwd(c, a))) return rc;        // S3
    SweepFork f(c);
    rc = launch_rad_force(c, a);                       // S5 radial + S4
    f.back();
    if (!rc) rc = launch_ang_force(c, a);              // S5 angular
    const int rj = f.join();
    if (rc || rj) return rc ? rc : rj;
    return c->pair_on ? launch_pair_correction(c) : NEP_OK;   // short-range pair term, only when the caller set one
}

int launch_loss_grad(nep_ctx* c)
{
    const StepArgs a = make_args(c);
    int rc;
    if ((rc = launch_loss(c, a))) return rc;           // S6 (clears g)
    if (c->b.nbs == 0) return NEP_OK;
    {
        SweepFork f(c);
        rc = launch_rad_tangent(c, a);                 // S7 radial
        f.back();
        if (!rc) rc = launch_ang_tangent(c, a);        // S7 angular
        const int rj = f.join();
        if (rc || rj) return rc ? rc : rj;
    }
    if ((rc = launch_ann_bwd(c, a))) return rc;        // S8
    if ((rc = launch_ang_adjoint(c, a))) return rc;    // S9
    return NEP_OK;
}

}  // namespace nep
