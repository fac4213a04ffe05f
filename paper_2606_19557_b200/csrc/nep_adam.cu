// nep_adam.cu -- S10: fused Adam + AMSGrad update (Eqs. 9-13), one pass over theta, m, v, vmax, g.
#include <math.h>

#include "nep_kernels.cuh"

namespace nep {

// variant 0: the paper's equations literally -- running max of the bias-corrected second moment, epsilon inside
// the root.  variant 1: torch.optim.Adam(amsgrad=True) -- max of the raw v, sqrt(vmax / bc2) + eps.
template <int VARIANT>
__global__ void __launch_bounds__(256) k_adam(int n, float* __restrict__ theta, const float* __restrict__ g, float* __restrict__ m,
                                              float* __restrict__ v, float* __restrict__ vmax, float lr, float beta1, float beta2,
                                              float omb1, float omb2, float eps, float inv_bc1, float inv_bc2)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float gi = g[i];
    const float mi = fmaf(beta1, m[i], omb1 * gi);                      // Eq. 9 (omb = 1 - beta rounded from fp64)
    const float vi = fmaf(beta2, v[i], omb2 * gi * gi);                 // Eq. 10
    m[i] = mi; v[i] = vi;
    const float mh = mi * inv_bc1;                                    // Eq. 11
    if (VARIANT == 0) {
        const float vh = vi * inv_bc2;                                // Eq. 11
        const float vm = fmaxf(vmax[i], vh);                          // Eq. 12
        vmax[i] = vm;
        theta[i] -= lr * mh / sqrtf(vm + eps);                        // Eq. 13
    } else {
        const float vm = fmaxf(vmax[i], vi);
        vmax[i] = vm;
        theta[i] -= lr * mh / (sqrtf(vm * inv_bc2) + eps);
    }
}

void adam_args(nep_ctx* c, double lr, double b1, double b2, double eps, int variant, int64_t t, AdamArgs* o)
{
    const double bc1 = 1.0 - pow(b1, (double)t), bc2 = 1.0 - pow(b2, (double)t);
    o->n = c->m.npar; o->theta = c->theta; o->g = c->g; o->m = c->am; o->v = c->av; o->vmax = c->avmax;
    o->lr = (float)lr; o->beta1 = (float)b1; o->beta2 = (float)b2; o->omb1 = (float)(1.0 - b1); o->omb2 = (float)(1.0 - b2);
    o->eps = (float)eps; o->inv_bc1 = (float)(1.0 / bc1); o->inv_bc2 = (float)(1.0 / bc2);
    o->func = variant == 0 ? (const void*)k_adam<0> : (const void*)k_adam<1>;
    o->ptrs[0] = &o->n; o->ptrs[1] = &o->theta; o->ptrs[2] = &o->g; o->ptrs[3] = &o->m; o->ptrs[4] = &o->v; o->ptrs[5] = &o->vmax;
    o->ptrs[6] = &o->lr; o->ptrs[7] = &o->beta1; o->ptrs[8] = &o->beta2; o->ptrs[9] = &o->omb1; o->ptrs[10] = &o->omb2;
    o->ptrs[11] = &o->eps; o->ptrs[12] = &o->inv_bc1; o->ptrs[13] = &o->inv_bc2;
}

int launch_adam(nep_ctx* c, double lr, double b1, double b2, double eps, int variant)
{
    c->t_adam += 1;
    AdamArgs A;
    adam_args(c, lr, b1, b2, eps, variant, c->t_adam, &A);
    const unsigned grid = (unsigned)((A.n + 255) / 256);
    prof_begin(c, "k_adam");
    cudaError_t e = cudaLaunchKernel(A.func, dim3(grid), dim3(256), A.ptrs, 0, c->stream);
    prof_end(c);
    NEP_CUDA(c, e);
    return NEP_OK;
}

}  // namespace nep
