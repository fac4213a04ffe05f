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

int launch_adam(nep_ctx* c, double lr, double b1, double b2, double eps, int variant)
{
    c->t_adam += 1;
    const double bc1 = 1.0 - pow(b1, (double)c->t_adam), bc2 = 1.0 - pow(b2, (double)c->t_adam);
    const int n = c->m.npar;
    const unsigned grid = (unsigned)((n + 255) / 256);
    if (variant == 0)
        NEP_LAUNCH(c, "k_adam", k_adam<0>, grid, 256, 0, n, c->theta, c->g, c->am, c->av, c->avmax, (float)lr, (float)b1, (float)b2,
                   (float)(1.0 - b1), (float)(1.0 - b2), (float)eps, (float)(1.0 / bc1), (float)(1.0 / bc2));
    else
        NEP_LAUNCH(c, "k_adam", k_adam<1>, grid, 256, 0, n, c->theta, c->g, c->am, c->av, c->avmax, (float)lr, (float)b1, (float)b2,
                   (float)(1.0 - b1), (float)(1.0 - b2), (float)eps, (float)(1.0 / bc1), (float)(1.0 / bc2));
    return NEP_OK;
}

}  // namespace nep
