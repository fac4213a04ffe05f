// nep_pair.cu -- short-range pair correction.  P:105: "TorchNEP fully supports the Ziegler-Biersack-Littmark (ZBL)
// potential [24] as a short-range correction".  The paper prints neither the screening constants nor the switching radii, so the
// library stores none: the term has a fixed form and every number in it comes from the caller (DESIGN reading G29)
//     phi_ij(r) = sw(r) (k_C Z_i Z_j / r) sum_m coef_m exp(-expo_m r / a_ij),   a_ij = a_prefac / (Z_i^p + Z_j^p),
//     sw = 1 below r_inner, 1/2 (1 + cos(pi (r - r_inner) / (r_outer - r_inner))) up to r_outer, 0 beyond.
// It has no model parameter in it: it adds to E_s, F_i, W_s after the force sweeps (so the loss seeds eps, u, G see the corrected
// predictions) and contributes nothing to grad_theta L.
// One kernel over the HALF list of the radial pairs (one record per undirected pair, as k_rad_force): the owner evaluates phi and
// phi', adds phi' r^ to its own force, scatters the reaction to the neighbour, and the warp folds phi and d (x) phi' r^ into the
// structure's energy (fp64) and virial.  Pairs beyond r_outer (nearly all of them) cost a compare.
#include <cmath>

#include "nep_kernels.cuh"

namespace nep {

constexpr int PAIRC_TB = 128;

__global__ void __launch_bounds__(PAIRC_TB) k_pair_correction(StepArgs a, PairCorrDev pc)
{
    __shared__ __align__(16) float4 stage_s[PAIRC_TB * 4];
    Lane L;
    if (!lane_init(a, L)) return;
    const SweepA sw = sweep_init(a.d.recoffH, a.d.recH, a.d.cntH, L);
    float fx = 0.f, fy = 0.f, fz = 0.f, wxx = 0.f, wyy = 0.f, wzz = 0.f, wxy = 0.f, wxz = 0.f, wyz = 0.f;
    double e = 0.0;
    bool hit = false;
    float* Fb = a.b.F;
    const int ti = L.ti, bbase = L.bbase;
    auto one = [&](const float4& rc4) {
        const PairGeo p = pair_geo(rc4);
        if (!(p.r < pc.r_outer)) return;
        const float r = p.r, rinv = 1.0f / r;
        const float ainv = pc.ainv[ti * MAX_T + p.tj];
        const float x = r * ainv;
        float scr = 0.0f, dscr = 0.0f;
        for (int m = 0; m < pc.n_terms; ++m) {
            const float t = pc.coef[m] * expf(-pc.expo[m] * x);
            scr += t;
            dscr = fmaf(-pc.expo[m] * ainv, t, dscr);
        }
        const float coul = pc.pref[ti * MAX_T + p.tj] * rinv;
        float s = 1.0f, ds = 0.0f;
        if (r > pc.r_inner) {
            const float t = (r - pc.r_inner) * pc.inv_width;
            s = 0.5f * (1.0f + cospif(t));
            ds = -0.5f * 3.14159265358979f * pc.inv_width * sinpif(t);
        }
        const float phi0 = coul * scr, dphi0 = coul * (dscr - scr * rinv);
        const float phi = s * phi0, fs = fmaf(ds, phi0, s * dphi0);          // fs = d phi / d r
        e += (double)phi;
        hit = true;
        const float px = fs * p.x, py = fs * p.y, pz = fs * p.z;
        fx += px; fy += py; fz += pz;
        force_add(Fb, (unsigned)(bbase + p.jl), -px, -py, -pz);
        wxx = fmaf(-p.dx, px, wxx); wyy = fmaf(-p.dy, py, wyy); wzz = fmaf(-p.dz, pz, wzz);
        wxy = fmaf(-p.dx, py, wxy); wxz = fmaf(-p.dx, pz, wxz); wyz = fmaf(-p.dy, pz, wyz);
    };
    sweep_pairs2<PAIRC_TB>(sw.rec, sw.width, sw.cnt, stage_s + threadIdx.x, [&](const float4& ra, const float4& rb, bool has2) {
        one(ra);
        if (has2) one(rb);
    });
    if (!__any_sync(0xffffffffu, hit)) return;           // no pair of this slice inside r_outer: nothing to add
    if (hit) force_add(Fb, L.ib, fx, fy, fz);
    wxx = warp_sum(wxx); wyy = warp_sum(wyy); wzz = warp_sum(wzz); wxy = warp_sum(wxy); wxz = warp_sum(wxz); wyz = warp_sum(wyz);
    e = warp_sum(e);
    if (L.lane == 0) {
        float* W = a.b.Ws + 9 * L.sb;
        atomicAdd(W + 0, wxx); atomicAdd(W + 1, wxy); atomicAdd(W + 2, wxz);
        atomicAdd(W + 3, wxy); atomicAdd(W + 4, wyy); atomicAdd(W + 5, wyz);
        atomicAdd(W + 6, wxz); atomicAdd(W + 7, wyz); atomicAdd(W + 8, wzz);
        atomicAdd(a.b.Es + L.sb, e);
    }
}

int launch_pair_correction(nep_ctx* c)
{
    if (c->b.nbs == 0) return NEP_OK;
    const StepArgs a = make_args(c);
    const unsigned gx = (unsigned)((c->b.nbs * WARP + PAIRC_TB - 1) / PAIRC_TB);
    NEP_LAUNCH(c, "k_pair_correction", k_pair_correction, gx, PAIRC_TB, 0, a, c->pair);
    return NEP_OK;
}

}  // namespace nep

using namespace nep;

extern "C" int nep_set_pair_correction(nep_ctx* c, const double* Z, double r_inner, double r_outer, int n_terms, const double* coef,
                                       const double* expo, double a_prefac, double a_pow, double coulomb_k)
{
    if (!c) return NEP_EINVAL;
    c->forward_valid = c->grad_valid = false;
    ++c->graph_gen;                                      // the constants travel by value in the captured launch
    if (!Z || n_terms == 0) { c->pair_on = false; return NEP_OK; }
    if (n_terms < 0 || n_terms > MAX_PAIR_TERMS) return fail(c, NEP_ECAPACITY, "nep_set_pair_correction: n_terms must be 1.." + std::to_string(MAX_PAIR_TERMS));
    if (!coef || !expo) return fail(c, NEP_EINVAL, "nep_set_pair_correction: coef / expo is NULL");
    if (!(r_inner >= 0.0) || !(r_outer > r_inner) || !(r_outer <= c->rcR))
        return fail(c, NEP_EINVAL, "nep_set_pair_correction: need 0 <= r_inner < r_outer <= rc_R (the term walks the radial neighbour list)");
    if (!(a_prefac > 0.0) || !std::isfinite(a_pow) || !(coulomb_k > 0.0) || !std::isfinite(coulomb_k))
        return fail(c, NEP_EINVAL, "nep_set_pair_correction: a_prefac and coulomb_k must be positive, a_pow finite");
    PairCorrDev pc{};
    pc.n_terms = n_terms;
    pc.r_inner = (float)r_inner; pc.r_outer = (float)r_outer; pc.inv_width = (float)(1.0 / (r_outer - r_inner));
    for (int m = 0; m < n_terms; ++m) {
        if (!std::isfinite(coef[m]) || !(expo[m] >= 0.0) || !std::isfinite(expo[m])) return fail(c, NEP_EINVAL, "nep_set_pair_correction: bad coef / expo");
        pc.coef[m] = (float)coef[m]; pc.expo[m] = (float)expo[m];
    }
    const int T = c->m.T;
    for (int t = 0; t < T; ++t)
        if (!(Z[t] > 0.0) || !std::isfinite(Z[t])) return fail(c, NEP_EINVAL, "nep_set_pair_correction: Z must be positive");
    for (int ti = 0; ti < T; ++ti)
        for (int tj = 0; tj < T; ++tj) {
            pc.pref[ti * MAX_T + tj] = (float)(coulomb_k * Z[ti] * Z[tj]);
            pc.ainv[ti * MAX_T + tj] = (float)((std::pow(Z[ti], a_pow) + std::pow(Z[tj], a_pow)) / a_prefac);
        }
    c->pair = pc; c->pair_on = true;
    return NEP_OK;
}
