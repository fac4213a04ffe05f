// nep_radial.cu -- the two sweeps over the radial pair list.
// S5 (radial part): F_i = sum_j (s_ij + s_ji) r^_ij with s_ij = sum_k a^i_k[t_j] f_k'(r_ij), a^i_k[T'] = sum_n Fp_n cR[t_i][T'][n][k].
//     The sweep walks the HALF list (one record per undirected pair, nep_neighbor.cu): the pair and its mirror share f_k'(r), so the
//     owner evaluates the basis once, gathers the other atom's coefficient row a^j[t_i] (rows of one structure are cache resident),
//     adds (s_ij + s_ji) r^ to its own force and scatters the reaction to j (one vector RED, like the angular force sweep).
//     W_s -= sum d (x) ((s_ij + s_ji) r^).  Also folds the per-atom energies into E_s (Eq. 1).
// S7 (radial part): Bd_k[T'] = sum_{j, t_j = T'} f_k'(r_ij) (r^_ij . d~_ij), the tangent of the aggregate B (DESIGN C10).
#include "nep_kernels.cuh"

namespace nep {

constexpr int RAD_TB = 128;

template <int K>
__global__ void __launch_bounds__(RAD_TB) k_rad_force(StepArgs a)
{
    __shared__ __align__(16) float4 stage_s[RAD_TB * 4];
    Lane L;
    if (!lane_init(a, L)) return;
    const ModelDev& m = a.m;
    const SweepA sw = sweep_init(a.d.recoffH, a.d.recH, a.d.cntH, L);
    constexpr int KP = (K + 3) & ~3;
    const int KRP = m.KRP, TKRP = m.T * m.KRP;
    float ai[KP];
#pragma unroll
    for (int k = 0; k < KP; ++k) ai[k] = 0.0f;
    int cur = -1;
    float fx = 0.f, fy = 0.f, fz = 0.f, wxx = 0.f, wyy = 0.f, wzz = 0.f, wxy = 0.f, wxz = 0.f, wyz = 0.f;
    const float* arow = a.b.arow;
    const float* arow_i = arow + (size_t)L.ib * TKRP;
    float* Fb = a.b.F;
    const int ti = L.ti, bbase = L.bbase;
    const float rcinv = m.rcinvR;
    auto one = [&](const float4& rc4) {
        const PairGeo p = pair_geo(rc4);
        if (p.tj != cur) {
            cur = p.tj;
            const float4* src = reinterpret_cast<const float4*>(arow_i + cur * KRP);
#pragma unroll
            for (int k4 = 0; k4 < KP / 4; ++k4)
                if (k4 * 4 < KRP) { const float4 v = src[k4]; ai[4 * k4] = v.x; ai[4 * k4 + 1] = v.y; ai[4 * k4 + 2] = v.z; ai[4 * k4 + 3] = v.w; }
        }
        float aj[KP];
        const float4* srcj = reinterpret_cast<const float4*>(arow + (size_t)(bbase + p.jl) * TKRP + ti * KRP);
#pragma unroll
        for (int k4 = 0; k4 < KP / 4; ++k4) {
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (k4 * 4 < KRP) v = __ldg(srcj + k4);
            aj[4 * k4] = v.x; aj[4 * k4 + 1] = v.y; aj[4 * k4 + 2] = v.z; aj[4 * k4 + 3] = v.w;
        }
        float sij = 0.0f, sji = 0.0f;
        cheb_basis<K, true>(p.r, rcinv, [&](int k, float, float dfk) {
            sij = fmaf(ai[k], dfk, sij);
            sji = fmaf(aj[k], dfk, sji);
        });
        const float fs = sij + sji;
        const float px = fs * p.x, py = fs * p.y, pz = fs * p.z;
        fx += px; fy += py; fz += pz;
        force_add(Fb, (unsigned)(bbase + p.jl), -px, -py, -pz);
        wxx = fmaf(-p.dx, px, wxx); wyy = fmaf(-p.dy, py, wyy); wzz = fmaf(-p.dz, pz, wzz);
        wxy = fmaf(-p.dx, py, wxy); wxz = fmaf(-p.dx, pz, wxz); wyz = fmaf(-p.dy, pz, wyz);
    };
    sweep_pairs2<RAD_TB>(sw.rec, sw.width, sw.cnt, stage_s + threadIdx.x, [&](const float4& ra, const float4& rb, bool has2) {
        one(ra);
        if (has2) one(rb);
    });
    if (L.ti >= 0) force_add(Fb, L.ib, fx, fy, fz);   // F was cleared by k_ang_fwd
    wxx = warp_sum(wxx); wyy = warp_sum(wyy); wzz = warp_sum(wzz); wxy = warp_sum(wxy); wxz = warp_sum(wxz); wyz = warp_sum(wyz);
    const double Es = warp_sum(L.ti >= 0 ? (double)a.b.Ei[L.ib] : 0.0);
    if (L.lane == 0) {
        float* W = a.b.Ws + 9 * L.sb;
        atomicAdd(W + 0, wxx); atomicAdd(W + 1, wxy); atomicAdd(W + 2, wxz);
        atomicAdd(W + 3, wxy); atomicAdd(W + 4, wyy); atomicAdd(W + 5, wyz);
        atomicAdd(W + 6, wxz); atomicAdd(W + 7, wyz); atomicAdd(W + 8, wzz);
        atomicAdd(a.b.Es + L.sb, Es);
    }
}

template <int K>
__global__ void __launch_bounds__(RAD_TB) k_rad_tangent(StepArgs a)
{
    __shared__ __align__(16) float4 stage_s[RAD_TB * 4];
    Lane L;
    if (!lane_init(a, L)) return;
    const ModelDev& m = a.m;
    const SweepA sw = sweep_init(a.d.recoffR, a.d.recR, a.d.cntR, L);
    float G[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) G[k] = __ldg(a.b.G + 9 * L.sb + k);
    const float* ui = sb_ptr(a.b.u, L.w, 3, L.lane);
    const float uix = ui[0], uiy = ui[WARP], uiz = ui[2 * WARP];
    float bd[K];
#pragma unroll
    for (int k = 0; k < K; ++k) bd[k] = 0.0f;
    float* Bdp = sb_ptr(a.b.Bd, L.w, m.T * m.KR, L.lane);
    const int KR = m.KR;
    // every row is written: types without neighbours get zeros
    for (int r = 0; r < m.T * KR; ++r) Bdp[(size_t)r * WARP] = 0.0f;
    int cur = -1;
    auto store = [&]() {
#pragma unroll
        for (int k = 0; k < K; ++k)
            if (k < KR) { Bdp[(size_t)(cur * KR + k) * WARP] = bd[k]; bd[k] = 0.0f; }
    };
    const float* ub = a.b.u;
    const int bbase = L.bbase;
    const float rcinv = m.rcinvR;
    auto one = [&](const float4& rc4) {
        const PairGeo p = pair_geo(rc4);
        if (p.tj != cur) {
            if (cur >= 0) store();
            cur = p.tj;
        }
        const Tangent T = pair_tangent(ub, bbase, p, uix, uiy, uiz, G);
        cheb_basis<K, true, true>(p.r, rcinv, [&](int k, float, float dfk) { bd[k] = fmaf(dfk, T.t, bd[k]); });
    };
    sweep_pairs2<RAD_TB>(sw.rec, sw.width, sw.cnt, stage_s + threadIdx.x, [&](const float4& ra, const float4& rb, bool has2) {
        one(ra);
        if (has2) one(rb);
    });
    if (cur >= 0) store();
}

#define NEP_DISPATCH_KR(KRv, ...)                              \
    if ((KRv) <= 9) { constexpr int K = 9; __VA_ARGS__; }      \
    else if ((KRv) <= 11) { constexpr int K = 11; __VA_ARGS__; } \
    else if ((KRv) <= 13) { constexpr int K = 13; __VA_ARGS__; } \
    else { constexpr int K = 17; __VA_ARGS__; }

int launch_rad_force(nep_ctx* c, const StepArgs& a)
{
    const unsigned gx = (unsigned)((c->b.nbs * WARP + RAD_TB - 1) / RAD_TB);
    NEP_DISPATCH_KR(c->m.KR, { NEP_LAUNCH(c, "k_rad_force", k_rad_force<K>, gx, RAD_TB, 0, a); });
    return NEP_OK;
}
int launch_rad_tangent(nep_ctx* c, const StepArgs& a)
{
    const unsigned gx = (unsigned)((c->b.nbs * WARP + RAD_TB - 1) / RAD_TB);
    NEP_DISPATCH_KR(c->m.KR, { NEP_LAUNCH(c, "k_rad_tangent", k_rad_tangent<K>, gx, RAD_TB, 0, a); });
    return NEP_OK;
}

}  // namespace nep
