// nep_ang_force.cu -- S5 (angular part): the closed-form pair force of P:145 (DESIGN C8)
//   p_ij = dE_i/dd_ij = sum_n sum_L EdS_nL [g_n'(r) b_L(r^) r^ + g_n(r) grad_d b_L(r^)],   EdS = dE_i/dS held in registers,
// F_i += p_ij, F_j -= p_ij (one vector RED per pair), W_s -= d_ij (x) p_ij.
#include "nep_kernels.cuh"

namespace nep {

// STAGED: the per-atom rows of the prologue (moments of the chunk, angular rows of Fp) come through shared memory (rows_request),
// requested before the coefficient table is filled; otherwise (tables too large for that) they are loaded into registers directly.
template <int NCH, int K, bool STAGED>
__global__ void __launch_bounds__(PAIR_TB) k_ang_force(StepArgs a)
{
    extern __shared__ __align__(16) float smem[];
    const ModelDev& m = a.m;
    constexpr int CST = CoefStride<NCH, K>::value;
    float4* stage = reinterpret_cast<float4*>(smem) + threadIdx.x;
    float* cs = smem + SWEEP2_SMEM_BYTES / 4;
    const int n0 = blockIdx.y * NCH;
    const int wib = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    float* area0 = cs + ((m.T * m.T * CST + 3) & ~3);
    float* area = area0 + (size_t)wib * staged_warp_floats(m, NCH);
    uint64_t* mbar = reinterpret_cast<uint64_t*>(area0 + (size_t)nwarp * staged_warp_floats(m, NCH)) + wib;
    if (STAGED) {
        const size_t w = (size_t)blockIdx.x * nwarp + wib;
        if (w < (size_t)a.b.nbs)
            rows_request(mbar, area, a.b.S + (w * m.nA + n0) * NL * WARP, chunk_rows(m, n0, NCH),
                         area + NCH * NL * WARP, a.b.Fp + (w * m.D + m.nR) * WARP, m.D - m.nR);
    }
    Lane L;
    const bool inb = lane_init(a, L);
    SweepA sw;
    if (inb) {
        sw = sweep_init(a.d.recoffA, a.d.recA, a.d.cntA, L);
        sweep2_begin<SWEEP2_TB>(sw.rec, sw.width, stage);
    }
    load_cA_chunk<NCH, K>(a, cs, n0);
    __syncthreads();
    if (!inb) return;
    float2 E2[NCH][NL / 2];   // dE_i/dS in packed pairs
    {
        float EdS[NCH][NL];
        if (STAGED) {
            rows_wait(mbar);
            load_EdS_staged<NCH>(m, L.ti, n0, area + L.lane, area + NCH * NL * WARP + L.lane, EdS);
        } else {
            load_EdS<NCH>(a, L, n0, EdS);
        }
#pragma unroll
        for (int n = 0; n < NCH; ++n) pack24(EdS[n], E2[n]);
    }
    float fx = 0.f, fy = 0.f, fz = 0.f, w[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) w[k] = 0.0f;
    const float* cbase = cs + (L.ti > 0 ? L.ti : 0) * m.T * CST;
    const float rcinv = m.rcinvA;
    float* Fb = a.b.F;
    const int bbase = L.bbase;
    // two pairs per iteration (sweep_pairs2): the scalar chains of both are issued together, then the two contractions
    struct Prep { PairGeo p; float g[NCH], dg[NCH]; };
    auto prep = [&](const float4& rc4, float on) {
        Prep P;
        P.p = pair_geo(rc4);
        radial_gn<NCH, K, true>(P.p.r, rcinv, cbase + P.p.tj * CST, P.g, P.dg, on);
        return P;
    };
    auto contract = [&](const Prep& P) {
        const PairGeo& p = P.p;
        float b[NL], A[NL];
        float2 b2[NL / 2], A2[NL / 2];
        const HarmZ hz = harm_z(p.z);
        const HarmXY hxy = harm_xy(p.x, p.y);
        harm24(hz, hxy, b);
        pack24(b, b2);
        float radial = 0.0f;
#pragma unroll
        for (int l = 0; l < NL / 2; ++l) A2[l] = make_float2(0.0f, 0.0f);
#pragma unroll
        for (int n = 0; n < NCH; ++n) {
            float2 eb = make_float2(0.0f, 0.0f);
            const float2 gg = dup2(P.g[n]);
#pragma unroll
            for (int l = 0; l < NL / 2; ++l) {
                eb = __ffma2_rn(E2[n][l], b2[l], eb);
                A2[l] = __ffma2_rn(gg, E2[n][l], A2[l]);
            }
            radial = fmaf(P.dg[n], eb.x + eb.y, radial);
        }
        unpack24(A2, A);
        float vx, vy, vz;
        harm24_grad_contract(hz, hxy, A, vx, vy, vz);
        const float vr = vx * p.x + vy * p.y + vz * p.z;
        const float px = fmaf(radial, p.x, (vx - vr * p.x) * p.rinv);
        const float py = fmaf(radial, p.y, (vy - vr * p.y) * p.rinv);
        const float pz = fmaf(radial, p.z, (vz - vr * p.z) * p.rinv);
        fx += px; fy += py; fz += pz;
        force_add(Fb, (unsigned)(bbase + p.jl), -px, -py, -pz);
        w[0] = fmaf(-p.dx, px, w[0]); w[1] = fmaf(-p.dx, py, w[1]); w[2] = fmaf(-p.dx, pz, w[2]);
        w[3] = fmaf(-p.dy, px, w[3]); w[4] = fmaf(-p.dy, py, w[4]); w[5] = fmaf(-p.dy, pz, w[5]);
        w[6] = fmaf(-p.dz, px, w[6]); w[7] = fmaf(-p.dz, py, w[7]); w[8] = fmaf(-p.dz, pz, w[8]);
    };
    sweep2_run<SWEEP2_TB>(sw.rec, sw.width, sw.cnt, stage, [&](const float4& ra, const float4& rb, bool has2) {
        const Prep A = prep(ra, 1.0f), B = prep(rb, has2 ? 1.0f : 0.0f);
        contract(A);
        if (has2) contract(B);
    });
    if (L.ti >= 0) force_add(Fb, L.ib, fx, fy, fz);
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const float v = warp_sum(w[k]);
        if (L.lane == 0) atomicAdd(a.b.Ws + 9 * L.sb + k, v);
    }
}

int launch_ang_force(nep_ctx* c, const StepArgs& a)
{
    const ModelDev& m = c->m;
    const int nch = pick_nch(c), kpad = pick_kpad(m.KA);
    const unsigned gx = (unsigned)((c->b.nbs * WARP + PAIR_TB - 1) / PAIR_TB);
    NEP_DISPATCH_NCH_K(nch, kpad, {
        const size_t base = SWEEP2_SMEM_BYTES + ((cA_chunk_bytes<NCH, K>(m) + 15) & ~(size_t)15);
        const size_t smem = base + 4 * (PAIR_TB / WARP) * staged_warp_floats(m, NCH) + STAGED_BAR_BYTES;
        if (2 * smem + 2048 <= (size_t)c->max_smem_sm) {      // two blocks per SM (the register limit) keep fitting
            auto kern = k_ang_force<NCH, K, true>;
            if (smem > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            NEP_LAUNCH(c, "k_ang_force", kern, dim3(gx, a.nchunks), PAIR_TB, smem, a);
        } else {
            auto kern = k_ang_force<NCH, K, false>;
            if (base > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)base));
            NEP_LAUNCH(c, "k_ang_force", kern, dim3(gx, a.nchunks), PAIR_TB, base, a);
        }
    });
    return NEP_OK;
}

}  // namespace nep
