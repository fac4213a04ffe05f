// nep_forward.cu -- S1-S5 of the training step: radial and angular descriptors (Eqs. 15-20),
// the per-species tanh network (Eqs. 2-3), structure energies (Eq. 1) and the closed-form
// pair forces and virials (DESIGN C8).  fp32 arithmetic, fp64 only for the energy reduction.
#include <algorithm>

#include "nep_kernels.cuh"

namespace nep {

// ------------------------------------------------------------------------------------------------
// S1: q_n = sum_{T'} sum_k cR[t_i][T'][n][k] B_k[T']   (B is the one-time aggregate of f_k over neighbours)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_radial_q(StepArgs a)
{
    extern __shared__ float cs[];   // cR, [ti][tj][n][k] as in theta
    const ModelDev& m = a.m;
    const int ncr = m.T * m.T * m.nR * m.KR;
    for (int i = threadIdx.x; i < ncr; i += blockDim.x) cs[i] = a.theta[m.o_cR + i];
    __syncthreads();
    Lane L;
    if (!lane_init(a, L)) return;
    const int TK = m.T * m.KR;
    for (int n = 0; n < m.nR; ++n) {
        float acc = 0.0f;
        if (L.ti >= 0) {
            for (int tj = 0; tj < m.T; ++tj) {
                const float* cc = cs + ((L.ti * m.T + tj) * m.nR + n) * m.KR;
                for (int k = 0; k < m.KR; ++k) acc = fmaf(cc[k], a.d.B[(int64_t)(tj * m.KR + k) * a.d.NP + L.ip], acc);
            }
        }
        a.b.q[(int64_t)n * a.b.NBP + L.ib] = acc;
    }
    (void)TK;
}

// ------------------------------------------------------------------------------------------------
// S2: angular moments S_nL = sum_j g_n(r_ij) b_L(r^_ij) and the invariants built from them
// grid = (slices / warps per block, channel chunks); thread = (atom, chunk of NCH channels)
// ------------------------------------------------------------------------------------------------
template <int NCH>
__global__ void __launch_bounds__(128) k_ang_fwd(StepArgs a)
{
    extern __shared__ float cs[];
    load_cA_smem(a, cs);
    __syncthreads();
    Lane L;
    if (!lane_init(a, L)) return;
    const ModelDev& m = a.m;
    const int n0 = blockIdx.y * NCH;
    const int cnt = (L.ti >= 0) ? a.d.cntA[L.ip] : 0;
    const int64_t base = a.d.recoffA[L.ds];
    const int width = (int)((a.d.recoffA[L.ds + 1] - base) >> 5);
    const float4* rec = a.d.recA + base + L.lane;
    float S[NCH][NL];
#pragma unroll
    for (int n = 0; n < NCH; ++n)
#pragma unroll
        for (int l = 0; l < NL; ++l) S[n][l] = 0.0f;
    for (int s = 0; s < width; ++s) {
        const float4 rc4 = rec[(int64_t)s * WARP];
        if (s < cnt) {
            const PairGeo p = pair_geo(rc4);
            float g[NCH];
            radial_gn<NCH, false>(p.r, m.rcinvA, m.KA, cs + (L.ti * m.T + p.tj) * m.KA * a.nAP + n0, a.nAP, g, nullptr);
            float b[NL];
            const HarmZ hz = harm_z(p.z);
            const HarmXY hxy = harm_xy(p.x, p.y);
            harm24(hz, hxy, b);
#pragma unroll
            for (int n = 0; n < NCH; ++n)
#pragma unroll
                for (int l = 0; l < NL; ++l) S[n][l] = fmaf(g[n], b[l], S[n][l]);
        }
    }
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        if (n0 + n < m.nA) {
            float qv[6];
            inv_values(S[n], m.has4, m.has5, qv);
            for (int aa = 0; aa < m.nang; ++aa) a.b.q[(int64_t)(m.nR + aa * m.nA + n0 + n) * a.b.NBP + L.ib] = qv[aa];
#pragma unroll
            for (int l = 0; l < NL; ++l) a.b.S[(int64_t)((n0 + n) * NL + l) * a.b.NBP + L.ib] = S[n][l];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S3 + S4: network forward, dE_i/dq, a-rows for the radial force sweep, structure energies.
// thread = atom.  shared: w0 [T][HP][DP] (zero padded), b0, w1 [T][HP], scaler [DP], cR, and two
// per-thread columns: qcol [DP][BLK], ecol [HP][BLK].
// ------------------------------------------------------------------------------------------------
struct AnnSmem {
    int w0, b0, w1, sc, cR, qcol, ecol, total;   // float offsets
};
__host__ __device__ inline AnnSmem ann_smem_layout(const ModelDev& m, int BLK)
{
    AnnSmem s;
    int o = 0;
    s.w0 = o; o += m.T * m.HP * m.DP;
    s.b0 = o; o += m.T * m.HP;
    s.w1 = o; o += m.T * m.HP;
    s.sc = o; o += m.DP;
    s.cR = o; o += (m.T * m.T * m.nR * m.KR + 3) & ~3;
    s.qcol = o; o += m.DP * BLK;
    s.ecol = o; o += m.HP * BLK;
    s.total = o;
    return s;
}
__device__ __forceinline__ void ann_load_weights(const StepArgs& a, float* sm, const AnnSmem& lay)
{
    const ModelDev& m = a.m;
    for (int i = threadIdx.x; i < m.T * m.HP * m.DP; i += blockDim.x) {
        const int v = i % m.DP, mu = (i / m.DP) % m.HP, t = i / (m.DP * m.HP);
        sm[lay.w0 + i] = (v < m.D && mu < m.H) ? a.theta[t * m.per_type + mu * m.D + v] : 0.0f;
    }
    for (int i = threadIdx.x; i < m.T * m.HP; i += blockDim.x) {
        const int mu = i % m.HP, t = i / m.HP;
        sm[lay.b0 + i] = (mu < m.H) ? a.theta[t * m.per_type + m.H * m.D + mu] : 0.0f;
        sm[lay.w1 + i] = (mu < m.H) ? a.theta[t * m.per_type + m.H * m.D + m.H + mu] : 0.0f;
    }
    for (int i = threadIdx.x; i < m.DP; i += blockDim.x) sm[lay.sc + i] = (i < m.D) ? a.scaler[i] : 0.0f;
    for (int i = threadIdx.x; i < m.T * m.T * m.nR * m.KR; i += blockDim.x) sm[lay.cR + i] = a.theta[m.o_cR + i];
}

template <int BLK>
__global__ void __launch_bounds__(BLK) k_ann_fwd(StepArgs a)
{
    extern __shared__ __align__(16) float sm[];
    const ModelDev& m = a.m;
    const AnnSmem lay = ann_smem_layout(m, BLK);
    ann_load_weights(a, sm, lay);
    __syncthreads();
    Lane L;
    if (!lane_init(a, L)) return;
    const int tid = threadIdx.x;
    float* qcol = sm + lay.qcol + tid;
    float* ecol = sm + lay.ecol + tid;
    float Ei = 0.0f;
    if (L.ti >= 0) {
        for (int v = 0; v < m.DP; ++v) qcol[v * BLK] = (v < m.D) ? sm[lay.sc + v] * a.b.q[(int64_t)v * a.b.NBP + L.ib] : 0.0f;
        const float* w0 = sm + lay.w0 + L.ti * m.HP * m.DP;
        const float* b0 = sm + lay.b0 + L.ti * m.HP;
        const float* w1 = sm + lay.w1 + L.ti * m.HP;
        for (int mu0 = 0; mu0 < m.HP; mu0 += 8) {
            float acc[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[j] = -b0[mu0 + j];
            for (int v = 0; v < m.DP; v += 4) {
                const float q0 = qcol[v * BLK], q1 = qcol[(v + 1) * BLK], q2 = qcol[(v + 2) * BLK], q3 = qcol[(v + 3) * BLK];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const float4 w = *reinterpret_cast<const float4*>(w0 + (mu0 + j) * m.DP + v);
                    acc[j] = fmaf(w.x, q0, fmaf(w.y, q1, fmaf(w.z, q2, fmaf(w.w, q3, acc[j]))));
                }
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const float h = tanhf(acc[j]);
                Ei = fmaf(w1[mu0 + j], h, Ei);
                ecol[(mu0 + j) * BLK] = w1[mu0 + j] * (1.0f - h * h);
                if (mu0 + j < m.H) a.b.h[(int64_t)(mu0 + j) * a.b.NBP + L.ib] = h;
            }
        }
        Ei -= a.theta[m.o_b1];
        // Fp = s o (w0^T e)
        for (int v0 = 0; v0 < m.DP; v0 += 8) {
            float acc[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[j] = 0.0f;
            for (int mu = 0; mu < m.HP; ++mu) {
                const float e = ecol[mu * BLK];
                const float4 wa = *reinterpret_cast<const float4*>(w0 + mu * m.DP + v0);
                const float4 wb = *reinterpret_cast<const float4*>(w0 + mu * m.DP + v0 + 4);
                acc[0] = fmaf(e, wa.x, acc[0]); acc[1] = fmaf(e, wa.y, acc[1]); acc[2] = fmaf(e, wa.z, acc[2]); acc[3] = fmaf(e, wa.w, acc[3]);
                acc[4] = fmaf(e, wb.x, acc[4]); acc[5] = fmaf(e, wb.y, acc[5]); acc[6] = fmaf(e, wb.z, acc[6]); acc[7] = fmaf(e, wb.w, acc[7]);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int v = v0 + j;
                if (v < m.D) {
                    const float fp = sm[lay.sc + v] * acc[j];
                    a.b.Fp[(int64_t)v * a.b.NBP + L.ib] = fp;
                    qcol[v * BLK] = fp;      // q~ no longer needed; keep Fp (radial part used below)
                }
            }
        }
        // a_k[T'] = sum_n Fp_n cR[t_i][T'][n][k]
        float* arow = a.b.arow + (L.ib * m.T) * m.KRP;
        for (int tj = 0; tj < m.T; ++tj) {
            const float* cc = sm + lay.cR + (L.ti * m.T + tj) * m.nR * m.KR;
            for (int k = 0; k < m.KRP; ++k) {
                float s = 0.0f;
                if (k < m.KR) for (int n = 0; n < m.nR; ++n) s = fmaf(qcol[n * BLK], cc[n * m.KR + k], s);
                arow[tj * m.KRP + k] = s;
            }
        }
        a.b.Ei[L.ib] = Ei;
    } else {
        a.b.Ei[L.ib] = 0.0f;
    }
    const double Es = warp_sum((double)Ei);
    if (L.lane == 0) atomicAdd(&a.b.Es[L.sb], Es);
}

// ------------------------------------------------------------------------------------------------
// S5 (radial part): F_i = sum_j (s_ij + s_ji) r^_ij with s_ij = sum_k a^i_k[t_j] f_k'(r_ij); the reverse pair's
// coefficient row a^j[t_i] is gathered (rows of one structure are L1/L2 resident): no atomics, deterministic.
// W_s -= sum d (x) (s_ij r^).
// ------------------------------------------------------------------------------------------------
template <int KMAX>
__global__ void __launch_bounds__(128) k_rad_force(StepArgs a)
{
    Lane L;
    if (!lane_init(a, L)) return;
    const ModelDev& m = a.m;
    const int cnt = (L.ti >= 0) ? a.d.cntR[L.ip] : 0;
    const int64_t base = a.d.recoffR[L.ds];
    const int width = (int)((a.d.recoffR[L.ds + 1] - base) >> 5);
    const float4* rec = a.d.recR + base + L.lane;
    constexpr int KP = (KMAX + 3) & ~3;
    float ai[KP];
#pragma unroll
    for (int k = 0; k < KP; ++k) ai[k] = 0.0f;
    int cur = -1;
    float fx = 0.f, fy = 0.f, fz = 0.f, wxx = 0.f, wyy = 0.f, wzz = 0.f, wxy = 0.f, wxz = 0.f, wyz = 0.f;
    for (int s = 0; s < width; ++s) {
        const float4 rc4 = rec[(int64_t)s * WARP];
        if (s < cnt) {
            const PairGeo p = pair_geo(rc4);
            if (p.tj != cur) {
                cur = p.tj;
                const float4* src = reinterpret_cast<const float4*>(a.b.arow + (L.ib * m.T + cur) * m.KRP);
#pragma unroll
                for (int k4 = 0; k4 < KP / 4; ++k4)
                    if (k4 * 4 < m.KRP) { const float4 v = src[k4]; ai[4 * k4] = v.x; ai[4 * k4 + 1] = v.y; ai[4 * k4 + 2] = v.z; ai[4 * k4 + 3] = v.w; }
            }
            float aj[KP];
            const float4* srcj = reinterpret_cast<const float4*>(a.b.arow + ((int64_t)(L.bbase + p.jl) * m.T + L.ti) * m.KRP);
#pragma unroll
            for (int k4 = 0; k4 < KP / 4; ++k4) {
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (k4 * 4 < m.KRP) v = __ldg(srcj + k4);
                aj[4 * k4] = v.x; aj[4 * k4 + 1] = v.y; aj[4 * k4 + 2] = v.z; aj[4 * k4 + 3] = v.w;
            }
            float sij = 0.0f, sji = 0.0f;
            cheb_foreach<KMAX>(p.r, m.rcinvR, m.KR, [&](int k, float, float dfk) {
                sij = fmaf(ai[k], dfk, sij);
                sji = fmaf(aj[k], dfk, sji);
            });
            const float fs = sij + sji;
            fx = fmaf(fs, p.x, fx); fy = fmaf(fs, p.y, fy); fz = fmaf(fs, p.z, fz);
            const float px = sij * p.x, py = sij * p.y, pz = sij * p.z;
            wxx = fmaf(-p.dx, px, wxx); wyy = fmaf(-p.dy, py, wyy); wzz = fmaf(-p.dz, pz, wzz);
            wxy = fmaf(-p.dx, py, wxy); wxz = fmaf(-p.dx, pz, wxz); wyz = fmaf(-p.dy, pz, wyz);
        }
    }
    a.b.F[L.ib] = fx; a.b.F[a.b.NBP + L.ib] = fy; a.b.F[2 * a.b.NBP + L.ib] = fz;
    wxx = warp_sum(wxx); wyy = warp_sum(wyy); wzz = warp_sum(wzz); wxy = warp_sum(wxy); wxz = warp_sum(wxz); wyz = warp_sum(wyz);
    if (L.lane == 0) {
        float* W = a.b.Ws + 9 * L.sb;
        atomicAdd(W + 0, wxx); atomicAdd(W + 1, wxy); atomicAdd(W + 2, wxz);
        atomicAdd(W + 3, wxy); atomicAdd(W + 4, wyy); atomicAdd(W + 5, wyz);
        atomicAdd(W + 6, wxz); atomicAdd(W + 7, wyz); atomicAdd(W + 8, wzz);
    }
}

// ------------------------------------------------------------------------------------------------
// S5 (angular part): p_ij = sum_n sum_L EdS_nL [g_n' b_L r^ + g_n grad_d b_L],  EdS = dE_i/dS (registers).
// F_i += p_ij, F_j -= p_ij (atomics), W_s -= d (x) p.
// ------------------------------------------------------------------------------------------------
template <int NCH>
__global__ void __launch_bounds__(128) k_ang_force(StepArgs a)
{
    extern __shared__ float cs[];
    load_cA_smem(a, cs);
    __syncthreads();
    Lane L;
    if (!lane_init(a, L)) return;
    const ModelDev& m = a.m;
    const int n0 = blockIdx.y * NCH;
    const int cnt = (L.ti >= 0) ? a.d.cntA[L.ip] : 0;
    const int64_t base = a.d.recoffA[L.ds];
    const int width = (int)((a.d.recoffA[L.ds + 1] - base) >> 5);
    const float4* rec = a.d.recA + base + L.lane;
    float EdS[NCH][NL];
    load_EdS<NCH>(a, L, n0, EdS);
    float fx = 0.f, fy = 0.f, fz = 0.f, w[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) w[k] = 0.0f;
    for (int s = 0; s < width; ++s) {
        const float4 rc4 = rec[(int64_t)s * WARP];
        if (s < cnt) {
            const PairGeo p = pair_geo(rc4);
            float g[NCH], dg[NCH];
            radial_gn<NCH, true>(p.r, m.rcinvA, m.KA, cs + (L.ti * m.T + p.tj) * m.KA * a.nAP + n0, a.nAP, g, dg);
            float b[NL], A[NL];
            const HarmZ hz = harm_z(p.z);
            const HarmXY hxy = harm_xy(p.x, p.y);
            harm24(hz, hxy, b);
            float radial = 0.0f;
#pragma unroll
            for (int l = 0; l < NL; ++l) A[l] = 0.0f;
#pragma unroll
            for (int n = 0; n < NCH; ++n) {
                float eb = 0.0f;
#pragma unroll
                for (int l = 0; l < NL; ++l) {
                    eb = fmaf(EdS[n][l], b[l], eb);
                    A[l] = fmaf(g[n], EdS[n][l], A[l]);
                }
                radial = fmaf(dg[n], eb, radial);
            }
            float vx, vy, vz;
            harm24_grad_contract(hz, hxy, A, vx, vy, vz);
            const float vr = vx * p.x + vy * p.y + vz * p.z;
            const float px = fmaf(radial, p.x, (vx - vr * p.x) * p.rinv);
            const float py = fmaf(radial, p.y, (vy - vr * p.y) * p.rinv);
            const float pz = fmaf(radial, p.z, (vz - vr * p.z) * p.rinv);
            fx += px; fy += py; fz += pz;
            const int64_t jb = L.bbase + p.jl;
            atomicAdd(a.b.F + jb, -px); atomicAdd(a.b.F + a.b.NBP + jb, -py); atomicAdd(a.b.F + 2 * a.b.NBP + jb, -pz);
            w[0] = fmaf(-p.dx, px, w[0]); w[1] = fmaf(-p.dx, py, w[1]); w[2] = fmaf(-p.dx, pz, w[2]);
            w[3] = fmaf(-p.dy, px, w[3]); w[4] = fmaf(-p.dy, py, w[4]); w[5] = fmaf(-p.dy, pz, w[5]);
            w[6] = fmaf(-p.dz, px, w[6]); w[7] = fmaf(-p.dz, py, w[7]); w[8] = fmaf(-p.dz, pz, w[8]);
        }
    }
    if (L.ti >= 0) {
        atomicAdd(a.b.F + L.ib, fx); atomicAdd(a.b.F + a.b.NBP + L.ib, fy); atomicAdd(a.b.F + 2 * a.b.NBP + L.ib, fz);
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) {
        const float v = warp_sum(w[k]);
        if (L.lane == 0) atomicAdd(a.b.Ws + 9 * L.sb + k, v);
    }
}

// ------------------------------------------------------------------------------------------------
// outputs in batch order, scaler, descriptors
// ------------------------------------------------------------------------------------------------
__global__ void k_gather_outputs(StepArgs a, float* E, float* F, float* W)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < a.b.Sb) {
        if (E) E[i] = (float)a.b.Es[i];
        if (W) for (int k = 0; k < 9; ++k) W[9 * i + k] = a.b.Ws[9 * i + k];
    }
    if (F && i < a.b.NBP) {
        const int w = (int)(i >> 5);
        const int64_t ip = (int64_t)a.b.bslice[w] * WARP + (i & 31);
        if (a.d.type_p[ip] >= 0) {
            const int64_t o = a.b.bfoff[a.b.bsb[w]] + (i - a.b.bbase[w]);
            F[3 * o] = a.b.F[i]; F[3 * o + 1] = a.b.F[a.b.NBP + i]; F[3 * o + 2] = a.b.F[2 * a.b.NBP + i];
        }
    }
}
__global__ void k_gather_q(StepArgs a, float* q)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= a.b.NBP) return;
    const int w = (int)(i >> 5);
    const int64_t ip = (int64_t)a.b.bslice[w] * WARP + (i & 31);
    if (a.d.type_p[ip] < 0) return;
    const int64_t o = a.b.bfoff[a.b.bsb[w]] + (i - a.b.bbase[w]);
    for (int v = 0; v < a.m.D; ++v) q[o * a.m.D + v] = a.b.q[(int64_t)v * a.b.NBP + i];
}
// S0c (Eq. 2): one block per descriptor component: s = 1 / (max - min), degenerate range -> 1 (DESIGN G10)
__global__ void __launch_bounds__(256) k_scaler_minmax(StepArgs a, float* s)
{
    const int v = blockIdx.x;
    float lo = INFINITY, hi = -INFINITY, am = 0.0f;
    for (int64_t i = threadIdx.x; i < a.b.NBP; i += blockDim.x) {
        const int64_t ip = (int64_t)a.b.bslice[i >> 5] * WARP + (i & 31);
        if (a.d.type_p[ip] >= 0) {
            const float x = a.b.q[(int64_t)v * a.b.NBP + i];
            lo = fminf(lo, x); hi = fmaxf(hi, x); am = fmaxf(am, fabsf(x));
        }
    }
    __shared__ float slo[256], shi[256], sam[256];
    slo[threadIdx.x] = lo; shi[threadIdx.x] = hi; sam[threadIdx.x] = am;
    __syncthreads();
    for (int o = 128; o; o >>= 1) {
        if (threadIdx.x < o) {
            slo[threadIdx.x] = fminf(slo[threadIdx.x], slo[threadIdx.x + o]);
            shi[threadIdx.x] = fmaxf(shi[threadIdx.x], shi[threadIdx.x + o]);
            sam[threadIdx.x] = fmaxf(sam[threadIdx.x], sam[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const float range = shi[0] - slo[0];
        s[v] = (a.b.Nb > 0 && range > 1e-12f * fmaxf(1.0f, sam[0])) ? 1.0f / range : 1.0f;
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
#define DISPATCH_NCH(nch, ...)              \
    switch (nch) {                           \
    case 2: { constexpr int NCH = 2; __VA_ARGS__; } break; \
    case 3: { constexpr int NCH = 3; __VA_ARGS__; } break; \
    case 4: { constexpr int NCH = 4; __VA_ARGS__; } break; \
    default: { constexpr int NCH = 5; __VA_ARGS__; } break; \
    }
#define DISPATCH_K(K, ...)                  \
    if ((K) <= 9) { constexpr int KMAX = 9; __VA_ARGS__; } \
    else if ((K) <= 13) { constexpr int KMAX = 13; __VA_ARGS__; } \
    else { constexpr int KMAX = 17; __VA_ARGS__; }

int launch_forward(nep_ctx* c, bool descriptors_only)
{
    const ModelDev& m = c->m;
    const BatchDev& b = c->b;
    if (b.nbs == 0) return NEP_OK;
    const int nch = pick_nch(m.nA);
    StepArgs a = make_args(c, nch);
    const int WPB = 4, TB = WPB * WARP;
    const unsigned gx = (unsigned)((b.nbs + WPB - 1) / WPB);
    NEP_CUDA(c, cudaMemsetAsync(b.Es, 0, 8 * (size_t)b.Sb, c->stream));
    NEP_CUDA(c, cudaMemsetAsync(b.Ws, 0, 36 * (size_t)b.Sb, c->stream));
    {
        const size_t smem = 4 * (size_t)(m.T * m.T * m.nR * m.KR);
        if (smem > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(k_radial_q, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        NEP_LAUNCH(c, "k_radial_q", k_radial_q, gx, TB, smem, a);
    }
    const size_t smemA = 4 * (size_t)(m.T * m.T * m.KA * a.nAP);
    DISPATCH_NCH(nch, {
        if (smemA > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(k_ang_fwd<NCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smemA));
        NEP_LAUNCH(c, "k_ang_fwd", k_ang_fwd<NCH>, dim3(gx, a.nchunks), TB, smemA, a);
    });
    if (descriptors_only) return NEP_OK;
    {
        // pick the largest block whose shared memory fits
        int blk = 128;
        while (blk > 32 && 4 * (size_t)ann_smem_layout(m, blk).total > (size_t)c->max_smem_optin) blk >>= 1;
        const size_t smem = 4 * (size_t)ann_smem_layout(m, blk).total;
        if (smem > (size_t)c->max_smem_optin) return fail(c, NEP_ECAPACITY, "network weights do not fit in shared memory");
        const unsigned g = (unsigned)(((int64_t)b.nbs * WARP + blk - 1) / blk);
        if (blk == 128) {
            NEP_CUDA(c, cudaFuncSetAttribute(k_ann_fwd<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            NEP_LAUNCH(c, "k_ann_fwd", k_ann_fwd<128>, g, 128, smem, a);
        } else if (blk == 64) {
            NEP_CUDA(c, cudaFuncSetAttribute(k_ann_fwd<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            NEP_LAUNCH(c, "k_ann_fwd", k_ann_fwd<64>, g, 64, smem, a);
        } else {
            NEP_CUDA(c, cudaFuncSetAttribute(k_ann_fwd<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            NEP_LAUNCH(c, "k_ann_fwd", k_ann_fwd<32>, g, 32, smem, a);
        }
    }
    DISPATCH_K(m.KR, { NEP_LAUNCH(c, "k_rad_force", k_rad_force<KMAX>, gx, TB, 0, a); });
    DISPATCH_NCH(nch, {
        if (smemA > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(k_ang_force<NCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smemA));
        NEP_LAUNCH(c, "k_ang_force", k_ang_force<NCH>, dim3(gx, a.nchunks), TB, smemA, a);
    });
    return NEP_OK;
}

int launch_scaler_minmax(nep_ctx* c, float* d_s)
{
    StepArgs a = make_args(c, pick_nch(c->m.nA));
    NEP_CUDA(c, cudaMemsetAsync(d_s, 0, 4 * (size_t)c->m.DP, c->stream));
    NEP_LAUNCH(c, "k_scaler_minmax", k_scaler_minmax, c->m.D, 256, 0, a, d_s);
    return NEP_OK;
}

int launch_gather_outputs(nep_ctx* c, float* dE, float* dF, float* dW)
{
    StepArgs a = make_args(c, pick_nch(c->m.nA));
    const int64_t n = std::max<int64_t>(c->b.NBP, c->b.Sb);
    if (n == 0) return NEP_OK;
    NEP_LAUNCH(c, "k_gather_outputs", k_gather_outputs, (unsigned)((n + 255) / 256), 256, 0, a, dE, dF, dW);
    return NEP_OK;
}

int launch_gather_q(nep_ctx* c, float* dq)
{
    StepArgs a = make_args(c, pick_nch(c->m.nA));
    if (c->b.NBP == 0) return NEP_OK;
    NEP_LAUNCH(c, "k_gather_q", k_gather_q, (unsigned)((c->b.NBP + 255) / 256), 256, 0, a, dq);
    return NEP_OK;
}

}  // namespace nep
