// nep_backward.cu -- S6-S9 of the training step: loss and seeds (Eqs. 4-7), the tangent sweep along
// d~_ij = u_i - u_j - G^T d_ij (the second-order path of P:145; DESIGN C10), the network tangent/adjoint with the
// network-weight gradient (C11), and the adjoint sweep giving the descriptor-coefficient gradient (C12).
#include <algorithm>

#include "nep_kernels.cuh"

namespace nep {

// ------------------------------------------------------------------------------------------------
// S6: loss terms and seeds
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_loss_struct(StepArgs a, float lamE, float lamV)
{
    const int sb = blockIdx.x * blockDim.x + threadIdx.x;
    double sE = 0.0, sW = 0.0;
    if (sb < a.b.Sb) {
        const int sid = a.b.bsid[sb];
        const double n = (double)a.b.bnat[sb];
        const double dE = a.b.Es[sb] - a.d.Elab[sid];
        sE = (dE / n) * (dE / n);                                                   // Eq. 5
        const float eps = (float)(2.0 * lamE * dE / ((double)a.b.Sb * n * n));
        a.b.eps[sb] = eps;
        atomicAdd(a.g + a.m.o_b1, -eps * (float)n);                                 // g_b1 = -sum_i eps_s
        const bool hv = a.d.hasv[sid] != 0;
        for (int k = 0; k < 9; ++k) {
            const double t = hv ? (double)a.b.Ws[9 * sb + k] - (double)a.d.Wlab[9 * (int64_t)sid + k] : 0.0;
            sW += (t / n) * (t / n);                                                // Eq. 7
            a.b.G[9 * sb + k] = (hv && a.b.Sv > 0) ? (float)(2.0 * lamV * t / (9.0 * a.b.Sv * n * n)) : 0.0f;
        }
    }
    sE = warp_sum(sE); sW = warp_sum(sW);
    if ((threadIdx.x & 31) == 0) { atomicAdd(a.b.lacc + 0, sE); atomicAdd(a.b.lacc + 2, sW); }
}

__global__ void __launch_bounds__(256) k_loss_atom(StepArgs a, float lamF)
{
    const int64_t ib = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double sF = 0.0;
    if (ib < a.b.NBP) {
        const int64_t ip = (int64_t)a.b.bslice[ib >> 5] * WARP + (ib & 31);
        const float c = 2.0f * lamF / (3.0f * (float)a.b.Nb);
        const bool valid = a.d.type_p[ip] >= 0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const float dF = valid ? a.b.F[k * a.b.NBP + ib] - a.d.Flab[k * a.d.NP + ip] : 0.0f;
            sF += (double)dF * (double)dF;                                          // Eq. 6
            a.b.u[k * a.b.NBP + ib] = c * dF;
        }
    }
    sF = warp_sum(sF);
    if ((threadIdx.x & 31) == 0) atomicAdd(a.b.lacc + 1, sF);
}

__global__ void k_loss_final(StepArgs a, double lamE, double lamF, double lamV)
{
    double* l = a.b.lacc;
    const double dE = a.b.Sb ? l[0] / a.b.Sb : 0.0, dF = a.b.Nb ? l[1] / (3.0 * a.b.Nb) : 0.0, dV = a.b.Sv ? l[2] / (9.0 * a.b.Sv) : 0.0;
    l[4] = lamE * dE + lamF * dF + lamV * dV; l[5] = dE; l[6] = dF; l[7] = dV;       // Eq. 4
}

// d~ = u_i - u_j - G^T d ;  returns t = r^ . d~ and (optionally) the tangent rho = (d~ - t r^) / r of r^
struct Tangent { float t, rx, ry, rz; };
__device__ __forceinline__ Tangent pair_tangent(const StepArgs& a, const PairGeo& p, int64_t jb, float uix, float uiy, float uiz, const float* G)
{
    const float ujx = __ldg(a.b.u + jb), ujy = __ldg(a.b.u + a.b.NBP + jb), ujz = __ldg(a.b.u + 2 * a.b.NBP + jb);
    const float tx = uix - ujx - (G[0] * p.dx + G[3] * p.dy + G[6] * p.dz);
    const float ty = uiy - ujy - (G[1] * p.dx + G[4] * p.dy + G[7] * p.dz);
    const float tz = uiz - ujz - (G[2] * p.dx + G[5] * p.dy + G[8] * p.dz);
    Tangent T;
    T.t = tx * p.x + ty * p.y + tz * p.z;
    T.rx = (tx - T.t * p.x) * p.rinv; T.ry = (ty - T.t * p.y) * p.rinv; T.rz = (tz - T.t * p.z) * p.rinv;
    return T;
}

// ------------------------------------------------------------------------------------------------
// S7 (radial part): Bd_k[T'] = sum_{j, t_j = T'} f_k'(r_ij) (r^_ij . d~_ij)   (tangent of the aggregate B)
// ------------------------------------------------------------------------------------------------
template <int KMAX>
__global__ void __launch_bounds__(128) k_rad_tangent(StepArgs a)
{
    Lane L;
    if (!lane_init(a, L)) return;
    const ModelDev& m = a.m;
    const int cnt = (L.ti >= 0) ? a.d.cntR[L.ip] : 0;
    const int64_t base = a.d.recoffR[L.ds];
    const int width = (int)((a.d.recoffR[L.ds + 1] - base) >> 5);
    const float4* rec = a.d.recR + base + L.lane;
    float G[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) G[k] = a.b.G[9 * L.sb + k];
    const float uix = a.b.u[L.ib], uiy = a.b.u[a.b.NBP + L.ib], uiz = a.b.u[2 * a.b.NBP + L.ib];
    float bd[KMAX];
#pragma unroll
    for (int k = 0; k < KMAX; ++k) bd[k] = 0.0f;
    int cur = -1;
    for (int s = 0; s < width; ++s) {
        const float4 rc4 = rec[(int64_t)s * WARP];
        if (s < cnt) {
            const PairGeo p = pair_geo(rc4);
            if (p.tj != cur) {
                if (cur >= 0) {
#pragma unroll
                    for (int k = 0; k < KMAX; ++k)
                        if (k < m.KR) { a.b.Bd[(int64_t)(cur * m.KR + k) * a.b.NBP + L.ib] = bd[k]; bd[k] = 0.0f; }
                }
                cur = p.tj;
            }
            const Tangent T = pair_tangent(a, p, L.bbase + p.jl, uix, uiy, uiz, G);
            cheb_foreach<KMAX>(p.r, m.rcinvR, m.KR, [&](int k, float, float dfk) { bd[k] = fmaf(dfk, T.t, bd[k]); });
        }
    }
    if (cur >= 0) {
#pragma unroll
        for (int k = 0; k < KMAX; ++k)
            if (k < m.KR) a.b.Bd[(int64_t)(cur * m.KR + k) * a.b.NBP + L.ib] = bd[k];
    }
}

// ------------------------------------------------------------------------------------------------
// S7 (angular part): Sd_nL = sum_j [g_n' (r^.d~) b_L + g_n (grad b_L . d~)],  qd_ang = J_q(S) Sd
// ------------------------------------------------------------------------------------------------
template <int NCH>
__global__ void __launch_bounds__(128) k_ang_tangent(StepArgs a)
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
    float G[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) G[k] = a.b.G[9 * L.sb + k];
    const float uix = a.b.u[L.ib], uiy = a.b.u[a.b.NBP + L.ib], uiz = a.b.u[2 * a.b.NBP + L.ib];
    float Sd[NCH][NL];
#pragma unroll
    for (int n = 0; n < NCH; ++n)
#pragma unroll
        for (int l = 0; l < NL; ++l) Sd[n][l] = 0.0f;
    for (int s = 0; s < width; ++s) {
        const float4 rc4 = rec[(int64_t)s * WARP];
        if (s < cnt) {
            const PairGeo p = pair_geo(rc4);
            const Tangent T = pair_tangent(a, p, L.bbase + p.jl, uix, uiy, uiz, G);
            float g[NCH], dg[NCH];
            radial_gn<NCH, true>(p.r, m.rcinvA, m.KA, cs + (L.ti * m.T + p.tj) * m.KA * a.nAP + n0, a.nAP, g, dg);
            float b[NL], bd[NL];
            const HarmZ hz = harm_z(p.z);
            const HarmXY hxy = harm_xy(p.x, p.y);
            harm24(hz, hxy, b);
            harm24_tangent(hz, hxy, T.rx, T.ry, T.rz, bd);
#pragma unroll
            for (int n = 0; n < NCH; ++n) {
                const float c1 = dg[n] * T.t;
#pragma unroll
                for (int l = 0; l < NL; ++l) Sd[n][l] = fmaf(c1, b[l], fmaf(g[n], bd[l], Sd[n][l]));
            }
        }
    }
#pragma unroll
    for (int n = 0; n < NCH; ++n) {
        if (n0 + n < m.nA) {
            float S[NL], qd[6];
#pragma unroll
            for (int l = 0; l < NL; ++l) {
                S[l] = a.b.S[(int64_t)((n0 + n) * NL + l) * a.b.NBP + L.ib];
                a.b.Sd[(int64_t)((n0 + n) * NL + l) * a.b.NBP + L.ib] = Sd[n][l];
            }
            inv_tangent(S, Sd[n], m.has4, m.has5, qd);
            for (int aa = 0; aa < m.nang; ++aa) a.b.qd[(int64_t)(m.nR + aa * m.nA + n0 + n) * a.b.NBP + L.ib] = qd[aa];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S8: network tangent and adjoint per atom (phase 1, thread = atom), then the block reduces the outer
// products into the gradient of w0, b0, w1 and cR (phase 2, thread = 4x4 output tile), one global atomic
// per output and block.
// ------------------------------------------------------------------------------------------------
struct BwdSmem {
    int w0, w1, sc, cR, gcol, ecol, wcol, qt, qds, qbr, fpr, bc, bdc, typ, total, ld;
};
__host__ __device__ inline BwdSmem bwd_smem_layout(const ModelDev& m, int BLK)
{
    BwdSmem s;
    s.ld = BLK + 1;   // padded row length: conflict-free both for column (thread = atom) and row (thread = tile) access
    int o = 0;
    s.w0 = o; o += m.T * m.HP * m.DP;
    s.w1 = o; o += m.T * m.HP;
    s.sc = o; o += m.DP;
    s.cR = o; o += (m.T * m.T * m.nR * m.KR + 3) & ~3;
    s.gcol = o; o += m.HP * s.ld;
    s.ecol = o; o += m.HP * s.ld;
    s.wcol = o; o += m.HP * s.ld;
    s.qt = o; o += m.DP * s.ld;
    s.qds = o; o += m.DP * s.ld;
    s.qbr = o; o += m.nR * s.ld;
    s.fpr = o; o += m.nR * s.ld;
    s.bc = o; o += m.T * m.KR * s.ld;
    s.bdc = o; o += m.T * m.KR * s.ld;
    s.typ = o; o += BLK;
    s.total = o;
    return s;
}

template <int BLK>
__global__ void __launch_bounds__(BLK) k_ann_bwd(StepArgs a)
{
    extern __shared__ __align__(16) float sm[];
    const ModelDev& m = a.m;
    const BwdSmem lay = bwd_smem_layout(m, BLK);
    const int tid = threadIdx.x, ld = lay.ld;
    for (int i = tid; i < m.T * m.HP * m.DP; i += BLK) {
        const int v = i % m.DP, mu = (i / m.DP) % m.HP, t = i / (m.DP * m.HP);
        sm[lay.w0 + i] = (v < m.D && mu < m.H) ? a.theta[t * m.per_type + mu * m.D + v] : 0.0f;
    }
    for (int i = tid; i < m.T * m.HP; i += BLK) {
        const int mu = i % m.HP, t = i / m.HP;
        sm[lay.w1 + i] = (mu < m.H) ? a.theta[t * m.per_type + m.H * m.D + m.H + mu] : 0.0f;
    }
    for (int i = tid; i < m.DP; i += BLK) sm[lay.sc + i] = (i < m.D) ? a.scaler[i] : 0.0f;
    for (int i = tid; i < m.T * m.T * m.nR * m.KR; i += BLK) sm[lay.cR + i] = a.theta[m.o_cR + i];
    __syncthreads();

    // ---------------- phase 1 ----------------
    const int w = (int)((blockIdx.x * (int64_t)BLK + tid) >> 5);
    int ti = -1;
    int64_t ib = 0, ip = 0;
    int sb = 0;
    if (w < a.b.nbs) {
        ib = (int64_t)w * WARP + (tid & 31);
        ip = (int64_t)a.b.bslice[w] * WARP + (tid & 31);
        ti = a.d.type_p[ip];
        sb = a.b.bsb[w];
    }
    int* typ = reinterpret_cast<int*>(sm + lay.typ);
    typ[tid] = ti;
    float* gcol = sm + lay.gcol + tid; float* ecol = sm + lay.ecol + tid; float* wcol = sm + lay.wcol + tid;
    float* qt = sm + lay.qt + tid;     float* qds = sm + lay.qds + tid;
    if (ti >= 0) {
        const float eps = a.b.eps[sb];
        const int TK = m.T * m.KR;
        for (int k = 0; k < TK; ++k) {
            sm[lay.bc + k * ld + tid] = a.d.B[(int64_t)k * a.d.NP + ip];
            sm[lay.bdc + k * ld + tid] = a.b.Bd[(int64_t)k * a.b.NBP + ib];
        }
        for (int v = 0; v < m.DP; ++v) {
            float qv = 0.0f, qdv = 0.0f;
            if (v < m.D) {
                qv = a.b.q[(int64_t)v * a.b.NBP + ib];
                if (v < m.nR) {   // radial tangent from the aggregate: qd_n = sum cR[ti][tj][n][k] Bd_k[tj]
                    for (int tj = 0; tj < m.T; ++tj) {
                        const float* cc = sm + lay.cR + ((ti * m.T + tj) * m.nR + v) * m.KR;
                        for (int k = 0; k < m.KR; ++k) qdv = fmaf(cc[k], sm[lay.bdc + (tj * m.KR + k) * ld + tid], qdv);
                    }
                    sm[lay.fpr + v * ld + tid] = a.b.Fp[(int64_t)v * a.b.NBP + ib];
                } else {
                    qdv = a.b.qd[(int64_t)v * a.b.NBP + ib];
                }
            }
            qt[v * ld] = sm[lay.sc + v] * qv;
            qds[v * ld] = sm[lay.sc + v] * qdv;
        }
        const float* w0 = sm + lay.w0 + ti * m.HP * m.DP;
        const float* w1 = sm + lay.w1 + ti * m.HP;
        for (int mu0 = 0; mu0 < m.HP; mu0 += 8) {
            float acc[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[j] = 0.0f;
            for (int v = 0; v < m.DP; v += 4) {
                const float q0 = qds[v * ld], q1 = qds[(v + 1) * ld], q2 = qds[(v + 2) * ld], q3 = qds[(v + 3) * ld];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const float4 ww = *reinterpret_cast<const float4*>(w0 + (mu0 + j) * m.DP + v);
                    acc[j] = fmaf(ww.x, q0, fmaf(ww.y, q1, fmaf(ww.z, q2, fmaf(ww.w, q3, acc[j]))));
                }
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int mu = mu0 + j;
                const float h = (mu < m.H) ? a.b.h[(int64_t)mu * a.b.NBP + ib] : 0.0f;
                const float omh2 = 1.0f - h * h;
                const float e = w1[mu] * omh2;
                const float xd = acc[j];
                const float gam = fmaf(eps, e, -2.0f * h * e * xd);
                gcol[mu * ld] = gam;
                ecol[mu * ld] = e;
                wcol[mu * ld] = fmaf(eps, h, omh2 * xd);
            }
        }
        for (int v0 = 0; v0 < m.DP; v0 += 8) {
            float acc[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[j] = 0.0f;
            for (int mu = 0; mu < m.HP; ++mu) {
                const float gm = gcol[mu * ld];
                const float4 wa = *reinterpret_cast<const float4*>(w0 + mu * m.DP + v0);
                const float4 wb = *reinterpret_cast<const float4*>(w0 + mu * m.DP + v0 + 4);
                acc[0] = fmaf(gm, wa.x, acc[0]); acc[1] = fmaf(gm, wa.y, acc[1]); acc[2] = fmaf(gm, wa.z, acc[2]); acc[3] = fmaf(gm, wa.w, acc[3]);
                acc[4] = fmaf(gm, wb.x, acc[4]); acc[5] = fmaf(gm, wb.y, acc[5]); acc[6] = fmaf(gm, wb.z, acc[6]); acc[7] = fmaf(gm, wb.w, acc[7]);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int v = v0 + j;
                if (v < m.D) {
                    const float qb = sm[lay.sc + v] * acc[j];
                    a.b.Qb[(int64_t)v * a.b.NBP + ib] = qb;
                    if (v < m.nR) sm[lay.qbr + v * ld + tid] = qb;
                }
            }
        }
    }
    __syncthreads();

    // ---------------- phase 2 ----------------
    const int tilesH = m.HP / 4, tilesD = m.DP / 4, ntiles = tilesH * tilesD;
    for (int t = 0; t < m.T; ++t) {
        bool present = false;
        for (int aidx = 0; aidx < BLK; ++aidx) present |= (typ[aidx] == t);   // uniform
        if (!present) continue;
        // g_w0[t][mu][v] += sum_a gamma_mu q~_v + e_mu (s qd)_v
        for (int tile = tid; tile < ntiles; tile += BLK) {
            const int mu0 = (tile / tilesD) * 4, v0 = (tile % tilesD) * 4;
            float acc[4][4];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = 0.0f;
            for (int aidx = 0; aidx < BLK; ++aidx) {
                if (typ[aidx] != t) continue;
                float gm[4], ee[4], qq[4], qd[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    gm[i] = sm[lay.gcol + (mu0 + i) * ld + aidx]; ee[i] = sm[lay.ecol + (mu0 + i) * ld + aidx];
                    qq[i] = sm[lay.qt + (v0 + i) * ld + aidx];    qd[i] = sm[lay.qds + (v0 + i) * ld + aidx];
                }
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(gm[i], qq[j], fmaf(ee[i], qd[j], acc[i][j]));
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (mu0 + i < m.H && v0 + j < m.D) atomicAdd(a.g + t * m.per_type + (mu0 + i) * m.D + v0 + j, acc[i][j]);
        }
        // g_b0[t][mu] -= sum_a gamma_mu ; g_w1[t][mu] += sum_a (eps h + (1-h^2) xd)
        for (int mu = tid; mu < m.H; mu += BLK) {
            float sg = 0.0f, sw = 0.0f;
            for (int aidx = 0; aidx < BLK; ++aidx)
                if (typ[aidx] == t) { sg += sm[lay.gcol + mu * ld + aidx]; sw += sm[lay.wcol + mu * ld + aidx]; }
            atomicAdd(a.g + t * m.per_type + m.H * m.D + mu, -sg);
            atomicAdd(a.g + t * m.per_type + m.H * m.D + m.H + mu, sw);
        }
        // g_cR[t][tj][n][k] += sum_a Qb_n B_k[tj] + Fp_n Bd_k[tj]
        const int nout = m.T * m.nR * m.KR;
        for (int o = tid; o < nout; o += BLK) {
            const int k = o % m.KR, n = (o / m.KR) % m.nR, tj = o / (m.KR * m.nR);
            float s = 0.0f;
            for (int aidx = 0; aidx < BLK; ++aidx)
                if (typ[aidx] == t)
                    s = fmaf(sm[lay.qbr + n * ld + aidx], sm[lay.bc + (tj * m.KR + k) * ld + aidx],
                             fmaf(sm[lay.fpr + n * ld + aidx], sm[lay.bdc + (tj * m.KR + k) * ld + aidx], s));
            atomicAdd(a.g + m.o_cR + ((t * m.T + tj) * m.nR + n) * m.KR + k, s);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S9: adjoint sweep for the angular coefficients:
//   g_cA[ti][tj][n][k] += [sum_L Sb_nL b_L + sum_L EdS_nL (grad b_L . d~)] f_k + [sum_L EdS_nL b_L] (r^.d~) f_k'
// pass 1 holds Sb = J^T Qb + Fp H Sd in registers, pass 2 holds EdS = dE_i/dS.  Per-thread accumulators
// acc[n][k] are flushed when the neighbour type changes (records are sorted by type).
// ------------------------------------------------------------------------------------------------
template <int NCH, int KMAX>
__device__ __forceinline__ void flush_acc(const StepArgs& a, float* gs, int ti, int tj, int n0, float (*acc)[KMAX])
{
    const ModelDev& m = a.m;
#pragma unroll
    for (int n = 0; n < NCH; ++n)
#pragma unroll
        for (int k = 0; k < KMAX; ++k) {
            if (k < m.KA && n0 + n < m.nA) atomicAdd(gs + ((ti * m.T + tj) * m.nA + n0 + n) * m.KA + k, acc[n][k]);
            acc[n][k] = 0.0f;
        }
}

template <int NCH, int KMAX>
__global__ void __launch_bounds__(128) k_ang_adjoint(StepArgs a)
{
    extern __shared__ float smem[];
    const ModelDev& m = a.m;
    float* cs = smem;                                  // cA as [pt][k][nAP]
    float* gs = smem + m.T * m.T * m.KA * a.nAP;         // block accumulator, theta layout [pt][n][k]
    load_cA_smem(a, cs);
    const int ngs = m.T * m.T * m.nA * m.KA;
    for (int i = threadIdx.x; i < ngs; i += blockDim.x) gs[i] = 0.0f;
    __syncthreads();
    Lane L;
    const bool active = lane_init(a, L);
    const int n0 = blockIdx.y * NCH;
    if (active) {
        const int cnt = (L.ti >= 0) ? a.d.cntA[L.ip] : 0;
        const int64_t base = a.d.recoffA[L.ds];
        const int width = (int)((a.d.recoffA[L.ds + 1] - base) >> 5);
        const float4* rec = a.d.recA + base + L.lane;
        const bool uniform = (m.T == 1);
        float acc[NCH][KMAX];
#pragma unroll
        for (int n = 0; n < NCH; ++n)
#pragma unroll
            for (int k = 0; k < KMAX; ++k) acc[n][k] = 0.0f;
        float X[NCH][NL];
        // ---- pass 1: Sb ----
#pragma unroll
        for (int n = 0; n < NCH; ++n) {
            if (n0 + n < m.nA && L.ti >= 0) {
                float S[NL], Sd[NL], cq[6], cf[6];
#pragma unroll
                for (int l = 0; l < NL; ++l) {
                    S[l] = a.b.S[(int64_t)((n0 + n) * NL + l) * a.b.NBP + L.ib];
                    Sd[l] = a.b.Sd[(int64_t)((n0 + n) * NL + l) * a.b.NBP + L.ib];
                }
#pragma unroll
                for (int aa = 0; aa < 6; ++aa) {
                    const int64_t idx = (int64_t)(m.nR + aa * m.nA + n0 + n) * a.b.NBP + L.ib;
                    cq[aa] = (aa < m.nang) ? a.b.Qb[idx] : 0.0f;
                    cf[aa] = (aa < m.nang) ? a.b.Fp[idx] : 0.0f;
                }
                inv_adjoint(S, m.has4, m.has5, cq, X[n]);
                inv_hessian_action(S, Sd, m.has4, m.has5, cf, X[n]);
            } else {
#pragma unroll
                for (int l = 0; l < NL; ++l) X[n][l] = 0.0f;
            }
        }
        int cur = -1;
        for (int s = 0; s < width; ++s) {
            const float4 rc4 = rec[(int64_t)s * WARP];
            if (s < cnt) {
                const PairGeo p = pair_geo(rc4);
                if (!uniform && p.tj != cur) {
                    if (cur >= 0) flush_acc<NCH, KMAX>(a, gs, L.ti, cur, n0, acc);
                    cur = p.tj;
                }
                float b[NL], al[NCH];
                harm24(harm_z(p.z), harm_xy(p.x, p.y), b);
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    float s1 = 0.0f;
#pragma unroll
                    for (int l = 0; l < NL; ++l) s1 = fmaf(X[n][l], b[l], s1);
                    al[n] = s1;
                }
                cheb_foreach<KMAX>(p.r, m.rcinvA, m.KA, [&](int k, float fk, float) {
#pragma unroll
                    for (int n = 0; n < NCH; ++n) acc[n][k] = fmaf(al[n], fk, acc[n][k]);
                });
            }
        }
        if (!uniform && cur >= 0) flush_acc<NCH, KMAX>(a, gs, L.ti, cur, n0, acc);
        // ---- pass 2: EdS ----
        load_EdS<NCH>(a, L, n0, X);
        float G[9];
#pragma unroll
        for (int k = 0; k < 9; ++k) G[k] = a.b.G[9 * L.sb + k];
        const float uix = a.b.u[L.ib], uiy = a.b.u[a.b.NBP + L.ib], uiz = a.b.u[2 * a.b.NBP + L.ib];
        cur = -1;
        for (int s = 0; s < width; ++s) {
            const float4 rc4 = rec[(int64_t)s * WARP];
            if (s < cnt) {
                const PairGeo p = pair_geo(rc4);
                if (!uniform && p.tj != cur) {
                    if (cur >= 0) flush_acc<NCH, KMAX>(a, gs, L.ti, cur, n0, acc);
                    cur = p.tj;
                }
                const Tangent T = pair_tangent(a, p, L.bbase + p.jl, uix, uiy, uiz, G);
                float b[NL], bd[NL], be[NCH], de[NCH];
                const HarmZ hz = harm_z(p.z);
                const HarmXY hxy = harm_xy(p.x, p.y);
                harm24(hz, hxy, b);
                harm24_tangent(hz, hxy, T.rx, T.ry, T.rz, bd);
#pragma unroll
                for (int n = 0; n < NCH; ++n) {
                    float s1 = 0.0f, s2 = 0.0f;
#pragma unroll
                    for (int l = 0; l < NL; ++l) { s1 = fmaf(X[n][l], b[l], s1); s2 = fmaf(X[n][l], bd[l], s2); }
                    be[n] = s1 * T.t; de[n] = s2;
                }
                cheb_foreach<KMAX>(p.r, m.rcinvA, m.KA, [&](int k, float fk, float dfk) {
#pragma unroll
                    for (int n = 0; n < NCH; ++n) acc[n][k] = fmaf(de[n], fk, fmaf(be[n], dfk, acc[n][k]));
                });
            }
        }
        if (!uniform) {
            if (cur >= 0) flush_acc<NCH, KMAX>(a, gs, L.ti, cur, n0, acc);
        } else {
            // single species: every lane targets the same block of coefficients -> shuffle-reduce, one lane adds
#pragma unroll
            for (int n = 0; n < NCH; ++n)
#pragma unroll
                for (int k = 0; k < KMAX; ++k) {
                    const float v = warp_sum(acc[n][k]);
                    if (L.lane == 0 && k < m.KA && n0 + n < m.nA) atomicAdd(gs + (n0 + n) * m.KA + k, v);
                }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < ngs; i += blockDim.x) {
        const int n = (i / m.KA) % m.nA;
        if (n >= n0 && n < n0 + NCH) atomicAdd(a.g + m.o_cA + i, gs[i]);
    }
}

// ------------------------------------------------------------------------------------------------
// launcher
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

int launch_loss_grad(nep_ctx* c)
{
    const ModelDev& m = c->m;
    const BatchDev& b = c->b;
    NEP_CUDA(c, cudaMemsetAsync(c->g, 0, 4 * (size_t)m.npar, c->stream));
    NEP_CUDA(c, cudaMemsetAsync(b.lacc, 0, 64, c->stream));
    const int nch = pick_nch(m.nA);
    StepArgs a = make_args(c, nch);
    if (b.nbs == 0) {
        NEP_LAUNCH(c, "k_loss_final", k_loss_final, 1, 1, 0, a, c->lamE, c->lamF, c->lamV);
        return NEP_OK;
    }
    NEP_CUDA(c, cudaMemsetAsync(b.Bd, 0, 4 * (size_t)b.NBP * m.T * m.KR, c->stream));
    const int WPB = 4, TB = WPB * WARP;
    const unsigned gx = (unsigned)((b.nbs + WPB - 1) / WPB);
    NEP_LAUNCH(c, "k_loss_struct", k_loss_struct, (unsigned)((b.Sb + 127) / 128), 128, 0, a, (float)c->lamE, (float)c->lamV);
    NEP_LAUNCH(c, "k_loss_atom", k_loss_atom, (unsigned)((b.NBP + 255) / 256), 256, 0, a, (float)c->lamF);
    NEP_LAUNCH(c, "k_loss_final", k_loss_final, 1, 1, 0, a, c->lamE, c->lamF, c->lamV);
    DISPATCH_K(m.KR, { NEP_LAUNCH(c, "k_rad_tangent", k_rad_tangent<KMAX>, gx, TB, 0, a); });
    const size_t smemA = 4 * (size_t)(m.T * m.T * m.KA * a.nAP);
    DISPATCH_NCH(nch, {
        if (smemA > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(k_ang_tangent<NCH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smemA));
        NEP_LAUNCH(c, "k_ang_tangent", k_ang_tangent<NCH>, dim3(gx, a.nchunks), TB, smemA, a);
    });
    {
        int blk = 128;
        while (blk > 32 && 4 * (size_t)bwd_smem_layout(m, blk).total > (size_t)c->max_smem_optin) blk >>= 1;
        const size_t smem = 4 * (size_t)bwd_smem_layout(m, blk).total;
        if (smem > (size_t)c->max_smem_optin) return fail(c, NEP_ECAPACITY, "network weights do not fit in shared memory");
        const unsigned g = (unsigned)(((int64_t)b.nbs * WARP + blk - 1) / blk);
        if (blk == 128) {
            NEP_CUDA(c, cudaFuncSetAttribute(k_ann_bwd<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            NEP_LAUNCH(c, "k_ann_bwd", k_ann_bwd<128>, g, 128, smem, a);
        } else if (blk == 64) {
            NEP_CUDA(c, cudaFuncSetAttribute(k_ann_bwd<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            NEP_LAUNCH(c, "k_ann_bwd", k_ann_bwd<64>, g, 64, smem, a);
        } else {
            NEP_CUDA(c, cudaFuncSetAttribute(k_ann_bwd<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            NEP_LAUNCH(c, "k_ann_bwd", k_ann_bwd<32>, g, 32, smem, a);
        }
    }
    const size_t smemD = smemA + 4 * (size_t)(m.T * m.T * m.nA * m.KA);
    DISPATCH_NCH(nch, {
        DISPATCH_K(m.KA, {
            auto kern = k_ang_adjoint<NCH, KMAX>;
            if (smemD > 48 * 1024) NEP_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smemD));
            NEP_LAUNCH(c, "k_ang_adjoint", kern, dim3(gx, a.nchunks), TB, smemD, a);
        });
    });
    return NEP_OK;
}

}  // namespace nep
