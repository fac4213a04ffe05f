// nep_math.cuh -- device-side fp32 building blocks of the NEP descriptor (sm_100a).
//
// Radial basis: Eqs. 17-18.  Angular functions: the 24 real harmonics l = 1..4 of Eq. 19
// as expanded polynomials  b_{l,m,c/s}(r^) = N_lm P_l^{(m)}(z) Re/Im (x+iy)^m, normalised so that
// Eq. 20 reads q_nl = sum_{L in l} S_nL^2  (N_lm^2 = (2l+1)/(4 pi) * (m ? 2 (l-m)!/(l+m)! : 1)).
// 4-/5-body invariants: DESIGN.md C5 / reading G7.  This file shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace nep {

constexpr int NL = 24;  // real harmonics, l = 1..4

// index of (l, m=0) inside the 24-vector; (l, m, cos) = base[l] + 2m-1, (l, m, sin) = base[l] + 2m
__host__ __device__ constexpr int lbase(int l) { return l == 1 ? 0 : l == 2 ? 3 : l == 3 ? 8 : 15; }

// sqrt of the addition-theorem weights
constexpr float N10 = 0.48860251190291992f, N11 = 0.48860251190291992f;
constexpr float N20 = 0.63078313050504009f, N21 = 0.36418281019735971f, N22 = 0.18209140509867985f;
constexpr float N30 = 0.7463526651802308f, N31 = 0.3046971996429772f, N32 = 0.096353714754685141f, N33 = 0.0393362393284429f;
constexpr float N40 = 0.84628437532163447f, N41 = 0.26761861742291565f, N42 = 0.063078313050504001f,
                N43 = 0.016858388283618388f, N44 = 0.0059603403376112018f;
constexpr float KAPPA4 = -0.26998130975990764f;  // -45 / (8 sqrt(14) pi^{3/2})
constexpr float C5 = 7.0f / 15.0f;               // q5 = kappa5 |s|^4 = (7/15) q_{l=1}^2, kappa5 = 21/(80 pi^2)
constexpr float PI_F = 3.14159265358979323846f;

// ------------------------------------------------------------------------------------------------
// cos(pi u), sin(pi u) for u in [0, 1]  (the only range Eq. 18 needs: 0 < r < rc).
// v = u - 1/2 in [-1/2, 1/2]:  cos(pi u) = -sin(pi v), sin(pi u) = cos(pi v); Taylor polynomials in x = pi v,
// |x| <= pi/2, truncated after x^13 / x^14 (first neglected terms 5.7e-8 x and 6.4e-9): ~1 ulp of the results that
// Eqs. 17-18 use them for, at 15 FMA-pipe operations (sincospif costs ~25 with its range reduction and selects).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void sincospi_unit(float u, float& sn, float& cs)
{
    const float x = PI_F * (u - 0.5f);
    const float x2 = x * x;
    float ps = -1.0f / 6227020800.0f;                       // -1/13!
    ps = fmaf(ps, x2, 1.0f / 39916800.0f);                  //  1/11!
    ps = fmaf(ps, x2, -1.0f / 362880.0f);
    ps = fmaf(ps, x2, 1.0f / 5040.0f);
    ps = fmaf(ps, x2, -1.0f / 120.0f);
    ps = fmaf(ps, x2, 1.0f / 6.0f);
    ps = ps * x2;                                           // (x - sin x) / x
    float pc = 1.0f / 479001600.0f;                         //  1/12!
    pc = fmaf(pc, x2, -1.0f / 3628800.0f);
    pc = fmaf(pc, x2, 1.0f / 40320.0f);
    pc = fmaf(pc, x2, -1.0f / 720.0f);
    pc = fmaf(pc, x2, 1.0f / 24.0f);
    pc = fmaf(pc, x2, -0.5f);
    cs = fmaf(ps, x, -x);                                   // cos(pi u) = -sin x
    sn = fmaf(pc, x2, 1.0f);                                // sin(pi u) =  cos x
}

// ------------------------------------------------------------------------------------------------
// Chebyshev x cosine-cutoff basis (Eqs. 17-18).  body(k, f_k, df_k/dr) is called for k = 0..K-1, K a compile-time
// constant (models with fewer functions run the next larger instantiation with zero-padded coefficients).
// Without DERIV the derivative argument is 0 and its arithmetic is not generated.
// ------------------------------------------------------------------------------------------------
// The same from the special-function unit (sin.approx / cos.approx, absolute error ~1e-6): used by the sweeps of the second-order
// path, whose results enter only the parameter gradient (tolerance 1e-3 relative); 4 instructions instead of 15.
__device__ __forceinline__ void sincospi_unit_fast(float u, float& sn, float& cs)
{
    const float x = PI_F * (u - 0.5f);
    cs = -__sinf(x);
    sn = __cosf(x);
}

// scale multiplies every f_k and f_k' (they are linear in the three cutoff factors): a sweep masks a padded pair slot with scale = 0.
template <int K, bool DERIV, bool FAST = false, class Body>
__device__ __forceinline__ void cheb_basis(float r, float rcinv, Body&& body, float scale = 1.0f)
{
    const float u = r * rcinv;
    float sn, cs;
    if (FAST) sincospi_unit_fast(u, sn, cs); else sincospi_unit(u, sn, cs);
    const float hfc = fmaf(0.25f, cs, 0.25f) * scale;      // 1/2 f_c
    const float um1 = u - 1.0f;
    const float x = fmaf(2.0f * um1, um1, -1.0f);
    const float x2 = 2.0f * x;
    float hdfc = 0.0f, hdxfc = 0.0f;
    if (DERIV) {
        hdfc = (-0.25f * PI_F) * rcinv * sn * scale;       // 1/2 f_c'
        hdxfc = 4.0f * um1 * rcinv * hfc;                  // 1/2 x' f_c
    }
    float T2 = 1.0f, T1 = x, dT2 = 0.0f, dT1 = 1.0f;
    body(0, 2.0f * hfc, 2.0f * hdfc);
    if (K > 1) body(1, fmaf(x, hfc, hfc), DERIV ? fmaf(x, hdfc, hdfc + hdxfc) : 0.0f);
#pragma unroll
    for (int k = 2; k < K; ++k) {
        const float T = fmaf(x2, T1, -T2);
        float dT = 0.0f;
        if (DERIV) dT = fmaf(x2, dT1, fmaf(2.0f, T1, -dT2));
        T2 = T1; T1 = T; dT2 = dT1; dT1 = dT;
        body(k, fmaf(T, hfc, hfc), DERIV ? fmaf(dT, hdxfc, fmaf(T, hdfc, hdfc)) : 0.0f);
    }
}

// ------------------------------------------------------------------------------------------------
// Harmonics.  zp = N_lm P_l^{(m)}(z) (14 values), (c_m, s_m) = Re/Im (x+iy)^m.
// ------------------------------------------------------------------------------------------------
struct HarmZ {
    float z10, z11, z20, z21, z22, z30, z31, z32, z33, z40, z41, z42, z43, z44;
};
__device__ __forceinline__ HarmZ harm_z(float z)
{
    HarmZ h;
    const float z2 = z * z;
    h.z10 = N10 * z;                         h.z11 = N11;
    h.z20 = N20 * (1.5f * z2 - 0.5f);        h.z21 = N21 * 3.0f * z;               h.z22 = N22 * 3.0f;
    h.z30 = N30 * (2.5f * z2 - 1.5f) * z;    h.z31 = N31 * (7.5f * z2 - 1.5f);     h.z32 = N32 * 15.0f * z;  h.z33 = N33 * 15.0f;
    h.z40 = N40 * ((4.375f * z2 - 3.75f) * z2 + 0.375f);
    h.z41 = N41 * (17.5f * z2 - 7.5f) * z;   h.z42 = N42 * (52.5f * z2 - 7.5f);    h.z43 = N43 * 105.0f * z; h.z44 = N44 * 105.0f;
    return h;
}
// ratios N_lm / N_l,m+1 = sqrt((l-m)(l+m+1)) (m >= 1), sqrt(l(l+1)/2) (m = 0): d/dz [N_lm P^(m)] = ratio * [N_l,m+1 P^(m+1)]
constexpr float R10 = 1.0f;                    // sqrt(1)
constexpr float R20 = 1.7320508075688772f, R21 = 2.0f;
constexpr float R30 = 2.4494897427831779f, R31 = 3.1622776601683795f, R32 = 2.4494897427831779f;
constexpr float R40 = 3.1622776601683795f, R41 = 4.2426406871192848f, R42 = 3.7416573867739413f, R43 = 2.8284271247461903f;

struct HarmXY {
    float c1, s1, c2, s2, c3, s3, c4, s4;
};
__device__ __forceinline__ HarmXY harm_xy(float x, float y)
{
    HarmXY a;
    a.c1 = x; a.s1 = y;
    a.c2 = x * x - y * y;           a.s2 = 2.0f * x * y;
    a.c3 = x * a.c2 - y * a.s2;     a.s3 = x * a.s2 + y * a.c2;
    a.c4 = x * a.c3 - y * a.s3;     a.s4 = x * a.s3 + y * a.c3;
    return a;
}

// b[24] at the unit vector (x, y, z)
__device__ __forceinline__ void harm24(const HarmZ& h, const HarmXY& a, float* b)
{
    b[0] = h.z10;  b[1] = h.z11 * a.c1;  b[2] = h.z11 * a.s1;
    b[3] = h.z20;  b[4] = h.z21 * a.c1;  b[5] = h.z21 * a.s1;  b[6] = h.z22 * a.c2;  b[7] = h.z22 * a.s2;
    b[8] = h.z30;  b[9] = h.z31 * a.c1;  b[10] = h.z31 * a.s1; b[11] = h.z32 * a.c2; b[12] = h.z32 * a.s2;
    b[13] = h.z33 * a.c3; b[14] = h.z33 * a.s3;
    b[15] = h.z40; b[16] = h.z41 * a.c1; b[17] = h.z41 * a.s1; b[18] = h.z42 * a.c2; b[19] = h.z42 * a.s2;
    b[20] = h.z43 * a.c3; b[21] = h.z43 * a.s3; b[22] = h.z44 * a.c4; b[23] = h.z44 * a.s4;
}

// directional derivative of b[24] along a tangent rho = D r^ (rho . r^ = 0):  bd = grad_{r^} b . rho
__device__ __forceinline__ void harm24_tangent(const HarmZ& h, const HarmXY& a, float rx, float ry, float rz, float* bd)
{
    // d c_m = m (c_{m-1} rx - s_{m-1} ry),  d s_m = m (s_{m-1} rx + c_{m-1} ry)
    const float dc1 = rx, ds1 = ry;
    const float dc2 = 2.0f * (a.c1 * rx - a.s1 * ry), ds2 = 2.0f * (a.s1 * rx + a.c1 * ry);
    const float dc3 = 3.0f * (a.c2 * rx - a.s2 * ry), ds3 = 3.0f * (a.s2 * rx + a.c2 * ry);
    const float dc4 = 4.0f * (a.c3 * rx - a.s3 * ry), ds4 = 4.0f * (a.s3 * rx + a.c3 * ry);
    // d z_lm = ratio * z_{l,m+1} * rz
    const float e10 = R10 * h.z11 * rz;
    const float e20 = R20 * h.z21 * rz, e21 = R21 * h.z22 * rz;
    const float e30 = R30 * h.z31 * rz, e31 = R31 * h.z32 * rz, e32 = R32 * h.z33 * rz;
    const float e40 = R40 * h.z41 * rz, e41 = R41 * h.z42 * rz, e42 = R42 * h.z43 * rz, e43 = R43 * h.z44 * rz;
    bd[0] = e10;   bd[1] = h.z11 * dc1;                 bd[2] = h.z11 * ds1;
    bd[3] = e20;   bd[4] = fmaf(e21, a.c1, h.z21 * dc1); bd[5] = fmaf(e21, a.s1, h.z21 * ds1);
    bd[6] = h.z22 * dc2;                                bd[7] = h.z22 * ds2;
    bd[8] = e30;   bd[9] = fmaf(e31, a.c1, h.z31 * dc1); bd[10] = fmaf(e31, a.s1, h.z31 * ds1);
    bd[11] = fmaf(e32, a.c2, h.z32 * dc2);              bd[12] = fmaf(e32, a.s2, h.z32 * ds2);
    bd[13] = h.z33 * dc3;                               bd[14] = h.z33 * ds3;
    bd[15] = e40;  bd[16] = fmaf(e41, a.c1, h.z41 * dc1); bd[17] = fmaf(e41, a.s1, h.z41 * ds1);
    bd[18] = fmaf(e42, a.c2, h.z42 * dc2);              bd[19] = fmaf(e42, a.s2, h.z42 * ds2);
    bd[20] = fmaf(e43, a.c3, h.z43 * dc3);              bd[21] = fmaf(e43, a.s3, h.z43 * ds3);
    bd[22] = h.z44 * dc4;                               bd[23] = h.z44 * ds4;
}

// v = sum_L A_L grad_{r^} b_L  (reverse mode of harm24; any smooth extension off the sphere is fine because the
// caller projects v onto the tangent plane)
__device__ __forceinline__ void harm24_grad_contract(const HarmZ& h, const HarmXY& a, const float* A, float& vx, float& vy, float& vz)
{
    // z-derivatives
    vz = R10 * h.z11 * A[0];
    vz = fmaf(R20 * h.z21, A[3], vz);
    vz = fmaf(R21 * h.z22, fmaf(A[4], a.c1, A[5] * a.s1), vz);
    vz = fmaf(R30 * h.z31, A[8], vz);
    vz = fmaf(R31 * h.z32, fmaf(A[9], a.c1, A[10] * a.s1), vz);
    vz = fmaf(R32 * h.z33, fmaf(A[11], a.c2, A[12] * a.s2), vz);
    vz = fmaf(R40 * h.z41, A[15], vz);
    vz = fmaf(R41 * h.z42, fmaf(A[16], a.c1, A[17] * a.s1), vz);
    vz = fmaf(R42 * h.z43, fmaf(A[18], a.c2, A[19] * a.s2), vz);
    vz = fmaf(R43 * h.z44, fmaf(A[20], a.c3, A[21] * a.s3), vz);
    // per-m sums over l of z_lm A_{lmc}, z_lm A_{lms}
    const float a1c = fmaf(h.z11, A[1], fmaf(h.z21, A[4], fmaf(h.z31, A[9], h.z41 * A[16])));
    const float a1s = fmaf(h.z11, A[2], fmaf(h.z21, A[5], fmaf(h.z31, A[10], h.z41 * A[17])));
    const float a2c = fmaf(h.z22, A[6], fmaf(h.z32, A[11], h.z42 * A[18]));
    const float a2s = fmaf(h.z22, A[7], fmaf(h.z32, A[12], h.z42 * A[19]));
    const float a3c = fmaf(h.z33, A[13], h.z43 * A[20]);
    const float a3s = fmaf(h.z33, A[14], h.z43 * A[21]);
    const float a4c = h.z44 * A[22], a4s = h.z44 * A[23];
    // d c_m/dx = m c_{m-1}, d s_m/dx = m s_{m-1};  d c_m/dy = -m s_{m-1}, d s_m/dy = m c_{m-1}   (c_0 = 1, s_0 = 0)
    vx = a1c;
    vy = a1s;
    vx = fmaf(2.0f, fmaf(a2c, a.c1, a2s * a.s1), vx);
    vy = fmaf(2.0f, fmaf(a2s, a.c1, -a2c * a.s1), vy);
    vx = fmaf(3.0f, fmaf(a3c, a.c2, a3s * a.s2), vx);
    vy = fmaf(3.0f, fmaf(a3s, a.c2, -a3c * a.s2), vy);
    vx = fmaf(4.0f, fmaf(a4c, a.c3, a4s * a.s3), vx);
    vy = fmaf(4.0f, fmaf(a4s, a.c3, -a4c * a.s3), vy);
}

// ------------------------------------------------------------------------------------------------
// Angular invariants of one channel from its 24 normalised moments S.
// Descriptor blocks a = 0..3: l = 1..4 (Eq. 20); a = 4: 4-body; a = 5: 5-body (if enabled).
// ------------------------------------------------------------------------------------------------
struct Sym6 { float xx, yy, zz, xy, xz, yz; };

__device__ __forceinline__ Sym6 anticomm(const Sym6& A, const Sym6& B)  // A B + B A for symmetric A, B
{
    Sym6 C;
    C.xx = 2.0f * (A.xx * B.xx + A.xy * B.xy + A.xz * B.xz);
    C.yy = 2.0f * (A.xy * B.xy + A.yy * B.yy + A.yz * B.yz);
    C.zz = 2.0f * (A.xz * B.xz + A.yz * B.yz + A.zz * B.zz);
    C.xy = (A.xx * B.xy + A.xy * B.yy + A.xz * B.yz) + (B.xx * A.xy + B.xy * A.yy + B.xz * A.yz);
    C.xz = (A.xx * B.xz + A.xy * B.yz + A.xz * B.zz) + (B.xx * A.xz + B.xy * A.yz + B.xz * A.zz);
    C.yz = (A.xy * B.xz + A.yy * B.yz + A.yz * B.zz) + (B.xy * A.xz + B.yy * A.yz + B.yz * A.zz);
    return C;
}
// T = sum_j g (r^ r^T - I/3) from the normalised l = 2 moments S[3..7]
__device__ __forceinline__ Sym6 tensor_from_l2(const float* S)
{
    const float s3 = S[3] * (1.0f / N20), s4 = S[4] * (1.0f / N21), s5 = S[5] * (1.0f / N21),
                s6 = S[6] * (1.0f / N22), s7 = S[7] * (1.0f / N22);
    Sym6 T;
    T.zz = (2.0f / 3.0f) * s3;
    T.xx = fmaf(-1.0f / 3.0f, s3, s6 * (1.0f / 6.0f));
    T.yy = fmaf(-1.0f / 3.0f, s3, -s6 * (1.0f / 6.0f));
    T.xz = s4 * (1.0f / 3.0f); T.yz = s5 * (1.0f / 3.0f); T.xy = s7 * (1.0f / 6.0f);
    return T;
}
// sum_ab P_ab dT_ab/dS_L for L = 3..7 added to out[3..7], scaled by c
__device__ __forceinline__ void l2_from_tensor_adjoint(const Sym6& P, float c, float* out)
{
    out[3] = fmaf(c * (1.0f / N20), (2.0f * P.zz - P.xx - P.yy) * (1.0f / 3.0f), out[3]);
    out[4] = fmaf(c * (1.0f / N21), P.xz * (2.0f / 3.0f), out[4]);
    out[5] = fmaf(c * (1.0f / N21), P.yz * (2.0f / 3.0f), out[5]);
    out[6] = fmaf(c * (1.0f / N22), (P.xx - P.yy) * (1.0f / 6.0f), out[6]);
    out[7] = fmaf(c * (1.0f / N22), P.xy * (1.0f / 3.0f), out[7]);
}
__device__ __forceinline__ float sym_dot(const Sym6& A, const Sym6& B)  // sum_ab A_ab B_ab
{
    return A.xx * B.xx + A.yy * B.yy + A.zz * B.zz + 2.0f * (A.xy * B.xy + A.xz * B.xz + A.yz * B.yz);
}
__device__ __forceinline__ float lsum(const float* S, int l)  // sum_{L in l} S_L^2
{
    float s = 0.0f;
    const int b = lbase(l);
#pragma unroll
    for (int k = 0; k < 2 * l + 1; ++k) s = fmaf(S[b + k], S[b + k], s);
    return s;
}
__device__ __forceinline__ float ldot(const float* S, const float* V, int l)
{
    float s = 0.0f;
    const int b = lbase(l);
#pragma unroll
    for (int k = 0; k < 2 * l + 1; ++k) s = fmaf(S[b + k], V[b + k], s);
    return s;
}

// Invariants of one channel.  q[0..3]: l = 1..4 (Eq. 20); q[4]: 4-body; q[5]: 5-body (always at these fixed slots;
// the caller maps them to descriptor rows).  coefficient arrays c[6] use the same slots (0 where a term is absent).
__device__ __forceinline__ void inv_values(const float* S, float* q)
{
    q[0] = lsum(S, 1); q[1] = lsum(S, 2); q[2] = lsum(S, 3); q[3] = lsum(S, 4);
    const Sym6 T = tensor_from_l2(S);
    const Sym6 T2 = anticomm(T, T);
    q[4] = 0.5f * KAPPA4 * sym_dot(T2, T);
    q[5] = C5 * q[0] * q[0];
}
// out[L] = sum_a c[a] dq_a/dS_L
__device__ __forceinline__ void inv_adjoint(const float* S, const float* c, float* out)
{
    const float c1 = fmaf(4.0f * C5 * c[5], lsum(S, 1), 2.0f * c[0]);   // d/dS (7/15) q1^2 = (28/15) q1 S
#pragma unroll
    for (int L = 0; L < 3; ++L) out[L] = c1 * S[L];
#pragma unroll
    for (int L = 3; L < 8; ++L) out[L] = 2.0f * c[1] * S[L];
#pragma unroll
    for (int L = 8; L < 15; ++L) out[L] = 2.0f * c[2] * S[L];
#pragma unroll
    for (int L = 15; L < 24; ++L) out[L] = 2.0f * c[3] * S[L];
    const Sym6 T = tensor_from_l2(S);
    const Sym6 P = anticomm(T, T);   // 2 T^2 ; dq4/dT = 3 kappa4 T^2
    l2_from_tensor_adjoint(P, 1.5f * KAPPA4 * c[4], out);
}
// qd[a] = sum_L dq_a/dS_L * V_L
__device__ __forceinline__ void inv_tangent(const float* S, const float* V, float* qd)
{
    qd[0] = 2.0f * ldot(S, V, 1); qd[1] = 2.0f * ldot(S, V, 2); qd[2] = 2.0f * ldot(S, V, 3); qd[3] = 2.0f * ldot(S, V, 4);
    const Sym6 T = tensor_from_l2(S), Td = tensor_from_l2(V);
    const Sym6 T2 = anticomm(T, T);
    qd[4] = 1.5f * KAPPA4 * sym_dot(T2, Td);
    qd[5] = 2.0f * C5 * lsum(S, 1) * qd[0];
}
// inv_adjoint(S, cq) plus the second-derivative action along V: out[L] = sum_a cq[a] dq_a/dS_L + sum_a cf[a] sum_L' (d2 q_a / dS_L dS_L') V_L'.
// The two 4-body terms are 3 k4 cq4 T^2 and 3 k4 cf4 (T Td + Td T): both are anticommutators with T, so one anticommutator of T with
// (cq4 / 2) T + cf4 Td (scaled by 3 k4) serves both.
__device__ __forceinline__ void inv_adjoint_hessian(const float* S, const float* V, const float* cq, const float* cf, float* out)
{
    const float q1 = lsum(S, 1), q1d = 2.0f * ldot(S, V, 1);
    const float a1 = fmaf(4.0f * C5 * cq[5], q1, 2.0f * cq[0]);          // coefficient of S_L, l = 1, from the first term
    const float b1 = fmaf(4.0f * C5 * cf[5], q1, 2.0f * cf[0]);          // coefficient of V_L
    const float a1s = fmaf(4.0f * C5 * cf[5], q1d, a1);                  // ... and of S_L from the second term
#pragma unroll
    for (int L = 0; L < 3; ++L) out[L] = fmaf(b1, V[L], a1s * S[L]);
#pragma unroll
    for (int L = 3; L < 8; ++L) out[L] = fmaf(2.0f * cf[1], V[L], 2.0f * cq[1] * S[L]);
#pragma unroll
    for (int L = 8; L < 15; ++L) out[L] = fmaf(2.0f * cf[2], V[L], 2.0f * cq[2] * S[L]);
#pragma unroll
    for (int L = 15; L < 24; ++L) out[L] = fmaf(2.0f * cf[3], V[L], 2.0f * cq[3] * S[L]);
    const Sym6 T = tensor_from_l2(S), Td = tensor_from_l2(V);
    const float wq = 0.5f * cq[4], wf = cf[4];
    Sym6 M;
    M.xx = fmaf(wq, T.xx, wf * Td.xx); M.yy = fmaf(wq, T.yy, wf * Td.yy); M.zz = fmaf(wq, T.zz, wf * Td.zz);
    M.xy = fmaf(wq, T.xy, wf * Td.xy); M.xz = fmaf(wq, T.xz, wf * Td.xz); M.yz = fmaf(wq, T.yz, wf * Td.yz);
    l2_from_tensor_adjoint(anticomm(T, M), 3.0f * KAPPA4, out);
}

}  // namespace nep
