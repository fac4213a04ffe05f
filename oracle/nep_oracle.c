/*
 * nep_oracle.c -- CPU fp64 ORACLE for one NEP training step.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain, slow, by-eye-checkable restatement of what the hot path computes.
 * It shares no code, header, table or constant with the CUDA library (paper_2606_19557_b200/csrc);
 * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it.  The product path never calls it.
 *
 * Citations: P:NNN = /root/reference/PAPER.md line NNN.  "C<k>" = DESIGN.md section "Oracle
 * algorithm" step k (the paper prints no force / virial / gradient formula; those steps
 * are derivatives of Eqs. 1-7 and are pinned against finite differences in tests/).
 *
 *   C1  neighbours: every periodic image within the cutoff, brute force        ("j != i")
 *   C2  f_k(r) = 1/2 (T_k[2(r/rc-1)^2-1] + 1) f_c(r), f_c = 1/2(cos(pi r/rc)+1)  (Eqs. 17-18)
 *   C3  q_n  = sum_j g_n(r_ij),  g_n = sum_k c_nk^{ti tj} f_k                   (Eqs. 15-16)
 *   C4  A_nlm = sum_j g_n^A(r_ij) Y_lm(r^_ij), l = 1..l_max                      (Eq. 19)
 *   C5  q_nl = sum_m |A_nlm|^2 (Eq. 20); 4-/5-body invariants (reading G7)
 *   C6  q~ = q / (q_max - q_min)                                                (Eq. 2)
 *   C7  E_i = sum_mu w1 tanh(sum_nu w0 q~ - b0) - b1 ;  E = sum_i E_i           (Eqs. 3, 1)
 *   C8  F = -dE/dr, W = -sum d (x) dE_i/dd                                      (derivative of C7)
 *   C9  L = lE dE + lF dF + lV dV                                               (Eqs. 4-7)
 *   C10-C12  g = grad_theta L                                                   (Eq. 8)
 *   C13 Adam / AMSGrad                                                          (Eqs. 9-13)
 *
 * Real-harmonic route used here (differs on purpose from the CUDA path, which uses expanded
 * polynomials): b_{l,m,c/s}(r^) = P_l^{(m)}(z) Re/Im (x+iy)^m with P_l^{(m)} the m-th derivative
 * of the Legendre polynomial from the textbook recurrences, and
 * sum_m |Y_lm|^2-type sums become sum_L w_L b_L^2 with w = (2l+1)/(4 pi) * (m ? 2 (l-m)!/(l+m)! : 1).
 * The 4-body and 5-body terms are accumulated directly as the tensor T = sum_j g (r^ r^T - I/3)
 * and the vector s = sum_j g r^ (not through the l = 2 / l = 1 harmonics).
 *
 * Parity pins for every function here live in tests/test_oracle_*.py; nothing is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC  (no FMA contraction: C1 must be
 * reproducible bit for bit).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NEPO_MAXK 40   /* basis functions per channel  */
#define NEPO_MAXN 24   /* channels                     */
#define NEPO_MAXL 8    /* l_max for the 3-body part    */
#define NEPO_MAXNL (NEPO_MAXL * (NEPO_MAXL + 2))
#define NEPO_MAXNA (NEPO_MAXNL + 12)

typedef struct {
    int T;            /* number of species */
    double rcR, rcA;  /* radial / angular cutoff (Angstrom) */
    int nmaxR, nmaxA; /* n_max (channels are 0..n_max inclusive) */
    int basR, basA;   /* basis_size (k = 0..basis_size inclusive) */
    int l3, l4, l5;   /* l_max entries of Table I: 3-body order, 4-body on (2) / off (0), 5-body on (1) / off (0) */
    int H;            /* neurons */
} nepo_cfg;

typedef struct {
    int S;                     /* structures */
    const int64_t* atom_off;   /* [S+1] */
    const double* pos;         /* [N][3] Cartesian */
    const double* box;         /* [S][9] rows a, b, c */
    const int* type;           /* [N] */
    const int64_t* offR; const int* jR; const signed char* shR;  /* radial CSR over all atoms; j local to the structure */
    const int64_t* offA; const int* jA; const signed char* shA;  /* angular CSR */
    const double* E;           /* [S] labels (may be NULL for forward-only) */
    const double* F;           /* [N][3] */
    const double* W;           /* [S][9] row-major xx xy xz yx .. */
    const unsigned char* has_virial; /* [S] or NULL = all */
} nepo_data;

/* ---- sizes (D2, D1 of the paper's parameter count; pinned by Table II) ---- */
static int n_ang(const nepo_cfg* c) { return c->l3 + (c->l4 > 0) + (c->l5 > 0); }
int nepo_num_descriptors(const nepo_cfg* c) { return (c->nmaxR + 1) + (c->nmaxA + 1) * n_ang(c); }
int64_t nepo_num_params(const nepo_cfg* c)
{
    int64_t D = nepo_num_descriptors(c), T = c->T, H = c->H;
    int64_t nR = c->nmaxR + 1, nA = c->nmaxA + 1, KR = c->basR + 1, KA = c->basA + 1;
    return T * (D + 2) * H + 1 + T * T * (nR * KR + nA * KA);
}
int nepo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void nepo_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- C2: radial basis, Eqs. 17-18.  K = basis_size + 1 values f[0..K-1], df = d f/d r ---- */
void nepo_radial_basis(double r, double rc, int basis_size, double* f, double* df)
{
    int K = basis_size + 1;
    double u = r / rc;
    double fc = 0.5 * (cos(M_PI * u) + 1.0);             /* Eq. 18 */
    double dfc = -0.5 * M_PI / rc * sin(M_PI * u);
    double x = 2.0 * (u - 1.0) * (u - 1.0) - 1.0;          /* argument of T_k in Eq. 17 */
    double dx = 4.0 * (u - 1.0) / rc;
    double Tkm2 = 1.0, Tkm1 = x, dTkm2 = 0.0, dTkm1 = 1.0; /* T_0, T_1 and d/dx */
    for (int k = 0; k < K; ++k) {
        double Tk, dTk;
        if (k == 0) { Tk = 1.0; dTk = 0.0; }
        else if (k == 1) { Tk = x; dTk = 1.0; }
        else {
            Tk = 2.0 * x * Tkm1 - Tkm2;                    /* Chebyshev recurrence */
            dTk = 2.0 * Tkm1 + 2.0 * x * dTkm1 - dTkm2;
            Tkm2 = Tkm1; Tkm1 = Tk; dTkm2 = dTkm1; dTkm1 = dTk;
        }
        f[k] = 0.5 * (Tk + 1.0) * fc;                      /* Eq. 17 */
        df[k] = 0.5 * dTk * dx * fc + 0.5 * (Tk + 1.0) * dfc;
    }
}

/* ---- C4: angular functions of the bond vector d (not normalised on input) ----
 * phi_A(r^), A = 0..NA-1:
 *   A <  NL          : real harmonics b_L, ordered l = 1..l3, m = 0, 1c, 1s, 2c, 2s, ...
 *   next 9 (if l4)   : tau_ab = r^_a r^_b - delta_ab / 3           (row-major)
 *   next 3 (if l5)   : r^_a
 * dphi[A][3] = gradient w.r.t. the vector d = (1/r)(I - r^ r^T) grad_{r^} phi.
 * w[L] (harmonics only) = (2l+1)/(4 pi) * (m == 0 ? 1 : 2 (l-m)!/(l+m)!).
 */
static double factorial(int n) { double f = 1.0; for (int i = 2; i <= n; ++i) f *= i; return f; }

int nepo_num_harmonics(int l3) { return l3 * (l3 + 2); }
static int num_angfun(const nepo_cfg* c) { return nepo_num_harmonics(c->l3) + (c->l4 > 0 ? 9 : 0) + (c->l5 > 0 ? 3 : 0); }

void nepo_harmonic_weights(int l3, double* w)
{
    int L = 0;
    for (int l = 1; l <= l3; ++l)
        for (int m = 0; m <= l; ++m) {
            double wl = (2.0 * l + 1.0) / (4.0 * M_PI);
            if (m == 0) w[L++] = wl;
            else { double v = wl * 2.0 * factorial(l - m) / factorial(l + m); w[L++] = v; w[L++] = v; }
        }
}

void nepo_angular_functions(const double d[3], int l3, int has4, int has5, double* phi, double* dphi /* [NA][3] */)
{
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double x = d[0] / r, y = d[1] / r, z = d[2] / r;
    double rh[3] = { x, y, z };
    /* Legendre polynomials and their derivatives in z: P[m][l] = d^m P_l / dz^m.
       P_{l+1} = ((2l+1) z P_l - l P_{l-1}) / (l+1);  P^{(m)}_{l+1} = P^{(m)}_{l-1} + (2l+1) P^{(m-1)}_l  */
    double P[NEPO_MAXL + 2][NEPO_MAXL + 2];
    memset(P, 0, sizeof P);
    P[0][0] = 1.0; P[0][1] = z;
    for (int l = 1; l < l3 + 1; ++l) P[0][l + 1] = ((2.0 * l + 1.0) * z * P[0][l] - l * P[0][l - 1]) / (l + 1.0);
    for (int m = 1; m <= l3 + 1; ++m) {
        P[m][0] = 0.0;
        P[m][1] = (m == 1) ? 1.0 : 0.0;
        for (int l = 1; l < l3 + 1; ++l) P[m][l + 1] = P[m][l - 1] + (2.0 * l + 1.0) * P[m - 1][l];
    }
    /* (x + i y)^m = cm[m] + i sm[m] */
    double cm[NEPO_MAXL + 1], sm[NEPO_MAXL + 1];
    cm[0] = 1.0; sm[0] = 0.0;
    for (int m = 1; m <= l3; ++m) { cm[m] = cm[m - 1] * x - sm[m - 1] * y; sm[m] = cm[m - 1] * y + sm[m - 1] * x; }
    int A = 0;
    double g[NEPO_MAXNA][3]; /* gradient w.r.t. (x^,y^,z^) treated as independent */
    for (int l = 1; l <= l3; ++l)
        for (int m = 0; m <= l; ++m) {
            /* d/dx (x+iy)^m = m (x+iy)^{m-1};  d/dy = i m (x+iy)^{m-1} */
            double dcx = m ? m * cm[m - 1] : 0.0, dsx = m ? m * sm[m - 1] : 0.0;
            double dcy = m ? -m * sm[m - 1] : 0.0, dsy = m ? m * cm[m - 1] : 0.0;
            phi[A] = P[m][l] * cm[m];
            g[A][0] = P[m][l] * dcx; g[A][1] = P[m][l] * dcy; g[A][2] = P[m + 1][l] * cm[m];
            ++A;
            if (m > 0) {
                phi[A] = P[m][l] * sm[m];
                g[A][0] = P[m][l] * dsx; g[A][1] = P[m][l] * dsy; g[A][2] = P[m + 1][l] * sm[m];
                ++A;
            }
        }
    if (has4)
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                phi[A] = rh[a] * rh[b] - (a == b ? 1.0 / 3.0 : 0.0);
                for (int c = 0; c < 3; ++c) g[A][c] = (c == a ? rh[b] : 0.0) + (c == b ? rh[a] : 0.0);
                ++A;
            }
    if (has5)
        for (int a = 0; a < 3; ++a) {
            phi[A] = rh[a];
            for (int c = 0; c < 3; ++c) g[A][c] = (c == a ? 1.0 : 0.0);
            ++A;
        }
    if (dphi)
        for (int a = 0; a < A; ++a) {
            double rg = rh[0] * g[a][0] + rh[1] * g[a][1] + rh[2] * g[a][2];
            for (int c = 0; c < 3; ++c) dphi[3 * a + c] = (g[a][c] - rg * rh[c]) / r;   /* (I - r^ r^T) g / r */
        }
}

/* ---- C1: neighbours.  All (j, n) != (i, 0) with |d| < rc, d = (((r_j - r_i) + na a) + nb b) + nc c,
 * every product and sum rounded separately (compiled with -ffp-contract=off).  Order: ascending
 * (j, na, nb, nc).  Two-call pattern: with nbr_j == NULL only pair_off is filled.  j is local to
 * the structure.  Returns the total number of pairs. */
static void cross3(const double* u, const double* v, double* w)
{
    w[0] = u[1] * v[2] - u[2] * v[1]; w[1] = u[2] * v[0] - u[0] * v[2]; w[2] = u[0] * v[1] - u[1] * v[0];
}
void nepo_image_range(const double* box, double rc, int* m /*[3]*/)
{
    const double *a = box, *b = box + 3, *c = box + 6;
    double bc[3], ca[3], ab[3];
    cross3(b, c, bc); cross3(c, a, ca); cross3(a, b, ab);
    double V = fabs(a[0] * bc[0] + a[1] * bc[1] + a[2] * bc[2]);
    double ha = V / sqrt(bc[0] * bc[0] + bc[1] * bc[1] + bc[2] * bc[2]);
    double hb = V / sqrt(ca[0] * ca[0] + ca[1] * ca[1] + ca[2] * ca[2]);
    double hc = V / sqrt(ab[0] * ab[0] + ab[1] * ab[1] + ab[2] * ab[2]);
    /* wrapped inputs: |n_k| <= ceil(rc / h_k); one more for safety (extra candidates fail the test) */
    m[0] = (int)ceil(rc / ha) + 1; m[1] = (int)ceil(rc / hb) + 1; m[2] = (int)ceil(rc / hc) + 1;
}

int64_t nepo_build_neighbors(int S, const int64_t* atom_off, const double* pos, const double* box, double rc,
                             int64_t* pair_off /*[N+1]*/, int* nbr_j, signed char* nbr_shift /*[P][3]*/)
{
    double rc2 = rc * rc;
    int64_t N = atom_off[S];
    int fill = (nbr_j != NULL);
    if (!fill) pair_off[0] = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < S; ++s) {
        const double *a = box + 9 * s, *b = a + 3, *c = a + 6;
        int m[3];
        nepo_image_range(a, rc, m);
        int64_t o = atom_off[s];
        int n = (int)(atom_off[s + 1] - o);
        for (int i = 0; i < n; ++i) {
            int64_t cnt = 0, w = fill ? pair_off[o + i] : 0;
            const double* ri = pos + 3 * (o + i);
            for (int j = 0; j < n; ++j) {
                const double* rj = pos + 3 * (o + j);
                for (int na = -m[0]; na <= m[0]; ++na)
                    for (int nb = -m[1]; nb <= m[1]; ++nb)
                        for (int nc = -m[2]; nc <= m[2]; ++nc) {
                            if (j == i && na == 0 && nb == 0 && nc == 0) continue;
                            double d[3];
                            for (int k = 0; k < 3; ++k) {
                                double t = rj[k] - ri[k];
                                t = t + (double)na * a[k];
                                t = t + (double)nb * b[k];
                                t = t + (double)nc * c[k];
                                d[k] = t;
                            }
                            double r2 = (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2];
                            if (r2 < rc2) {
                                if (fill) {
                                    nbr_j[w] = j;
                                    nbr_shift[3 * w] = (signed char)na; nbr_shift[3 * w + 1] = (signed char)nb; nbr_shift[3 * w + 2] = (signed char)nc;
                                    ++w;
                                }
                                ++cnt;
                            }
                        }
            }
            if (!fill) pair_off[o + i + 1] = cnt; /* counts; prefix-summed below */
        }
    }
    if (!fill)
        for (int64_t i = 0; i < N; ++i) pair_off[i + 1] += pair_off[i];
    return pair_off[N];
}

/* bond vector of a stored pair, same formula as C1 */
static void bond(const double* pos_s, const double* bx, int i, int j, const signed char* sh, double* d)
{
    for (int k = 0; k < 3; ++k) {
        double t = pos_s[3 * j + k] - pos_s[3 * i + k];
        t = t + (double)sh[0] * bx[k];
        t = t + (double)sh[1] * bx[3 + k];
        t = t + (double)sh[2] * bx[6 + k];
        d[k] = t;
    }
}

/* ---- theta layout (C0) ---- */
typedef struct {
    int T, H, D, nR, nA, KR, KA, l3, has4, has5, NL, NA, nang;
    const double *w0, *b0, *w1; /* per species stride (D+2)*H from w0 */
    const double* b1; const double* cR; const double* cA;
    int64_t o_b1, o_cR, o_cA, npar;
    double wL[NEPO_MAXNL];
} layout;

static void make_layout(const nepo_cfg* c, const double* theta, layout* L)
{
    L->T = c->T; L->H = c->H; L->D = nepo_num_descriptors(c);
    L->nR = c->nmaxR + 1; L->nA = c->nmaxA + 1; L->KR = c->basR + 1; L->KA = c->basA + 1;
    L->l3 = c->l3; L->has4 = c->l4 > 0; L->has5 = c->l5 > 0;
    L->NL = nepo_num_harmonics(c->l3); L->NA = num_angfun(c); L->nang = n_ang(c);
    int64_t per = (int64_t)(L->D + 2) * L->H;
    L->o_b1 = per * L->T; L->o_cR = L->o_b1 + 1; L->o_cA = L->o_cR + (int64_t)L->T * L->T * L->nR * L->KR;
    L->npar = L->o_cA + (int64_t)L->T * L->T * L->nA * L->KA;
    L->w0 = theta; L->b0 = theta ? theta + (int64_t)L->H * L->D : NULL; L->w1 = theta ? theta + (int64_t)L->H * L->D + L->H : NULL;
    L->b1 = theta ? theta + L->o_b1 : NULL; L->cR = theta ? theta + L->o_cR : NULL; L->cA = theta ? theta + L->o_cA : NULL;
    nepo_harmonic_weights(c->l3, L->wL);
}
#define W0(L, t) ((L)->w0 + (int64_t)(t) * ((L)->D + 2) * (L)->H)
#define B0(L, t) ((L)->b0 + (int64_t)(t) * ((L)->D + 2) * (L)->H)
#define W1(L, t) ((L)->w1 + (int64_t)(t) * ((L)->D + 2) * (L)->H)
#define CR(L, ti, tj) ((L)->cR + ((int64_t)(ti) * (L)->T + (tj)) * (L)->nR * (L)->KR)
#define CA(L, ti, tj) ((L)->cA + ((int64_t)(ti) * (L)->T + (tj)) * (L)->nA * (L)->KA)

/* reading G7 constants: normalisation of the cubic l=2 and quartic l=1 invariants */
static double kappa4(void) { return -45.0 / (8.0 * sqrt(14.0) * pow(M_PI, 1.5)); }
static double kappa5(void) { return 21.0 / (80.0 * M_PI * M_PI); }

/* ---- C5: angular invariants of one channel from its moments M[NA];  optional first and second
 * derivative actions:  J[nang][NA] = dq/dM ;  HV(q index a) = sum_B d2q_a/dM_A dM_B * V_B ---- */
static void invariants(const layout* L, const double* M, double* q /*[nang]*/, double* J /*[nang][NA] or NULL*/)
{
    int NA = L->NA, A = 0;
    if (J) memset(J, 0, sizeof(double) * L->nang * NA);
    for (int l = 1; l <= L->l3; ++l) {       /* Eq. 20 in the real basis */
        double s = 0.0;
        for (int k = 0; k < 2 * l + 1; ++k, ++A) {
            s += L->wL[A] * M[A] * M[A];
            if (J) J[(l - 1) * NA + A] = 2.0 * L->wL[A] * M[A];
        }
        q[l - 1] = s;
    }
    int a = L->l3;
    if (L->has4) {                           /* q4 = kappa4 tr(T^3) */
        const double* Tm = M + A;
        double tr = 0.0;
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k) tr += Tm[3 * i + j] * Tm[3 * j + k] * Tm[3 * k + i];
        q[a] = kappa4() * tr;
        if (J)
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
                double t2 = 0.0;
                for (int k = 0; k < 3; ++k) t2 += Tm[3 * j + k] * Tm[3 * k + i];   /* (T^2)_{ji} */
                J[a * NA + A + 3 * i + j] = 3.0 * kappa4() * t2;
            }
        A += 9; ++a;
    }
    if (L->has5) {                           /* q5 = kappa5 (s.s)^2 */
        const double* sv = M + A;
        double ss = sv[0] * sv[0] + sv[1] * sv[1] + sv[2] * sv[2];
        q[a] = kappa5() * ss * ss;
        if (J) for (int i = 0; i < 3; ++i) J[a * NA + A + i] = 4.0 * kappa5() * ss * sv[i];
        A += 3; ++a;
    }
}
/* out[A] += sum_a coef[a] * sum_B (d2 q_a / dM_A dM_B) V[B] */
static void hessian_action(const layout* L, const double* M, const double* V, const double* coef /*[nang]*/, double* out /*[NA]*/)
{
    int A = 0;
    for (int l = 1; l <= L->l3; ++l)
        for (int k = 0; k < 2 * l + 1; ++k, ++A) out[A] += coef[l - 1] * 2.0 * L->wL[A] * V[A];
    int a = L->l3;
    if (L->has4) {
        const double *Tm = M + A, *Tv = V + A;   /* d/dT_ij of 3 k4 (T^2)_ji  along Tv: 3 k4 (T Tv + Tv T)_ji */
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
            double t = 0.0;
            for (int k = 0; k < 3; ++k) t += Tm[3 * j + k] * Tv[3 * k + i] + Tv[3 * j + k] * Tm[3 * k + i];
            out[A + 3 * i + j] += coef[a] * 3.0 * kappa4() * t;
        }
        A += 9; ++a;
    }
    if (L->has5) {
        const double *sv = M + A, *sd = V + A;
        double ss = sv[0] * sv[0] + sv[1] * sv[1] + sv[2] * sv[2], sds = sv[0] * sd[0] + sv[1] * sd[1] + sv[2] * sd[2];
        for (int i = 0; i < 3; ++i) out[A + i] += coef[a] * 4.0 * kappa5() * (ss * sd[i] + 2.0 * sds * sv[i]);
        A += 3; ++a;
    }
}

/* descriptor index (C0): radial n -> n ; angular (block a = l-1 | 4-body | 5-body, channel n) -> nR + a*nA + n */
static int qidx(const layout* L, int a, int n) { return L->nR + a * L->nA + n; }

/* per-pair geometry scratch for one atom */
typedef struct {
    int j, tj; double d[3], r;
    double f[NEPO_MAXK], df[NEPO_MAXK];
    double phi[NEPO_MAXNA], dphi[NEPO_MAXNA * 3];
} pairgeo;

/* ---- C3-C5: descriptor of atom i (local index) of structure s; fills q[D], M[nA][NA]; geometry lists out ---- */
static void atom_geometry(const nepo_cfg* c, const layout* L, const nepo_data* X, int s, int i, pairgeo** gR, int* nRn, pairgeo** gA, int* nAn)
{
    int64_t o = X->atom_off[s];
    const double *ps = X->pos + 3 * o, *bx = X->box + 9 * s;
    int64_t b = X->offR[o + i], e = X->offR[o + i + 1];
    *nRn = (int)(e - b);
    *gR = (pairgeo*)malloc(sizeof(pairgeo) * (size_t)(*nRn > 0 ? *nRn : 1));
    for (int64_t p = b; p < e; ++p) {
        pairgeo* g = *gR + (p - b);
        g->j = X->jR[p]; g->tj = X->type[o + g->j];
        bond(ps, bx, i, g->j, X->shR + 3 * p, g->d);
        g->r = sqrt(g->d[0] * g->d[0] + g->d[1] * g->d[1] + g->d[2] * g->d[2]);
        nepo_radial_basis(g->r, c->rcR, c->basR, g->f, g->df);
    }
    b = X->offA[o + i]; e = X->offA[o + i + 1];
    *nAn = (int)(e - b);
    *gA = (pairgeo*)malloc(sizeof(pairgeo) * (size_t)(*nAn > 0 ? *nAn : 1));
    for (int64_t p = b; p < e; ++p) {
        pairgeo* g = *gA + (p - b);
        g->j = X->jA[p]; g->tj = X->type[o + g->j];
        bond(ps, bx, i, g->j, X->shA + 3 * p, g->d);
        g->r = sqrt(g->d[0] * g->d[0] + g->d[1] * g->d[1] + g->d[2] * g->d[2]);
        nepo_radial_basis(g->r, c->rcA, c->basA, g->f, g->df);
        nepo_angular_functions(g->d, L->l3, L->has4, L->has5, g->phi, g->dphi);
    }
}
static double dotk(const double* a, const double* b, int n) { double s = 0.0; for (int k = 0; k < n; ++k) s += a[k] * b[k]; return s; }

static void atom_descriptor(const layout* L, int ti, const pairgeo* gR, int nRn, const pairgeo* gA, int nAn, double* q, double* M /*[nA][NA]*/)
{
    memset(q, 0, sizeof(double) * L->D);
    memset(M, 0, sizeof(double) * L->nA * L->NA);
    for (int p = 0; p < nRn; ++p)                                        /* Eqs. 15-16 */
        for (int n = 0; n < L->nR; ++n) q[n] += dotk(CR(L, ti, gR[p].tj) + n * L->KR, gR[p].f, L->KR);
    for (int p = 0; p < nAn; ++p)                                        /* Eq. 19 */
        for (int n = 0; n < L->nA; ++n) {
            double gn = dotk(CA(L, ti, gA[p].tj) + n * L->KA, gA[p].f, L->KA);
            for (int A = 0; A < L->NA; ++A) M[n * L->NA + A] += gn * gA[p].phi[A];
        }
    double qa[NEPO_MAXL + 2];
    for (int n = 0; n < L->nA; ++n) {                                    /* Eq. 20 + higher-body */
        invariants(L, M + n * L->NA, qa, NULL);
        for (int a = 0; a < L->nang; ++a) q[qidx(L, a, n)] = qa[a];
    }
}

/* descriptors of every atom of the data set -> q[N][D]  (used for the scaler, C6) */
void nepo_descriptors(const nepo_cfg* c, const nepo_data* X, const double* theta, double* q)
{
    layout L; make_layout(c, theta, &L);
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < X->S; ++s) {
        int64_t o = X->atom_off[s];
        int n = (int)(X->atom_off[s + 1] - o);
        double* M = (double*)malloc(sizeof(double) * L.nA * L.NA);
        for (int i = 0; i < n; ++i) {
            pairgeo *gR, *gA; int nRn, nAn;
            atom_geometry(c, &L, X, s, i, &gR, &nRn, &gA, &nAn);
            atom_descriptor(&L, X->type[o + i], gR, nRn, gA, nAn, q + (o + i) * L.D, M);
            free(gR); free(gA);
        }
        free(M);
    }
}

/* C6 (Eq. 2): s_nu = 1 / (max_i q_nu - min_i q_nu) over all N atoms; degenerate range -> 1 (reading G10) */
void nepo_scaler(int D, int64_t N, const double* q, double* s)
{
    for (int v = 0; v < D; ++v) {
        double lo = INFINITY, hi = -INFINITY, amax = 0.0;
        for (int64_t i = 0; i < N; ++i) {
            double x = q[i * D + v];
            if (x < lo) lo = x;
            if (x > hi) hi = x;
            if (fabs(x) > amax) amax = fabs(x);
        }
        double range = hi - lo;
        s[v] = (N > 0 && range > 1e-12 * (amax > 1.0 ? amax : 1.0)) ? 1.0 / range : 1.0;
    }
}

/* ---- one structure: forward (E, F, W) and, if seeds are given, its contribution to grad_theta L ---- */
typedef struct { double epsE; const double* u; /*[n][3]*/ const double* G; /*[9]*/ } seeds;

static void structure_pass(const nepo_cfg* c, const layout* L, const nepo_data* X, const double* scal, int s,
                           double* E_out, double* F /*[n][3] or NULL*/, double* Wv /*[9] or NULL*/,
                           const seeds* sd, double* grad /*[npar] accumulated, or NULL*/)
{
    int64_t o = X->atom_off[s];
    int n = (int)(X->atom_off[s + 1] - o);
    int D = L->D, H = L->H, NA = L->NA, nA = L->nA, nR = L->nR, KR = L->KR, KA = L->KA, T = L->T;
    double E = 0.0;
    if (F) memset(F, 0, sizeof(double) * 3 * n);
    if (Wv) memset(Wv, 0, sizeof(double) * 9);
    double* q = (double*)malloc(sizeof(double) * D);
    double* qt = (double*)malloc(sizeof(double) * D);
    double* Fp = (double*)malloc(sizeof(double) * D);
    double* qd = (double*)malloc(sizeof(double) * D);
    double* Qb = (double*)malloc(sizeof(double) * D);
    double* M = (double*)malloc(sizeof(double) * nA * NA);
    double* Md = (double*)malloc(sizeof(double) * nA * NA);   /* tangent of M */
    double* EdM = (double*)malloc(sizeof(double) * nA * NA);  /* dE_i/dM  (adjoint of Md) */
    double* Mb = (double*)malloc(sizeof(double) * nA * NA);   /* adjoint of M */
    double* J = (double*)malloc(sizeof(double) * L->nang * NA);
    double* h = (double*)malloc(sizeof(double) * H);
    double* e = (double*)malloc(sizeof(double) * H);
    double* xd = (double*)malloc(sizeof(double) * H);
    double* gx = (double*)malloc(sizeof(double) * H);
    for (int i = 0; i < n; ++i) {
        int ti = X->type[o + i];
        pairgeo *gR, *gA; int nRn, nAn;
        atom_geometry(c, L, X, s, i, &gR, &nRn, &gA, &nAn);
        atom_descriptor(L, ti, gR, nRn, gA, nAn, q, M);
        /* C7: Eq. 2 then Eq. 3 */
        const double *w0 = W0(L, ti), *b0 = B0(L, ti), *w1 = W1(L, ti);
        for (int v = 0; v < D; ++v) qt[v] = scal[v] * q[v];
        double Ei = 0.0;
        for (int mu = 0; mu < H; ++mu) {
            double x = dotk(w0 + (int64_t)mu * D, qt, D) - b0[mu];
            h[mu] = tanh(x);
            Ei += w1[mu] * h[mu];
            e[mu] = w1[mu] * (1.0 - h[mu] * h[mu]);       /* dE_i/dx_mu */
        }
        Ei -= L->b1[0];
        E += Ei;
        for (int v = 0; v < D; ++v) {                      /* Fp = dE_i/dq */
            double t = 0.0;
            for (int mu = 0; mu < H; ++mu) t += e[mu] * w0[(int64_t)mu * D + v];
            Fp[v] = scal[v] * t;
        }
        /* C8: dE_i/dM_nA = sum_a Fp[q index (a,n)] dq_a/dM_A */
        for (int nn = 0; nn < nA; ++nn) {
            double qa[NEPO_MAXL + 2];
            invariants(L, M + nn * NA, qa, J);
            for (int A = 0; A < NA; ++A) {
                double t = 0.0;
                for (int a = 0; a < L->nang; ++a) t += Fp[qidx(L, a, nn)] * J[a * NA + A];
                EdM[nn * NA + A] = t;
            }
        }
        if (F || Wv) {
            for (int p = 0; p < nRn; ++p) {                /* radial: p_ij = [sum_n Fp_n g_n'(r)] r^ */
                const pairgeo* g = gR + p;
                double sc = 0.0;
                for (int nn = 0; nn < nR; ++nn) sc += Fp[nn] * dotk(CR(L, ti, g->tj) + nn * KR, g->df, KR);
                for (int a = 0; a < 3; ++a) {
                    double pa = sc * g->d[a] / g->r;
                    if (F) { F[3 * i + a] += pa; F[3 * g->j + a] -= pa; }
                    if (Wv) for (int b = 0; b < 3; ++b) Wv[3 * b + a] -= g->d[b] * pa;   /* W_ba -= d_b p_a */
                }
            }
            for (int p = 0; p < nAn; ++p) {                /* angular: sum_n sum_A EdM [g' phi r^ + g dphi] */
                const pairgeo* g = gA + p;
                double pv[3] = { 0, 0, 0 };
                for (int nn = 0; nn < nA; ++nn) {
                    double gn = dotk(CA(L, ti, g->tj) + nn * KA, g->f, KA), dgn = dotk(CA(L, ti, g->tj) + nn * KA, g->df, KA);
                    for (int A = 0; A < NA; ++A) {
                        double w = EdM[nn * NA + A];
                        for (int a = 0; a < 3; ++a) pv[a] += w * (dgn * g->phi[A] * g->d[a] / g->r + gn * g->dphi[3 * A + a]);
                    }
                }
                for (int a = 0; a < 3; ++a) {
                    if (F) { F[3 * i + a] += pv[a]; F[3 * g->j + a] -= pv[a]; }
                    if (Wv) for (int b = 0; b < 3; ++b) Wv[3 * b + a] -= g->d[b] * pv[a];
                }
            }
        }
        if (sd && grad) {
            double* gw0 = grad + (W0(L, ti) - L->w0), *gb0 = grad + (B0(L, ti) - L->w0), *gw1 = grad + (W1(L, ti) - L->w0);
            const double *u = sd->u, *G = sd->G;
            /* C10 tangent sweep along dt_ij = u_i - u_j - G^T d_ij */
            memset(qd, 0, sizeof(double) * D);
            memset(Md, 0, sizeof(double) * nA * NA);
            for (int p = 0; p < nRn; ++p) {
                pairgeo* g = gR + p;
                double dt[3], rd = 0.0;
                for (int a = 0; a < 3; ++a) {
                    double Gtd = G[0 * 3 + a] * g->d[0] + G[1 * 3 + a] * g->d[1] + G[2 * 3 + a] * g->d[2];
                    dt[a] = u[3 * i + a] - u[3 * g->j + a] - Gtd;
                    rd += g->d[a] / g->r * dt[a];
                }
                for (int nn = 0; nn < nR; ++nn) qd[nn] += dotk(CR(L, ti, g->tj) + nn * KR, g->df, KR) * rd;
            }
            for (int p = 0; p < nAn; ++p) {
                pairgeo* g = gA + p;
                double dt[3], rd = 0.0;
                for (int a = 0; a < 3; ++a) {
                    double Gtd = G[0 * 3 + a] * g->d[0] + G[1 * 3 + a] * g->d[1] + G[2 * 3 + a] * g->d[2];
                    dt[a] = u[3 * i + a] - u[3 * g->j + a] - Gtd;
                    rd += g->d[a] / g->r * dt[a];
                }
                for (int nn = 0; nn < nA; ++nn) {
                    double gn = dotk(CA(L, ti, g->tj) + nn * KA, g->f, KA), dgn = dotk(CA(L, ti, g->tj) + nn * KA, g->df, KA);
                    for (int A = 0; A < NA; ++A)
                        Md[nn * NA + A] += dgn * rd * g->phi[A] + gn * dotk(g->dphi + 3 * A, dt, 3);
                }
            }
            for (int nn = 0; nn < nA; ++nn) {
                double qa[NEPO_MAXL + 2];
                invariants(L, M + nn * NA, qa, J);
                for (int a = 0; a < L->nang; ++a) qd[qidx(L, a, nn)] = dotk(J + a * NA, Md + nn * NA, NA);
            }
            /* C11 network tangent + adjoint */
            for (int mu = 0; mu < H; ++mu) {
                double t = 0.0;
                for (int v = 0; v < D; ++v) t += w0[(int64_t)mu * D + v] * scal[v] * qd[v];
                xd[mu] = t;
                double a_ = -2.0 * h[mu] * e[mu] * xd[mu];
                gx[mu] = sd->epsE * e[mu] + a_;
                gw1[mu] += sd->epsE * h[mu] + (1.0 - h[mu] * h[mu]) * xd[mu];
                gb0[mu] += -gx[mu];
                for (int v = 0; v < D; ++v) gw0[(int64_t)mu * D + v] += gx[mu] * qt[v] + e[mu] * scal[v] * qd[v];
            }
            grad[L->o_b1] += -sd->epsE;
            for (int v = 0; v < D; ++v) {
                double t = 0.0;
                for (int mu = 0; mu < H; ++mu) t += gx[mu] * w0[(int64_t)mu * D + v];
                Qb[v] = scal[v] * t;
            }
            /* C12 adjoint of M:  Mb = J^T Qb + sum_a Fp_a Hess(q_a) Md */
            for (int nn = 0; nn < nA; ++nn) {
                double qa[NEPO_MAXL + 2], coef[NEPO_MAXL + 2];
                invariants(L, M + nn * NA, qa, J);
                for (int A = 0; A < NA; ++A) {
                    double t = 0.0;
                    for (int a = 0; a < L->nang; ++a) t += Qb[qidx(L, a, nn)] * J[a * NA + A];
                    Mb[nn * NA + A] = t;
                }
                for (int a = 0; a < L->nang; ++a) coef[a] = Fp[qidx(L, a, nn)];
                hessian_action(L, M + nn * NA, Md + nn * NA, coef, Mb + nn * NA);
            }
            for (int p = 0; p < nRn; ++p) {
                pairgeo* g = gR + p;
                double dt[3], rd = 0.0;
                for (int a = 0; a < 3; ++a) {
                    double Gtd = G[0 * 3 + a] * g->d[0] + G[1 * 3 + a] * g->d[1] + G[2 * 3 + a] * g->d[2];
                    dt[a] = u[3 * i + a] - u[3 * g->j + a] - Gtd;
                    rd += g->d[a] / g->r * dt[a];
                }
                double* gc = grad + L->o_cR + ((int64_t)ti * T + g->tj) * nR * KR;
                for (int nn = 0; nn < nR; ++nn)
                    for (int k = 0; k < KR; ++k) gc[nn * KR + k] += Qb[nn] * g->f[k] + Fp[nn] * g->df[k] * rd;
            }
            for (int p = 0; p < nAn; ++p) {
                pairgeo* g = gA + p;
                double dt[3], rd = 0.0;
                for (int a = 0; a < 3; ++a) {
                    double Gtd = G[0 * 3 + a] * g->d[0] + G[1 * 3 + a] * g->d[1] + G[2 * 3 + a] * g->d[2];
                    dt[a] = u[3 * i + a] - u[3 * g->j + a] - Gtd;
                    rd += g->d[a] / g->r * dt[a];
                }
                double* gc = grad + L->o_cA + ((int64_t)ti * T + g->tj) * nA * KA;
                for (int nn = 0; nn < nA; ++nn) {
                    double al = 0.0, be = 0.0, de = 0.0;
                    for (int A = 0; A < NA; ++A) {
                        al += Mb[nn * NA + A] * g->phi[A];
                        be += EdM[nn * NA + A] * g->phi[A];
                        de += EdM[nn * NA + A] * dotk(g->dphi + 3 * A, dt, 3);
                    }
                    for (int k = 0; k < KA; ++k) gc[nn * KA + k] += (al + de) * g->f[k] + be * rd * g->df[k];
                }
            }
        }
        free(gR); free(gA);
    }
    *E_out = E;
    free(q); free(qt); free(Fp); free(qd); free(Qb); free(M); free(Md); free(EdM); free(Mb); free(J); free(h); free(e); free(xd); free(gx);
}

/* ---- forward over a batch of structures: E[nb], F[batch atoms][3] (batch order), W[nb][9] ---- */
void nepo_forward(const nepo_cfg* c, const nepo_data* X, const double* theta, const double* scal,
                  int nb, const int* batch, double* E, double* F, double* Wv)
{
    layout L; make_layout(c, theta, &L);
    int64_t* fo = (int64_t*)malloc(sizeof(int64_t) * (size_t)(nb + 1));
    fo[0] = 0;
    for (int b = 0; b < nb; ++b) { int s = batch ? batch[b] : b; fo[b + 1] = fo[b] + (X->atom_off[s + 1] - X->atom_off[s]); }
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < nb; ++b) {
        int s = batch ? batch[b] : b;
        structure_pass(c, &L, X, scal, s, E + b, F ? F + 3 * fo[b] : NULL, Wv ? Wv + 9 * b : NULL, NULL, NULL);
    }
    free(fo);
}

/* ---- C9-C12: loss (Eqs. 4-7) and its gradient (Eq. 8).  loss4 = {L, dE, dF, dV}.
 * Optional outputs Ehat/Fhat/What as in nepo_forward (may be NULL). ---- */
void nepo_loss_grad(const nepo_cfg* c, const nepo_data* X, const double* theta, const double* scal,
                    int nb, const int* batch, double lamE, double lamF, double lamV,
                    double* loss4, double* grad /*[npar] or NULL*/)
{
    layout L; make_layout(c, theta, &L);
    int64_t Na = 0; int Sv = 0;
    for (int b = 0; b < nb; ++b) {
        int s = batch ? batch[b] : b;
        Na += X->atom_off[s + 1] - X->atom_off[s];
        if (!X->has_virial || X->has_virial[s]) ++Sv;
    }
    int nth = nepo_max_threads();
    double* gth = grad ? (double*)calloc((size_t)nth * (size_t)L.npar, sizeof(double)) : NULL;
    double* part = (double*)calloc((size_t)nb * 3, sizeof(double));
#pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < nb; ++b) {
        int s = batch ? batch[b] : b;
        int64_t o = X->atom_off[s];
        int n = (int)(X->atom_off[s + 1] - o);
        int hv = (!X->has_virial || X->has_virial[s]);
        double Eh, Wh[9];
        double* Fh = (double*)malloc(sizeof(double) * 3 * n);
        double* u = (double*)malloc(sizeof(double) * 3 * n);
        structure_pass(c, &L, X, scal, s, &Eh, Fh, Wh, NULL, NULL);
        double dE = (Eh - X->E[s]) / n;                                   /* Eq. 5 */
        part[3 * b + 0] = dE * dE;
        double sF = 0.0;
        for (int k = 0; k < 3 * n; ++k) { double t = Fh[k] - X->F[3 * o + k]; sF += t * t; u[k] = 2.0 * lamF * t / (3.0 * (double)Na); } /* Eq. 6 */
        part[3 * b + 1] = sF;
        double sW = 0.0, G[9];
        for (int k = 0; k < 9; ++k) {
            double t = hv ? (Wh[k] - X->W[9 * s + k]) / n : 0.0;                 /* Eq. 7 */
            sW += t * t;
            G[k] = (hv && Sv > 0) ? 2.0 * lamV * (Wh[k] - X->W[9 * s + k]) / (9.0 * Sv * (double)n * n) : 0.0;
        }
        part[3 * b + 2] = sW;
        if (grad) {
            seeds sd; sd.epsE = 2.0 * lamE * (Eh - X->E[s]) / ((double)nb * n * n); sd.u = u; sd.G = G;
            int th = 0;
#ifdef _OPENMP
            th = omp_get_thread_num();
#endif
            double Edummy;
            structure_pass(c, &L, X, scal, s, &Edummy, NULL, NULL, &sd, gth + (size_t)th * L.npar);
        }
        free(Fh); free(u);
    }
    double sE = 0, sF = 0, sW = 0;
    for (int b = 0; b < nb; ++b) { sE += part[3 * b]; sF += part[3 * b + 1]; sW += part[3 * b + 2]; }
    double dE = nb ? sE / nb : 0.0, dF = Na ? sF / (3.0 * Na) : 0.0, dV = Sv ? sW / (9.0 * Sv) : 0.0;
    loss4[0] = lamE * dE + lamF * dF + lamV * dV; loss4[1] = dE; loss4[2] = dF; loss4[3] = dV;   /* Eq. 4 */
    if (grad) {
        for (int64_t k = 0; k < L.npar; ++k) {
            double t = 0.0;
            for (int th = 0; th < nth; ++th) t += gth[(size_t)th * L.npar + k];
            grad[k] = t;
        }
        free(gth);
    }
    free(part);
}

/* ---- C13: Adam with AMSGrad.  variant 0 = the paper's Eqs. 9-13 literally (max over the
 * bias-corrected v^, epsilon inside the root); variant 1 = torch.optim.Adam(amsgrad=True)
 * (max over raw v, sqrt(vmax/bc2) + eps).  t is the step count BEFORE the call; returns t+1. ---- */
int64_t nepo_adam_step(int64_t npar, double* theta, const double* g, double* m, double* v, double* vmax,
                       int64_t t, double lr, double beta1, double beta2, double eps, int variant)
{
    t += 1;
    double bc1 = 1.0 - pow(beta1, (double)t), bc2 = 1.0 - pow(beta2, (double)t);
    for (int64_t k = 0; k < npar; ++k) {
        m[k] = beta1 * m[k] + (1.0 - beta1) * g[k];            /* Eq. 9  */
        v[k] = beta2 * v[k] + (1.0 - beta2) * g[k] * g[k];     /* Eq. 10 */
        double mh = m[k] / bc1;                                /* Eq. 11 */
        if (variant == 0) {
            double vh = v[k] / bc2;                            /* Eq. 11 */
            if (vh > vmax[k]) vmax[k] = vh;                    /* Eq. 12 */
            theta[k] -= lr * mh / sqrt(vmax[k] + eps);         /* Eq. 13 */
        } else {
            if (v[k] > vmax[k]) vmax[k] = v[k];
            theta[k] -= lr * mh / (sqrt(vmax[k] / bc2) + eps);
        }
    }
    return t;
}
