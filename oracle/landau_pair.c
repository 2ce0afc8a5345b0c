/*
 * oracle/landau_pair.c -- CPU ORACLE (test infrastructure, NOT the product path).
 *
 * Plain, slow, obviously-correct evaluation of the inner integral of the axisymmetric
 * Landau operator (Alg. 1 lines 3-12, L109-121; Eqs. 7-8; Eq. 10):
 *
 *   G_D(i) = sum_{j != i} w[j] * T_D(j) * U^D(v_i, v_j)        T_D(j) = sum_b e_b^2 f_b(j)
 *   G_K(i) = sum_{j != i} w[j] * U^K(v_i, v_j) . T_K(j)        T_K(j) = sum_b e_b^2 (m0/m_b) grad f_b(j)
 *
 * in the paper's loop order (i outer, j inner, beta innermost, T reset per j -- DESIGN.md
 * reading Q4), with no tiling, hoisting or symmetry.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this file's library.  It shares no
 * code with paper_2104_10000_b200/csrc.
 *
 * U^D, U^K are NOT printed in the paper ("much more complex than (3) [4]", L69).  They are Eq. 3
 * (L44) integrated over the azimuth (reading Q1): v at azimuth 0, vbar at azimuth phi,
 *   u = (r - rb cos phi, -rb sin phi, dz),  |u|^2 = s (1 - m cos^2(phi/2)),
 *   s = (r+rb)^2 + dz^2,  d2 = (r-rb)^2 + dz^2,  m = 4 r rb / s,
 *   P0  = int dphi 1/|u|^3            = 4 E(m) / (sqrt(s) d2)
 *   Pc  = int dphi (1-cos phi)/|u|^3  = 8 D(m) / s^{3/2}        D = (K-E)/m
 *   Pss = int dphi sin^2 phi/|u|^3    = 16 S(m) / s^{3/2}       S = (2D-K)/m
 *   U^D_rr = rb^2 Pss + dz^2 P0;  U^D_rz = -dz[(r-rb) P0 + rb Pc];  U^D_zz = (r-rb)^2 P0 + 2 r rb Pc
 *   U^K_{r rb} = dz^2 (P0-Pc) + r rb Pss;  U^K_{z rb} = dz[(rb-r) P0 + r Pc]
 *   U^K_{r zb} = U^D_rz;  U^K_{z zb} = U^D_zz
 * (K, E complete elliptic integrals in the parameter convention.)  These are pinned in
 * tests/test_oracle_pins.py against brute-force azimuthal quadrature of Eq. 3.
 *
 * Elliptic integrals: Carlson symmetric forms by the duplication algorithm (a different route
 * from the CUDA path's AGM): K = R_F(0,1-m,1), D = R_D(0,1-m,1)/3, E = K - m D;
 * S = (2D-K)/m for m >= 0.05 and the Gauss hypergeometric series S = (pi/16) 2F1(3/2,3/2;3;m)
 * below (the closed form loses eps/m^2 there).
 *
 * Compile twice: -DREAL_LD (long double: parity reference) and plain (double: timed baseline).
 */
#include <math.h>
#include <stddef.h>

#ifdef REAL_LD
typedef long double real;
#define SQRT sqrtl
#define FABS fabsl
#define REAL_EPS 1.0e-19L
#define SUFFIX(n) n##_ld
#else
typedef double real;
#define SQRT sqrt
#define FABS fabs
#define REAL_EPS 2.2e-16
#define SUFFIX(n) n##_d
#endif

static const real PI_R = (real)3.14159265358979323846264338327950288L;

/* Carlson R_F(x,y,z), duplication theorem with the 5th-order series (Carlson 1995). */
static real carlson_rf(real x, real y, real z)
{
    real A0 = (x + y + z) / 3, A = A0;
    real Q = FABS(A0 - x);
    if (FABS(A0 - y) > Q) Q = FABS(A0 - y);
    if (FABS(A0 - z) > Q) Q = FABS(A0 - z);
    /* |error| < (3 r)^{-1/6}-scaled tolerance: iterate until 4^-n Q < tol |A| */
    real tol = (real)pow((double)(3 * REAL_EPS), 1.0 / 6.0);
    Q /= tol;
    real p4 = 1;
    for (int n = 0; n < 100; ++n) {
        if (p4 * Q < FABS(A)) break;
        real sx = SQRT(x), sy = SQRT(y), sz = SQRT(z);
        real lam = sx * sy + sx * sz + sy * sz;
        A = (A + lam) / 4; x = (x + lam) / 4; y = (y + lam) / 4; z = (z + lam) / 4;
        p4 /= 4;
    }
    /* deviations of the reduced variables from their mean */
    real Xd = 1 - x / A, Yd = 1 - y / A, Zd = -Xd - Yd;
    real E2 = Xd * Yd - Zd * Zd, E3 = Xd * Yd * Zd;
    return (1 - E2 / 10 + E3 / 14 + E2 * E2 / 24 - 3 * E2 * E3 / 44) / SQRT(A);
}

/* Carlson R_D(x,y,z), duplication (Carlson 1995, eq. 2.30-2.35). */
static real carlson_rd(real x, real y, real z)
{
    real A0 = (x + y + 3 * z) / 5, A = A0;
    real Q = FABS(A0 - x);
    if (FABS(A0 - y) > Q) Q = FABS(A0 - y);
    if (FABS(A0 - z) > Q) Q = FABS(A0 - z);
    real tol = (real)pow((double)(REAL_EPS / 4), 1.0 / 6.0);
    Q /= tol;
    real p4 = 1, sum = 0;
    for (int n = 0; n < 100; ++n) {
        if (p4 * Q < FABS(A)) break;
        real sx = SQRT(x), sy = SQRT(y), sz = SQRT(z);
        real lam = sx * sy + sx * sz + sy * sz;
        sum += p4 / (sz * (z + lam));
        A = (A + lam) / 4; x = (x + lam) / 4; y = (y + lam) / 4; z = (z + lam) / 4;
        p4 /= 4;
    }
    real Xd = 1 - x / A, Yd = 1 - y / A, Zd = -(Xd + Yd) / 3;
    real E2 = Xd * Yd - 6 * Zd * Zd;
    real E3 = (3 * Xd * Yd - 8 * Zd * Zd) * Zd;
    real E4 = 3 * (Xd * Yd - Zd * Zd) * Zd * Zd;
    real E5 = Xd * Yd * Zd * Zd * Zd;
    real ser = 1 - 3 * E2 / 14 + E3 / 6 + 9 * E2 * E2 / 88 - 3 * E4 / 22 - 9 * E2 * E3 / 52 + 3 * E5 / 26;
    return p4 * ser / (A * SQRT(A)) + 3 * sum;
}

/* K, E, D = (K-E)/m, S = int sin^2 cos^2 (1 - m sin^2)^{-3/2}, parameter m in [0,1). */
static void ellip_KEDS(real m, real *K, real *E, real *D, real *S)
{
    real k = carlson_rf(0, 1 - m, 1);
    real d = carlson_rd(0, 1 - m, 1) / 3;
    *K = k; *D = d; *E = k - m * d;
    if (m >= (real)0.05) {
        *S = (2 * d - k) / m;
    } else {
        /* S = (pi/16) 2F1(3/2,3/2;3;m): t_{n+1}/t_n = (n+3/2)^2 m / ((n+1)(n+3)) */
        real t = PI_R / 16, s = 0;
        for (int n = 0; n < 200; ++n) {
            s += t;
            if (t < REAL_EPS * s * (real)1e-3) break;
            real a = n + (real)1.5;
            t *= a * a * m / ((real)(n + 1) * (real)(n + 3));
        }
        *S = s;
    }
}

/* U^D = (rr, rz, zz), U^K = (r rb, r zb, z rb, z zb), header formulas. */
static void tensor2d(real r, real z, real rb, real zb, real UD[3], real UK[4])
{
    real dz = z - zb, dr = r - rb;
    real s = (r + rb) * (r + rb) + dz * dz;
    real d2 = dr * dr + dz * dz;
    real m = 4 * r * rb / s;
    real K, E, D, S;
    ellip_KEDS(m, &K, &E, &D, &S);
    real rs = SQRT(s);
    real P0 = 4 * E / (rs * d2);
    real Pc = 8 * D / (s * rs);
    real Pss = 16 * S / (s * rs);
    UD[0] = rb * rb * Pss + dz * dz * P0;
    UD[1] = -dz * (dr * P0 + rb * Pc);
    UD[2] = dr * dr * P0 + 2 * r * rb * Pc;
    UK[0] = dz * dz * (P0 - Pc) + r * rb * Pss;
    UK[1] = UD[1];
    UK[2] = dz * (-dr * P0 + r * Pc);
    UK[3] = UD[2];
}

void SUFFIX(oracle_ellip)(double m, double out[4])
{
    real K, E, D, S;
    ellip_KEDS((real)m, &K, &E, &D, &S);
    out[0] = (double)K; out[1] = (double)E; out[2] = (double)D; out[3] = (double)S;
}

void SUFFIX(oracle_tensor2d)(double r, double z, double rb, double zb, double UD[3], double UK[4])
{
    real ud[3], uk[4];
    tensor2d(r, z, rb, zb, ud, uk);
    for (int c = 0; c < 3; ++c) UD[c] = (double)ud[c];
    for (int c = 0; c < 4; ++c) UK[c] = (double)uk[c];
}

/*
 * Alg. 1 lines 3-12 for every integration point i (the paper runs one element per block; here
 * a plain loop).  Arrays: r,z,w[N]; f[S][N]; dfr,dfz[S][N] (physical gradient); e2[S] = e_b^2;
 * m0m[S] = m0/m_b.  Output GD[N][3] = (rr,rz,zz), GK[N][2] = (r,z).  i_begin/i_end select a
 * sub-range of rows (for sampled parity at full size and for the bounded timing sample).
 */
void SUFFIX(oracle_inner_integral)(int N, int S, const double *r, const double *z, const double *w,
                                   const double *f, const double *dfr, const double *dfz,
                                   const double *e2, const double *m0m, int i_begin, int i_end,
                                   double *GD, double *GK)
{
#pragma omp parallel for schedule(dynamic, 4)
    for (int i = i_begin; i < i_end; ++i) {
        real gd[3] = {0, 0, 0}, gk[2] = {0, 0};
        for (int j = 0; j < N; ++j) {
            /* coincident pair (d2 = 0): zero contribution (Q3).  On one mesh only j == i
             * coincides; with several grids (section III-C) points of different grids may too. */
            if (j == i || (r[j] == r[i] && z[j] == z[i])) continue;
            real UD[3], UK[4];
            tensor2d(r[i], z[i], r[j], z[j], UD, UK);
            real TD = 0, TKr = 0, TKz = 0; /* reset per j (Q4) */
            for (int b = 0; b < S; ++b) {
                TKr += (real)e2[b] * (real)m0m[b] * (real)dfr[(size_t)b * N + j];
                TKz += (real)e2[b] * (real)m0m[b] * (real)dfz[(size_t)b * N + j];
                TD += (real)e2[b] * (real)f[(size_t)b * N + j];
            }
            real wj = w[j];
            gk[0] += wj * (UK[0] * TKr + UK[1] * TKz);
            gk[1] += wj * (UK[2] * TKr + UK[3] * TKz);
            gd[0] += wj * TD * UD[0];
            gd[1] += wj * TD * UD[1];
            gd[2] += wj * TD * UD[2];
        }
        for (int c = 0; c < 3; ++c) GD[(size_t)i * 3 + c] = (double)gd[c];
        for (int c = 0; c < 2; ++c) GK[(size_t)i * 2 + c] = (double)gk[c];
    }
}
