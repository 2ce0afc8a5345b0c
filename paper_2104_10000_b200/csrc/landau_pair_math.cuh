// Device-side arithmetic of one point pair of the inner integral (step a3): fast fp64 reciprocal / square roots,
// the azimuth-integrated Landau tensor through a scaled AGM, its five distinct entries and the accumulation.
// PAPER.md Alg. 1 line 4 (L116), Eqs. 3, 7-8 (L44, L65-67); reading Q1.  Included by the kernels that
// evaluate pairs (landau_kernels.cu: per-problem pair kernel; landau_shared.cu: the batch-shared tensor).
#pragma once
#include <cuda_runtime.h>

namespace landau {

// ------------------------------------------------------------------------------------------------
// fast fp64 reciprocal / square roots: MUFU seed (relative error < 2^-19 including the truncation
// of the operand to its high word) + ONE cubic correction on the DFMA pipe (error ~ seed^3 < 1e-17).
// Not IEEE-rounded (~1 ulp), no special cases: arguments here are finite and > 0.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp_fast(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double p = fma(e, e, e);      // e + e^2
    return fma(y, p, y);                // y (1 + e + e^2)
}

// g = sqrt(x), yy = 1/sqrt(x)
__device__ __forceinline__ void sqrt_rsqrt_fast(double x, double &g, double &yy) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double r = fma(-t, y, 1.0);   // 1 - x y^2
    double p = fma(0.375, r, 0.5);
    p = p * r;                          // r/2 + 3 r^2/8
    g = fma(t, p, t);
    yy = fma(y, p, y);
}

// 2 sqrt(x) = t (2 + r + 3 r^2/4), t = x y, r = 1 - x y^2: the factor 2 sits in the correction
// polynomial, so the scaled AGM below needs no multiplication by 1/2 or 2 and no integer fix-up.
__device__ __forceinline__ double sqrt_times2_fast(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double r = fma(-t, y, 1.0);
#ifdef SQRT_SHALLOW      // one instruction more, one level less on the dependent chain: 2t + (t r)(1 + 3r/4)
    const double tr = t * r;
    const double p = fma(0.75, r, 1.0);
    return fma(tr, p, t + t);
#else
    const double p = fma(0.75, r, 1.0);
    const double q = fma(p, r, 2.0);
    return t * q;
#endif
}

// x * 2^e for a normal positive x that stays normal (integer add on the exponent field)
__device__ __forceinline__ double scale_pow2(double x, int e) {
    return __hiloint2double(__double2hiint(x) + (e << 20), __double2loint(x));
}

// ------------------------------------------------------------------------------------------------
// a3: pair kernel.  PAPER.md Alg. 1 lines 3-12 (L114-121), Eqs. 7-8 (L65-67).
//
// Azimuth-integrated Landau tensor through a SCALED arithmetic-geometric mean (DESIGN.md "Elliptic
// integrals on the device").  With a0 = sqrt(s), b0 = sqrt(d2), q = 4 r rb = s - d2 and
// A_k = 2^k a_k, B_k = 2^k b_k:
//     A_{k+1} = A_k + B_k,  B_{k+1} = 2 sqrt(A_k B_k),  C_{k+1} = A_k - B_k = 2^{k+1} c_{k+1}
//     (powers of two are applied at the end by integer adds on the exponent field)
//     K(m)/sqrt(s) = pi/(2 lim a_k) = pi 2^k / A_{k+1}
//     W = [sum_{k>=1} 2^k c_k^2]/q^2 = 1/(2 A_1^2) + (sum_{k>=2} C_k^2 / 2^k)/q^2   (c_1 = q/(4 a_1))
//     Pss = 16 Kt W,  Pc = 4 Kt (1 + q W)/s,  P0 = 2 Kt (s + d2 - q^2 W)/(s d2),  Kt = K/sqrt(s)
// every sum has positive terms except the bracket of P0 (= 2 s E/K: bounded cancellation ~ K/E).
// Evaluated with rho2 = 2 r rb = q/2, 2W and 4Kt so that no multiplication by a power of two remains:
//     g = 1 + q W = 1 + rho2 (2W),  Pss/2 = (4Kt)(2W),  Pc = (4Kt/s) g,  P0 = (4Kt/s)(s - rho2 g)/d2
//     (s - rho2 g = (s + d2 - q^2 W)/2 because s - d2 = q).
// The AGM is NOT run to convergence: after P passes (A = A_{P+1}, B = B_{P+1}) with e = c_{P+2}/a_{P+2} =
// (A - B)/(A + B) small, both limits are finished in closed form (x = e^2):
//     pi/(2 agm(a, b)) = K(e)/a_{P+2}               ->  4 Kt = 4 pi 2^(P+1) F(x)/(A + B),   F = (2/pi) K(e)
//     sum_{j>=P+2} 2^j c_j^2 = 2 a_{P+2}^2 2^(P+2) (1 - E(e)/K(e)) = (C^2 / 2^(P+2)) G(x),   C = A - B,
//     F(x) = 1 + x/4 + 9x^2/64 + 25x^3/256 + 1225x^4/16384 + ..,  G(x) = 2(1 - E/K)/x = 1 + x/8 + x^2/16 + 41x^3/1024 + ..
// (the standard AGM relation E = K (1 - sum_{i>=0} 2^(i-1) c_i^2) applied to the sequence restarted at step P+2).
// With e <= 2^-6 the truncations used (F to x^3, G to x^3) are below 2^-51.7 (F) and 2^-54 of W (G's term is at most
// 2^-7 of W).
// The number of passes follows from d2/s = k'^2 ALONE (e_1 = (1-k')/(1+k'), e_{k+1} = e_k^2/(1+sqrt(1-e_k^2))^2):
// P = 0 for d2/s >= 0.366, 1 for >= 0.0129, 2 for >= 1.05e-5, 3 for >= 6.9e-12, 4 for >= 2.9e-24, else 5 -- so it is
// decided BEFORE the first square root from the exponent fields of d2 and s (integer compares of the high words,
// thresholds 0.0862 = max |m - log2(1+m)| on the safe side), the warp takes the maximum over its lanes
// (one REDUX), and the loop has a known trip count: no vote waits for the end of a dependent sqrt chain.
// Measured against the version that iterated to c <= 2^-26 a with an exit vote per pass: DESIGN.md 6.1.
// The constant 4 pi is not applied here: it sits in the weights w_in of T (k_fields_beta).
//
// FP64 issue cost on sm_100a (measured): 2 cycles per warp instruction and SM
// sub-partition, 3 cycles for a DFMA with three distinct register operands; 8 cycles dependent
// latency.  Hence the lock-step evaluation of several pairs per thread and the care for operand count.
// ------------------------------------------------------------------------------------------------
struct PairAcc { double drr, drz, dzz, kr, kz; };

// hi32(d2) - hi32(s) below these -> one more AGM pass (2^20 (log2 of the d2/s thresholds above + 0.0862), rounded up)
constexpr int AGM_T0 = -1430341, AGM_T1 = -6495283, AGM_T2 = -17255704, AGM_T3 = -38796084, AGM_T4 = -81876859;

// What a thread keeps of one of its i points.
struct IPoint {
    double r, z;
    double r2x;     // 2 r
    double rr2;     // 2 r^2
    double c;       // 1/(16 r^2): 1/q^2 = c_i / r_j^2
    double tD, tKr, tKz;
};
// One j point, read from shared memory (SoA there, see k_pair_sym).
struct JPoint { double r, z, invr2, rr2, tD, tKr, tKz; };

// P0, Pc and Pss/2 of a pair plus the geometry the tensor entries need (rho2 = 2 r_i r_j).
struct PairParts { double P0, Pc, Pssh, dz, dr, dr2, rho2; };

// NP pairs (i_u, j), u < NP, evaluated in lock-step: NP independent dependency chains per thread
// through the AGM, one exit vote for all of them.
template <int NP, bool CHECK_SELF>
__device__ __forceinline__ void pair_parts(const IPoint (&pi)[NP], const JPoint &pj, PairParts (&pp)[NP]) {
    double s[NP], ys[NP], yd[NP], iA1[NP], A[NP], B[NP], V[NP];
    bool self[NP];
    int dHmin = 0;
#pragma unroll
    for (int u = 0; u < NP; ++u) {
        pp[u].dz = pi[u].z - pj.z; pp[u].dr = pi[u].r - pj.r;
        const double dz2 = pp[u].dz * pp[u].dz;
        pp[u].dr2 = pp[u].dr * pp[u].dr;
        double d2 = pp[u].dr2 + dz2;
        pp[u].rho2 = pi[u].r2x * pj.r;
        self[u] = false;
        if (CHECK_SELF) {             // coincident pair (j == i): contributes nothing (reading Q3)
            self[u] = !(d2 > 0.0);
            if (self[u]) d2 = 1.0;
        }
        s[u] = fma(2.0, pp[u].rho2, d2);                 // (r_i + r_j)^2 + dz^2 = d2 + 4 r_i r_j
        dHmin = min(dHmin, __double2hiint(d2) - __double2hiint(s[u]));  // ~ 2^20 log2(d2/s) <= 0
        double a0, b0;
        sqrt_rsqrt_fast(s[u], a0, ys[u]);
        sqrt_rsqrt_fast(d2, b0, yd[u]);
        A[u] = a0 + b0;                                  // A_1 = 2 a_1
        B[u] = sqrt_times2_fast(a0 * b0);
        iA1[u] = rcp_fast(A[u]);
        V[u] = 0.0;
    }
    // the smallest d2/s of the warp decides (every lane is here: lock-step callers); the compares run once per
    // warp on the uniform datapath instead of once per pair
    dHmin = __reduce_min_sync(0xffffffffu, dHmin);
    const int npass = int(dHmin < AGM_T0) + int(dHmin < AGM_T1) + int(dHmin < AGM_T2) + int(dHmin < AGM_T3) + int(dHmin < AGM_T4);
    // V_P = 2 V_{P-1} + C_{P+1}^2: after P passes sum_{j=2}^{P+1} C_j^2 / 2^j = V / 2^(P+1)
#pragma unroll 1
    for (int p = 0; p < npass; ++p) {
#pragma unroll
        for (int u = 0; u < NP; ++u) {
            const double C = A[u] - B[u];
            V[u] = fma(V[u], 2.0, C * C);
            const double X = A[u] * B[u];
            A[u] = A[u] + B[u];
            B[u] = sqrt_times2_fast(X);
        }
    }
#pragma unroll
    for (int u = 0; u < NP; ++u) {
        const double C = A[u] - B[u];                    // C_{P+2}
        const double iAp = rcp_fast(A[u] + B[u]);        // 1 / A_{P+2}
        const double e = C * iAp;
        const double x = e * e;
        const double F = fma(x, fma(x, fma(x, 25.0 / 256.0, 9.0 / 64.0), 0.25), 1.0);     // next term <= 0.075 2^-48
        const double G = fma(x, fma(x, fma(x, 41.0 / 1024.0, 0.0625), 0.125), 1.0);
        const double K4 = scale_pow2(iAp * F, npass + 1);              // 4 K/sqrt(s) / (4 pi)
        const double Vf = fma(V[u], 2.0, (C * C) * G);                 // sum_{j>=2} C_j^2 / 2^j = Vf / 2^(P+2)
        // 2 W = 1/A_1^2 + Vf 2^-(P+1) / q^2.  1/q^2 is a normal number far from the exponent limits (Vf may be
        // tiny for far pairs: scale 1/q^2, not the product).
        const double invq2 = pi[u].c * pj.invr2;
        const double W2 = fma(iA1[u], iA1[u], Vf * scale_pow2(invq2, -(npass + 1)));
        const double g = fma(pp[u].rho2, W2, 1.0);       // 1 + q W
        const double Kh = K4 * (ys[u] * ys[u]);          // 4 K / s^(3/2)
        pp[u].Pssh = K4 * W2;
        pp[u].Pc = Kh * g;
        pp[u].P0 = (Kh * (yd[u] * yd[u])) * fma(-pp[u].rho2, g, s[u]);   // (s + d2 - q^2 W)/2 = s - rho2 (1 + q W)
        if (CHECK_SELF && self[u]) { pp[u].Pssh = 0.0; pp[u].Pc = 0.0; pp[u].P0 = 0.0; }
    }
}

// The five distinct tensor entries of a pair (Q1) from its parts:
//   UDrr = U^D_rr(i,j), UDrrT = U^D_rr(j,i), A2 = -U^D_rz(i,j) = -U^K_zr(j,i), A3 = U^D_zz = U^K_zz (both ways),
//   A4 = U^K_rr (both ways), A5 = U^K_zr(i,j) = U^D_rz(j,i)
struct PairTensor { double UDrr, UDrrT, A2, A3, A4, A5; };

__device__ __forceinline__ PairTensor pair_tensor(const IPoint &pi, const JPoint &pj, const PairParts &pp) {
    PairTensor t;
    const double dzP0 = pp.dz * pp.P0;
    const double A1 = pp.dz * dzP0;                      // dz^2 P0
    const double b = pp.dr * dzP0;                       // dz dr P0
    const double e = pp.dz * pp.Pc;
    t.A2 = fma(pj.r, e, b);                              // dz (dr P0 + r_j Pc)
    t.A5 = fma(pi.r, e, -b);                             // dz (-dr P0 + r_i Pc)
    t.A3 = fma(pp.dr2, pp.P0, pp.rho2 * pp.Pc);          // dr^2 P0 + 2 r_i r_j Pc
    t.A4 = fma(pp.rho2, pp.Pssh, fma(-pp.dz, e, A1));    // dz^2 (P0 - Pc) + r_i r_j Pss
    t.UDrr = fma(pj.rr2, pp.Pssh, A1);                   // r_j^2 Pss + dz^2 P0
    t.UDrrT = fma(pi.rr2, pp.Pssh, A1);
    return t;
}

__device__ __forceinline__ void accumulate_i(PairAcc &acc, const JPoint &pj, const PairTensor &t) {
    acc.drr = fma(pj.tD, t.UDrr, acc.drr);
    acc.drz = fma(-pj.tD, t.A2, acc.drz);
    acc.dzz = fma(pj.tD, t.A3, acc.dzz);
    acc.kr = fma(t.A4, pj.tKr, fma(-t.A2, pj.tKz, acc.kr));
    acc.kz = fma(t.A5, pj.tKr, fma(t.A3, pj.tKz, acc.kz));
}

}  // namespace landau
