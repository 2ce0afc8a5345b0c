// Device kernels of the Landau Jacobian hot path for sm_100a (fp64).  Steps a1-a8 of
// include/landau.h; Algorithm 1 (L109-131).  See DESIGN.md "Kernels" for the layout
// and the roofline of each.
//
//   k_fields_beta   a1+a2  f -> w_in*T_D, w_in*T_K at every integration point (beta sum hoisted
//                          out of the pair loop: it does not depend on i)
//   k_pair_sym      a3     all-pairs inner integral over tile pairs, one tensor evaluation per
//                          unordered pair, thread owns i, j broadcast from shared memory
//   k_element       a4+a5  scale, transform, element matrix C_e and element vector C_e u
//   k_gather        a6/a7  deterministic gather of element entries into CSR values / C(f)
//   k_mass_element  a8     shift * element mass matrices (gathered by k_gather)
//   k_dfma_probe           FP64 peak probe (measurement aid)
#include <cuda_runtime.h>

#include <cstdint>

#include "landau_kernels.h"

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
    const double p = fma(0.75, r, 1.0);
    const double q = fma(p, r, 2.0);
    return t * q;
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
// The iteration stops for the whole warp once every lane's next c would be < 2^-27 a (the then
// neglected term is < 6e-17 a).  The test compares exponents with integer ops, one pass ahead.
// ------------------------------------------------------------------------------------------------
struct PairAcc { double drr, drz, dzz, kr, kz; };
struct __align__(16) JPoint { double r, z, invr, tD, tKr, tKz; };

constexpr int AGM_MAX_STEPS = 8;

// P0, Pc, Pss of one pair (header above) plus the geometry the tensor entries need.
struct PairParts { double P0, Pc, Pss, dz, dr, dz2, dr2, rho; };

template <bool CHECK_SELF>
__device__ __forceinline__ PairParts pair_parts(double ri, double zi, double ri4, double inv4ri, const JPoint &pj) {
    PairParts pp;
    const double rj = pj.r;
    const double sr = ri + rj;
    pp.dz = zi - pj.z; pp.dr = ri - rj;
    pp.dz2 = pp.dz * pp.dz; pp.dr2 = pp.dr * pp.dr;
    double d2 = pp.dr2 + pp.dz2;
    const double s = fma(sr, sr, pp.dz2);
    bool self = false;
    if (CHECK_SELF) {                 // coincident pair (j == i): contributes nothing (reading Q3)
        self = !(d2 > 0.0);
        if (self) d2 = 1.0;
    }
    double a0, b0, ys, yd;
    sqrt_rsqrt_fast(s, a0, ys);
    sqrt_rsqrt_fast(d2, b0, yd);
    double A = a0 + b0;               // A_1 = 2 a_1
    double B = sqrt_times2_fast(a0 * b0);
    const double iA1 = rcp_fast(A);
    // Rolled loop, state in fixed registers.  V_P = 2 V_{P-1} + C_{P+1}^2, so after P passes
    // sum_{k>=2} C_k^2/2^k = V / 2^{P+1}, and 2 K/sqrt(s) = 2 pi 2^P / A_{P+1}.
    // The exit is decided ONE PASS AHEAD so that the branch never waits on fresh data:
    // c_{k+2} = c_{k+1}^2/(4 a_{k+2}) exactly, hence C_{k+1} <= 2^-12 A_k in every lane guarantees
    // c_{k+2} < 2^-27 a after the next pass, which is then the last (its C only feeds V).
    double V = 0.0;
    int P = 0;
    bool last = false;
#pragma unroll 1
    for (;;) {
        const double C = A - B;
        V = fma(V, 2.0, C * C);
        ++P;
        if (last || P == AGM_MAX_STEPS) break;
        last = __all_sync(0xffffffffu, __double2hiint(C) + (13 << 20) <= __double2hiint(A));
        const double X = A * B;
        A = A + B;
        B = sqrt_times2_fast(X);
    }
    A = A + B;
    const double KP2 = scale_pow2(6.283185307179586476925286766559 * rcp_fast(A), P);   // 2 K/sqrt(s)
    const double q = ri4 * rj;
    pp.rho = ri * rj;
    const double invq = inv4ri * pj.invr;
    // 1/q^2 is a normal number far from the exponent limits (V may be 0 for far pairs: scale 1/q^2, not the product)
    const double W = fma(0.5 * iA1, iA1, V * scale_pow2(invq * invq, -(P + 1)));
    const double Ks = KP2 * (ys * ys);
    const double x = q * W;
    pp.Pc = Ks * fma(2.0, x, 2.0);
    pp.P0 = Ks * (yd * yd) * fma(-q, x, s + d2);
    pp.Pss = 8.0 * (KP2 * W);
    if (CHECK_SELF && self) { pp.Pss = 0.0; pp.Pc = 0.0; pp.P0 = 0.0; }
    return pp;
}

// ------------------------------------------------------------------------------------------------
// Symmetric tile-pair kernel.  P0, Pc, Pss are exchange-symmetric and
//   U^D_rr(j,i) = ri^2 Pss + dz^2 P0,  U^D_rz(j,i) = U^K_zr(i,j),  U^D_zz(j,i) = U^D_zz(i,j),
//   U^K_rr(j,i) = U^K_rr(i,j),  U^K_zr(j,i) = U^D_rz(i,j)
// so one elliptic evaluation serves the ordered pairs (i,j) and (j,i) (the paper notes the
// symmetry, L193, and does not exploit it).
//
// Points are cut into tiles of TS; block (I <= J, problem b), TS threads, thread t owns
// i = I*TS + t and walks the j of tile J held in shared memory.  It keeps the i-side sums in
// registers; the j-side sums rotate around the warp's lanes together with their j (see below) and
// are parked in shared memory per warp, then added over the warps in warp order.  Diagonal blocks (I == J) do
// all ordered pairs of the tile with the coincident-pair test.
//
// Deterministic order: Gpart[b][src tile][5][N] holds, for every target
// point, the partial sum over the points of one source tile; each slot is written by exactly one
// block, and k_element / k_sum_partials add the slabs in tile order.  TS depends on N only, so a
// batched build is bitwise equal to single builds.
// ------------------------------------------------------------------------------------------------
#ifndef PAIR_K_UNROLL
#define PAIR_K_UNROLL 2   // j steps per loop trip (sweep 1/2: 247/253 GPair/s)
#endif
constexpr int kPairUnroll = PAIR_K_UNROLL;
#ifndef PAIR_MIN_BLOCKS
#define PAIR_MIN_BLOCKS 5   // resident blocks per SM the register budget is capped for (sweep 4/5/6: 239/247/246 GPair/s)
#endif
template <int TS>
__global__ void __launch_bounds__(TS, PAIR_MIN_BLOCKS)
k_pair_sym(int N, int ntiles, const double *__restrict__ r, const double *__restrict__ z, const double *__restrict__ invr,
           const double *__restrict__ T, double *__restrict__ Gpart) {
    constexpr int NW = TS / 32;
    __shared__ JPoint sj[2 * TS];        // every 32-point sub-tile is stored twice in a row: rotated walks need no wrap
    __shared__ double sacc[NW][5][TS];
    const int b = blockIdx.y;
    // linear tile-pair index p = J (J+1)/2 + I, I <= J
    const int p = blockIdx.x;
    int J = int((sqrt(8.0 * double(p) + 1.0) - 1.0) * 0.5);
    while ((J + 1) * (J + 2) / 2 <= p) ++J;
    while (J * (J + 1) / 2 > p) --J;
    const int I = p - J * (J + 1) / 2;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double *Tb = T + (size_t)b * 3 * N;
    const int i = I * TS + tid;
    const bool valid = i < N;
    const int ic = valid ? i : N - 1;
    const double ri = r[ic], zi = z[ic];
    const double ri4 = 4.0 * ri, inv4ri = 0.25 * invr[ic], ri2 = ri * ri;
    const double tDi = valid ? Tb[ic] : 0.0, tKri = valid ? Tb[N + ic] : 0.0, tKzi = valid ? Tb[2 * N + ic] : 0.0;
    const int jbase = J * TS;
    const int cnt = min(TS, N - jbase);
    {
        JPoint pj;
        if (tid < cnt) {
            const int j = jbase + tid;
            pj.r = r[j]; pj.z = z[j]; pj.invr = invr[j];
            pj.tD = Tb[j]; pj.tKr = Tb[N + j]; pj.tKz = Tb[2 * N + j];
        } else {
            // padding of a ragged tile: a far-away point with zero weight (finite tensor, no effect)
            pj.r = 1.0; pj.z = 1.0e6; pj.invr = 1.0; pj.tD = 0.0; pj.tKr = 0.0; pj.tKz = 0.0;
        }
        sj[warp * 64 + lane] = pj;
        sj[warp * 64 + 32 + lane] = pj;
    }
    __syncthreads();
    PairAcc acc = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (I == J) {
        for (int t = 0; t < cnt; ++t) {
            const JPoint pj = sj[(t >> 5) * 64 + (t & 31)];
            const PairParts pp = pair_parts<true>(ri, zi, ri4, inv4ri, pj);
            const double UDrr = fma(pj.r * pj.r, pp.Pss, pp.dz2 * pp.P0);
            const double nUDrz = pp.dz * fma(pp.dr, pp.P0, pj.r * pp.Pc);         // -U^D_rz(i,j)
            const double UDzz = fma(2.0, pp.rho * pp.Pc, pp.dr2 * pp.P0);
            const double UKrr = fma(pp.dz2, pp.P0 - pp.Pc, pp.rho * pp.Pss);
            const double UKzr = pp.dz * fma(-pp.dr, pp.P0, ri * pp.Pc);
            acc.drr = fma(pj.tD, UDrr, acc.drr);
            acc.drz = fma(-pj.tD, nUDrz, acc.drz);
            acc.dzz = fma(pj.tD, UDzz, acc.dzz);
            acc.kr = fma(UKrr, pj.tKr, fma(-nUDrz, pj.tKz, acc.kr));
            acc.kz = fma(UKzr, pj.tKr, fma(UDzz, pj.tKz, acc.kz));
        }
    } else {
        // Lane t walks the 32 j of a sub-tile in rotated order, j = (t + k) mod 32, so that the warp
        // touches 32 different j per step; the j-side sums travel around the lanes with their j
        // (one shuffle per value per step) and need no cross-lane reduction.
        const int nsub = (cnt + 31) >> 5;
        const int src = (lane + 1) & 31;
        for (int sub = 0; sub < nsub; ++sub) {
            double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0, v4 = 0.0;
            // explicit 32-bit shared address, advanced by one JPoint per step (three 16-byte loads)
            unsigned sa = (unsigned)__cvta_generic_to_shared(sj + sub * 64 + lane);
#pragma unroll kPairUnroll
            for (int k = 0; k < 32; ++k, sa += (unsigned)sizeof(JPoint)) {
                JPoint pj;
                asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(pj.r), "=d"(pj.z) : "r"(sa));
                asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+16];" : "=d"(pj.invr), "=d"(pj.tD) : "r"(sa));
                asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+32];" : "=d"(pj.tKr), "=d"(pj.tKz) : "r"(sa));
                const PairParts pp = pair_parts<false>(ri, zi, ri4, inv4ri, pj);
                const double dzP0 = pp.dz2 * pp.P0;
                const double UDrr = fma(pj.r * pj.r, pp.Pss, dzP0);
                const double UDrrT = fma(ri2, pp.Pss, dzP0);                          // U^D_rr(j,i)
                const double nUDrz = pp.dz * fma(pp.dr, pp.P0, pj.r * pp.Pc);         // -U^D_rz(i,j)
                const double UDzz = fma(2.0, pp.rho * pp.Pc, pp.dr2 * pp.P0);
                const double UKrr = fma(pp.dz2, pp.P0 - pp.Pc, pp.rho * pp.Pss);
                const double UKzr = pp.dz * fma(-pp.dr, pp.P0, ri * pp.Pc);           // = U^D_rz(j,i)
                acc.drr = fma(pj.tD, UDrr, acc.drr);
                acc.drz = fma(-pj.tD, nUDrz, acc.drz);
                acc.dzz = fma(pj.tD, UDzz, acc.dzz);
                acc.kr = fma(UKrr, pj.tKr, fma(-nUDrz, pj.tKz, acc.kr));
                acc.kz = fma(UKzr, pj.tKr, fma(UDzz, pj.tKz, acc.kz));
                // terms of target j from source i, then pass the sums on with their j
                v0 = fma(tDi, UDrrT, v0);
                v1 = fma(tDi, UKzr, v1);
                v2 = fma(tDi, UDzz, v2);
                v3 = fma(UKrr, tKri, fma(UKzr, tKzi, v3));
                v4 = fma(-nUDrz, tKri, fma(UDzz, tKzi, v4));
                v0 = __shfl_sync(0xffffffffu, v0, src);
                v1 = __shfl_sync(0xffffffffu, v1, src);
                v2 = __shfl_sync(0xffffffffu, v2, src);
                v3 = __shfl_sync(0xffffffffu, v3, src);
                v4 = __shfl_sync(0xffffffffu, v4, src);
            }
            const int jl = sub * 32 + lane;
            sacc[warp][0][jl] = v0; sacc[warp][1][jl] = v1; sacc[warp][2][jl] = v2;
            sacc[warp][3][jl] = v3; sacc[warp][4][jl] = v4;
        }
    }
    if (valid) {
        double *G = Gpart + ((size_t)b * ntiles + J) * 5 * N;
        G[i] = acc.drr; G[N + i] = acc.drz; G[2 * N + i] = acc.dzz; G[3 * N + i] = acc.kr; G[4 * N + i] = acc.kz;
    }
    if (I != J) {
        __syncthreads();
        if (tid < cnt) {
            double *G = Gpart + ((size_t)b * ntiles + I) * 5 * N + jbase + tid;
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                double sum = sacc[0][c][tid];
#pragma unroll
                for (int w = 1; w < NW; ++w) sum += sacc[w][c][tid];
                G[(size_t)c * N] = sum;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a1 + a2: field values at the integration points and the beta sums (L101, Alg. 1 lines 5-8,
// Eq. 10).  grid = (ceil(Ne/EPB), nb), block = (Nq, EPB).  Thread (q, e): local node a = q
// gathers u_a = sum P_e[a,d] f_b[d]; then f = B u, grad f = J^-T (E u).
// Output T[b][3][N] = w_in * (T_D, T_Kr, T_Kz): the weight of the inner sum is folded in here.
// ------------------------------------------------------------------------------------------------
constexpr int FIELD_EPB = 8;

__global__ void k_fields_beta(DeviceSpace ds, const double *__restrict__ f, double *__restrict__ T) {
    __shared__ double s_u[FIELD_EPB][16];
    const int b = blockIdx.y;
    const int e = blockIdx.x * FIELD_EPB + threadIdx.y;
    const int q = threadIdx.x;
    const bool valid = e < ds.Ne;
    const int Nb = ds.Nb;
    const double *fb = f + (size_t)b * ds.S * ds.n;
    double tD = 0.0, tKr = 0.0, tKz = 0.0;
    double ijr = 0.0, ijz = 0.0;
    if (valid) { ijr = ds.invJ[2 * e]; ijz = ds.invJ[2 * e + 1]; }
    for (int sp = 0; sp < ds.S; ++sp) {
        if (valid) {
            double u = 0.0;
            const int t0 = ds.lptr[e * Nb + q], t1 = ds.lptr[e * Nb + q + 1];
            for (int t = t0; t < t1; ++t) u = fma(ds.lw[t], fb[(size_t)sp * ds.n + ds.ldof[t]], u);
            s_u[threadIdx.y][q] = u;
        }
        __syncthreads();
        if (valid) {
            double fq = 0.0, g0 = 0.0, g1 = 0.0;
            for (int a = 0; a < Nb; ++a) {
                const double u = s_u[threadIdx.y][a];
                fq = fma(ds.B[q * Nb + a], u, fq);
                g0 = fma(ds.E0[q * Nb + a], u, g0);
                g1 = fma(ds.E1[q * Nb + a], u, g1);
            }
            const double e2 = ds.e2[sp], em = ds.e2[sp] * ds.m0m[sp];
            tD = fma(e2, fq, tD);
            tKr = fma(em, ijr * g0, tKr);
            tKz = fma(em, ijz * g1, tKz);
        }
        __syncthreads();
    }
    if (valid) {
        const int gi = e * ds.Nq + q;
        const double w = ds.w_in[gi];
        double *Tb = T + (size_t)b * 3 * ds.N;
        Tb[gi] = w * tD; Tb[ds.N + gi] = w * tKr; Tb[2 * ds.N + gi] = w * tKz;
    }
}

// ------------------------------------------------------------------------------------------------
// a4 + a5 (+ element part of a7): Alg. 1 lines 13-23 (L122-131).  grid = (Ne, nb), block = Nb*Nb
// threads; the block loops over the species (tabulations and G are loaded once per cell).
// Two phases per species, both thread-per-entry on Nq x Nb = Nb x Nb arrays:
//   X[q][b] = DDrr_q E0_qb + DDrz_q E1_qb + KKr_q B_qb,   Y[q][b] = DDrz_q E0_qb + DDzz_q E1_qb + KKz_q B_qb
//   C_e[a][b] = sum_q ( E0_qa X_qb + E1_qa Y_qb )
// (the same sum as line 23, factored so that the q loop is two FMAs).  Also writes ce = C_e u
// (u = P_e f_alpha), the element vector of C(f).  G is the tile-order sum of the pair kernel's slabs.
// ------------------------------------------------------------------------------------------------
__global__ void k_element(DeviceSpace ds, int jsplit, const double *__restrict__ f, const double *__restrict__ Gpart,
                          double *__restrict__ Ce, double *__restrict__ ce) {
    __shared__ double s_g[16][5];      // w_out * (invJ-transformed G_D rr, rz, zz, G_K r, z), species-independent
    __shared__ double s_B[256], s_E0[256], s_E1[256], s_X[256], s_Y[256], s_Ce[256], s_u[16];
    const int e = blockIdx.x, b = blockIdx.y;
    const int Nb = ds.Nb, Nq = ds.Nq, N = ds.N;
    const int tid = threadIdx.x;
    s_B[tid] = ds.B[tid]; s_E0[tid] = ds.E0[tid]; s_E1[tid] = ds.E1[tid];
    if (tid < Nq) {
        const int gi = e * Nq + tid;
        double g[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        for (int js = 0; js < jsplit; ++js) {
            const double *G = Gpart + ((size_t)b * jsplit + js) * 5 * N;
#pragma unroll
            for (int c = 0; c < 5; ++c) g[c] += G[c * N + gi];
        }
        const double ir = ds.invJ[2 * e], iz = ds.invJ[2 * e + 1], w = ds.w_out[gi];
        s_g[tid][0] = ir * ir * w * g[0];
        s_g[tid][1] = ir * iz * w * g[1];
        s_g[tid][2] = iz * iz * w * g[2];
        s_g[tid][3] = ir * w * g[3];
        s_g[tid][4] = iz * w * g[4];
    }
    const int a = tid / Nb, bb = tid % Nb;   // phase 1: (q, b) = (a, bb); phase 2: (a, b) = (a, bb)
    for (int sp = 0; sp < ds.S; ++sp) {
        __syncthreads();                      // s_g / tabulations ready; previous species done with s_X, s_Y, s_Ce, s_u
        if (tid < Nb) {
            const double *fa = f + ((size_t)b * ds.S + sp) * ds.n;
            double u = 0.0;
            for (int t = ds.lptr[e * Nb + tid]; t < ds.lptr[e * Nb + tid + 1]; ++t) u = fma(ds.lw[t], fa[ds.ldof[t]], u);
            s_u[tid] = u;
        }
        {
            const double kf = ds.kfac[sp], df = ds.dfac[sp];
            const int q = a;
            const double e0 = s_E0[q * Nb + bb], e1 = s_E1[q * Nb + bb], bq = s_B[q * Nb + bb];
            const double drr = df * s_g[q][0], drz = df * s_g[q][1], dzz = df * s_g[q][2];
            s_X[tid] = fma(drr, e0, fma(drz, e1, kf * s_g[q][3] * bq));
            s_Y[tid] = fma(drz, e0, fma(dzz, e1, kf * s_g[q][4] * bq));
        }
        __syncthreads();
        double acc = 0.0;
        for (int q = 0; q < Nq; ++q)
            acc = fma(s_E0[q * Nb + a], s_X[q * Nb + bb], fma(s_E1[q * Nb + a], s_Y[q * Nb + bb], acc));
        const size_t mat = ((size_t)b * ds.S + sp) * ds.Ne + e;
        Ce[mat * Nb * Nb + tid] = acc;
        s_Ce[tid] = acc;
        __syncthreads();
        if (tid < Nb) {
            double v = 0.0;
            for (int c = 0; c < Nb; ++c) v = fma(s_Ce[tid * Nb + c], s_u[c], v);
            ce[mat * Nb + tid] = v;
        }
    }
}

// a8: element mass matrices, M_e[a][b] = shift sum_q w_out B_qa B_qb (L280).  grid = Ne.
__global__ void k_mass_element(DeviceSpace ds, double shift, double *__restrict__ Ce) {
    const int e = blockIdx.x, Nb = ds.Nb, tid = threadIdx.x;
    const int a = tid / Nb, b = tid % Nb;
    double acc = 0.0;
    for (int q = 0; q < ds.Nq; ++q) acc = fma(ds.w_out[e * ds.Nq + q] * ds.B[q * Nb + a], ds.B[q * Nb + b], acc);
    Ce[(size_t)e * Nb * Nb + tid] = shift * acc;
}

// a6 / a7: out[m][k] = sum_{t in [ptr[k], ptr[k+1])} w[t] * src[m*stride + idx[t]], fixed order
// (owner computes; replaces the paper's atomic MatSetValues, L165-167).  grid = (ceil(K/256), nmat).
__global__ void k_gather(int K, size_t stride, const int32_t *__restrict__ ptr, const int32_t *__restrict__ idx,
                         const double *__restrict__ w, const double *__restrict__ src, double *__restrict__ out) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= K) return;
    const double *s = src + (size_t)blockIdx.y * stride;
    double acc = 0.0;
    for (int t = ptr[k]; t < ptr[k + 1]; ++t) acc = fma(w[t], s[idx[t]], acc);
    out[(size_t)blockIdx.y * K + k] = acc;
}

// Sums the j-split partials (used by landau_inner_integral when jsplit > 1).  grid over 5N x nb.
__global__ void k_sum_partials(int n5, int jsplit, const double *__restrict__ Gpart, double *__restrict__ G) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n5) return;
    const size_t b = blockIdx.y;
    double acc = 0.0;
    for (int js = 0; js < jsplit; ++js) acc += Gpart[(b * jsplit + js) * n5 + t];
    G[b * n5 + t] = acc;
}

// FP64 peak probe: 8 independent DFMA chains per thread, all operands in registers.
__global__ void k_dfma_probe(int iters, double *out) {
    double x0 = threadIdx.x * 1e-9, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    const double a = 0.999999999, c = 1e-12;
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, a, c); x1 = fma(x1, a, c); x2 = fma(x2, a, c); x3 = fma(x3, a, c);
        x4 = fma(x4, a, c); x5 = fma(x5, a, c); x6 = fma(x6, a, c); x7 = fma(x7, a, c);
    }
    const double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == 12345.678) out[0] = s;  // keep the chains alive
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
// Tile size of the pair kernel: a function of N ONLY (it fixes the summation order).
int pair_tile_size(int N) { return N >= 4096 ? 128 : (N >= 1024 ? 64 : 32); }
int pair_tiles(int N) { const int ts = pair_tile_size(N); return (N + ts - 1) / ts; }

int launch_fields_beta(const DeviceSpace &ds, int nb, const double *f, double *T, cudaStream_t st) {
    dim3 grid((ds.Ne + FIELD_EPB - 1) / FIELD_EPB, nb), block(ds.Nq, FIELD_EPB);
    k_fields_beta<<<grid, block, 0, st>>>(ds, f, T);
    return 1;
}

int launch_pair(const DeviceSpace &ds, int nb, const double *T, double *Gpart, cudaStream_t st) {
    const int ts = pair_tile_size(ds.N), nt = pair_tiles(ds.N);
    dim3 grid(nt * (nt + 1) / 2, nb);
    if (ts == 128) k_pair_sym<128><<<grid, 128, 0, st>>>(ds.N, nt, ds.r, ds.z, ds.invr, T, Gpart);
    else if (ts == 64) k_pair_sym<64><<<grid, 64, 0, st>>>(ds.N, nt, ds.r, ds.z, ds.invr, T, Gpart);
    else k_pair_sym<32><<<grid, 32, 0, st>>>(ds.N, nt, ds.r, ds.z, ds.invr, T, Gpart);
    return 1;
}

int launch_element(const DeviceSpace &ds, int nb, int jsplit, const double *f, const double *G, double *Ce, double *ce,
                   cudaStream_t st) {
    dim3 grid(ds.Ne, nb);
    k_element<<<grid, ds.Nb * ds.Nb, 0, st>>>(ds, jsplit, f, G, Ce, ce);
    return 1;
}

int launch_gather_vals(const DeviceSpace &ds, int nmat, const double *Ce, double *vals, cudaStream_t st) {
    dim3 grid((ds.nnz + 255) / 256, nmat);
    k_gather<<<grid, 256, 0, st>>>(ds.nnz, (size_t)ds.Ne * ds.Nb * ds.Nb, ds.gptr, ds.gidx, ds.gw, Ce, vals);
    return 1;
}

int launch_gather_cf(const DeviceSpace &ds, int nvec, const double *ce, double *Cf, cudaStream_t st) {
    dim3 grid((ds.n + 255) / 256, nvec);
    k_gather<<<grid, 256, 0, st>>>(ds.n, (size_t)ds.Ne * ds.Nb, ds.cptr, ds.cidx, ds.cw, ce, Cf);
    return 1;
}

int launch_mass_element(const DeviceSpace &ds, double shift, double *Ce, cudaStream_t st) {
    k_mass_element<<<ds.Ne, ds.Nb * ds.Nb, 0, st>>>(ds, shift, Ce);
    return 1;
}

int launch_sum_partials(const DeviceSpace &ds, int nb, int jsplit, const double *Gpart, double *G, cudaStream_t st) {
    const int n5 = 5 * ds.N;
    dim3 grid((n5 + 255) / 256, nb);
    k_sum_partials<<<grid, 256, 0, st>>>(n5, jsplit, Gpart, G);
    return 1;
}

int launch_dfma_probe(int blocks, int threads, int iters, double *out, cudaStream_t st) {
    k_dfma_probe<<<blocks, threads, 0, st>>>(iters, out);
    return 1;
}

}  // namespace landau
