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
#include "landau_launch.cuh"
#include "landau_pair_math.cuh"

namespace landau {

namespace { thread_local cudaError_t g_launch_err = cudaSuccess; }
void note_launch_error(cudaError_t e) { if (e != cudaSuccess && g_launch_err == cudaSuccess) g_launch_err = e; }
cudaError_t take_launch_error() { const cudaError_t e = g_launch_err; g_launch_err = cudaSuccess; return e; }


// ------------------------------------------------------------------------------------------------
// Symmetric tile-pair kernel.  P0, Pc, Pss are exchange-symmetric and
//   U^D_rr(j,i) = ri^2 Pss + dz^2 P0,  U^D_rz(j,i) = U^K_zr(i,j),  U^D_zz(j,i) = U^D_zz(i,j),
//   U^K_rr(j,i) = U^K_rr(i,j),  U^K_zr(j,i) = U^D_rz(i,j)
// so one elliptic evaluation serves the ordered pairs (i,j) and (j,i) (the paper notes the
// symmetry, L193, and does not exploit it).
//
// Points are cut into tiles of TS; block (I <= J, problem b), TS/IPT threads, thread t owns the IPT
// points i_u = I*TS + u*TS/IPT + t and walks the j of tile J held in shared memory, evaluating its
// IPT pairs (i_u, j) in lock-step.  It keeps the i-side sums in registers; the j-side sums rotate
// around the warp's lanes together with their j (see below) and are parked in shared memory per
// warp, then added over the warps in warp order.  Diagonal blocks (I == J) do all ordered pairs of
// the tile with the coincident-pair test.
//
// Deterministic order: Gpart[b][src tile][5][N] holds, for every target
// point, the partial sum over the points of one source tile; each slot is written by exactly one
// block, and k_sum_partials adds the slabs in tile order.  TS and IPT depend on N only, so a
// batched build is bitwise equal to single builds.
// ------------------------------------------------------------------------------------------------
#ifndef PAIR_MIN_BLOCKS
#define PAIR_MIN_BLOCKS 1
#endif
template <int TS, int IPT, bool CHECK_ALL>
__global__ void __launch_bounds__(TS / IPT, PAIR_MIN_BLOCKS)
k_pair_sym(int N, int ntiles, const double *__restrict__ r, const double *__restrict__ z, const double *__restrict__ invr,
           const double *__restrict__ T, double *__restrict__ Gpart) {
    pdl_prologue();
    constexpr int NT = TS / IPT;         // threads
    constexpr int NW = NT / 32;          // warps
    static_assert(NT % 32 == 0 && NW >= 1, "whole warps");
    __shared__ double sj[7][TS];         // r, z, 1/r^2, 2 r^2, tD, tKr, tKz of the j tile (SoA: conflict-free LDS.64)
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
    IPoint pi[IPT];
    bool valid[IPT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        const int i = I * TS + u * NT + tid;
        valid[u] = i < N;
        const int ic = valid[u] ? i : N - 1;
        const double ri = r[ic], iri = invr[ic];
        pi[u].r = ri; pi[u].z = z[ic]; pi[u].r2x = 2.0 * ri; pi[u].rr2 = 2.0 * ri * ri; pi[u].c = 0.0625 * iri * iri;
        pi[u].tD = valid[u] ? Tb[ic] : 0.0; pi[u].tKr = valid[u] ? Tb[N + ic] : 0.0; pi[u].tKz = valid[u] ? Tb[2 * N + ic] : 0.0;
    }
    const int jbase = J * TS;
    const int cnt = min(TS, N - jbase);
    for (int t = tid; t < TS; t += NT) {
        if (t < cnt) {
            const int j = jbase + t;
            const double rj = r[j], irj = invr[j];
            sj[0][t] = rj; sj[1][t] = z[j]; sj[2][t] = irj * irj; sj[3][t] = 2.0 * rj * rj;
            sj[4][t] = Tb[j]; sj[5][t] = Tb[N + j]; sj[6][t] = Tb[2 * N + j];
        } else {
            // padding of a ragged tile: a far-away point with zero weight (finite tensor, no effect)
            sj[0][t] = 1.0; sj[1][t] = 1.0e6; sj[2][t] = 1.0; sj[3][t] = 2.0;
            sj[4][t] = 0.0; sj[5][t] = 0.0; sj[6][t] = 0.0;
        }
    }
    __syncthreads();
    PairAcc acc[IPT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) acc[u] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (I == J) {
        for (int t = 0; t < cnt; ++t) {
            const JPoint pj = {sj[0][t], sj[1][t], sj[2][t], sj[3][t], sj[4][t], sj[5][t], sj[6][t]};
            PairParts pp[IPT];
            pair_parts<IPT, true>(pi, pj, pp);
#pragma unroll
            for (int u = 0; u < IPT; ++u) accumulate_i(acc[u], pj, pair_tensor(pi[u], pj, pp[u]));
        }
    } else {
        // Lane t walks the 32 j of a sub-tile in rotated order, j = (t + k) mod 32, so that the warp
        // touches 32 different j per step; the j-side sums travel around the lanes with their j
        // (one shuffle per value per step) and need no cross-lane reduction.
        const int nsub = (cnt + 31) >> 5;
        const int src = (lane + 1) & 31;
        for (int sub = 0; sub < nsub; ++sub) {
            double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0, v4 = 0.0;
#pragma unroll 1
            for (int k = 0; k < 32; ++k) {
                const int t = sub * 32 + ((lane + k) & 31);
                const JPoint pj = {sj[0][t], sj[1][t], sj[2][t], sj[3][t], sj[4][t], sj[5][t], sj[6][t]};
                PairParts pp[IPT];
                pair_parts<IPT, CHECK_ALL>(pi, pj, pp);
#pragma unroll
                for (int u = 0; u < IPT; ++u) {
                    const PairTensor tt = pair_tensor(pi[u], pj, pp[u]);
                    accumulate_i(acc[u], pj, tt);
                    // terms of target j from source i_u
                    v0 = fma(pi[u].tD, tt.UDrrT, v0);
                    v1 = fma(pi[u].tD, tt.A5, v1);
                    v2 = fma(pi[u].tD, tt.A3, v2);
                    v3 = fma(tt.A4, pi[u].tKr, fma(tt.A5, pi[u].tKz, v3));
                    v4 = fma(-tt.A2, pi[u].tKr, fma(tt.A3, pi[u].tKz, v4));
                }
                // pass the sums on with their j
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
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        if (valid[u]) {
            const int i = I * TS + u * NT + tid;
            double *G = Gpart + ((size_t)b * ntiles + J) * 5 * N;
            G[i] = acc[u].drr; G[N + i] = acc[u].drz; G[2 * N + i] = acc[u].dzz; G[3 * N + i] = acc[u].kr; G[4 * N + i] = acc[u].kz;
        }
    }
    if (I != J) {
        __syncthreads();
        for (int t = tid; t < cnt; t += NT) {
            double *G = Gpart + ((size_t)b * ntiles + I) * 5 * N + jbase + t;
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                double sum = sacc[0][c][t];
#pragma unroll
                for (int w = 1; w < NW; ++w) sum += sacc[w][c][t];
                G[(size_t)c * N] = sum;
            }
        }
    }
}

// Small N (N < 2560: single builds are latency-bound there, a warp needs ~350 ns per step of its j walk): tiles of
// 32 points, one i per thread, and the 32 steps of a tile pair are SHARED BY WS WARPS -- warp w takes the rotation
// offsets [w 32/WS, (w+1) 32/WS) (diagonal tiles: the j with j mod WS = w).  Every warp then holds partial sums
// for the same 32 targets i and for the j it visited; they are added over the warps in warp order, so the
// summation order is again a function of N alone.  N = 450: 17.5 -> 6 us, N = 2048: 28.7 -> 17 us.
template <int WS, bool CHECK_ALL>
// (compiled for 14 or 16 blocks of two warps per SM -- 72 / 64 registers instead of 80, all 2,080 tile pairs of N = 2,048
// resident at once -- it is slower: 28.3 against 26.7 us; the kernel is bound by its issue slots, not by a partial wave)
__global__ void __launch_bounds__(32 * WS)
k_pair_split(int N, int ntiles, const double *__restrict__ r, const double *__restrict__ z, const double *__restrict__ invr,
             const double *__restrict__ T, double *__restrict__ Gpart) {
    pdl_prologue();
    constexpr int TS = 32, NS = 32 / WS;
    __shared__ double sj[7][TS];
    __shared__ double sacc[WS][2][5][TS];     // [warp][0: targets i, 1: targets j][component][point]
    const int b = blockIdx.y;
    const int p = blockIdx.x;
    int J = int((sqrt(8.0 * double(p) + 1.0) - 1.0) * 0.5);
    while ((J + 1) * (J + 2) / 2 <= p) ++J;
    while (J * (J + 1) / 2 > p) --J;
    const int I = p - J * (J + 1) / 2;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double *Tb = T + (size_t)b * 3 * N;
    const int i = I * TS + lane;
    const bool valid = i < N;
    IPoint pi[1];
    {
        const int ic = valid ? i : N - 1;
        const double ri = r[ic], iri = invr[ic];
        pi[0].r = ri; pi[0].z = z[ic]; pi[0].r2x = 2.0 * ri; pi[0].rr2 = 2.0 * ri * ri; pi[0].c = 0.0625 * iri * iri;
        pi[0].tD = valid ? Tb[ic] : 0.0; pi[0].tKr = valid ? Tb[N + ic] : 0.0; pi[0].tKz = valid ? Tb[2 * N + ic] : 0.0;
    }
    const int jbase = J * TS;
    const int cnt = min(TS, N - jbase);
    if (tid < TS) {
        const int t = tid;
        if (t < cnt) {
            const int j = jbase + t;
            const double rj = r[j], irj = invr[j];
            sj[0][t] = rj; sj[1][t] = z[j]; sj[2][t] = irj * irj; sj[3][t] = 2.0 * rj * rj;
            sj[4][t] = Tb[j]; sj[5][t] = Tb[N + j]; sj[6][t] = Tb[2 * N + j];
        } else {      // padding of a ragged tile: a far-away point with zero weight (finite tensor, no effect)
            sj[0][t] = 1.0; sj[1][t] = 1.0e6; sj[2][t] = 1.0; sj[3][t] = 2.0;
            sj[4][t] = 0.0; sj[5][t] = 0.0; sj[6][t] = 0.0;
        }
    }
    __syncthreads();
    PairAcc acc = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (I == J) {
        for (int t = warp; t < cnt; t += WS) {
            const JPoint pj = {sj[0][t], sj[1][t], sj[2][t], sj[3][t], sj[4][t], sj[5][t], sj[6][t]};
            PairParts pp[1];
            pair_parts<1, true>(pi, pj, pp);
            accumulate_i(acc, pj, pair_tensor(pi[0], pj, pp[0]));
        }
    } else {
        const int src = (lane + 1) & 31, k0 = warp * NS;
        double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0, v4 = 0.0;
#pragma unroll 1
        for (int k = k0; k < k0 + NS; ++k) {
            const int t = (lane + k) & 31;
            const JPoint pj = {sj[0][t], sj[1][t], sj[2][t], sj[3][t], sj[4][t], sj[5][t], sj[6][t]};
            PairParts pp[1];
            pair_parts<1, CHECK_ALL>(pi, pj, pp);
            const PairTensor tt = pair_tensor(pi[0], pj, pp[0]);
            accumulate_i(acc, pj, tt);
            v0 = fma(pi[0].tD, tt.UDrrT, v0);
            v1 = fma(pi[0].tD, tt.A5, v1);
            v2 = fma(pi[0].tD, tt.A3, v2);
            v3 = fma(tt.A4, pi[0].tKr, fma(tt.A5, pi[0].tKz, v3));
            v4 = fma(-tt.A2, pi[0].tKr, fma(tt.A3, pi[0].tKz, v4));
            v0 = __shfl_sync(0xffffffffu, v0, src);
            v1 = __shfl_sync(0xffffffffu, v1, src);
            v2 = __shfl_sync(0xffffffffu, v2, src);
            v3 = __shfl_sync(0xffffffffu, v3, src);
            v4 = __shfl_sync(0xffffffffu, v4, src);
        }
        const int jl = (lane + k0 + NS) & 31;      // the j whose sums this lane holds after NS steps
        sacc[warp][1][0][jl] = v0; sacc[warp][1][1][jl] = v1; sacc[warp][1][2][jl] = v2;
        sacc[warp][1][3][jl] = v3; sacc[warp][1][4][jl] = v4;
    }
    sacc[warp][0][0][lane] = acc.drr; sacc[warp][0][1][lane] = acc.drz; sacc[warp][0][2][lane] = acc.dzz;
    sacc[warp][0][3][lane] = acc.kr; sacc[warp][0][4][lane] = acc.kz;
    __syncthreads();
    // warp 0 adds the partial sums of the targets i, warp 1 (if there is one) those of the targets j
    const int side = WS > 1 ? warp : 0;
    for (int sd = side; sd < 2; sd += WS) {
        if (sd == 1 && I == J) break;
        const int pt = sd == 0 ? i : jbase + lane;
        if (sd == 0 ? valid : lane < cnt) {
            double *G = Gpart + ((size_t)b * ntiles + (sd == 0 ? J : I)) * 5 * N + pt;
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                double sum = sacc[0][sd][c][lane];
#pragma unroll
                for (int w = 1; w < WS; ++w) sum += sacc[w][sd][c][lane];
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
constexpr int FIELD_EPB = 8;      // cells per block
constexpr int FIELD_SG = 2;       // species sharing one read of the tabulations

// TILED: T in the layout of the batch-shared contraction (landau_shared.cu): T[c][jo][b][k][h], j = 8 jo + 4 h + k.
// The kernel is latency-bound (three dependent loads per gathered value, a few hundred flop per cell): small blocks
// with few registers (tabulations transposed in shared memory: conflict-free), every species gathered before the
// one barrier, so that many independent list walks are in flight per SM.
template <bool TILED>
__global__ void __launch_bounds__(16 * FIELD_EPB)
k_fields_beta(DeviceSpace ds, int Kq8, int nbpad, const double *__restrict__ f, double *__restrict__ T, double *__restrict__ uout) {
    pdl_prologue();
    __shared__ double s_tab[3][16][16];                     // [B, E0, E1][a][q]
    // u = P_e f of every species of the block's cells; a cell's row padded by two words: the two cells of a warp read
    // the same (species, node) and would otherwise hit one bank
    __shared__ double s_u[FIELD_EPB][MAX_SPECIES * 16 + 2];
    const int b = blockIdx.y;
    const int q = threadIdx.x;
    const int Nb = ds.Nb, Nq = ds.Nq;
    const double *fb = f + (size_t)b * ds.fstride;
    for (int t = threadIdx.y * Nq + q; t < Nq * Nb; t += Nq * FIELD_EPB) {
        const int qq = t / Nb, a = t % Nb;
        s_tab[0][a][qq] = ds.B[t]; s_tab[1][a][qq] = ds.E0[t]; s_tab[2][a][qq] = ds.E1[t];
    }
    const int e = blockIdx.x * FIELD_EPB + threadIdx.y;
    const bool valid = e < ds.Ne;
    if (valid) {
        // the first item of the node's list (for a node that does not hang: the only one) comes with the bounds
        const int t0 = ds.lptr[e * Nb + q], t1 = ds.lptr[e * Nb + q + 1];
        const double2 hw = *reinterpret_cast<const double2 *>(ds.lhead + e * Nb + q);
        const int d0 = __double2loint(hw.y);
        for (int sp = 0; sp < ds.S; ++sp) {
            double u = fma(hw.x, fb[(size_t)sp * ds.n + d0], 0.0);
            for (int t = t0 + 1; t < t1; ++t) u = fma(ds.lw[t], fb[(size_t)sp * ds.n + ds.ldof[t]], u);
            s_u[threadIdx.y][sp * 16 + q] = u;
            // u = P_e f is needed again by the element kernel (C_e u): kept in the element vector's own slots, which
            // k_element_q3 reads before it overwrites them -- one coalesced load there instead of a second list walk
            uout[(((size_t)b * ds.S + sp) * ds.Ne + e) * Nb + q] = u;
        }
    }
    __syncthreads();
    if (!valid) return;
    const double ijr = ds.invJ[2 * e], ijz = ds.invJ[2 * e + 1];
    double tD = 0.0, tKr = 0.0, tKz = 0.0;
    // the kernel's time is shared-memory bandwidth (three tabulation words per node and species): FIELD_SG species share them
    for (int sp0 = 0; sp0 < ds.S; sp0 += FIELD_SG) {
        double fq[FIELD_SG], g0[FIELD_SG], g1[FIELD_SG];
#pragma unroll
        for (int s = 0; s < FIELD_SG; ++s) { fq[s] = 0.0; g0[s] = 0.0; g1[s] = 0.0; }
#pragma unroll
        for (int a = 0; a < 16; ++a) {
            if (a < Nb) {
                const double tb = s_tab[0][a][q], t0 = s_tab[1][a][q], t1 = s_tab[2][a][q];
#pragma unroll
                for (int s = 0; s < FIELD_SG; ++s) {
                    const double u = s_u[threadIdx.y][min(sp0 + s, ds.S - 1) * 16 + a];
                    fq[s] = fma(tb, u, fq[s]);
                    g0[s] = fma(t0, u, g0[s]);
                    g1[s] = fma(t1, u, g1[s]);
                }
            }
        }
#pragma unroll
        for (int s = 0; s < FIELD_SG; ++s) {
            if (sp0 + s < ds.S) {
                const int sp = sp0 + s;
                const double e2 = ds.e2[sp], em = ds.e2[sp] * ds.m0m[sp];
                tD = fma(e2, fq[s], tD);
                tKr = fma(em, ijr * g0[s], tKr);
                tKz = fma(em, ijz * g1[s], tKz);
            }
        }
    }
    const int gi = e * Nq + q;
    const double w = 12.566370614359172953850573533118 * ds.w_in[gi];    // 4 pi of the tensor (landau_pair_math.cuh) folded in
    if (TILED) {
        const int j = ds.poff + gi;
        const size_t o = (((size_t)(j >> 3) * nbpad + b) * 4 + (j & 3)) * 2 + ((j >> 2) & 1), cs = (size_t)Kq8 * nbpad * 8;
        T[o] = w * tD; T[cs + o] = w * tKr; T[2 * cs + o] = w * tKz;
    } else {
        double *Tb = T + (size_t)b * 3 * ds.Ntot + ds.poff;
        Tb[gi] = w * tD; Tb[ds.Ntot + gi] = w * tKr; Tb[2 * ds.Ntot + gi] = w * tKz;
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
// FULL = true builds the operator of a fully implicit step of Eq. 4 (L52, L75, L280) in the same pass:
//   C_e[a][b] = sum_q w_q [ shift B_qa B_qb + (e_s m0/m_s) E_z B_qa (J^-1 E1)_qb ] - (collision part),
//   ce = (advection - collision part) u     (the shift term is left to the integrator's residual)
// through a third factor Z[q][b] (and ZM for the mass part), Ez[b] read per problem.
// ------------------------------------------------------------------------------------------------
template <bool FULL>
__global__ void k_element(DeviceSpace ds, int jsplit, const double *__restrict__ f, const double *__restrict__ Gpart,
                          double *__restrict__ Ce, double *__restrict__ ce, const double *__restrict__ Ez, double shift) {
    pdl_prologue();
    __shared__ double s_g[16][5];      // w_out * (invJ-transformed G_D rr, rz, zz, G_K r, z), species-independent
    __shared__ double s_w[16];         // w_out (FULL only)
    __shared__ double s_B[256], s_E0[256], s_E1[256], s_X[256], s_Y[256], s_Ce[256], s_u[16];
    __shared__ double s_Z[FULL ? 256 : 1], s_ZM[FULL ? 256 : 1];
    const int e = blockIdx.x, b = blockIdx.y;
    const int Nb = ds.Nb, Nq = ds.Nq, N = ds.Ntot;
    const int tid = threadIdx.x;
    s_B[tid] = ds.B[tid]; s_E0[tid] = ds.E0[tid]; s_E1[tid] = ds.E1[tid];
    if (tid < Nq) {
        const int gi = e * Nq + tid;
        double g[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        for (int js = 0; js < jsplit; ++js) {
            const double *G = Gpart + ((size_t)b * jsplit + js) * 5 * N + ds.poff;
#pragma unroll
            for (int c = 0; c < 5; ++c) g[c] += G[c * N + gi];
        }
        const double ir = ds.invJ[2 * e], iz = ds.invJ[2 * e + 1], w = ds.w_out[gi];
        s_g[tid][0] = ir * ir * w * g[0];
        s_g[tid][1] = ir * iz * w * g[1];
        s_g[tid][2] = iz * iz * w * g[2];
        s_g[tid][3] = ir * w * g[3];
        s_g[tid][4] = iz * w * g[4];
        if (FULL) s_w[tid] = w;
    }
    const double sgn = FULL ? -1.0 : 1.0;
    const double ezb = FULL ? Ez[b] : 0.0, izc = ds.invJ[2 * e + 1];
    const int a = tid / Nb, bb = tid % Nb;   // phase 1: (q, b) = (a, bb); phase 2: (a, b) = (a, bb)
    for (int sp = 0; sp < ds.S; ++sp) {
        __syncthreads();                      // s_g / tabulations ready; previous species done with s_X, s_Y, s_Ce, s_u
        if (tid < Nb) {
            const double *fa = f + (size_t)b * ds.fstride + (size_t)sp * ds.n;
            double u = 0.0;
            for (int t = ds.lptr[e * Nb + tid]; t < ds.lptr[e * Nb + tid + 1]; ++t) u = fma(ds.lw[t], fa[ds.ldof[t]], u);
            s_u[tid] = u;
        }
        {
            const double kf = sgn * ds.kfac[sp], df = sgn * ds.dfac[sp];
            const int q = a;
            const double e0 = s_E0[q * Nb + bb], e1 = s_E1[q * Nb + bb], bq = s_B[q * Nb + bb];
            const double drr = df * s_g[q][0], drz = df * s_g[q][1], dzz = df * s_g[q][2];
            s_X[tid] = fma(drr, e0, fma(drz, e1, kf * s_g[q][3] * bq));
            s_Y[tid] = fma(drz, e0, fma(dzz, e1, kf * s_g[q][4] * bq));
            if (FULL) {
                s_Z[tid] = s_w[q] * (ds.qm[sp] * ezb) * (izc * e1);
                s_ZM[tid] = s_w[q] * shift * bq;
            }
        }
        __syncthreads();
        double acc = 0.0, accM = 0.0;
        for (int q = 0; q < Nq; ++q) {
            acc = fma(s_E0[q * Nb + a], s_X[q * Nb + bb], fma(s_E1[q * Nb + a], s_Y[q * Nb + bb], acc));
            if (FULL) {
                acc = fma(s_B[q * Nb + a], s_Z[q * Nb + bb], acc);
                accM = fma(s_B[q * Nb + a], s_ZM[q * Nb + bb], accM);
            }
        }
        const size_t mat = ((size_t)b * ds.S + sp) * ds.Ne + e;
        Ce[mat * Nb * Nb + tid] = acc + accM;
        s_Ce[tid] = acc;
        __syncthreads();
        if (tid < Nb) {
            double v = 0.0;
            for (int c = 0; c < Nb; ++c) v = fma(s_Ce[tid * Nb + c], s_u[c], v);
            ce[mat * Nb + tid] = v;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a4 + a5 for Q3 (Nb = Nq = 16) on the FP64 tensor cores.  Line 23's contraction
//   C_e[a][b] = sum_q ( E0_qa X_qb + E1_qa Y_qb [+ B_qa Z_qb] )
// is a 16 x 16 x 32 (48, 64 with FULL) matrix product per (cell, species):
// mma.sync.m8n8k4.f64, A = tabulations (row-major, a x q), B = X / Y / Z (col-major, q x b).
// One WARP per (cell, problem), looping over the species.  In the m8n8k4 layouts lane (g = lane/4,
// k = lane%4) holds A[g][k] and B[k][g]: with q = 4 ks + k both are the tabulation entry
// (q, 8 t + g), t = 0, 1 -- so each lane keeps 8 entries of B, E0, E1 in registers for the whole
// kernel, builds its X, Y entries there and nothing but G, f and the outputs touches memory.
// Replaces the shared-memory version (k_element) for Q3: 1.49 -> see DESIGN.md 6.2.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

constexpr int ELQ3_WARPS = 4;    // cells per block and round
#ifndef ELQ3_ROUNDS
#define ELQ3_ROUNDS 4              // cells per warp in a large batch (the next cell's inputs are fetched while this one is multiplied)
#endif
#ifndef ELQ3_MIN_BLOCKS
#define ELQ3_MIN_BLOCKS 4
#endif
// inputs of a cell, staged per warp in shared memory: G (5 x 16), w_out (16), u (S x 16), invJ (2)
constexpr int ELQ3_ROUNDS_MIN_NB = 64;
constexpr int ELQ3_IN_W = 80, ELQ3_IN_U = 96, ELQ3_IN_J = 96 + 16 * MAX_SPECIES, ELQ3_IN = ELQ3_IN_J + 2;

__device__ __forceinline__ void cp_async8(double *dst_shared, const double *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_shared)), "l"(src) : "memory");
}

// One warp per cell, `rounds` cells one after the other (cell e_r = (blockIdx.x rounds + r) ELQ3_WARPS + warp).  The
// kernel is bound by the latency of its loads (a cell is 2 us of them against 0.5 us of tensor work): the inputs of
// cell r + 1 are copied asynchronously into the warp's second buffer while cell r is multiplied and stored.
template <bool FULL>
__global__ void __launch_bounds__(ELQ3_WARPS * 32, FULL ? 3 : ELQ3_MIN_BLOCKS)
k_element_q3(DeviceSpace ds, int rounds, const double *__restrict__ Gsum, double *__restrict__ Ce, double *__restrict__ ce,
             const double *__restrict__ Ez, double shift) {
    pdl_prologue();
    __shared__ double s_in[ELQ3_WARPS][2][ELQ3_IN];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.y;
    const int k = lane & 3, g = lane >> 2;
    const size_t ustep = (size_t)ds.Ne * 16;
    // u = P_e f (hanging-node interpolation folded in) was left by k_fields_beta in the cell's element-vector slots; it
    // is fetched before those slots are overwritten with C_e u below (this warp is the only one that touches them)
    auto prefetch = [&](int e, int buf) {
        double *dst = s_in[warp][buf];
        const double *G = Gsum + (size_t)b * 5 * ds.Ntot + ds.poff + e * 16;
        for (int t = lane; t < 80; t += 32) cp_async8(dst + t, G + (size_t)(t >> 4) * ds.Ntot + (t & 15));
        if (lane < 16) cp_async8(dst + ELQ3_IN_W + lane, ds.w_out + e * 16 + lane);
        else if (lane < 18) cp_async8(dst + ELQ3_IN_J + lane - 16, ds.invJ + 2 * e + lane - 16);
        const double *ub = ce + ((size_t)b * ds.S * ds.Ne + e) * 16;
        for (int t = lane; t < 16 * ds.S; t += 32) cp_async8(dst + ELQ3_IN_U + t, ub + (size_t)(t >> 4) * ustep + (t & 15));
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    const int e_first = blockIdx.x * rounds * ELQ3_WARPS + warp;
    if (e_first >= ds.Ne) return;
    prefetch(e_first, 0);
    // tabulation entries (q = 4 ks + k, col = 8 t + g)
    double tB[4][2], tE0[4][2], tE1[4][2];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks)
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            const int o = (4 * ks + k) * 16 + 8 * t + g;
            tB[ks][t] = ds.B[o]; tE0[ks][t] = ds.E0[o]; tE1[ks][t] = ds.E1[o];
        }
    const double sgn = FULL ? -1.0 : 1.0;
    const double ezb = FULL ? Ez[b] : 0.0;
    for (int round = 0; round < rounds; ++round) {
        const int e = e_first + round * ELQ3_WARPS;
        if (e >= ds.Ne) break;
        const bool more = round + 1 < rounds && e + ELQ3_WARPS < ds.Ne;
        if (more) {
            prefetch(e + ELQ3_WARPS, (round + 1) & 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncwarp();
        const double *in = s_in[warp][round & 1];
        // species-independent coefficients at this lane's four q: w J^-1 G_D J^-T (rr, rz, zz), w J^-1 G_K (r, z)
        // (summing the pair kernel's slabs here instead of in k_sum_partials was measured slower for every batch size)
        const double ir = in[ELQ3_IN_J], iz = in[ELQ3_IN_J + 1];
        // FULL: the mass and E-field advection parts of the operator are, per cell, fixed matrices times a scalar --
        // M_e[a][b] = sum_q w_q B_qa B_qb and A_e[a][b] = sum_q w_q (J^-1)_zz B_qa E1_qb (tabulated at landau_create) -- so
        // they are added to the C fragment (this lane's 2 x 2 x 2 entries) instead of being multiplied out again for every
        // problem and species: half the tensor-core work of the implicit-step operator.
        double2 mF[2][2], aF[2][2];
        if (FULL) {
            const double *Mp = ds.Me + (size_t)e * 256 + 2 * k, *Ap = ds.Ae + (size_t)e * 256 + 2 * k;
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) {
                    mF[mt][nt] = *reinterpret_cast<const double2 *>(Mp + (8 * mt + g) * 16 + 8 * nt);
                    aF[mt][nt] = *reinterpret_cast<const double2 *>(Ap + (8 * mt + g) * 16 + 8 * nt);
                }
        }
        double g0[4], g1[4], g2[4], g3[4], g4[4];
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
            const int q = 4 * ks + k;
            const double w = in[ELQ3_IN_W + q];
            g0[ks] = ir * ir * w * in[q];
            g1[ks] = ir * iz * w * in[16 + q];
            g2[ks] = iz * iz * w * in[32 + q];
            g3[ks] = ir * w * in[48 + q];
            g4[ks] = iz * w * in[64 + q];
        }
        for (int sp = 0; sp < ds.S; ++sp) {
            const double u = in[ELQ3_IN_U + 16 * sp + (lane & 15)];
            const double kf = sgn * ds.kfac[sp], df = sgn * ds.dfac[sp];
            double acc[2][2][2] = {};       // [mt][nt][2]
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
                const double drr = df * g0[ks], drz = df * g1[ks], dzz = df * g2[ks], kr = kf * g3[ks], kz = kf * g4[ks];
                double X[2], Y[2];
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    X[t] = fma(drr, tE0[ks][t], fma(drz, tE1[ks][t], kr * tB[ks][t]));
                    Y[t] = fma(drz, tE0[ks][t], fma(dzz, tE1[ks][t], kz * tB[ks][t]));
                }
#pragma unroll
                for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                    for (int nt = 0; nt < 2; ++nt) {
                        dmma884(acc[mt][nt], tE0[ks][mt], X[nt]);
                        dmma884(acc[mt][nt], tE1[ks][mt], Y[nt]);
                    }
            }
            if (FULL) {     // + (e_s m0 / m_s) E_z x the cell's advection matrix (geometry only: tabulated, see above)
                const double ca = ds.qm[sp] * ezb;
#pragma unroll
                for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                    for (int nt = 0; nt < 2; ++nt) {
                        acc[mt][nt][0] = fma(ca, aF[mt][nt].x, acc[mt][nt][0]);
                        acc[mt][nt][1] = fma(ca, aF[mt][nt].y, acc[mt][nt][1]);
                    }
            }
            // C fragment: lane holds rows a = 8 mt + g, columns b = 8 nt + 2 k + {0, 1}
            const size_t mat = ((size_t)b * ds.S + sp) * ds.Ne + e;
            double *C = Ce + mat * 256;
            double part[2] = {0.0, 0.0};
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                const double u0 = __shfl_sync(0xffffffffu, u, 8 * nt + 2 * k), u1 = __shfl_sync(0xffffffffu, u, 8 * nt + 2 * k + 1);
#pragma unroll
                for (int mt = 0; mt < 2; ++mt) {
                    part[mt] = fma(acc[mt][nt][0], u0, fma(acc[mt][nt][1], u1, part[mt]));
                    double2 v;
                    v.x = FULL ? fma(shift, mF[mt][nt].x, acc[mt][nt][0]) : acc[mt][nt][0];      // the mass part is kept out of
                    v.y = FULL ? fma(shift, mF[mt][nt].y, acc[mt][nt][1]) : acc[mt][nt][1];      // acc: the element vector excludes it
                    *reinterpret_cast<double2 *>(C + (8 * mt + g) * 16 + 8 * nt + 2 * k) = v;
                }
            }
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                part[mt] += __shfl_xor_sync(0xffffffffu, part[mt], 1);
                part[mt] += __shfl_xor_sync(0xffffffffu, part[mt], 2);
                if (k == 0) ce[mat * 16 + 8 * mt + g] = part[mt];
            }
        }
        __syncwarp();       // the buffer is refilled two rounds on
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

// a6 / a7: out[b][sp][k] = sum_{t in [ptr[k], ptr[k+1])} w[t] * src[(b*S+sp)*stride + idx[t]], fixed order
// (owner computes; replaces the paper's atomic MatSetValues, L165-167).  grid = (ceil(K/256), ceil(S/2), nb);
// problem b's outputs start at out + b*ostride.
#ifndef GATHER_EPT
#define GATHER_EPT 2               // outputs per thread (independent list walks in flight)
#endif
#ifndef GATHER_MIN_BLOCKS
#define GATHER_MIN_BLOCKS 8
#endif
__global__ void __launch_bounds__(256, GATHER_MIN_BLOCKS)
k_gather(int K, int S, size_t stride, size_t ostride, const int32_t *__restrict__ ptr, const int32_t *__restrict__ idx,
         const double *__restrict__ w, const GatherHead *__restrict__ head, const double *__restrict__ src, double *__restrict__ out) {
    pdl_prologue();
    // the lists are the same for every species: one walk serves two species blocks (blockIdx.y = species pair)
    const int sp0 = 2 * blockIdx.y;
    const bool two = sp0 + 1 < S;
    const double *s0 = src + ((size_t)blockIdx.z * S + sp0) * stride;
    const double *s1 = s0 + (two ? stride : 0);
    // the first item comes with the list bounds (GatherHead), the others -- cells sharing the entry, hanging-node
    // interpolation -- from the list; same items in the same order as one walk of the list
    int k[GATHER_EPT], t0[GATHER_EPT], t1[GATHER_EPT];
    double2 hw[GATHER_EPT];
    double acc0[GATHER_EPT], acc1[GATHER_EPT];
#pragma unroll
    for (int u = 0; u < GATHER_EPT; ++u) {
        k[u] = (blockIdx.x * GATHER_EPT + u) * 256 + threadIdx.x;
        const int kc = min(k[u], K - 1);
        t0[u] = ptr[kc]; t1[u] = ptr[kc + 1];
        hw[u] = *reinterpret_cast<const double2 *>(head + kc);
    }
#pragma unroll
    for (int u = 0; u < GATHER_EPT; ++u) {
        const int i0 = __double2loint(hw[u].y);
        acc0[u] = s0[i0]; acc1[u] = s1[i0];
    }
#pragma unroll
    for (int u = 0; u < GATHER_EPT; ++u) {
        acc0[u] = fma(hw[u].x, acc0[u], 0.0); acc1[u] = fma(hw[u].x, acc1[u], 0.0);
        for (int t = t0[u] + 1; t < t1[u]; ++t) {
            const double wt = w[t];
            const int it = idx[t];
            acc0[u] = fma(wt, s0[it], acc0[u]);
            acc1[u] = fma(wt, s1[it], acc1[u]);
        }
        if (k[u] < K) {
            double *o = out + (size_t)blockIdx.z * ostride + (size_t)sp0 * K + k[u];
            o[0] = acc0[u];
            if (two) o[K] = acc1[u];
        }
    }
}

// Sums the j-split partials (used by landau_inner_integral when jsplit > 1).  grid over 5N x nb.
__global__ void k_sum_partials(int n5, int jsplit, const double *__restrict__ Gpart, double *__restrict__ G) {
    pdl_prologue();
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n5) return;
    const size_t b = blockIdx.y;
    double acc = 0.0;
    for (int js = 0; js < jsplit; ++js) acc += Gpart[(b * jsplit + js) * n5 + t];
    G[b * n5 + t] = acc;
}

// The same sum for many partials (per-problem path: one slab per source tile, 15 ... 154 of them).  A single build has only
// 5 N outputs: one thread per output walking all slabs leaves most of the GPU idle and pays the slabs' latencies one
// after the other (N = 2,048: 9.4 us, N = 4,928: 19.5 us).  Here 8 warps share 32 outputs: warp g adds the slabs g, g + 8,
// g + 16, ... (four loads in flight), the eight group sums are then added in group order -- a fixed order that depends on
// the number of slabs only, so a batched build stays bitwise equal to single builds.
constexpr int SUMP_GROUPS = 8;
constexpr int SUMP_MIN_SLABS = 8;      // fewer slabs (the shared path's 1 ... 4 j-splits): k_sum_partials
__global__ void __launch_bounds__(32 * SUMP_GROUPS)
k_sum_partials_split(int n5, int jsplit, const double *__restrict__ Gpart, double *__restrict__ G) {
    pdl_prologue();
    __shared__ double sp[SUMP_GROUPS][32];
    const int o = threadIdx.x & 31, sg = threadIdx.x >> 5;
    const int t = blockIdx.x * 32 + o;
    const size_t b = blockIdx.y;
    double acc = 0.0;
    if (t < n5) {
        const double *p = Gpart + b * jsplit * n5 + t;
        int js = sg;
        for (; js + 3 * SUMP_GROUPS < jsplit; js += 4 * SUMP_GROUPS) {
            const double a0 = p[(size_t)js * n5], a1 = p[(size_t)(js + SUMP_GROUPS) * n5];
            const double a2 = p[(size_t)(js + 2 * SUMP_GROUPS) * n5], a3 = p[(size_t)(js + 3 * SUMP_GROUPS) * n5];
            acc += a0; acc += a1; acc += a2; acc += a3;
        }
        for (; js < jsplit; js += SUMP_GROUPS) acc += p[(size_t)js * n5];
    }
    sp[sg][o] = acc;
    __syncthreads();
    if (sg == 0 && t < n5) {
        double sum = sp[0][o];
#pragma unroll
        for (int g = 1; g < SUMP_GROUPS; ++g) sum += sp[g][o];
        G[b * n5 + t] = sum;
    }
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

// FP64 issue-rate probes (measurement aid; the numbers behind the "issue bound" of DESIGN.md 6.1).  Three warps
// per SM sub-partition, 8 independent register-resident chains per thread; clock64() of one block per SM.
//   MODE 0  DFMA, two register operands + an immediate          x = fma(x, y, 1.5)
//   MODE 1  DFMA, two DISTINCT registers (one used twice)       x = fma(y, y, x)
//   MODE 2  DFMA, three distinct registers                      x = fma(y, z, x)
//   MODE 3  DFMA, three registers, one shared by neighbours     x = fma(x, Y, z)   (operand reuse cache)
//   MODE 4  one dependent DFMA chain, one warp per sub-partition (latency)
//   MODE 5  DMMA m8n8k4, 8 independent accumulators per warp
//   MODE 6  as 0, plus ONE independent integer multiply-add per DFMA   (do other pipes issue under FP64 issue?)
//   MODE 7  as 0, plus TWO independent integer multiply-adds per DFMA
template <int MODE>
__global__ void k_issue_probe(int iters, const double *__restrict__ in, double *out, long long *cycles) {
    constexpr int CH = 8;
    double x[CH], y[CH], z[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) { x[c] = in[threadIdx.x + c]; y[c] = in[threadIdx.x + 32 + c]; z[c] = in[threadIdx.x + 64 + c]; }
    double Y = in[threadIdx.x + 100];
    int n[2 * CH];
#pragma unroll
    for (int c = 0; c < 2 * CH; ++c) n[c] = threadIdx.x + c + iters;
    __syncthreads();
    const long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
        if (MODE == 4) {
#pragma unroll
            for (int c = 0; c < CH; ++c) x[0] = fma(x[0], y[0], 1.5);
        } else if (MODE == 5) {
#pragma unroll
            for (int c = 0; c < CH; c += 2)
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                             : "+d"(x[c]), "+d"(x[c + 1]) : "d"(y[c]), "d"(z[c]));
        } else {
#pragma unroll
            for (int c = 0; c < CH; ++c) {
                if (MODE == 0 || MODE >= 6) x[c] = fma(x[c], y[c], 1.5);
                if (MODE >= 6) n[c] = n[c] * 3 + 7;
                if (MODE == 7) n[CH + c] = n[CH + c] * 5 + 3;
                if (MODE == 1) x[c] = fma(y[c], y[c], x[c]);
                if (MODE == 2) x[c] = fma(y[c], z[c], x[c]);
                if (MODE == 3) x[c] = fma(x[c], Y, z[c]);
            }
            if (MODE == 3) Y += 1e-30;
        }
    }
    const long long t1 = clock64();
    __syncthreads();
    double sum = 0.0;
#pragma unroll
    for (int c = 0; c < CH; ++c) sum += x[c] + y[c] + z[c] + double(n[c] ^ n[CH + c]);
    if (sum == 12345.678) out[0] = sum;     // keep the chains alive
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
// Tile size of the pair kernel: a function of N and of the context's tiling policy ONLY (it fixes the summation
// order; the policy is fixed at landau_create, so inside a context a batched build equals single builds bitwise).
// Small N is latency-bound (one warp walks its j tile step by step, ~700 cycles per step): short tiles give
// more warps and fewer steps (N = 2048: 39 -> 31 us); large N is throughput-bound: two i per thread.
// latency = true (contexts created for fewer than LANDAU_SHARED_MIN_BATCH problems: single builds): 32-point tiles up to
// N = 8,192 -- a single build of N = 4,928 is 780 blocks of 128-point tile pairs on 888 slots, under one wave with a
// 5 : 6 imbalance between SMs; 11,935 short blocks balance (pair kernel 115 -> 101 us).
int pair_tile_size(int N, bool latency) {
    if (latency) return N >= 16384 ? 128 : (N >= 8192 ? 64 : 32);
    return N >= 4096 ? 128 : (N >= 2560 ? 64 : 32);
}
int pair_tiles(int N, bool latency) { const int ts = pair_tile_size(N, latency); return (N + ts - 1) / ts; }
// Warps sharing a tile pair where the tiles are 32 points (k_pair_split): a function of N and the policy, like the tile size.
int pair_split_warps(int N, bool latency) { return N < (latency ? 2048 : 1536) ? 4 : 2; }

int launch_fields_beta(const DeviceSpace &ds, int nb, const double *f, double *T, double *u, cudaStream_t st) {
    dim3 grid((ds.Ne + FIELD_EPB - 1) / FIELD_EPB, nb), block(ds.Nq, FIELD_EPB);
    launch_k(k_fields_beta<false>, grid, block, 0, st, nb <= PDL_MAX_NB, ds, 0, 0, f, T, u);
    return 1;
}

int launch_fields_beta_tiled(const DeviceSpace &ds, int nb, int nbpad, const double *f, double *T, double *u, cudaStream_t st) {
    dim3 grid((ds.Ne + FIELD_EPB - 1) / FIELD_EPB, nb), block(ds.Nq, FIELD_EPB);
    launch_k(k_fields_beta<true>, grid, block, 0, st, nb <= PDL_MAX_NB, ds, shared_kpad(ds.Ntot) / 8, nbpad, f, T, u);
    return 1;
}

template <bool CHECK_ALL>
static void launch_pair_t(int N, bool latency, const double *r, const double *z, const double *invr, int nb, const double *T, double *Gpart,
                          cudaStream_t st) {
    const int ts = pair_tile_size(N, latency), nt = pair_tiles(N, latency);
    dim3 grid(nt * (nt + 1) / 2, nb);
    const bool pdl = nb <= PDL_MAX_NB;
    if (ts == 128) launch_k(k_pair_sym<128, 2, CHECK_ALL>, grid, dim3(64), 0, st, pdl, N, nt, r, z, invr, T, Gpart);
    else if (ts == 64) launch_k(k_pair_sym<64, 2, CHECK_ALL>, grid, dim3(32), 0, st, pdl, N, nt, r, z, invr, T, Gpart);
    else if (pair_split_warps(N, latency) == 4) launch_k(k_pair_split<4, CHECK_ALL>, grid, dim3(128), 0, st, pdl, N, nt, r, z, invr, T, Gpart);
    else launch_k(k_pair_split<2, CHECK_ALL>, grid, dim3(64), 0, st, pdl, N, nt, r, z, invr, T, Gpart);
}

int launch_pair(int Ntot, bool latency, const double *r, const double *z, const double *invr, bool check_all, int nb, const double *T,
                double *Gpart, cudaStream_t st) {
    if (check_all) launch_pair_t<true>(Ntot, latency, r, z, invr, nb, T, Gpart, st);
    else launch_pair_t<false>(Ntot, latency, r, z, invr, nb, T, Gpart, st);
    return 1;
}

int launch_element(const DeviceSpace &ds, int nb, int jsplit, const double *f, const double *G, double *Ce, double *ce,
                   const double *Ez, double shift, cudaStream_t st) {
    if (ds.Nb == 16 && jsplit == 1) {   // Q3: FP64 tensor cores, warp per cell
        // several cells per warp pay in a batch (prefetch); a small batch needs every warp it can get
        const int rounds = nb >= ELQ3_ROUNDS_MIN_NB ? ELQ3_ROUNDS : 1;
        dim3 grid((ds.Ne + ELQ3_WARPS * rounds - 1) / (ELQ3_WARPS * rounds), nb);
        if (Ez) launch_k(k_element_q3<true>, grid, dim3(ELQ3_WARPS * 32), 0, st, nb <= PDL_MAX_NB, ds, rounds, G, Ce, ce, Ez, shift);
        else launch_k(k_element_q3<false>, grid, dim3(ELQ3_WARPS * 32), 0, st, nb <= PDL_MAX_NB, ds, rounds, G, Ce, ce, (const double *)nullptr, 0.0);
        return 1;
    }
    dim3 grid(ds.Ne, nb);
    if (Ez) launch_k(k_element<true>, grid, dim3(ds.Nb * ds.Nb), 0, st, nb <= PDL_MAX_NB, ds, jsplit, f, G, Ce, ce, Ez, shift);
    else launch_k(k_element<false>, grid, dim3(ds.Nb * ds.Nb), 0, st, nb <= PDL_MAX_NB, ds, jsplit, f, G, Ce, ce, (const double *)nullptr, 0.0);
    return 1;
}

// both gathers of a build in one launch: blocks [0, bv) of grid.x do the CSR values, the rest C(f)
__global__ void k_gather2(DeviceSpace ds, int bv, size_t vstride, size_t fstride, const double *__restrict__ Ce,
                          const double *__restrict__ ce, double *__restrict__ vals, double *__restrict__ Cf) {
    pdl_prologue();
    const bool isv = (int)blockIdx.x < bv;
    const int K = isv ? ds.nnz : ds.n;
    const int kk = (isv ? blockIdx.x : blockIdx.x - bv) * blockDim.x + threadIdx.x;
    if (kk >= K) return;
    const int32_t *ptr = isv ? ds.gptr : ds.cptr, *idx = isv ? ds.gidx : ds.cidx;
    const double *w = isv ? ds.gw : ds.cw;
    const size_t stride = isv ? (size_t)ds.Ne * ds.Nb * ds.Nb : (size_t)ds.Ne * ds.Nb;
    const double *s = (isv ? Ce : ce) + ((size_t)blockIdx.z * gridDim.y + blockIdx.y) * stride;
    const GatherHead *head = isv ? ds.ghead : ds.chead;
    const int t0 = ptr[kk], t1 = ptr[kk + 1];
    const double2 hw = *reinterpret_cast<const double2 *>(head + kk);
    double acc = fma(hw.x, s[__double2loint(hw.y)], 0.0);
    // entries shared by several cells or fed by hanging nodes have long lists: four items in flight, added in list order
    int t = t0 + 1;
    for (; t + 3 < t1; t += 4) {
        const int i0 = idx[t], i1 = idx[t + 1], i2 = idx[t + 2], i3 = idx[t + 3];
        const double w0 = w[t], w1 = w[t + 1], w2 = w[t + 2], w3 = w[t + 3];
        const double v0 = s[i0], v1 = s[i1], v2 = s[i2], v3 = s[i3];
        acc = fma(w0, v0, acc); acc = fma(w1, v1, acc); acc = fma(w2, v2, acc); acc = fma(w3, v3, acc);
    }
    for (; t < t1; ++t) acc = fma(w[t], s[idx[t]], acc);
    (isv ? vals : Cf)[(size_t)blockIdx.z * (isv ? vstride : fstride) + (size_t)blockIdx.y * K + kk] = acc;
}

int launch_gather_both(const DeviceSpace &ds, int nb, size_t vstride, size_t fstride, const double *Ce, const double *ce,
                       double *vals, double *Cf, cudaStream_t st) {
    const int bv = (ds.nnz + 255) / 256, bc = (ds.n + 255) / 256;
    dim3 grid(bv + bc, ds.S, nb);
    launch_k(k_gather2, grid, dim3(256), 0, st, nb <= PDL_MAX_NB, ds, bv, vstride, fstride, Ce, ce, vals, Cf);
    return 1;
}

int launch_gather_vals(const DeviceSpace &ds, int nb, int nspecies, size_t ostride, const double *Ce, double *vals, cudaStream_t st) {
    dim3 grid((ds.nnz + 256 * GATHER_EPT - 1) / (256 * GATHER_EPT), (nspecies + 1) / 2, nb);
    launch_k(k_gather, grid, dim3(256), 0, st, false, ds.nnz, nspecies, (size_t)ds.Ne * ds.Nb * ds.Nb, ostride, ds.gptr, ds.gidx, ds.gw, ds.ghead, Ce, vals);
    return 1;
}

int launch_gather_cf(const DeviceSpace &ds, int nb, size_t ostride, const double *ce, double *Cf, cudaStream_t st) {
    dim3 grid((ds.n + 256 * GATHER_EPT - 1) / (256 * GATHER_EPT), (ds.S + 1) / 2, nb);
    launch_k(k_gather, grid, dim3(256), 0, st, false, ds.n, ds.S, (size_t)ds.Ne * ds.Nb, ostride, ds.cptr, ds.cidx, ds.cw, ds.chead, ce, Cf);
    return 1;
}

int launch_mass_element(const DeviceSpace &ds, double shift, double *Ce, cudaStream_t st) {
    launch_k(k_mass_element, dim3(ds.Ne), dim3(ds.Nb * ds.Nb), 0, st, false, ds, shift, Ce);
    return 1;
}

int launch_sum_partials(int Ntot, int nb, int jsplit, bool latency, const double *Gpart, double *G, cudaStream_t st) {
    const int n5 = 5 * Ntot;
    // chosen by the ctx's tiling policy (contexts made for single builds) and the number of slabs, never by nb: in a large
    // batch the plain kernel is DRAM-bound already and the split one a few per cent slower (8,192 x N = 450: 9.04 -> 9.55 ms)
    if (latency && jsplit >= SUMP_MIN_SLABS) {
        dim3 grid((n5 + 31) / 32, nb);
        launch_k(k_sum_partials_split, grid, dim3(32 * SUMP_GROUPS), 0, st, nb <= PDL_MAX_NB, n5, jsplit, Gpart, G);
        return 1;
    }
    dim3 grid((n5 + 255) / 256, nb);
    launch_k(k_sum_partials, grid, dim3(256), 0, st, nb <= PDL_MAX_NB, n5, jsplit, Gpart, G);
    return 1;
}

// returns the warp instructions each warp issues per iteration of the probe loop (0: unknown mode)
int launch_issue_probe(int mode, int blocks, int threads, int iters, const double *in, double *out, long long *cycles, cudaStream_t st) {
    switch (mode) {
        case 0: launch_k(k_issue_probe<0>, dim3(blocks), dim3(threads), 0, st, false, iters, in, out, cycles); return 8;
        case 1: launch_k(k_issue_probe<1>, dim3(blocks), dim3(threads), 0, st, false, iters, in, out, cycles); return 8;
        case 2: launch_k(k_issue_probe<2>, dim3(blocks), dim3(threads), 0, st, false, iters, in, out, cycles); return 8;
        case 3: launch_k(k_issue_probe<3>, dim3(blocks), dim3(threads), 0, st, false, iters, in, out, cycles); return 8;
        case 4: launch_k(k_issue_probe<4>, dim3(blocks), dim3(threads), 0, st, false, iters, in, out, cycles); return 8;
        case 5: launch_k(k_issue_probe<5>, dim3(blocks), dim3(threads), 0, st, false, iters, in, out, cycles); return 4;
        case 6: launch_k(k_issue_probe<6>, dim3(blocks), dim3(threads), 0, st, false, iters, in, out, cycles); return 8;
        case 7: launch_k(k_issue_probe<7>, dim3(blocks), dim3(threads), 0, st, false, iters, in, out, cycles); return 8;
        default: return 0;
    }
}

int launch_dfma_probe(int blocks, int threads, int iters, double *out, cudaStream_t st) {
    launch_k(k_dfma_probe, dim3(blocks), dim3(threads), 0, st, false, iters, out);
    return 1;
}

}  // namespace landau
