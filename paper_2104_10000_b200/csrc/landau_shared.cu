// Step a3 for a BATCH of problems on one mesh: the Landau tensor of a point pair depends on the geometry
// only, so it is evaluated ONCE per ordered pair and call (k_pair_tensor) and applied to every problem's
// beta sums by a dense fp64 contraction on the tensor cores (k_apply_dmma):
//
//   G_c(i, b) = sum_j U_c(i, j) T_c'(j, b)        PAPER.md Alg. 1 lines 3-12 (L114-121), Eqs. 7-8 (L65-67)
//
//   G_D,rr = U^D_rr t_D     G_D,rz = U^D_rz t_D     G_D,zz = U^D_zz t_D
//   G_K,r  = U^K_rr t_Kr + U^D_rz t_Kz              G_K,z  = U^K_zr t_Kr + U^D_zz t_Kz
//
// (U^K_rz = U^D_rz and U^K_zz = U^D_zz, reading Q1): five N x N matrices, seven products per ordered
// pair and problem -- 14 flop instead of the ~75 of evaluating K(m), E(m) again for every problem.  This is what
// "species loop fused so each pair is visited once" (L103) becomes when the batch dimension is fused as well;
// the paper's batching (L244, L377) keeps one mesh for all problems, which is what makes U shareable.
//
// Layouts (doubles; j = 8 jo + 4 h + k, h in {0,1}, k in 0..3 -- the k index of mma.m8n8k4, two k-groups per
// 16-byte word so that one LDS.128 feeds two DMMAs):
//   U [5][Kq8][Mpad ][4][2]   U[c][jo][i][k][h],  zero for i >= N or j >= N      (Kq8 = Kpad/8, Kpad = 16 ceil(N/16))
//   T [3][Kq8][nbpad][4][2]   T[c][jo][b][k][h] = w_in (T_D, T_Kr, T_Kz)(j) of problem b, zero for j >= N
// so that the (i-tile, 16-point chunk) block a CTA needs is 10 + 6 contiguous segments, fetched by bulk TMA copies.
#include <cuda_runtime.h>

#include <cstdint>

#include "landau_kernels.h"
#include "landau_launch.cuh"
#include "landau_pair_math.cuh"

namespace landau {

int shared_kpad(int N) { return (N + 15) / 16 * 16; }
int shared_mpad(int N) { return (N + 127) / 128 * 128; }
int shared_nbpad(int nb) { return (nb + 63) / 64 * 64; }
// Number of segments the j range is cut into (each summed by its own CTA, partial sums added in segment order).
// A function of N ONLY: it fixes the summation order, so a batched build stays bitwise equal to single builds.
int shared_ksplit(int N) {
    const int chunks = shared_kpad(N) / 16;
    return chunks >= 128 ? 4 : (chunks >= 48 ? 2 : 1);
}

// ------------------------------------------------------------------------------------------------
// U for all ordered pairs.  Thread = one target point i, block = 128 points x 64 source points (8 octets).
// The pair arithmetic is the per-problem kernel's (landau_pair_math.cuh): two pairs in lock-step through the
// AGM, coincident pairs (j = i, or points of different grids at one location, reading Q3) give zero.
// ------------------------------------------------------------------------------------------------
constexpr int PT_THREADS = 128;
constexpr int PT_OCTETS = 8;

__global__ void __launch_bounds__(PT_THREADS)
k_pair_tensor(int N, int Kq8, int Mpad, const double *__restrict__ r, const double *__restrict__ z,
              const double *__restrict__ invr, double *__restrict__ U) {
    __shared__ double sj[5][8 * PT_OCTETS];               // r, z, 2r, 2r^2, 1/(16 r^2) of the source points
    // one octet of results, [c][k][thread] = (h=0, h=1).  Rows padded by two words: the copy-out reads (k, point) =
    // (lane % 4, lane / 4), and with rows of 128 x 16 bytes the four k of a point would share a bank (4-way conflict)
    __shared__ double2 so[5][4][PT_THREADS + 2];
    const int tid = threadIdx.x;
    const int i = blockIdx.x * PT_THREADS + tid;
    const int jbase = blockIdx.y * 8 * PT_OCTETS;
    if (tid < 8 * PT_OCTETS) {
        const int j = jbase + tid;
        if (j < N) {
            const double rj = r[j], irj = invr[j];
            sj[0][tid] = rj; sj[1][tid] = z[j]; sj[2][tid] = 2.0 * rj; sj[3][tid] = 2.0 * rj * rj; sj[4][tid] = 0.0625 * irj * irj;
        } else {          // beyond the last point: a far-away dummy (finite arithmetic), its entries are written as zero
            sj[0][tid] = 1.0; sj[1][tid] = 1.0e6; sj[2][tid] = 2.0; sj[3][tid] = 2.0; sj[4][tid] = 0.0625;
        }
    }
    const int ic = i < N ? i : N - 1;
    JPoint me;                                             // the target point plays the "j" role of pair_parts
    {
        const double ri = r[ic], iri = invr[ic];
        me.r = ri; me.z = z[ic]; me.invr2 = iri * iri; me.rr2 = 2.0 * ri * ri; me.tD = 0.0; me.tKr = 0.0; me.tKz = 0.0;
    }
    __syncthreads();
    const int i0 = blockIdx.x * PT_THREADS;
    for (int oct = 0; oct < PT_OCTETS; ++oct) {
        const int jo = blockIdx.y * PT_OCTETS + oct;
        if (jo >= Kq8) break;                              // uniform over the block
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            IPoint src[2];
            bool live[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int jl = oct * 8 + 4 * h + k;
                src[h].r = sj[0][jl]; src[h].z = sj[1][jl]; src[h].r2x = sj[2][jl]; src[h].rr2 = sj[3][jl]; src[h].c = sj[4][jl];
                src[h].tD = 0.0; src[h].tKr = 0.0; src[h].tKz = 0.0;
                live[h] = jbase + jl < N;
            }
            PairParts pp[2];
            pair_parts<2, true>(src, me, pp);
            double v[5][2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                // tensor of (first = source j, second = target i); the entries of the ordered pair (i, j) are
                // U^D_rr(i,j) = UDrrT, U^D_rz(i,j) = A5, U^D_zz = A3, U^K_rr = A4, U^K_zr(i,j) = -A2
                const PairTensor t = pair_tensor(src[h], me, pp[h]);
                v[0][h] = live[h] ? t.UDrrT : 0.0;
                v[1][h] = live[h] ? t.A5 : 0.0;
                v[2][h] = live[h] ? t.A3 : 0.0;
                v[3][h] = live[h] ? t.A4 : 0.0;
                v[4][h] = live[h] ? -t.A2 : 0.0;
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) so[c][k][tid] = make_double2(v[c][0], v[c][1]);
        }
        __syncthreads();
        // coalesced copy-out: the block's 128 points x 8 doubles of one (c, jo) are contiguous in U
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            double2 *dst = reinterpret_cast<double2 *>(U + ((size_t)(c * Kq8 + jo) * Mpad + i0) * 8);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                const int q = tid + PT_THREADS * w;        // double2 index inside the segment: point q/4, k = q%4
                if (i0 + q / 4 < N) dst[q] = so[c][q & 3][q >> 2];
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// mbarrier / bulk-copy (TMA) helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// ------------------------------------------------------------------------------------------------
// The contraction.  mma.m8n8k4 computes C[m][n] += sum_k A[m][k] B[k][n] with lane (g = lane/4, k = lane%4)
// holding A[g][k], B[k][g] and C[g][2k], C[g][2k+1]: here m = problem b (A = T), n = point i (B = U), k = source
// point j -- so a lane's two accumulator entries are two consecutive points of one problem.
//
// CTA = 8 warps as 2 (problems) x 4 (points); warp tile = 8 TB problems x 8 TI points; CTA tile = 16 TB x 32 TI.
// The j range of split `ks` is walked in chunks of 16 points through a 3-stage ring of shared-memory buffers
// filled by bulk TMA copies (one elected thread, mbarrier completion).
// grid = (ceil(nb / (16 TB)), ceil(N / (32 TI)), ksplit); problem tiles fastest, so CTAs that run together share
// their U tile in L2.  Output: Gpart[b][ks][5][N] (k_sum_partials adds the splits in order; ksplit = 1 writes G).
// ------------------------------------------------------------------------------------------------
constexpr int AP_STAGES = 3;
constexpr int AP_THREADS = 256;

template <int TB, int TI>
constexpr size_t apply_smem_bytes() { return size_t(AP_STAGES) * (10 * 32 * TI + 6 * 16 * TB) * 64 + 64; }

template <int TB, int TI>
__global__ void __launch_bounds__(AP_THREADS, 1)
k_apply_dmma(int N, int nb, int Kq8, int Mpad, int nbpad, int ksplit, const double *__restrict__ U,
             const double *__restrict__ T, double *__restrict__ Gpart) {
    constexpr int BB = 16 * TB, BI = 32 * TI;
    constexpr int U_STAGE = 10 * BI * 8, T_STAGE = 6 * BB * 8;      // doubles
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *sU = reinterpret_cast<double *>(smem_raw);
    double *sT = sU + AP_STAGES * U_STAGE;
    uint64_t *full = reinterpret_cast<uint64_t *>(sT + AP_STAGES * T_STAGE);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, k = lane & 3;
    const int wb = warp & 1, wi = warp >> 1;
    const int b0 = blockIdx.x * BB, i0 = blockIdx.y * BI, ks = blockIdx.z;
    const int nchunks = Kq8 / 2, cps = (nchunks + ksplit - 1) / ksplit;
    const int ch0 = ks * cps, ch1 = min(ch0 + cps, nchunks);
    const int nit = ch1 - ch0;
    if (tid == 0) {
        for (int s = 0; s < AP_STAGES; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pdl_prologue();
    auto issue = [&](int it) {                     // thread 0: fetch chunk ch0 + it into stage it % AP_STAGES
        const int s = it % AP_STAGES, ch = ch0 + it;
        mbar_expect_tx(&full[s], (U_STAGE + T_STAGE) * 8);
#pragma unroll
        for (int c = 0; c < 5; ++c)
#pragma unroll
            for (int jl = 0; jl < 2; ++jl)
                bulk_g2s(sU + s * U_STAGE + (c * 2 + jl) * BI * 8, U + ((size_t)(c * Kq8 + 2 * ch + jl) * Mpad + i0) * 8, BI * 64, &full[s]);
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int jl = 0; jl < 2; ++jl)
                bulk_g2s(sT + s * T_STAGE + (c * 2 + jl) * BB * 8, T + ((size_t)(c * Kq8 + 2 * ch + jl) * nbpad + b0) * 8, BB * 64, &full[s]);
    };
    if (tid == 0)
        for (int it = 0; it < AP_STAGES && it < nit; ++it) issue(it);

    double acc[5][TB][TI][2];
#pragma unroll
    for (int c = 0; c < 5; ++c)
#pragma unroll
        for (int bt = 0; bt < TB; ++bt)
#pragma unroll
            for (int it = 0; it < TI; ++it) acc[c][bt][it][0] = acc[c][bt][it][1] = 0.0;

    for (int it = 0; it < nit; ++it) {
        const int s = it % AP_STAGES;
        mbar_wait(&full[s], (it / AP_STAGES) & 1);
        const double2 *pU = reinterpret_cast<const double2 *>(sU + s * U_STAGE) + (wi * 8 * TI + g) * 4 + k;
        const double2 *pT = reinterpret_cast<const double2 *>(sT + s * T_STAGE) + (wb * 8 * TB + g) * 4 + k;
#pragma unroll
        for (int jl = 0; jl < 2; ++jl) {
            double2 u[5][TI];
#pragma unroll
            for (int c = 0; c < 5; ++c)
#pragma unroll
                for (int ti = 0; ti < TI; ++ti) u[c][ti] = pU[((c * 2 + jl) * BI + ti * 8) * 4];
#pragma unroll
            for (int bt = 0; bt < TB; ++bt) {
                const double2 tD = pT[((0 * 2 + jl) * BB + bt * 8) * 4];
                const double2 tKr = pT[((1 * 2 + jl) * BB + bt * 8) * 4];
                const double2 tKz = pT[((2 * 2 + jl) * BB + bt * 8) * 4];
#pragma unroll
                for (int ti = 0; ti < TI; ++ti) {
                    dmma(acc[0][bt][ti], tD.x, u[0][ti].x);
                    dmma(acc[1][bt][ti], tD.x, u[1][ti].x);
                    dmma(acc[2][bt][ti], tD.x, u[2][ti].x);
                    dmma(acc[3][bt][ti], tKr.x, u[3][ti].x);
                    dmma(acc[4][bt][ti], tKr.x, u[4][ti].x);
                }
#pragma unroll
                for (int ti = 0; ti < TI; ++ti) {
                    dmma(acc[3][bt][ti], tKz.x, u[1][ti].x);
                    dmma(acc[4][bt][ti], tKz.x, u[2][ti].x);
                    dmma(acc[0][bt][ti], tD.y, u[0][ti].y);
                    dmma(acc[1][bt][ti], tD.y, u[1][ti].y);
                    dmma(acc[2][bt][ti], tD.y, u[2][ti].y);
                }
#pragma unroll
                for (int ti = 0; ti < TI; ++ti) {
                    dmma(acc[3][bt][ti], tKr.y, u[3][ti].y);
                    dmma(acc[4][bt][ti], tKr.y, u[4][ti].y);
                }
#pragma unroll
                for (int ti = 0; ti < TI; ++ti) {
                    dmma(acc[3][bt][ti], tKz.y, u[1][ti].y);
                    dmma(acc[4][bt][ti], tKz.y, u[2][ti].y);
                }
            }
        }
        __syncthreads();                            // every warp is done with stage s
        if (tid == 0 && it + AP_STAGES < nit) issue(it + AP_STAGES);
    }
    // epilogue: lane holds (problem b0 + .. + g, points .. + 2k, 2k + 1)
#pragma unroll
    for (int bt = 0; bt < TB; ++bt) {
        const int b = b0 + (wb * TB + bt) * 8 + g;
        if (b >= nb) continue;
        double *Gb = Gpart + ((size_t)b * ksplit + ks) * 5 * N;
#pragma unroll
        for (int ti = 0; ti < TI; ++ti) {
            const int i = i0 + (wi * TI + ti) * 8 + 2 * k;
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                if (i < N) Gb[(size_t)c * N + i] = acc[c][bt][ti][0];
                if (i + 1 < N) Gb[(size_t)c * N + i + 1] = acc[c][bt][ti][1];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
int launch_pair_tensor(int N, const double *r, const double *z, const double *invr, double *U, cudaStream_t st) {
    const int Kq8 = shared_kpad(N) / 8, Mpad = shared_mpad(N);
    dim3 grid((N + PT_THREADS - 1) / PT_THREADS, (Kq8 + PT_OCTETS - 1) / PT_OCTETS);
    launch_k(k_pair_tensor, grid, dim3(PT_THREADS), 0, st, false, N, Kq8, Mpad, r, z, invr, U);
    return 1;
}

template <int TB, int TI>
static void launch_apply_t(int N, int nb, int nbpad, const double *U, const double *T, double *Gpart, cudaStream_t st) {
    static bool configured = false;
    constexpr size_t smem = apply_smem_bytes<TB, TI>();
    if (!configured) {
        note_launch_error(cudaFuncSetAttribute(k_apply_dmma<TB, TI>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)));
        configured = true;
    }
    const int Kq8 = shared_kpad(N) / 8, Mpad = shared_mpad(N), ksplit = shared_ksplit(N);
    dim3 grid((nb + 16 * TB - 1) / (16 * TB), (N + 32 * TI - 1) / (32 * TI), ksplit);
    launch_k(k_apply_dmma<TB, TI>, grid, dim3(AP_THREADS), smem, st, nb <= PDL_MAX_NB, N, nb, Kq8, Mpad, nbpad, ksplit, U, T, Gpart);
}

int launch_apply(int N, int nb, int nbpad, const double *U, const double *T, double *Gpart, cudaStream_t st) {
    // the tile shape is free to follow nb (it does not change any summation order): narrow problem tiles for
    // small batches so that no tensor work is spent on padding columns
    if (nb <= 16) launch_apply_t<1, 2>(N, nb, nbpad, U, T, Gpart, st);
    else if (nb <= 32) launch_apply_t<2, 2>(N, nb, nbpad, U, T, Gpart, st);
    else launch_apply_t<4, 2>(N, nb, nbpad, U, T, Gpart, st);
    return 1;
}

}  // namespace landau
