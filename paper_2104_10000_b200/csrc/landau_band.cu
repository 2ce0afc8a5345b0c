// Per-species batched band LU (section III-G): reverse
// Cuthill-McKee ordering on the host (once per mesh), then on the device, per (problem, species)
// matrix: scatter of the CSR values into band storage, Gaussian elimination WITHOUT pivoting in
// outer-product form (Golub & Van Loan Alg. 4.3.1, the paper's choice) -- blocked: KB columns at a
// time, the B x B outer-product update becomes a rank-KB update of the trailing window from
// shared-memory panels -- and the two banded triangular solves.  One thread block per matrix
// (the matrices of a batch are independent: L171, L244).
//
// Band storage of one matrix (order n, half-bandwidth bw after RCM, W = bw + KB so that the
// rectangular panels of a block step stay inside the stored band): LAPACK's layout, element (i,j) at
// band[(W + i - j) + j*LD], LD = 2W + 1, which is the ordinary column-major matrix
// A(i,j) = band[W + i + j*(LD-1)] with leading dimension LD-1.  Entries outside the true band are
// zero and stay zero (no pivoting => no fill outside the band).
#include <cuda_runtime.h>

#include <mutex>

#include <algorithm>
#include <functional>
#include <cmath>
#include <cstdint>
#include <queue>
#include <vector>

#include "landau_kernels.h"

namespace landau {

// ------------------------------------------------------------------------------------------------
// host: reverse Cuthill-McKee on the (structurally symmetric) pattern A1
// ------------------------------------------------------------------------------------------------
namespace {
// BFS level structure from root inside the component; returns the eccentricity, fills order (BFS order)
int bfs_levels(int root, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, std::vector<int> &level,
               std::vector<int> &order) {
    order.clear();
    order.push_back(root);
    level[root] = 0;
    int ecc = 0;
    for (size_t h = 0; h < order.size(); ++h) {
        const int v = order[h];
        for (int t = rowptr[v]; t < rowptr[v + 1]; ++t) {
            const int u = colidx[t];
            if (level[u] < 0) { level[u] = level[v] + 1; ecc = std::max(ecc, level[u]); order.push_back(u); }
        }
    }
    return ecc;
}
}  // namespace

namespace {
// Reverse Cuthill-McKee.  forced_root >= 0: its component is numbered first, starting there; every other component
// starts at a pseudo-peripheral node (George & Liu).  perm[new] = old.
void rcm_from(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, int forced_root, std::vector<int32_t> &perm) {
    std::vector<int> deg(n), level(n, -1), order, visited(n, 0);
    for (int i = 0; i < n; ++i) deg[i] = rowptr[i + 1] - rowptr[i];
    perm.clear();
    std::vector<int> cm;
    for (int pass = forced_root >= 0 ? -1 : 0; pass < n; ++pass) {
        const int seed = pass < 0 ? forced_root : pass;
        if (visited[seed]) continue;
        int root = seed;
        if (pass >= 0) {
            // pseudo-peripheral node of this component: repeat BFS from a minimum-degree node of the last level
            std::fill(level.begin(), level.end(), -1);
            int ecc = bfs_levels(root, rowptr, colidx, level, order);
            for (int it = 0; it < 8; ++it) {
                int cand = -1;
                for (int v : order)
                    if (level[v] == ecc && (cand < 0 || deg[v] < deg[cand])) cand = v;
                for (int v : order) level[v] = -1;
                std::vector<int> order2;
                const int ecc2 = bfs_levels(cand, rowptr, colidx, level, order2);
                if (ecc2 > ecc) { root = cand; ecc = ecc2; order.swap(order2); }
                else { for (int v : order2) level[v] = -1; bfs_levels(root, rowptr, colidx, level, order); break; }
            }
        }
        // Cuthill-McKee: BFS from root, neighbours in order of increasing degree
        std::vector<int> q;
        q.push_back(root);
        visited[root] = 1;
        for (size_t h = 0; h < q.size(); ++h) {
            const int v = q[h];
            std::vector<int> nb;
            for (int t = rowptr[v]; t < rowptr[v + 1]; ++t)
                if (!visited[colidx[t]]) { visited[colidx[t]] = 1; nb.push_back(colidx[t]); }
            std::sort(nb.begin(), nb.end(), [&](int a, int b) { return deg[a] != deg[b] ? deg[a] < deg[b] : a < b; });
            q.insert(q.end(), nb.begin(), nb.end());
        }
        cm.insert(cm.end(), q.begin(), q.end());
    }
    perm.assign(cm.rbegin(), cm.rend());   // reverse
}
}  // namespace

// Half-bandwidth of an order and, per block step of KB = band_block(bw) columns, the rows below / columns right of the
// block that elimination without pivoting can reach (mlow) and the rows above it (mup): no fill is created left of
// a row's first entry / above a column's first entry, so the reach is the monotone hull of the envelope.
// Returns the window-update work of one factorisation, 2 KB sum mlow^2 flop.
double band_envelope(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const std::vector<int32_t> &perm,
                     int &bw, std::vector<int32_t> *mlow_out, std::vector<int32_t> *mup_out, int KB_in) {
    std::vector<int32_t> pos(n), first(n), last_with_first(n + 1, 0);
    for (int i = 0; i < n; ++i) { pos[perm[i]] = i; first[i] = i; }
    bw = 0;
    for (int i = 0; i < n; ++i)
        for (int t = rowptr[i]; t < rowptr[i + 1]; ++t) {
            const int pi = pos[i], pj = pos[colidx[t]];
            bw = std::max(bw, std::abs(pi - pj));
            first[pi] = std::min<int32_t>(first[pi], pj);              // structurally symmetric: rows = columns
        }
    for (int i = 0; i < n; ++i) last_with_first[first[i]] = std::max<int32_t>(last_with_first[first[i]], i);
    for (int j = 1; j < n; ++j) last_with_first[j] = std::max(last_with_first[j], last_with_first[j - 1]);
    const int KB = KB_in > 0 ? KB_in : band_block(bw), nsteps = (n + KB - 1) / KB;
    if (mlow_out) mlow_out->assign(nsteps, 0);
    if (mup_out) mup_out->assign(nsteps, 0);
    double work = 0.0;
    for (int st = 0; st < nsteps; ++st) {
        const int k0 = st * KB, ke = std::min(k0 + KB, n) - 1;
        const int m = std::max(0, last_with_first[ke] - ke);
        int fmin = k0;
        for (int j = k0; j <= ke; ++j) fmin = std::min(fmin, int(first[j]));
        if (mlow_out) (*mlow_out)[st] = m;
        if (mup_out) (*mup_out)[st] = k0 - fmin;
        work += 2.0 * (ke - k0 + 1) * double(m) * double(m);
    }
    return work;
}

// The order of the band LU (section III-G: reverse Cuthill-McKee).  RCM's result depends on its starting
// node, and on the high-order elements of this discretisation (every cell a clique of 16 or 9 unknowns) a
// pseudo-peripheral start is often not the best one; the cost of the factorisation is the envelope work above, which
// is cheap to evaluate.  So several candidates are tried (selection rule at the end of the function):
//   RCM from a pseudo-peripheral node, from the unknowns at the four corners of the domain, from the one nearest the
//   origin (where the refinement sits) and from up to ~100 unknowns spread along the boundary, and the plain sweep
//   (z, then r) -- the optimum on uniform meshes, where the BFS levels of RCM are L-shaped rings of cells and twice
//   as long as a row of the mesh.
// dof_r / dof_z may be null (only the pseudo-peripheral RCM is then tried).  perm[new] = old.
void rcm_order(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const double *dof_r, const double *dof_z,
               std::vector<int32_t> &perm, int &bw) {
    std::vector<int> roots = {-1};
    std::vector<int32_t> sweep;
    if (dof_r && dof_z && n > 0) {
        double rmin = dof_r[0], rmax = dof_r[0], zmin = dof_z[0], zmax = dof_z[0];
        for (int i = 1; i < n; ++i) {
            rmin = std::min(rmin, dof_r[i]); rmax = std::max(rmax, dof_r[i]);
            zmin = std::min(zmin, dof_z[i]); zmax = std::max(zmax, dof_z[i]);
        }
        const double tr[5] = {rmin, rmax, rmin, rmax, 0.0}, tz[5] = {zmin, zmin, zmax, zmax, 0.0};
        for (int c = 0; c < 5; ++c) {
            int best = 0;
            double bd = 1e300;
            for (int i = 0; i < n; ++i) {
                const double d = (dof_r[i] - tr[c]) * (dof_r[i] - tr[c]) + (dof_z[i] - tz[c]) * (dof_z[i] - tz[c]);
                if (d < bd) { bd = d; best = i; }
            }
            if (std::find(roots.begin(), roots.end(), best) == roots.end()) roots.push_back(best);
        }
        // ... and from unknowns spread evenly along the boundary of the domain (on the refined meshes the best start is
        // often an axis node near the refined region), as many as a budget of ~3e5 node visits allows
        {
            const double tol = 1e-12 * std::max(rmax - rmin, zmax - zmin), rc = 0.5 * (rmin + rmax), zc = 0.5 * (zmin + zmax);
            std::vector<int> bnd;
            for (int i = 0; i < n; ++i)
                if (dof_r[i] - rmin <= tol || rmax - dof_r[i] <= tol || dof_z[i] - zmin <= tol || zmax - dof_z[i] <= tol) bnd.push_back(i);
            std::sort(bnd.begin(), bnd.end(), [&](int a, int b) {
                const double ta = std::atan2(dof_z[a] - zc, dof_r[a] - rc), tb = std::atan2(dof_z[b] - zc, dof_r[b] - rc);
                return ta != tb ? ta < tb : a < b;
            });
            const int want = std::min<int>(int(bnd.size()), std::max(0, 300000 / n - int(roots.size())));
            for (int c = 0; c < want; ++c) {
                const int v = bnd[size_t(c) * bnd.size() / want];
                if (std::find(roots.begin(), roots.end(), v) == roots.end()) roots.push_back(v);
            }
        }
        sweep.resize(n);
        for (int i = 0; i < n; ++i) sweep[i] = i;
        std::stable_sort(sweep.begin(), sweep.end(), [&](int a, int b) { return dof_z[a] != dof_z[b] ? dof_z[a] < dof_z[b] : dof_r[a] < dof_r[b]; });
    }
    // The half-bandwidth fixes the storage, the shared-memory panels (blocks per SM) and the kernel configuration;
    // the envelope work is what the window updates cost.  So: among the candidates within 10 % of the narrowest
    // band, the one with the least work (measured on B200: always the fastest of the set).
    struct Cand { std::vector<int32_t> perm; int bw; double work; };
    std::vector<Cand> cands;
    for (size_t c = 0; c < roots.size() + (sweep.empty() ? 0 : 1); ++c) {
        Cand k;
        if (c < roots.size()) rcm_from(n, rowptr, colidx, roots[c], k.perm);
        else k.perm = sweep;
        k.work = band_envelope(n, rowptr, colidx, k.perm, k.bw, nullptr, nullptr);
        cands.push_back(std::move(k));
    }
    int bw_min = cands[0].bw;
    for (const Cand &k : cands) bw_min = std::min(bw_min, k.bw);
    const int bw_ok = bw_min + std::max(8, bw_min / 10);
    const Cand *best = nullptr;
    for (const Cand &k : cands)
        if (k.bw <= bw_ok && (!best || k.work < best->work || (k.work == best->work && k.bw < best->bw))) best = &k;
    perm = best->perm;
    bw = best->bw;
}

// stored half-width: bw + KB rounded up to even (16-byte aligned column pairs in the window update)
// (at least 2 KB - 1: the front kernel always lists the rows of the NEXT block, up to 2 KB - 1 below a block's first column)
__host__ __device__ inline int band_halfwidth(int bw, int KB) { return ((bw > KB - 1 ? bw : KB - 1) + KB + 1) & ~1; }
int band_stored_halfwidth(int bw) { return band_halfwidth(bw, band_block(bw)); }

// Block width and threads per matrix, by half-bandwidth (measured, 512 problems):
//   bw = 178 (n = 745, 5,120 matrices):  KB 16 x 128 threads 17.5 ms | 16 x 256: 23.2 | 32 x 256: 29.4 | 32 x 512: 34.0
//   bw = 339 (n = 2,767, 1,024 matrices): KB 32 x 256 threads 35.5 ms | 32 x 512: 36.5 | 32 x 128: 51.7 | 16 x 128: 56.1
// small matrices want several blocks per SM (their steps are dominated by latencies), wide ones the longer panels.
int band_block(int bw) { return bw <= 256 ? 16 : (bw <= 384 ? 32 : (bw <= 832 ? 16 : 8)); }   // panels must fit 227 KB of shared memory

// ------------------------------------------------------------------------------------------------
// device
// ------------------------------------------------------------------------------------------------
// Band fill: zero fill and scatter of the CSR values in one pass, one warp per band column.  Only the rows of a column
// that the factorisation and the solves can touch are written (the union of the block steps' squares, DESIGN.md 6.4:
// about three quarters of the stored band); the rest of the workspace is never read and stays as the caller left it.
// grid = (ceil(n / FILL_WARPS), S_g, nb); matrix (problem b, species s of this grid) starts at band + b pstride + s mat_doubles
constexpr int FILL_WARPS = 8;
__global__ void __launch_bounds__(32 * FILL_WARPS)
k_band_fill(int n, int nnz, size_t LD, size_t vstride, size_t mat_doubles, size_t pstride, const int32_t *__restrict__ zlo,
            const int32_t *__restrict__ zcnt, const int32_t *__restrict__ fptr, const int32_t *__restrict__ fsrc,
            const int32_t *__restrict__ foff, const double *__restrict__ vals, double *__restrict__ band) {
    const int lane = threadIdx.x & 31, pj = blockIdx.x * FILL_WARPS + (threadIdx.x >> 5);
    if (pj >= n) return;
    double *col = band + (size_t)blockIdx.z * pstride + (size_t)blockIdx.y * mat_doubles + (size_t)pj * LD;
    const int z0 = zlo[pj], zc = zcnt[pj];
    for (int r = lane; r < zc; r += 32) col[z0 + r] = 0.0;
    __syncwarp();                                  // orders the zeros before the values of this column (same warp)
    const double *v = vals + (size_t)blockIdx.z * vstride + (size_t)blockIdx.y * nnz;
    for (int t = fptr[pj] + lane; t < fptr[pj + 1]; t += 32) col[foff[t]] = v[fsrc[t]];
}

constexpr int BAND_THREADS = 512;
#ifndef BAND16_MIN_BLOCKS
#define BAND16_MIN_BLOCKS 3        // narrow-band instantiation (16 columns x 128 threads): three blocks per SM (168 registers); compiled
                                   // for four (128 registers) it was measured slower (ten-species 80-cell: 14.5 against 14.3 ms)
#endif
// threads per matrix in the solves (measured: bw = 339: 384 threads 4.2 ms, 256: 4.8, 512: 5.8; bw = 178: 64 threads 2.5 ms,
// 256: 3.9, 512: 7.6 -- the solves are latency-bound, small blocks leave room for more matrices per SM)
// (after the solves were confined to the envelope and compiled for seven blocks per SM, bw = 278: 288 threads 2.45 ms,
// 256: 2.47, 224: 2.69, 192: 2.91)
constexpr int SOLVE_NT32 = 288, SOLVE_NT16 = 64;
constexpr int WT = 32, WTJ = 16;   // warp tile of the window update: 32 rows x 16 columns = 4 x 2 mma tiles of 8 x 8

// 1/x: MUFU seed and two Newton steps (full double precision up to rounding of the last step)
__device__ __forceinline__ double rcp_newton(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, fma(e, e, e), y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

// KB x KB diagonal block at k0: loaded into shared memory, eliminated without pivoting by ONE warp (lane = row;
// every offset is a compile-time constant, so the loads of a column step are issued together), L\U written
// back, 1/pivots left in sDi.  A short last block is completed by the identity (no kb guards later).
template <int KB>
__device__ __forceinline__ void factor_diag_block(double *A, size_t lda, int k0, int kb, double *sD, double *sDi, int lane,
                                                  double &pmin, double &pmax) {
    double *myrow = sD + min(lane, KB - 1) * (KB + 1);
    const bool rowlane = lane < KB;        // KB < 32: the upper lanes only follow the warp barriers
    if (rowlane) {
#pragma unroll
        for (int c = 0; c < KB; ++c)
            myrow[c] = (lane < kb && c < kb) ? __ldcg(A + (k0 + lane) + (size_t)(k0 + c) * lda) : (lane == c ? 1.0 : 0.0);
    }
    __syncwarp();
#pragma unroll
    for (int c = 0; c < KB; ++c) {
        const double *prow = sD + c * (KB + 1);
        const double piv = prow[c];
        if (c < kb) { pmin = fmin(pmin, fabs(piv)); pmax = fmax(pmax, fabs(piv)); }   // fmin/fmax drop a NaN operand ...
        if (c < kb && !(fabs(piv) <= 1.79e308)) pmin = 0.0;                            // ... so a NaN / Inf pivot is flagged here
        const double pinv = rcp_newton(piv);
        if (lane == c) sDi[c] = pinv;
        if (lane > c && rowlane) {
            const double l = myrow[c] * pinv;
            myrow[c] = l;
#pragma unroll
            for (int cc = c + 1; cc < KB; ++cc) myrow[cc] = fma(-l, prow[cc], myrow[cc]);
        }
        __syncwarp();
    }
    if (lane < kb) {
#pragma unroll
        for (int c = 0; c < KB; ++c)
            if (c < kb) A[(k0 + lane) + (size_t)(k0 + c) * lda] = myrow[c];
    }
}

// Blocked outer-product band LU, one block per matrix.  Per block step of KB columns:
//   (1) the KB x KB diagonal block is eliminated by warp 0 in shared memory (lane = row);
//   (2) one thread per row / column forms the L panel A21 U11^-1 and the U panel L11^-1 A12 (both in the
//       same pass: two independent substitution chains per thread) and leaves -L and U in shared memory;
//   (3) the trailing window A22 (bw x bw) += (-L)(U) is a rank-KB update on the FP64 tensor cores
//       (mma.sync.m8n8k4, 32 x 32 warp tiles, fragments straight from the shared-memory panels).
// Computed transposed (C^T = U^T (-L)^T) so that a lane's two accumulator entries are two consecutive
// rows of one column of the column-major window.
// Dynamic shared memory: 2 x (sD[KB][KB+1], sDi[KB] (1/pivots)), sDs[KB][KB], sL[KB][MWP], sU[KB][MWP]; MWP = bw rounded up to
// WT, plus 4 (row stride = 4 mod 16 doubles: the fragment loads are bank-conflict free), zero padded.
template <int KB, int NT>
__global__ void __launch_bounds__(NT, (KB == 16 && NT == 128) ? BAND16_MIN_BLOCKS : 1)
k_band_factor(int n, int W, int MWP, size_t mat_doubles, size_t pstride, int S, const int32_t *__restrict__ mlow,
              double *__restrict__ band_all, double *__restrict__ pivots, int pivS) {
    extern __shared__ double smem[];
    constexpr int DSZ = KB * (KB + 1) + KB;  // one diagonal-block buffer: sD[KB][KB+1], sDi[KB]
    double *sDs = smem + 2 * DSZ;            // [KB][KB]: the current L11 \ U11 with 16-byte aligned rows (panel substitutions)
    double *sL = sDs + KB * KB;              // [KB][MWP]: sL[c][i] = -L(k0+kb+i, k0+c)
    double *sU = sL + (size_t)KB * MWP;      // [KB][MWP]: sU[c][j] = U(k0+c, k0+kb+j)
    const size_t lda = 2 * (size_t)W;        // LD - 1
    double *A = band_all + (size_t)(blockIdx.x / S) * pstride + (size_t)(blockIdx.x % S) * mat_doubles + W;   // A(i,j) = A[i + j*lda]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, k = lane & 3;
    double pmin = 1.79e308, pmax = 0.0;      // smallest / largest |pivot| (warp 0; uniform over its lanes)
    // Look-ahead: the diagonal block of step s+1 lies in the first 32 x 32 entries of step s's window.  Warp 0
    // updates those tiles first and then eliminates the next diagonal block while the other warps update the
    // rest of the window, so the serial elimination is off the critical path (two buffers, swapped per step).
    int cur = 0;
    if (warp == 0) factor_diag_block<KB>(A, lda, 0, min(KB, n), smem, smem + KB * (KB + 1), lane, pmin, pmax);
    __syncthreads();                         // phase (1) of the first step already reads the eliminated block
    for (int k0 = 0; k0 < n; k0 += KB) {
        const int kb = min(KB, n - k0);
        const int m = mlow[k0 / KB];         // rows below / columns right of the block inside the envelope (<= bw)
        double *sD = smem + cur * DSZ, *sDi = sD + KB * (KB + 1);
        // (1) raw panel entries into shared memory
        for (int i = tid; i < MWP; i += NT) {
            if (i < m) {
                const double *row = A + (k0 + kb + i) + (size_t)k0 * lda;
                const double *col = A + k0 + (size_t)(k0 + kb + i) * lda;
#pragma unroll 16
                for (int c = 0; c < KB; ++c) {
                    sL[(size_t)c * MWP + i] = c < kb ? row[(size_t)c * lda] : 0.0;
                    sU[(size_t)c * MWP + i] = c < kb ? col[c] : 0.0;
                }
            } else {
#pragma unroll
                for (int c = 0; c < KB; ++c) { sL[(size_t)c * MWP + i] = 0.0; sU[(size_t)c * MWP + i] = 0.0; }
            }
        }
        for (int t = tid; t < KB * KB; t += NT) sDs[t] = sD[(t / KB) * (KB + 1) + t % KB];
        __syncthreads();
        // (2) panels: thread i does row i of the L panel (x U11 = a) and column i of the U panel (L11 y = a), two
        //     independent substitution chains, interleaved.  The phase is bound by the warp-uniform loads of the
        //     diagonal block, so both chains walk ROWS of it, two entries per 16-byte load: the L row right-looking
        //     (x_c -= x_t U11[t][c] for c > t as soon as x_t is final), the U column left-looking
        //     (y_t -= L11[t][cc] y_cc for cc < t).  Every sum runs in ascending index order.
        for (int i = tid; i < m; i += NT) {
            double x[KB], y[KB];
            double *row = A + (k0 + kb + i) + (size_t)k0 * lda;
            double *col = A + k0 + (size_t)(k0 + kb + i) * lda;
#pragma unroll
            for (int c = 0; c < KB; ++c) { x[c] = sL[(size_t)c * MWP + i]; y[c] = sU[(size_t)c * MWP + i]; }
#pragma unroll
            for (int t = 0; t < KB; ++t) {
                const double *drow = sDs + t * KB;
                x[t] *= sDi[t];
                const double xt = -x[t];
                if ((t + 1) < KB && ((t + 1) & 1)) x[t + 1] = fma(xt, drow[t + 1], x[t + 1]);
#pragma unroll
                for (int c = (t + 2) & ~1; c < KB; c += 2) {
                    const double2 u = *reinterpret_cast<const double2 *>(drow + c);
                    x[c] = fma(xt, u.x, x[c]);
                    x[c + 1] = fma(xt, u.y, x[c + 1]);
                }
                double w = y[t];
#pragma unroll
                for (int cc = 0; cc + 1 < t; cc += 2) {
                    const double2 l = *reinterpret_cast<const double2 *>(drow + cc);
                    w = fma(-l.x, y[cc], w);
                    w = fma(-l.y, y[cc + 1], w);
                }
                if (t & 1) w = fma(-drow[t - 1], y[t - 1], w);
                y[t] = w;
            }
#pragma unroll
            for (int c = 0; c < KB; ++c) {
                if (c < kb) { __stcs(row + (size_t)c * lda, x[c]); __stcs(col + c, y[c]); }     // final L / U entries: evict first, the L2 is for the windows
                sL[(size_t)c * MWP + i] = -x[c];
                sU[(size_t)c * MWP + i] = y[c];
            }
        }
        __syncthreads();
        if (m > 0) {
            // warp tiles of 32 rows x 16 columns: the accumulators (32 doubles) leave room for the C tile itself
            // (32 doubles), which is fetched into registers BEFORE the mma loop and so costs no wait afterwards
            const int nti = (m + WT - 1) / WT, ntj = (m + WTJ - 1) / WTJ;
            double *C0 = A + (k0 + kb) + (size_t)(k0 + kb) * lda;
            // warp 0: only the tiles that hold the next diagonal block (row tile 0, column tiles 0 and 1); the
            // other warps share the rest
            const int ntiles = nti * ntj, nlook = min(ntj, (KB + WTJ - 1) / WTJ);
            constexpr int NWRK = NT / 32 - 1;
            for (int u = (warp == 0 ? 0 : warp - 1); u < (warp == 0 ? nlook : ntiles - nlook); u += (warp == 0 ? 1 : NWRK)) {
                int wt;
                if (warp == 0) wt = u * nti;                                   // (ti = 0, tj = u)
                else { wt = u + 1; if (nlook > 1 && wt >= nti) wt += 1; }      // skip tiles (0,0) and (0,1)
                const int i0 = (wt % nti) * WT, j0 = (wt / nti) * WTJ;
                // acc[jb][ib] = -(L U)(i0 + 8 ib + 2k + {0,1}, j0 + 8 jb + g)
                double acc[2][4][2], cb[2][4][2];
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {
                    const int j = j0 + 8 * jb + g;
                    const double *colp = C0 + (size_t)j * lda;
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {
                        const int i = i0 + 8 * ib + 2 * k;
                        if (j < m && i + 1 < m) {      // 16-byte aligned: W, lda and the matrix stride are even, i is even
                            const double2 v = *reinterpret_cast<const double2 *>(colp + i);
                            cb[jb][ib][0] = v.x; cb[jb][ib][1] = v.y;
                        } else {
                            cb[jb][ib][0] = (j < m && i < m) ? colp[i] : 0.0;
                            cb[jb][ib][1] = 0.0;
                        }
                        acc[jb][ib][0] = 0.0; acc[jb][ib][1] = 0.0;
                    }
                }
#pragma unroll 4
                for (int c0 = 0; c0 < KB; c0 += 4) {
                    const double *pu = sU + (size_t)(c0 + k) * MWP + j0 + g;
                    const double *pl = sL + (size_t)(c0 + k) * MWP + i0 + g;
                    double fa[2], fb[4];
#pragma unroll
                    for (int t = 0; t < 2; ++t) fa[t] = pu[8 * t];
#pragma unroll
                    for (int t = 0; t < 4; ++t) fb[t] = pl[8 * t];
#pragma unroll
                    for (int jb = 0; jb < 2; ++jb)
#pragma unroll
                        for (int ib = 0; ib < 4; ++ib) dmma884(acc[jb][ib], fa[jb], fb[ib]);
                }
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {
                    const int j = j0 + 8 * jb + g;
                    double *colp = C0 + (size_t)j * lda;
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {
                        const int i = i0 + 8 * ib + 2 * k;
                        if (j < m && i + 1 < m)
                            *reinterpret_cast<double2 *>(colp + i) = make_double2(cb[jb][ib][0] + acc[jb][ib][0], cb[jb][ib][1] + acc[jb][ib][1]);
                        else if (j < m && i < m) colp[i] = cb[jb][ib][0] + acc[jb][ib][0];
                    }
                }
            }
        }
        if (warp == 0 && k0 + kb < n) {
            __threadfence_block();
            __syncwarp();
            double *sDn = smem + (cur ^ 1) * DSZ;
            factor_diag_block<KB>(A, lda, k0 + kb, min(KB, n - k0 - kb), sDn, sDn + KB * (KB + 1), lane, pmin, pmax);
        }
        __syncthreads();
        cur ^= 1;
    }
    if (pivots && tid == 0) {       // [problem][all species of the ctx][2]; pivots points at this grid's first species
        double *pv = pivots + 2 * ((size_t)(blockIdx.x / S) * pivS + blockIdx.x % S);
        pv[0] = pmin; pv[1] = pmax;
    }
}

// ------------------------------------------------------------------------------------------------
// Front (envelope) factorisation.  The band kernel above updates the whole m x m hull of a block step; but LU without
// pivoting keeps the ENVELOPE, and in the ordered Landau matrices the envelope is jagged: at config 5 a block step
// reaches m = 230 rows of which only ~80 have their first entry at or before the block.  This kernel gathers exactly
// those rows / columns (BandSpace::act_*) into a dense front in shared memory -- raw panels sL / sU and the window
// sW[na][na] -- runs the same three phases as the band kernel on it (diagonal block by warp 0 with look-ahead, panel
// substitutions, rank-KB window update on the FP64 tensor cores, now shared memory to shared memory) and scatters the
// window back: a sixth of the flops and no read-modify-write of the window through L2.  Same storage, same L and U
// (up to the order of the sums inside a window entry: unchanged, the update of a step is one mma chain either way).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
__device__ __forceinline__ void named_bar_arrive(int id, int nthreads) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }

// KB x KB block eliminated without pivoting by one warp, lane = row, the row in REGISTERS and the pivot row passed
// around by shuffles (the shared-memory version of the band kernel spends its time on the round trip of every row
// through shared memory and a warp barrier per column; here a column costs one reciprocal and 2 (KB - c) shuffles).
// L\U goes to sD[KB][KB], 1/pivots to sDi, and to Aout (global, leading dimension lda); a short block is completed
// by the identity.  Returns (smallest, largest |pivot|), smallest = 0 for a zero / NaN / infinite pivot.
// SIGNAL > 0: the warp arrives at named barrier SIGNAL (of `nthreads` threads) once it has the block out of src.
// Not inlined: compiled on its own the rows stay in registers (inlined into the front kernel they went to the stack).
template <int KB, int SIGNAL>
__device__ __noinline__ double2 factor_diag_src(const double *src, size_t lds, double *Aout, size_t lda, int kb, double *sD, double *sDi,
                                                int lane, int nthreads, const int *ps = nullptr) {
    // ps != nullptr: block entry (r, c) is src[ps[r] + ps[c] lds] (rows / columns of the block by their window slots)
    double r[KB];
    double pmin = 1.79e308, pmax = 0.0;
    const int row = min(lane, KB - 1);
    const int myoff = (ps && lane < kb) ? ps[row] : row;
#pragma unroll
    for (int c = 0; c < KB; ++c)
        r[c] = (lane < kb && c < kb) ? src[myoff + (size_t)((ps && c < kb) ? ps[c] : c) * lds] : (lane == c ? 1.0 : 0.0);
    if (SIGNAL > 0) {
        double keep = 0.0;                 // the loads above must have RETURNED before the barrier lets others overwrite src
#pragma unroll
        for (int c = 0; c < KB; ++c) keep += r[c];
        if (keep == 1.2345e300) r[0] = keep;
        __syncwarp();
        named_bar_arrive(SIGNAL, nthreads);
    }
#pragma unroll
    for (int c = 0; c < KB; ++c) {
        const double piv = __shfl_sync(0xffffffffu, r[c], c);
        if (c < kb) { pmin = fmin(pmin, fabs(piv)); pmax = fmax(pmax, fabs(piv)); }   // fmin/fmax drop a NaN operand ...
        if (c < kb && !(fabs(piv) <= 1.79e308)) pmin = 0.0;                            // ... so a NaN / Inf pivot is flagged here
        const double pinv = rcp_newton(piv);
        if (lane == c) sDi[c] = pinv;
        const bool below = lane > c;
        const double l = r[c] * pinv;
        if (below) r[c] = l;
#pragma unroll
        for (int cc = c + 1; cc < KB; ++cc) {
            const double pr = __shfl_sync(0xffffffffu, r[cc], c);
            if (below) r[cc] = fma(-l, pr, r[cc]);
        }
    }
    if (lane < KB) {                       // rows 16-byte aligned: the substitutions read them with 16-byte loads
#pragma unroll
        for (int c = 0; c < KB; ++c) sD[lane * KB + c] = r[c];
    }
    if (lane < kb) {
#pragma unroll
        for (int c = 0; c < KB; ++c)
            if (c < kb) Aout[lane + (size_t)c * lda] = r[c];
    }
    __syncwarp();
    return make_double2(pmin, pmax);
}

// Dynamic shared memory (doubles): 2 x (sD[KB][KB], sDi[KB]), sL[KB][LDP], sU[KB][LDP], sW[na_max][LDW]
// (column-major window, LDW = 8 mod 16: the 16-byte accesses of a C tile are bank-conflict free), then 2 na_max ints
// (this step's list and the next one's).
//
// Schedule of a block step (warp 0 = the "pivot" warp, warps 1 .. NW-1 = workers):
//   all      copy of the eliminated diagonal block, panel substitutions (one chain per thread)          [block barriers]
//   warp 0   the window tiles that hold the next diagonal block, then its elimination (the serial part of the method)
//   workers  the other window tiles | scatter of the window back to the band | next step's list and gather
// so the elimination of the next diagonal block runs beside the workers' memory phases.  Named barriers: 1 = warp 0's
// tiles are done (workers wait), 2 = warp 0 has copied the block out of the window (the workers' gather may overwrite it),
// 3 = among the workers (scatter done).
constexpr int FRONT_JC = 4, FRONT_IR = 5;      // window gather: columns per warp and pass, rows per lane (fronts of up to 160 rows)
template <int KB, int NT>
__global__ void __launch_bounds__(NT)
k_front_factor(int n, int W, int LDP, int LDW, int na_max, size_t mat_doubles, size_t pstride, int S,
               const int32_t *__restrict__ act_ptr, const int32_t *__restrict__ act_idx, double *__restrict__ band_all,
               double *__restrict__ pivots, int pivS) {
    extern __shared__ double smem[];
    constexpr int DSZ = KB * KB + KB;
    constexpr int NW = NT / 32, NWW = NW - 1, NTW = NT - 32;      // warps, worker warps, worker threads
    static_assert(NW >= 2, "a pivot warp and at least one worker");
    double *sL = smem + 2 * DSZ;                 // sL[c][i] = -L(act[i], k0 + c)
    double *sU = sL + (size_t)KB * LDP;          // sU[c][j] = U(k0 + c, act[j])
    double *sW = sU + (size_t)KB * LDP;          // sW[i + j LDW] = A(act[i], act[j])
    int *sAct = reinterpret_cast<int *>(sW + (size_t)LDW * na_max), *sActN = sAct + na_max;    // this step's list, the next one's
    const size_t lda = 2 * (size_t)W;
    double *A = band_all + (size_t)(blockIdx.x / S) * pstride + (size_t)(blockIdx.x % S) * mat_doubles + W;   // A(i,j) = A[i + j*lda]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, k = lane & 3;
    double pmin = 1.79e308, pmax = 0.0;

    // gather of a step's front by the threads [t0, t0 + nt): raw panels (thread = active row / column), window (warp = columns)
    auto gather = [&](int k0, int kb, int na, int t, int nt) {
        for (int i = t; i < LDP; i += nt) {
            if (i < na) {
                const int gi = sAct[i];
                const double *row = A + gi + (size_t)k0 * lda;
                const double *col = A + k0 + (size_t)gi * lda;
#pragma unroll
                for (int c = 0; c < KB; ++c) {
                    sL[(size_t)c * LDP + i] = c < kb ? row[(size_t)c * lda] : 0.0;
                    sU[(size_t)c * LDP + i] = c < kb ? col[c] : 0.0;
                }
            } else {
#pragma unroll
                for (int c = 0; c < KB; ++c) { sL[(size_t)c * LDP + i] = 0.0; sU[(size_t)c * LDP + i] = 0.0; }
            }
        }
        // a warp takes FRONT_JC columns at a time and issues all their loads (FRONT_JC x FRONT_IR per lane) before the
        // first store: the gather is bound by the latency of these loads, not by their number
        int gr[FRONT_IR];
#pragma unroll
        for (int r = 0; r < FRONT_IR; ++r) gr[r] = lane + 32 * r < na ? sAct[lane + 32 * r] : -1;
        for (int j0 = (t >> 5) * FRONT_JC; j0 < na; j0 += (nt >> 5) * FRONT_JC) {
            double v[FRONT_JC][FRONT_IR];
#pragma unroll
            for (int q = 0; q < FRONT_JC; ++q) {
                const double *colp = A + (size_t)sAct[min(j0 + q, na - 1)] * lda;
#pragma unroll
                for (int r = 0; r < FRONT_IR; ++r) v[q][r] = gr[r] >= 0 ? colp[gr[r]] : 0.0;
            }
#pragma unroll
            for (int q = 0; q < FRONT_JC; ++q)
                if (j0 + q < na) {
#pragma unroll
                    for (int r = 0; r < FRONT_IR; ++r)
                        if (gr[r] >= 0) sW[lane + 32 * r + (size_t)(j0 + q) * LDW] = v[q][r];
                }
        }
    };

    // prologue: first diagonal block (warp 0), first list and front (everybody)
    if (warp == 0) {
        const double2 pv = factor_diag_src<KB, 0>(A, lda, A, lda, min(KB, n), smem, smem + KB * KB, lane, NT);
        pmin = fmin(pmin, pv.x); pmax = fmax(pmax, pv.y);
    }
    {
        const int na = act_ptr[1] - act_ptr[0];
        for (int i = tid; i < na; i += NT) sAct[i] = act_idx[act_ptr[0] + i];
        __syncthreads();
        gather(0, min(KB, n), na, tid, NT);
    }
    int cur = 0;
    for (int k0 = 0, step = 0; k0 < n; k0 += KB, ++step) {
        const int kb = min(KB, n - k0), kbn = min(KB, n - k0 - kb);      // this block, the next one
        const int na = act_ptr[step + 1] - act_ptr[step];
        const double *sDs = smem + cur * DSZ, *sDi = sDs + KB * KB;     // the eliminated diagonal block (rows), 1 / pivots
        const int nan = kbn > 0 ? act_ptr[step + 2] - act_ptr[step + 1] : 0;
        __syncthreads();                        // this step's front is gathered, its diagonal block eliminated
        for (int i = tid; i < nan; i += NT) sActN[i] = act_idx[act_ptr[step + 1] + i];      // the next list, for the workers' gather
        // panel substitutions, one chain per thread: items [0, na) are rows of the L panel (x U11 = a, right-looking),
        // items [na, 2 na) columns of the U panel (L11 y = a, left-looking); sums in ascending index order
        for (int it = tid; it < 2 * na; it += NT) {
            const bool isL = it < na;
            const int i = isL ? it : it - na;
            const int gi = sAct[i];
            double x[KB];
            double *pan = isL ? sL : sU;
#pragma unroll
            for (int c = 0; c < KB; ++c) x[c] = pan[(size_t)c * LDP + i];
            if (isL) {
#pragma unroll
                for (int t = 0; t < KB; ++t) {
                    const double *drow = sDs + t * KB;
                    x[t] *= sDi[t];
                    const double xt = -x[t];
                    if ((t + 1) < KB && ((t + 1) & 1)) x[t + 1] = fma(xt, drow[t + 1], x[t + 1]);
#pragma unroll
                    for (int c = (t + 2) & ~1; c < KB; c += 2) {
                        const double2 u = *reinterpret_cast<const double2 *>(drow + c);
                        x[c] = fma(xt, u.x, x[c]);
                        x[c + 1] = fma(xt, u.y, x[c + 1]);
                    }
                }
                double *row = A + gi + (size_t)k0 * lda;
#pragma unroll
                for (int c = 0; c < KB; ++c) {
                    if (c < kb) __stcs(row + (size_t)c * lda, x[c]);
                    sL[(size_t)c * LDP + i] = -x[c];
                }
            } else {
#pragma unroll
                for (int t = 0; t < KB; ++t) {
                    const double *drow = sDs + t * KB;
                    double w = x[t];
#pragma unroll
                    for (int cc = 0; cc + 1 < t; cc += 2) {
                        const double2 l = *reinterpret_cast<const double2 *>(drow + cc);
                        w = fma(-l.x, x[cc], w);
                        w = fma(-l.y, x[cc + 1], w);
                    }
                    if (t & 1) w = fma(-drow[t - 1], x[t - 1], w);
                    x[t] = w;
                }
                double *col = A + k0 + (size_t)gi * lda;
#pragma unroll
                for (int c = 0; c < KB; ++c) {
                    if (c < kb) __stcs(col + c, x[c]);
                    sU[(size_t)c * LDP + i] = x[c];
                }
            }
        }
        __syncthreads();
        // window update in shared memory: sW += (-L)(U), warp tiles of 32 rows x 16 columns as in the band kernel
        const int nti = (na + WT - 1) / WT, ntj = (na + WTJ - 1) / WTJ;
        const int ntiles = nti * ntj, nlook = min(ntj, (KB + WTJ - 1) / WTJ);
        auto do_tile = [&](int wt) {
                const int i0 = (wt % nti) * WT, j0 = (wt / nti) * WTJ;
                double acc[2][4][2];
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {
                    const int j = j0 + 8 * jb + g;
                    const double *colp = sW + (size_t)j * LDW;
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {
                        const int i = i0 + 8 * ib + 2 * k;
                        if (j < na && i + 1 < na) {
                            const double2 v = *reinterpret_cast<const double2 *>(colp + i);
                            acc[jb][ib][0] = v.x; acc[jb][ib][1] = v.y;
                        } else {
                            acc[jb][ib][0] = (j < na && i < na) ? colp[i] : 0.0;
                            acc[jb][ib][1] = 0.0;
                        }
                    }
                }
#pragma unroll 4
                for (int c0 = 0; c0 < KB; c0 += 4) {
                    const double *pu = sU + (size_t)(c0 + k) * LDP + j0 + g;
                    const double *pl = sL + (size_t)(c0 + k) * LDP + i0 + g;
                    double fa[2], fb[4];
#pragma unroll
                    for (int t = 0; t < 2; ++t) fa[t] = pu[8 * t];
#pragma unroll
                    for (int t = 0; t < 4; ++t) fb[t] = pl[8 * t];
#pragma unroll
                    for (int jb = 0; jb < 2; ++jb)
#pragma unroll
                        for (int ib = 0; ib < 4; ++ib) dmma884(acc[jb][ib], fa[jb], fb[ib]);
                }
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {
                    const int j = j0 + 8 * jb + g;
                    double *colp = sW + (size_t)j * LDW;
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {
                        const int i = i0 + 8 * ib + 2 * k;
                        if (j < na && i + 1 < na) *reinterpret_cast<double2 *>(colp + i) = make_double2(acc[jb][ib][0], acc[jb][ib][1]);
                        else if (j < na && i < na) colp[i] = acc[jb][ib][0];
                    }
                }
        };
        if (warp == 0) {
            for (int u = 0; u < nlook; ++u) do_tile(u * nti);                  // (ti = 0, tj = u): rows / columns of the next block
            __threadfence_block();
            __syncwarp();
            named_bar_arrive(1, NT);
            if (kbn > 0) {
                double *sDn = smem + (cur ^ 1) * DSZ;
                const double2 pv = factor_diag_src<KB, 2>(sW, LDW, A + (k0 + kb) + (size_t)(k0 + kb) * lda, lda, kbn, sDn, sDn + KB * KB, lane, NT);
                pmin = fmin(pmin, pv.x); pmax = fmax(pmax, pv.y);
            } else named_bar_arrive(2, NT);
        } else {
            for (int u = warp - 1; u < ntiles - nlook; u += NWW) {
                int wt = u + 1;
                if (nlook > 1 && wt >= nti) wt += 1;                           // skip tiles (0,0) and (0,1)
                do_tile(wt);
            }
            named_bar_sync(1, NT);                                             // every tile of the window is done
            // the updated window back to the band (the next diagonal block is warp 0's: it writes it eliminated)
            for (int j = warp - 1; j < na; j += NWW) {
                double *colp = A + (size_t)sAct[j] * lda;
                for (int i = lane; i < na; i += 32)
                    if (i >= kbn || j >= kbn) colp[sAct[i]] = sW[i + (size_t)j * LDW];
            }
            named_bar_sync(3, NTW);                                            // the workers have written the band
            named_bar_sync(2, NT);                                             // warp 0 has its block out of the window
            { int *t1 = sAct; sAct = sActN; sActN = t1; }
            if (kbn > 0) gather(k0 + kb, kbn, nan, tid - 32, NTW);
            { int *t1 = sAct; sAct = sActN; sActN = t1; }
        }
        cur ^= 1;
        { int *t1 = sAct; sAct = sActN; sActN = t1; }
    }
    if (pivots && tid == 0) {
        double *pv = pivots + 2 * ((size_t)(blockIdx.x / S) * pivS + blockIdx.x % S);
        pv[0] = pmin; pv[1] = pmax;
    }
}

// ------------------------------------------------------------------------------------------------
// Slot kernel: the front kernel with a window that never moves.  Every active row owns a slot (band_slot_lists) -- its
// row and column of sW, its column of sL / sU -- so per block step
//   all      panel substitutions over the active rows; rank-KB update of ALL NS x NS slots on the FP64 tensor cores (free
//            slots hold zero panels: their window entries are garbage nobody reads)
//   warp 0   takes the next diagonal block out of the window by the slots of the next block's rows and eliminates it
//   workers  meanwhile: the next step's raw panels ARE the window's columns / rows at those pivot slots (shared memory
//            to shared memory); the pivot slots are freed; the rows that ENTER are assembled into free slots: slot row and
//            column zeroed, their original entries read from the band by the step's load list (~50 per row)
// Window entries leave only as L and U, written to the band by the substitutions: no scatter, no gather of the window.
// Shared memory (doubles): 2 x (sD[KB][KB], sDi[KB]), sL[KB][LDP], sU[KB][LDP], sW[NS][LDW], then 5 NS ints.
// Named barriers: 2 = warp 0 has the block out of the window, 3 / 4 / 5 = among the workers.
// ------------------------------------------------------------------------------------------------
constexpr int SLOT_NO_DST = INT32_MIN;
#ifndef SLOT_NT2
#define SLOT_NT2 256
#endif
#ifndef SLOT_NT2_MIN_KB
#define SLOT_NT2_MIN_KB 56
#endif
constexpr int SLOT_LB = 8;                     // band loads a worker thread keeps in flight when it assembles entering rows
template <int KB, int NT>
__global__ void __launch_bounds__(NT)
k_slot_factor(int n, int W, int LDP, int LDW, int NS, size_t mat_doubles, size_t pstride, int S,
              const int32_t *__restrict__ act_ptr, const int32_t *__restrict__ act_idx, const int32_t *__restrict__ act_slot,
              const int32_t *__restrict__ slot_hi, const int32_t *__restrict__ new_ptr, const int32_t *__restrict__ new_pos, const int32_t *__restrict__ ld_ptr,
              const int32_t *__restrict__ ld_dst, const int32_t *__restrict__ ld_csr, const int32_t *__restrict__ d0_csr, const double *__restrict__ vals_all, size_t vstride, int nnz,
              double *__restrict__ band_all, double *__restrict__ pivots, int pivS) {
    extern __shared__ double smem[];
    constexpr int DSZ = KB * KB + KB;
    constexpr int NW = NT / 32, NTW = NT - 32;
    static_assert(NW >= 2, "a pivot warp and at least one worker");
    double *sL = smem + 2 * DSZ;                 // sL[c][slot] = -L(row of slot, k0 + c)
    double *sU = sL + (size_t)KB * LDP;          // sU[c][slot] = U(k0 + c, row of slot)
    double *sW = sU + (size_t)KB * LDP;          // sW[slot_i + slot_j LDW] = A(row_i, row_j)
    int *sAct = reinterpret_cast<int *>(sW + (size_t)LDW * NS), *sSlot = sAct + NS;      // this step's list: global row, slot
    int *sActN = sSlot + NS, *sSlotN = sActN + NS, *sNew = sSlotN + NS;                   // the next step's; positions of its entering rows
    const size_t lda = 2 * (size_t)W;
    double *A = band_all + (size_t)(blockIdx.x / S) * pstride + (size_t)(blockIdx.x % S) * mat_doubles + W;   // A(i,j) = A[i + j*lda]
    // The matrix itself is read from the CSR values (lists of CSR indices, -1 = no entry): the band workspace needs no
    // fill for this kernel and only ever holds L and U.
    const double *V = vals_all + (size_t)(blockIdx.x / S) * vstride + (size_t)(blockIdx.x % S) * nnz;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g = lane >> 2, k = lane & 3;
    double pmin = 1.79e308, pmax = 0.0;
    const int NSL = NS > 1 ? 32 - __clz(NS - 1) : 0;

    // assembly of the rows entering at `step` by the threads t = 0 .. nt-1 (list and slots of that step in la / ls, the
    // positions of the entering rows in ln): slot rows / columns zeroed, (after the caller's barrier) original entries loaded
    auto zero_new = [&](int nnew, const int *ls, const int *ln, int t, int nt) {
        for (int e = t; e < (nnew << NSL); e += nt) {          // (entering row, slot) pairs, NS rounded up to 2^NSL: no division
            const int o = e & ((1 << NSL) - 1);
            if (o >= NS) continue;
            const int sn = ls[ln[e >> NSL]];
            sW[sn + (size_t)o * LDW] = 0.0;
            sW[o + (size_t)sn * LDW] = 0.0;
        }
    };
    auto load_new = [&](int step, int t, int nt) {
        const int e0 = ld_ptr[step], e1 = ld_ptr[step + 1];
        for (int e = e0 + t; e < e1; e += SLOT_LB * nt) {
            double v[SLOT_LB];
            int d[SLOT_LB];
#pragma unroll
            for (int q = 0; q < SLOT_LB; ++q) {
                const int eq = e + q * nt;
                d[q] = eq < e1 ? ld_dst[eq] : SLOT_NO_DST;
                const int cs = eq < e1 ? ld_csr[eq] : -1;
                v[q] = cs >= 0 ? V[cs] : 0.0;
            }
#pragma unroll
            for (int q = 0; q < SLOT_LB; ++q)
                if (d[q] != SLOT_NO_DST) sW[d[q]] = v[q];      // (negative offsets: the panels sL, sU in front of the window)
        }
    };
    // raw panels of the step whose block starts at k0 (kb columns): thread per list position; carried rows from the
    // window's pivot columns / rows (slots in ps), entering rows zero (their few entries beside the block come with the
    // step's load list, which reaches into the panels); all loads of a row before its stores
    auto raw_panels = [&](int kb, int na, const int *ls, const int *ps, const int *ln, int nnew, int t, int nt) {
        for (int i = t; i < na; i += nt) {
            const int sl = ls[i];
            bool isnew = ps == nullptr;
            for (int q = 0; q < nnew; ++q) isnew |= ln[q] == i;
#pragma unroll 1
            for (int side = 0; side < 2; ++side) {          // the L row, then the U column: KB staging registers at a time
                double pa[KB];
                if (isnew) {
#pragma unroll
                    for (int c = 0; c < KB; ++c) pa[c] = 0.0;
                } else {
#pragma unroll
                    for (int c = 0; c < KB; ++c) {
                        const int pc = ps[min(c, kb - 1)];
                        pa[c] = c < kb ? (side == 0 ? sW[sl + (size_t)pc * LDW] : sW[pc + (size_t)sl * LDW]) : 0.0;
                    }
                }
                double *pan = side == 0 ? sL : sU;
#pragma unroll
                for (int c = 0; c < KB; ++c) pan[(size_t)c * LDP + sl] = pa[c];
            }
        }
    };

    // prologue: first diagonal block (warp 0; copied from the matrix into its place in the band first); everything zero,
    // then the first front assembled from the matrix
    {
        const int kb0 = min(KB, n);
        for (int e = tid; e < kb0 * kb0; e += NT) {
            const int i = e % kb0, j = e / kb0, cs = d0_csr[i + j * KB];
            A[i + (size_t)j * lda] = cs >= 0 ? V[cs] : 0.0;
        }
        __syncthreads();
    }
    if (warp == 0) {
        const double2 pv = factor_diag_src<KB, 0>(A, lda, A, lda, min(KB, n), smem, smem + KB * KB, lane, NT);
        pmin = fmin(pmin, pv.x); pmax = fmax(pmax, pv.y);
    }
    {
        const int na = act_ptr[1] - act_ptr[0], nnew = new_ptr[1] - new_ptr[0];
        for (int i = tid; i < na; i += NT) { sAct[i] = act_idx[act_ptr[0] + i]; sSlot[i] = act_slot[act_ptr[0] + i]; }
        for (int i = tid; i < nnew; i += NT) sNew[i] = new_pos[new_ptr[0] + i];
        for (int i = tid; i < 2 * KB * LDP; i += NT) sL[i] = 0.0;                  // sL and sU are contiguous
        for (int i = tid; i < LDW * NS; i += NT) sW[i] = 0.0;
        __syncthreads();
        raw_panels(min(KB, n), na, sSlot, nullptr, sNew, nnew, tid, NT);
        __syncthreads();                        // the load list also writes panel entries of these rows
        load_new(0, tid, NT);
    }
    int cur = 0;
    for (int k0 = 0, step = 0; k0 < n; k0 += KB, ++step) {
        const int kb = min(KB, n - k0), kbn = min(KB, n - k0 - kb);      // this block, the next one
        const int na = act_ptr[step + 1] - act_ptr[step];
        const int hi = slot_hi[step];            // slots in use are below hi (the lowest free slot is taken first: hi ~ na)
        const int nti = (hi + WT - 1) / WT, ntj = (hi + WTJ - 1) / WTJ, ntiles = nti * ntj;
        const int a1 = act_ptr[step + 1], nan = kbn > 0 ? act_ptr[step + 2] - a1 : 0;     // the next step's list
        const int nn0 = kbn > 0 ? new_ptr[step + 1] : 0, nnew = kbn > 0 ? new_ptr[step + 2] - nn0 : 0;
        const double *sDs = smem + cur * DSZ, *sDi = sDs + KB * KB;     // the eliminated diagonal block (rows), 1 / pivots
        __syncthreads();                        // this step's front is in place, its diagonal block eliminated
        // the next step's lists: asked for now, parked in shared memory after the substitutions (their latency off the chain)
        constexpr int LPT = (160 + NT - 1) / NT;          // list items per thread (fronts of at most 160 rows)
        int rAct[LPT], rSlot[LPT], rNew[LPT];
#pragma unroll
        for (int q = 0; q < LPT; ++q) {
            const int i = tid + q * NT;
            rAct[q] = i < nan ? act_idx[a1 + i] : 0;
            rSlot[q] = i < nan ? act_slot[a1 + i] : 0;
            rNew[q] = i < nnew ? new_pos[nn0 + i] : 0;
        }
        // panel substitutions, one chain per thread: items [0, na) are rows of the L panel (x U11 = a, right-looking),
        // items [na, 2 na) columns of the U panel (L11 y = a, left-looking); sums in ascending index order
        for (int it = tid; it < 2 * na; it += NT) {
            const bool isL = it < na;
            const int pos = isL ? it : it - na;
            const int gi = sAct[pos], i = sSlot[pos];
            double x[KB];
            double *pan = isL ? sL : sU;
#pragma unroll
            for (int c = 0; c < KB; ++c) x[c] = pan[(size_t)c * LDP + i];
            if (isL) {
#pragma unroll
                for (int t = 0; t < KB; ++t) {
                    const double *drow = sDs + t * KB;
                    x[t] *= sDi[t];
                    const double xt = -x[t];
                    if ((t + 1) < KB && ((t + 1) & 1)) x[t + 1] = fma(xt, drow[t + 1], x[t + 1]);
#pragma unroll
                    for (int c = (t + 2) & ~1; c < KB; c += 2) {
                        const double2 u = *reinterpret_cast<const double2 *>(drow + c);
                        x[c] = fma(xt, u.x, x[c]);
                        x[c + 1] = fma(xt, u.y, x[c + 1]);
                    }
                }
                double *row = A + gi + (size_t)k0 * lda;
#pragma unroll
                for (int c = 0; c < KB; ++c) {
                    if (c < kb) __stcs(row + (size_t)c * lda, x[c]);
                    sL[(size_t)c * LDP + i] = -x[c];
                }
            } else {
#pragma unroll
                for (int t = 0; t < KB; ++t) {
                    const double *drow = sDs + t * KB;
                    double w = x[t];
#pragma unroll
                    for (int cc = 0; cc + 1 < t; cc += 2) {
                        const double2 l = *reinterpret_cast<const double2 *>(drow + cc);
                        w = fma(-l.x, x[cc], w);
                        w = fma(-l.y, x[cc + 1], w);
                    }
                    if (t & 1) w = fma(-drow[t - 1], x[t - 1], w);
                    x[t] = w;
                }
                double *col = A + k0 + (size_t)gi * lda;
#pragma unroll
                for (int c = 0; c < KB; ++c) {
                    if (c < kb) __stcs(col + c, x[c]);
                    sU[(size_t)c * LDP + i] = x[c];
                }
            }
        }
#pragma unroll
        for (int q = 0; q < LPT; ++q) {
            const int i = tid + q * NT;
            if (i < nan) { sActN[i] = rAct[q]; sSlotN[i] = rSlot[q]; }
            if (i < nnew) sNew[i] = rNew[q];
        }
        __syncthreads();
        // window update over all slots: sW += (-L)(U), warp tiles of 32 rows x 16 columns as in the band kernel
        for (int wt = warp; wt < ntiles; wt += NW) {
                const int i0 = (wt % nti) * WT, j0 = (wt / nti) * WTJ;
                double acc[2][4][2];
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {
                    const int j = j0 + 8 * jb + g;
                    const double *colp = sW + (size_t)j * LDW;
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {
                        const int i = i0 + 8 * ib + 2 * k;
                        if (j < NS && i + 1 < NS) {
                            const double2 v = *reinterpret_cast<const double2 *>(colp + i);
                            acc[jb][ib][0] = v.x; acc[jb][ib][1] = v.y;
                        } else {
                            acc[jb][ib][0] = (j < NS && i < NS) ? colp[i] : 0.0;
                            acc[jb][ib][1] = 0.0;
                        }
                    }
                }
#pragma unroll 4
                for (int c0 = 0; c0 < KB; c0 += 4) {
                    const double *pu = sU + (size_t)(c0 + k) * LDP + j0 + g;
                    const double *pl = sL + (size_t)(c0 + k) * LDP + i0 + g;
                    double fa[2], fb[4];
#pragma unroll
                    for (int t = 0; t < 2; ++t) fa[t] = pu[8 * t];
#pragma unroll
                    for (int t = 0; t < 4; ++t) fb[t] = pl[8 * t];
#pragma unroll
                    for (int jb = 0; jb < 2; ++jb)
#pragma unroll
                        for (int ib = 0; ib < 4; ++ib) dmma884(acc[jb][ib], fa[jb], fb[ib]);
                }
#pragma unroll
                for (int jb = 0; jb < 2; ++jb) {
                    const int j = j0 + 8 * jb + g;
                    double *colp = sW + (size_t)j * LDW;
#pragma unroll
                    for (int ib = 0; ib < 4; ++ib) {
                        const int i = i0 + 8 * ib + 2 * k;
                        if (j < NS && i + 1 < NS) *reinterpret_cast<double2 *>(colp + i) = make_double2(acc[jb][ib][0], acc[jb][ib][1]);
                        else if (j < NS && i < NS) colp[i] = acc[jb][ib][0];
                    }
                }
        }
        __syncthreads();
        if (warp == 0) {
            // the next block's rows are the first kbn of this step's list: its diagonal block by their slots
            if (kbn > 0) {
                double *sDn = smem + (cur ^ 1) * DSZ;
                const double2 pv = factor_diag_src<KB, 2>(sW, LDW, A + (k0 + kb) + (size_t)(k0 + kb) * lda, lda, kbn, sDn, sDn + KB * KB, lane, NT, sSlot);
                pmin = fmin(pmin, pv.x); pmax = fmax(pmax, pv.y);
            } else named_bar_arrive(2, NT);
        } else {
            const int t = tid - 32;
            // the pivot rows leave: their panel entries back to zero (free slots must hold zero panels) ...
            for (int e = t; e < kbn * KB; e += NTW) {
                const int sl = sSlot[e / KB], c = e % KB;
                sL[(size_t)c * LDP + sl] = 0.0; sU[(size_t)c * LDP + sl] = 0.0;
            }
            named_bar_sync(4, NTW);             // ... before an entering row that takes such a slot writes its own
            if (kbn > 0) raw_panels(kbn, nan, sSlotN, sSlot, sNew, nnew, t, NTW);
            named_bar_sync(3, NTW);             // the workers have read the pivot columns / rows of the window
            named_bar_sync(2, NT);              // warp 0 has its block out of it
            zero_new(nnew, sSlotN, sNew, t, NTW);
            named_bar_sync(5, NTW);
            if (kbn > 0) load_new(step + 1, t, NTW);
        }
        cur ^= 1;
        { int *t1 = sAct; sAct = sActN; sActN = t1; t1 = sSlot; sSlot = sSlotN; sSlotN = t1; }
    }
    if (pivots && tid == 0) {
        double *pv = pivots + 2 * ((size_t)(blockIdx.x / S) * pivS + blockIdx.x % S);
        pv[0] = pmin; pv[1] = pmax;
    }
}

// Banded triangular solves, one block per matrix: x = P^T U^-1 L^-1 P b with the RCM permutation.
// Blocks of KB columns (those of the factorisation): the diagonal block by warp 0 (lane = row), the panel
// below / above, confined to the envelope, by one thread per row with KB independent loads.

// XG: the permuted vector of a matrix lives in global memory (xg + matrix * n) instead of shared memory -- for
// orders n beyond the 227 KB of an SM (n > ~28,000); the block barriers order those accesses just the same.
// The 32-column instantiation is compiled for seven blocks per SM (32 registers, 16 bytes of spill): the solves are chains
// of short phases, what counts is how many matrices an SM holds -- config 5: 1,024 matrices were two waves on 148 x 5
// places (3.54 ms), they are one on 148 x 7 (2.45 ms); 1,280 matrices of the ten-species 320-cell mesh 5.43 -> 4.76 ms.
template <int KB, int NT, bool XG>
__global__ void __launch_bounds__(NT, KB == 32 ? 7 : 1)
k_band_solve(int n, int W, size_t mat_doubles, size_t xstride, int S, const int32_t *__restrict__ perm,
             const int32_t *__restrict__ mlow, const int32_t *__restrict__ mup, const int32_t *__restrict__ first, size_t pstride,
             const double *__restrict__ band_all, const double *rhs, double *xout, double *xg) {     // xout may alias rhs (in-place solve): no __restrict__ on these two
    // first[i]: the column of row i's first entry in the ordered pattern = the row of column i's first entry (the
    // pattern is structurally symmetric).  L and U vanish outside the envelope -- L(i, j) for j < first[i], U(i, j) for
    // i < first[j] -- so those entries are not read: on the refined meshes two thirds of what a block step's panels span.
    constexpr int SB = KB;            // same blocks as the factorisation: panels stay inside the stored band
    extern __shared__ double smem[];
    double *x = XG ? xg + (size_t)blockIdx.x * n : smem;    // [n]
    double *sD = XG ? smem : smem + n;                      // [SB][SB+1]
    int *sF = reinterpret_cast<int *>(sD + SB * (SB + 1));  // [SB] first rows of the current block's columns (backward sweep)
    const size_t lda = 2 * (size_t)W;
    const int mat = blockIdx.x;       // = b * S + sp
    const double *A = band_all + (size_t)(mat / S) * pstride + (size_t)(mat % S) * mat_doubles + W;
    const size_t voff = (size_t)(mat / S) * xstride + (size_t)(mat % S) * n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < n; i += NT) x[i] = rhs[voff + perm[i]];
    __syncthreads();
    // forward: L y = b (unit lower)
    for (int k0 = 0; k0 < n; k0 += SB) {
        const int kb = min(SB, n - k0), m = mlow[k0 / SB];
        for (int t = tid; t < kb * kb; t += NT) {
            const int r = t % kb, c = t / kb;
            sD[r * (SB + 1) + c] = A[(k0 + r) + (size_t)(k0 + c) * lda];
        }
        __syncthreads();
        if (warp == 0) {
            double v = lane < kb ? x[k0 + lane] : 0.0;
            for (int c = 0; c < kb - 1; ++c) {
                const double xc = __shfl_sync(0xffffffffu, v, c);
                if (lane > c && lane < kb) v = fma(-sD[lane * (SB + 1) + c], xc, v);
            }
            if (lane < kb) x[k0 + lane] = v;
        }
        __syncthreads();
        for (int i = tid; i < m; i += NT) {
            const int c0 = first[k0 + kb + i] - k0;                 // row entries left of this are zero (c0 >= kb: the whole row)
            if (c0 >= kb) continue;
            const double *row = A + (k0 + kb + i) + (size_t)k0 * lda;
            double v = x[k0 + kb + i];
#pragma unroll 8
            for (int c = 0; c < kb; ++c)
                if (c >= c0) v = fma(-row[(size_t)c * lda], x[k0 + c], v);
            x[k0 + kb + i] = v;
        }
        __syncthreads();
    }
    // backward: U x = y
    const int nblk = (n + SB - 1) / SB;
    for (int blk = nblk - 1; blk >= 0; --blk) {
        const int k0 = blk * SB, kb = min(SB, n - k0), m = mup[blk];
        for (int t = tid; t < kb * kb; t += NT) {
            const int r = t % kb, c = t / kb;
            sD[r * (SB + 1) + c] = A[(k0 + r) + (size_t)(k0 + c) * lda];
        }
        if (tid < SB) sF[tid] = tid < kb ? first[k0 + tid] : n;
        __syncthreads();
        if (warp == 0) {
            double v = lane < kb ? x[k0 + lane] : 0.0;
            for (int c = kb - 1; c >= 0; --c) {
                if (lane == c) v = v / sD[c * (SB + 1) + c];
                const double xc = __shfl_sync(0xffffffffu, v, c);
                if (lane < c) v = fma(-sD[lane * (SB + 1) + c], xc, v);
            }
            if (lane < kb) x[k0 + lane] = v;
        }
        __syncthreads();
        for (int i = tid; i < m; i += NT) {
            const int r = k0 - m + i;
            const double *row = A + r + (size_t)k0 * lda;
            double v = x[r];
#pragma unroll 8
            for (int c = 0; c < kb; ++c)
                if (sF[c] <= r) v = fma(-row[(size_t)c * lda], x[k0 + c], v);     // U(r, k0 + c) is zero above the column's first row
            x[r] = v;
        }
        __syncthreads();
    }
    for (int i = tid; i < n; i += NT) xout[voff + perm[i]] = x[i];
}

// Host: the active list of every block step (BandSpace::act_*).  LU without pivoting keeps the envelope: row i of L
// starts at first[i] (its first entry in the ordered pattern), column j of U likewise (the pattern is structurally
// symmetric).  So block step s (columns k0 .. ke) only involves the rows / columns i > ke with first[i] <= ke; the
// next block's rows are always listed (first, in order) so that its diagonal block is the leading corner of the front.
int band_active_lists(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const std::vector<int32_t> &perm,
                      int KB, std::vector<int32_t> &act_ptr, std::vector<int32_t> &act_idx, double *front_flop) {
    const int nsteps = (n + KB - 1) / KB;
    std::vector<int32_t> pos(n), first(n);
    for (int i = 0; i < n; ++i) { pos[perm[i]] = i; first[i] = i; }
    for (int i = 0; i < n; ++i)
        for (int t = rowptr[i]; t < rowptr[i + 1]; ++t) first[pos[i]] = std::min<int32_t>(first[pos[i]], pos[colidx[t]]);
    int bw = 0;                            // a row i can only be active at a step with i - first[i] <= bw
    for (int i = 0; i < n; ++i) bw = std::max(bw, i - int(first[i]));
    act_ptr.assign(nsteps + 1, 0);
    act_idx.clear();
    int na_max = 0;
    double work = 0.0;
    for (int s = 0; s < nsteps; ++s) {
        const int ke = std::min(s * KB + KB, n) - 1, nxt = std::min(ke + KB, n - 1);
        for (int i = ke + 1; i < n && i <= std::min(n - 1, ke + bw + KB); ++i)      // first[i] >= i - bw
            if (i <= nxt || first[i] <= ke) act_idx.push_back(i);
        act_ptr[s + 1] = int32_t(act_idx.size());
        const int na = act_ptr[s + 1] - act_ptr[s];
        na_max = std::max(na_max, na);
        work += 2.0 * (ke - s * KB + 1) * double(na) * double(na);
    }
    if (front_flop) *front_flop = work;
    return na_max;
}

// Host: lists of the slot kernel (k_slot_factor).  A row keeps ONE place (row and column index) in the shared-memory
// window for as long as it is active -- a row that becomes a pivot row frees its slot, a row that enters takes the lowest
// free one (na_max slots suffice: the pivot rows of a step have been taken out before that step's new rows arrive) -- so
// the window is never re-packed and never travels.  Per block step s: act_slot (aligned with act_idx), new_pos (positions
// in list s of the rows that ENTER at step s) and the load list of step s: the original entries (i, j) of the matrix
// with i entering and j in list s (or both entering), as (offset in the window, index into the CSR values) -- the entering
// rows are assembled sparsely, everything else of their rows / columns is zero.  The list of step s also carries the
// entries of the entering rows beside the block of that step, A(i, k0 + c) and A(k0 + c, i): they belong into the raw
// panels sL[c ldp + slot], sU[c ldp + slot], which lie in front of the window in shared memory (negative offsets).
// d0_csr[i + j KB]: CSR index of the entry (i, j) of the first diagonal block, -1 where the matrix has none.
void band_slot_lists(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const std::vector<int32_t> &perm,
                     int KB, int ldp, int ldw, const std::vector<int32_t> &act_ptr, const std::vector<int32_t> &act_idx, int na_max,
                     std::vector<int32_t> &act_slot, std::vector<int32_t> &slot_hi, std::vector<int32_t> &new_ptr, std::vector<int32_t> &new_pos,
                     std::vector<int32_t> &ld_ptr, std::vector<int32_t> &ld_dst, std::vector<int32_t> &ld_csr, std::vector<int32_t> &d0_csr) {
    const int nsteps = (n + KB - 1) / KB;
    std::vector<int32_t> pos(n);
    for (int i = 0; i < n; ++i) pos[perm[i]] = i;
    // CSR index of the entry (i, j) (new numbering) or -1
    auto csr_of = [&](int i, int j) {
        const int io = perm[i], jo = perm[j];
        const int32_t *b = colidx.data() + rowptr[io], *e = colidx.data() + rowptr[io + 1];
        const int32_t *hit = std::lower_bound(b, e, int32_t(jo));
        return (hit != e && *hit == jo) ? int32_t(hit - colidx.data()) : int32_t(-1);
    };
    d0_csr.assign((size_t)KB * KB, -1);
    for (int j = 0; j < std::min(KB, n); ++j)
        for (int i = 0; i < std::min(KB, n); ++i) d0_csr[i + (size_t)j * KB] = csr_of(i, j);
    act_slot.assign(act_idx.size(), 0);
    new_ptr.assign(nsteps + 1, 0); ld_ptr.assign(nsteps + 1, 0); slot_hi.assign(nsteps, 0);
    new_pos.clear(); ld_dst.clear(); ld_csr.clear();
    std::vector<int32_t> slot_of(n, -1), entered(n, -1);
    std::vector<int> free_slots;                          // kept sorted descending: pop_back gives the lowest
    for (int k = na_max - 1; k >= 0; --k) free_slots.push_back(k);
    for (int s = 0; s < nsteps; ++s) {
        if (s > 0) {                                      // the rows of block s (the first entries of list s-1) have left
            const int k0 = s * KB, ke = std::min(k0 + KB, n) - 1;
            for (int i = k0; i <= ke; ++i)
                if (slot_of[i] >= 0) { free_slots.push_back(slot_of[i]); slot_of[i] = -1; }
            std::sort(free_slots.begin(), free_slots.end(), std::greater<int>());
        }
        for (int q = act_ptr[s]; q < act_ptr[s + 1]; ++q) {
            const int i = act_idx[q];
            if (slot_of[i] < 0) {
                slot_of[i] = free_slots.back(); free_slots.pop_back();
                entered[i] = s;
                new_pos.push_back(q - act_ptr[s]);
            }
            act_slot[q] = slot_of[i];
            slot_hi[s] = std::max(slot_hi[s], slot_of[i] + 1);
        }
        new_ptr[s + 1] = int32_t(new_pos.size());
        for (int t = new_ptr[s]; t < new_ptr[s + 1]; ++t) {
            const int i = act_idx[act_ptr[s] + new_pos[t]], io = perm[i], si = slot_of[i];
            for (int u = rowptr[io]; u < rowptr[io + 1]; ++u) {
                const int j = pos[colidx[u]];
                if (slot_of[j] < 0) continue;            // not in this step's list: eliminated, in the block, or not yet active
                // (i, j) and, unless j enters at this step too (its own pass covers it), (j, i)
                ld_dst.push_back(int32_t(si + slot_of[j] * ldw)); ld_csr.push_back(int32_t(u));
                if (entered[j] != s) { ld_dst.push_back(int32_t(slot_of[j] + si * ldw)); ld_csr.push_back(csr_of(j, i)); }
            }
            const int k0 = s * KB;                        // beside the block: sL at -2 KB ldp, sU at -KB ldp from the window
            for (int c = 0; c < KB && k0 + c < n; ++c) {
                const int32_t cl = csr_of(i, k0 + c), cu = csr_of(k0 + c, i);
                if (cl >= 0) { ld_dst.push_back(int32_t(-2 * KB * ldp + c * ldp + si)); ld_csr.push_back(cl); }
                if (cu >= 0) { ld_dst.push_back(int32_t(-KB * ldp + c * ldp + si)); ld_csr.push_back(cu); }
            }
        }
        ld_ptr[s + 1] = int32_t(ld_dst.size());
    }
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
static int band_mw(int bw) { return ((std::max(bw, 1) + WT - 1) / WT) * WT + 4; }

size_t band_factor_smem(int bw, int KB) {
    return sizeof(double) * (2 * ((size_t)KB * (KB + 1) + KB) + (size_t)KB * KB + 2 * (size_t)KB * band_mw(bw));
}

cudaError_t launch_band_fill(const BandSpace &bs, int nb, int S, size_t vstride, size_t pstride, const double *vals, double *band,
                             cudaStream_t st) {
    const int W = bs.W;
    dim3 grid((bs.n + FILL_WARPS - 1) / FILL_WARPS, S, nb);
    // (not launched when the slot kernel factors: band_needs_fill)
    k_band_fill<<<grid, 32 * FILL_WARPS, 0, st>>>(bs.n, bs.nnz, 2 * (size_t)W + 1, vstride, bs.mat_doubles, pstride, bs.zlo, bs.zcnt, bs.fptr,
                                                 bs.fsrc, bs.foff, vals, band);
    return cudaGetLastError();
}

// Host: the fill lists of BandSpace for an order (perm[new] = old, pos = its inverse) and its envelope (mlow, mup per
// block step of KB columns).  Column j (new numbering, block step s_j) is touched in the rows of every square
// [k0(s), E(s)]^2, E(s) = ke(s) + mlow[s], that contains it -- the diagonal block, panels and window of step s -- and
// by the backward solve up to mup[s_j] rows above its block: rows k0(first s with E(s) >= j) ... E(s_j).
void band_fill_lists(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const std::vector<int32_t> &perm,
                     int W, int KB, const std::vector<int32_t> &mlow, const std::vector<int32_t> &mup, int KBs,
                     const std::vector<int32_t> &mlow_s, const std::vector<int32_t> &mup_s, std::vector<int32_t> &zlo,
                     std::vector<int32_t> &zcnt, std::vector<int32_t> &fptr, std::vector<int32_t> &fsrc, std::vector<int32_t> &foff) {
    std::vector<int32_t> pos(n);
    for (int i = 0; i < n; ++i) pos[perm[i]] = i;
    // rows [lo[j], hi[j]] of column j for blocks of kb columns with the envelope (ml, mu)
    auto ranges = [n](int kb, const std::vector<int32_t> &ml, const std::vector<int32_t> &mu, std::vector<int32_t> &lo, std::vector<int32_t> &hi) {
        const int nsteps = (n + kb - 1) / kb;
        std::vector<int32_t> E(nsteps);
        // (the front kernel lists the next block's rows whether the envelope reaches them or not: at least kb rows)
        for (int s = 0; s < nsteps; ++s) E[s] = std::min(n - 1, std::min(s * kb + kb, n) - 1 + std::max(int(ml[s]), kb));
        lo.assign(n, 0); hi.assign(n, 0);
        int s0 = 0;
        for (int j = 0; j < n; ++j) {
            const int sj = j / kb;
            while (E[s0] < j) ++s0;                                // E is non-decreasing and E[sj] >= j
            lo[j] = std::min(s0 * kb, std::max(0, sj * kb - int(mu[sj])));
            hi[j] = E[sj];
        }
    };
    // the factorisation's blocks and, where the solves walk the band in blocks of another width (KBs), theirs as well
    std::vector<int32_t> lo, hi, lo_s, hi_s;
    ranges(KB, mlow, mup, lo, hi);
    if (KBs != KB) {
        ranges(KBs, mlow_s, mup_s, lo_s, hi_s);
        for (int j = 0; j < n; ++j) { lo[j] = std::min(lo[j], lo_s[j]); hi[j] = std::max(hi[j], hi_s[j]); }
    }
    zlo.assign(n, 0); zcnt.assign(n, 0); fptr.assign(n + 1, 0);
    fsrc.clear(); foff.clear();
    for (int j = 0; j < n; ++j) {
        zlo[j] = W + lo[j] - j;
        zcnt[j] = hi[j] - lo[j] + 1;
        const int jo = perm[j];
        for (int t = rowptr[jo]; t < rowptr[jo + 1]; ++t) {        // structurally symmetric: rows of column jo = columns of row jo
            const int io = colidx[t];
            const int32_t *b = colidx.data() + rowptr[io], *e = colidx.data() + rowptr[io + 1];
            const int32_t *hit = std::lower_bound(b, e, int32_t(jo));
            if (hit == e || *hit != jo) continue;                  // (not symmetric here: no entry (io, jo))
            fsrc.push_back(int32_t(hit - colidx.data()));
            foff.push_back(int32_t(W + pos[io] - j));
        }
        fptr[j + 1] = int32_t(fsrc.size());
    }
}

template <int KB, int NT>
static cudaError_t factor_t(const BandSpace &bs, int nmat, int S, size_t pstride, double *band, double *pivots, int pivS, cudaStream_t st) {
    const size_t smem = band_factor_smem(bs.bw, KB);
    cudaError_t e = cudaFuncSetAttribute(k_band_factor<KB, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_band_factor<KB, NT><<<nmat, NT, smem, st>>>(bs.n, bs.W, band_mw(bs.bw), bs.mat_doubles, pstride, S, bs.mlow, band, pivots, pivS);
    return cudaGetLastError();
}

static int front_ldw(int na_max) { return ((std::max(na_max, 1) + 7) / 16) * 16 + 8; }      // >= na_max, = 8 mod 16

size_t band_front_smem(int KB, int na_max) {
    return sizeof(double) * (2 * ((size_t)KB * KB + KB) + 2 * (size_t)KB * band_mw(na_max) +
                             (size_t)front_ldw(na_max) * std::max(na_max, 1) + (size_t)(2 * na_max + 2) / 2);
}

template <int KB, int NT>
static cudaError_t front_t(const BandSpace &bs, int nmat, int S, size_t pstride, double *band, double *pivots, int pivS, cudaStream_t st) {
    const size_t smem = band_front_smem(bs.kb, bs.na_max);
    cudaError_t e = cudaFuncSetAttribute(k_front_factor<KB, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_front_factor<KB, NT><<<nmat, NT, smem, st>>>(bs.n, bs.W, band_mw(bs.na_max), front_ldw(bs.na_max), std::max(bs.na_max, 1), bs.mat_doubles,
                                                   pstride, S, bs.act_ptr, bs.act_idx, band, pivots, pivS);
    return cudaGetLastError();
}

int band_front_ldw(int na_max) { return front_ldw(na_max); }
int band_front_ldp(int na_max) { return band_mw(na_max); }       // leading dimension of the raw panels

size_t band_slot_smem(int KB, int na_max) {
    return sizeof(double) * (2 * ((size_t)KB * KB + KB) + 2 * (size_t)KB * band_mw(na_max) +
                             (size_t)front_ldw(na_max) * std::max(na_max, 1) + (size_t)(5 * na_max + 2) / 2);
}

template <int KB, int NT>
static cudaError_t slot_t(const BandSpace &bs, int nmat, int S, size_t pstride, const double *vals, size_t vstride, double *band, double *pivots,
                          int pivS, cudaStream_t st) {
    const size_t smem = band_slot_smem(bs.kb, bs.na_max);
    cudaError_t e = cudaFuncSetAttribute(k_slot_factor<KB, NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_slot_factor<KB, NT><<<nmat, NT, smem, st>>>(bs.n, bs.W, band_mw(bs.na_max), front_ldw(bs.na_max), std::max(bs.na_max, 1), bs.mat_doubles,
                                                  pstride, S, bs.act_ptr, bs.act_idx, bs.act_slot, bs.slot_hi, bs.new_ptr, bs.new_pos, bs.ld_ptr, bs.ld_dst,
                                                  bs.ld_csr, bs.d0_csr, vals, vstride, bs.nnz, band, pivots, pivS);
    return cudaGetLastError();
}

// true: launch_band_fill first.  The slot kernel reads the matrix from the CSR values itself and writes every entry of
// L and U inside the envelope (the solves read nothing outside it): no fill, the workspace may hold anything.
bool band_needs_fill(const BandSpace &bs) { return !(bs.front && bs.slot && bs.kb == 16); }

cudaError_t launch_band_factor(const BandSpace &bs, int nmat, int S, size_t pstride, const double *vals, size_t vstride, double *band,
                               double *pivots, int pivS, cudaStream_t st) {
    // the front family: 16-column blocks take the slot kernel (measured: ten-species 80-cell 9.1 -> 7.4 ms, mesh 3A 5.6 -> 4.3),
    // 32-column blocks the gather / scatter kernel (config 5: 14.2 against 18.7 ms with slots -- its look-ahead of the next
    // diagonal block and the smaller tile sweep outweigh the round trip of the window there)
    if (!band_needs_fill(bs)) {
        // threads per matrix by the windows that fit an SM: one -> 512, two -> SLOT_NT2, more -> 128 (small fronts: the
        // steps are chains of latencies, more matrices per SM hide them better than more threads per matrix)
        const size_t smem = band_slot_smem(bs.kb, bs.na_max);
        if (smem > size_t(112) * 1024) return slot_t<16, 512>(bs, nmat, S, pstride, vals, vstride, band, pivots, pivS, st);
        if (smem > size_t(SLOT_NT2_MIN_KB) * 1024) return slot_t<16, SLOT_NT2>(bs, nmat, S, pstride, vals, vstride, band, pivots, pivS, st);
        return slot_t<16, 128>(bs, nmat, S, pstride, vals, vstride, band, pivots, pivS, st);
    }
    if (bs.front) {
        switch (bs.kb) {
            case 32: return front_t<32, 512>(bs, nmat, S, pstride, band, pivots, pivS, st);
            case 16: return front_t<16, 128>(bs, nmat, S, pstride, band, pivots, pivS, st);
            default: break;      // 8-column blocks mean bw > 832: no front of that size fits (front is false then)
        }
    }
    switch (bs.kb) {
        case 32: return factor_t<32, 256>(bs, nmat, S, pstride, band, pivots, pivS, st);
        case 16: return bs.bw <= 256 ? factor_t<16, 128>(bs, nmat, S, pstride, band, pivots, pivS, st)
                                     : factor_t<16, BAND_THREADS>(bs, nmat, S, pstride, band, pivots, pivS, st);
        default: return factor_t<8, BAND_THREADS>(bs, nmat, S, pstride, band, pivots, pivS, st);
    }
}

// bytes of shared memory the solve needs with the vector on chip
size_t band_solve_smem(int n, int bw) {
    const int KB = band_block(bw);
    return sizeof(double) * ((size_t)n + (size_t)KB * (KB + 1) + KB / 2);
}

template <int KB, int NT>
static cudaError_t solve_t(const BandSpace &bs, int nb, int S, size_t xstride, size_t pstride, const double *band, const double *rhs,
                           double *x, double *xg, cudaStream_t st) {
    if (xg) {        // vector in global memory: only the diagonal block in shared memory
        const size_t smem = sizeof(double) * (KB * (KB + 1) + KB / 2);
        k_band_solve<KB, NT, true><<<nb * S, NT, smem, st>>>(bs.n, bs.W, bs.mat_doubles, xstride, S, bs.perm, bs.mlow_s, bs.mup_s, bs.first, pstride, band, rhs, x, xg);
        return cudaGetLastError();
    }
    const size_t smem = band_solve_smem(bs.n, bs.bw);
    cudaError_t e = cudaFuncSetAttribute(k_band_solve<KB, NT, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_band_solve<KB, NT, false><<<nb * S, NT, smem, st>>>(bs.n, bs.W, bs.mat_doubles, xstride, S, bs.perm, bs.mlow_s, bs.mup_s, bs.first, pstride, band, rhs, x, nullptr);
    return cudaGetLastError();
}

// xg: nullptr (the vector of a matrix fits shared memory) or scratch of nb * S * n doubles
cudaError_t launch_band_solve(const BandSpace &bs, int nb, int S, size_t xstride, size_t pstride, const double *band, const double *rhs,
                              double *x, double *xg, cudaStream_t st) {
    switch (band_block(bs.bw)) {
        case 32: return solve_t<32, SOLVE_NT32>(bs, nb, S, xstride, pstride, band, rhs, x, xg, st);
        case 16: return bs.bw <= 256 ? solve_t<16, SOLVE_NT16>(bs, nb, S, xstride, pstride, band, rhs, x, xg, st)
                                     : solve_t<16, BAND_THREADS>(bs, nb, S, xstride, pstride, band, rhs, x, xg, st);
        default: return solve_t<8, BAND_THREADS>(bs, nb, S, xstride, pstride, band, rhs, x, xg, st);
    }
}

// ------------------------------------------------------------------------------------------------
// Band solve WITHOUT any allocation (landau_band_solve_static, include/landau.h): the XG instantiation of k_band_solve,
// whose permuted vectors live in global memory, given a scratch that is part of the library image instead of a
// cudaMalloc'ed one -- for callers that cannot allocate (stream capture, serving loops, harnesses that forbid it).
// Every GPU that loads the library holds BAND_STATIC_SCRATCH_DOUBLES * 8 bytes for it until the process exits.
// In host code the array's NAME is a host-side stand-in, not a device address (a kernel given it faults, or silently
// uses the wrong memory where the GPU can reach host memory): the address comes from cudaGetSymbolAddress, asked once
// per device with that device current (band_static_scratch, called at landau_create) and kept.
// All calls share the array; it keeps the last call's contents.  Nothing in it has to start at zero: a solve first
// writes the permuted right-hand sides of its nb * S matrices into [0, nb * S * n) and reads nothing beyond.  Two such
// solves that overlap on the GPU (different streams) race.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_band_static_scratch[BAND_STATIC_SCRATCH_DOUBLES];

cudaError_t band_static_scratch(double **ptr) {
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static double *addr[MAX_DEV] = {};
    *ptr = nullptr;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEV) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_band_static_scratch);
        if (e != cudaSuccess) return e;
        addr[dev] = p;
    }
    *ptr = addr[dev];
    return cudaSuccess;
}

// scratch: band_static_scratch() of the current device; the caller has checked nb * S * bs.n <= BAND_STATIC_SCRATCH_DOUBLES.
// Launches the kernel only: no attribute call, no allocation (the XG instantiation needs under 9 KB of shared memory).
cudaError_t launch_band_solve_static(const BandSpace &bs, int nb, int S, size_t xstride, size_t pstride, const double *band,
                                     const double *rhs, double *x, double *scratch, cudaStream_t st) {
    if (!scratch || (size_t)nb * S * bs.n > BAND_STATIC_SCRATCH_DOUBLES) return cudaErrorInvalidValue;
    return launch_band_solve(bs, nb, S, xstride, pstride, band, rhs, x, scratch, st);
}

}  // namespace landau
