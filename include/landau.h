/*
 * landau.h -- C ABI of the B200-native Landau Jacobian hot path (arxiv 2104.10000).
 *
 * PAPER.md = the paper's text.  The library builds, on ONE sm_100a GPU and in fp64, the
 * frozen-coefficient Jacobian of the conservative finite-element Landau collision
 * operator (Eq. 2, weak form Eqs. 4-8) on a 2-D axisymmetric (r,z) velocity mesh with
 * S species, following Algorithm 1 (L109-131):
 *
 *   a1  f_b(q), grad f_b(q) at all N integration points                          (L101)
 *   a2  T_D(j) = sum_b e_b^2 f_b(j),  T_K(j) = sum_b e_b^2 (m0/m_b) grad f_b(j)  (lines 5-8, Eq. 10)
 *   a3  G_D(i) = sum_{j!=i} w_j T_D(j) U^D(i,j),  G_K(i) = sum_{j!=i} w_j U^K(i,j).T_K(j)
 *                                                                                 (lines 3-12)
 *   a4  K_a = nu e_a^2 (m0/m_a) G_K,  D_a = -nu e_a^2 (m0/m_a)^2 G_D;
 *       KK = J^-1 K_a w,  DD = J^-1 D_a J^-T w                                    (lines 13-20)
 *   a5  C_e[a][b] = sum_q ( Ehat_qa.DD_q.Ehat_qb + Ehat_qa.KK_q B_qb )           (line 23)
 *   a6  vals_a[k] = sum over (e,a,b) of P_e[a,row k] P_e[b,col k] C_e[a][b], fixed order
 *                                                                                 (L101, L165-167, L297)
 *   a7  C(f)_a[i] = sum_q w grad psi_i.(K_a f_a + D_a grad f_a)   (right side of Eq. 4, = J_a f_a)
 *   a8  mass: M[a][b] = shift sum_q w psi_a psi_b                                 (L280)
 *
 * U^D, U^K are Eq. 3 (L44) integrated over the azimuth (complete elliptic integrals K, E);
 * DESIGN.md "Readings" Q1 gives the formulas, Q2 the weights: w_in = omega detJ r in a3,
 * w = 2 pi omega detJ r in a4-a8.
 *
 * Discretisation conventions (part of the problem statement; the CPU oracle follows the same):
 *   - mesh: leaves of a quadtree forest on [rmin,rmax]x[zmin,zmax], nbr x nbz level-0 cells,
 *     2:1 FACE balanced, rmin >= 0.  Leaf (level l, ir, iz) covers
 *     r in rmin + hr0/2^l [ir,ir+1], z in zmin + hz0/2^l [iz,iz+1].
 *   - order p in {2,3}: tensor Lagrange elements on EQUISPACED nodes, (p+1)^2 Gauss-Legendre
 *     points; local basis a = az (p+1) + ar; point gi = e Nq + qz (p+1) + qr (abscissae ascending).
 *   - hanging nodes: nodes of a fine edge whose face neighbour is one level coarser and that do
 *     not coincide with a coarse node take the coarse edge's 1-D Lagrange interpolant; chains are
 *     closed.  Natural boundary conditions everywhere (nothing imposed at r = 0).
 *   - unknowns: per species, the n unconstrained nodes numbered by ascending (z, r) node
 *     coordinate; f, Cf are [S][n] species-major.
 *   - matrix: block diagonal I_S (x) A1 (L75); one CSR pattern A1 (rows in DOF order, columns
 *     ascending) and vals[S][nnz].
 *
 * General rules: every function returns 0 (LANDAU_OK) or a negative LANDAU_E* code and never
 * throws.  "dev" pointers are CUDA device pointers, "host" pointers plain host memory.  Device
 * entry points enqueue work on `stream` (a cudaStream_t passed as void*, NULL = default
 * stream) and do NOT synchronise; inputs are never modified; the CALLER owns f/vals/Cf/mvals,
 * the ctx owns pattern, gather lists, point arrays and scratch.  A ctx must not be used from two
 * streams at once (it owns one scratch arena).  There is no CPU fallback: without a CUDA device
 * landau_create fails with LANDAU_ECUDA.  The device entry points make no synchronising call and allocate
 * nothing, so a build can be captured in a CUDA graph; results are bitwise reproducible and a batched call
 * equals the same problems built one by one.
 *
 * Two ways through step a3 (the choice changes rounding only, never the sum that is computed):
 *   LANDAU_PAIR_PER_PROBLEM  every problem evaluates the tensor of every point pair itself (symmetric tile-pair
 *                            kernel, K and E in registers, ~75 flop per ordered pair and problem);
 *   LANDAU_PAIR_SHARED       the tensor depends on the mesh only, and all problems of a ctx share the mesh
 *                            (the paper's batching model, L244, L377): it is evaluated ONCE per ordered pair and
 *                            call into five N x N matrices, and G = U T for all problems is a dense fp64
 *                            contraction on the tensor cores (14 flop per ordered pair and problem).
 * A ctx uses ONE path for all its calls, so "batched == loop of singles, bitwise" holds inside a ctx.
 *
 * Beyond a1-a8: the operator of a fully implicit step in one pass (landau_implicit_operator_batched:
 * E-field advection of Eq. 4 and the shifted mass matrix added), several grids for species clustered by
 * thermal speed (landau_create_multigrid, section III-C), and the per-species batched band LU of section
 * III-G (landau_band_*), so that a Newton iteration can stay on the device.
 */
#ifndef LANDAU_H
#define LANDAU_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LANDAU_OK 0
#define LANDAU_EINVAL (-1) /* bad argument: order, S < 1, mass <= 0, rmin < 0, mesh not a 2:1 tiling, nb > max_batch */
#define LANDAU_ENOMEM (-2) /* host or device allocation failed */
#define LANDAU_ECUDA (-3)  /* CUDA runtime error; text via landau_last_cuda_error() */

#define LANDAU_PAIR_AUTO 0        /* landau_create's choice: SHARED when max_batch >= LANDAU_SHARED_MIN_BATCH and   */
#define LANDAU_PAIR_PER_PROBLEM 1 /* the tensor scratch (40 N^2 bytes) is at most a quarter of the free device      */
#define LANDAU_PAIR_SHARED 2      /* memory, else PER_PROBLEM                                                       */
#define LANDAU_SHARED_MIN_BATCH 4

typedef struct landau_ctx landau_ctx; /* opaque; owns all device + host state */

/* Quadtree-forest leaves (host memory, borrowed for the call). */
typedef struct {
    double rmin, rmax, zmin, zmax;
    int32_t nbr, nbz;       /* level-0 cells in r and z */
    int32_t ncells;         /* number of leaves */
    const int32_t *level;   /* [ncells] */
    const int32_t *ir, *iz; /* [ncells] integer coordinates at the leaf's own level */
} landau_mesh;

/* Species table (host, borrowed).  The operator uses mass, charge, m0, nu (Alg. 1 lines 5-16;
 * nu_ab = nu e_a^2 e_b^2, L83; Appendix A: nu = 1, m0 = m_e).  density/temperature are carried for
 * the harness's Maxwellian generator only and may be NULL. */
typedef struct {
    int32_t S;
    const double *mass, *charge, *density, *temperature; /* [S] */
    double m0, nu;
} landau_species;

/* Set-up, once per mesh: DOF numbering, constraint closure, CSR pattern, gather
 * lists, point arrays, tabulations; uploads them.  max_batch in [1, 65535] sizes the scratch arena for
 * landau_jacobian_batched and chooses the path through step a3 (LANDAU_PAIR_AUTO above).  Device scratch:
 *   per-problem path : chunk * (3 + 5 ceil(N/TS)) * N doubles, TS = 128 / 64 / 32 by N (max_batch < 4, a context for
 *                      single builds: 32 up to N = 8,192 -- more, shorter blocks balance one build over the SMs -- which
 *                      is why results of contexts with different max_batch may differ in the last bits); a batch is processed in groups
 *                      of chunk = min(max_batch, 1 GB / (40 ceil(N/TS) N bytes)) >= 1 problems: at most ~1 GB whatever
 *                      the batch (139 problems per group at N = 4,928)
 *   batch-shared path: 40 N^2 bytes for the tensor (0.97 GB at N = 4,928) + max_batch * 5 (1 + ksplit) N doubles
 * plus max_batch * S * Ne * Nb (Nb + 1) doubles of element matrices.  LANDAU_ENOMEM if it does not fit;
 * on failure *out is NULL. */
int landau_create(const landau_mesh *mesh, int order, const landau_species *species, int max_batch,
                  landau_ctx **out);
int landau_destroy(landau_ctx *ctx);

/* Several grids (section III-C, Table I): species clustered by thermal speed live on
 * separate meshes of one order; the inner integral of Eqs. 7-8 runs over the UNION of all grids'
 * integration points, each species contributing at the points of its own grid, and the Jacobian
 * block of a species has its grid's pattern.  meshes: [ngrids] host; species_grid: [S] host,
 * non-decreasing, every grid used (species are grouped by grid).  Per-problem layouts become
 *   f, Cf, F: [species][n of its grid]   vals: [species][nnz of its grid]   mvals: [grid][nnz of the grid]
 * with the sizes from landau_strides / landau_grid_sizes.  Points of different grids that coincide
 * exactly are treated like j = i (no contribution).  landau_create is the ngrids = 1 case. */
int landau_create_multigrid(const landau_mesh *meshes, int ngrids, const int32_t *species_grid, int order,
                            const landau_species *species, int max_batch, landau_ctx **out);
int landau_grid_count(const landau_ctx *ctx, int32_t *ngrids);
/* Per grid: its species count and first species, n, nnz, integration points, cells (any may be NULL). */
int landau_grid_sizes(const landau_ctx *ctx, int grid, int32_t *S_g, int32_t *first_species, int64_t *n,
                      int64_t *nnz, int64_t *N, int64_t *Ne);
/* Doubles per problem in f / Cf (f_stride) and vals (vals_stride), length of mvals, points of all grids. */
int landau_strides(const landau_ctx *ctx, int32_t *S, int64_t *f_stride, int64_t *vals_stride,
                   int64_t *mvals_size, int64_t *N_total);
int landau_grid_csr_pattern(const landau_ctx *ctx, int grid, const int32_t **rowptr_dev, const int32_t **colidx_dev);
int landau_grid_csr_pattern_host(const landau_ctx *ctx, int grid, int32_t *rowptr_host, int32_t *colidx_host);
int landau_grid_dof_coords(const landau_ctx *ctx, int grid, double *r_host, double *z_host);

/* The path through step a3 (see the top of this file).  landau_set_pair_path synchronises the device, frees the
 * scratch of the old path and allocates the new one (LANDAU_ENOMEM leaves the ctx without pair scratch: call it
 * again with a path that fits).  landau_pair_path reports the path in use and its scratch bytes (either may be
 * NULL).  landau_set_tensor_cache(on): batch-shared path only -- keep the tensor between calls instead of
 * evaluating it in every call (the geometry of a ctx never changes); default OFF, so that every call does the
 * whole of step a3. */
int landau_set_pair_path(landau_ctx *ctx, int path);
int landau_pair_path(const landau_ctx *ctx, int32_t *path, int64_t *scratch_bytes);
int landau_set_tensor_cache(landau_ctx *ctx, int on);

/* Host-only part of landau_create (no CUDA device needed): runs the same set-up and returns the
 * sizes and, where the pointer is not NULL, the CSR pattern of A1 (rowptr[n+1], colidx[nnz]) and
 * the unknowns' node coordinates ([n] each).  Call once with NULL arrays to get the sizes. */
int landau_setup_host(const landau_mesh *mesh, int order, int64_t *n, int64_t *nnz, int64_t *N,
                      int32_t *rowptr_host, int32_t *colidx_host, double *dof_r_host, double *dof_z_host);

/* Sizes: S species, n unknowns per species, nnz of A1, N integration points, Ne cells. */
int landau_sizes(const landau_ctx *ctx, int32_t *S, int64_t *n, int64_t *nnz, int64_t *N, int64_t *Ne);
/* Device pointers (owned by ctx) to the CSR pattern of A1: rowptr[n+1], colidx[nnz], int32. */
int landau_csr_pattern(const landau_ctx *ctx, const int32_t **rowptr_dev, const int32_t **colidx_dev);
/* Host copies of the pattern (rowptr_host[n+1], colidx_host[nnz]); either may be NULL. */
int landau_csr_pattern_host(const landau_ctx *ctx, int32_t *rowptr_host, int32_t *colidx_host);
/* Coordinates of the unknowns' nodes (host, [n] each) -- to build nodal f. */
int landau_dof_coords(const landau_ctx *ctx, double *r_host, double *z_host);
/* Integration points (host, [N] each; any may be NULL): r, z, inner weight omega detJ r. */
int landau_points(const landau_ctx *ctx, double *r_host, double *z_host, double *w_host);

/* Steps a1-a3 only: G[nb][5][N] = (G_D rr, G_D rz, G_D zz, G_K r, G_K z) for nb problems.
 * f_dev [nb][S][n].  Exposed so the O(N^2) kernel can be checked and timed alone. */
int landau_inner_integral(landau_ctx *ctx, int nb, const double *f_dev, double *G_dev, void *stream);

/* Steps a1-a7 for one problem: f_dev [S][n] -> vals_dev [S][nnz], Cf_dev [S][n].
 * vals_dev or Cf_dev may be NULL to skip that output. */
int landau_jacobian(landau_ctx *ctx, const double *f_dev, double *vals_dev, double *Cf_dev, void *stream);
/* The same for nb <= max_batch independent problems on the same mesh and species (PAPER.md L244,
 * L377): f_dev [nb][S][n] -> vals_dev [nb][S][nnz], Cf_dev [nb][S][n].  Bitwise equal to nb
 * single calls. */
int landau_jacobian_batched(landau_ctx *ctx, int nb, const double *f_dev, double *vals_dev,
                            double *Cf_dev, void *stream);
/* Step a8: mvals_dev [nnz] = shift * mass matrix on the pattern A1 (same for every species). */
int landau_mass(landau_ctx *ctx, double shift, double *mvals_dev, void *stream);

/* Everything a fully implicit step of Eq. 4 ("the mass matrix ... is added to the Jacobian
 * in all time integrators", L280) needs about the states f, in ONE pass (no source term):
 *   vals_dev [nb][S][nnz]:  shift * M + A_a(E_z[b]) - J_a(f_b)   on the pattern A1
 *   F_dev    [nb][S][n]  :  A_a(E_z[b]) f_a - C_a(f_b)           (the residual without the d/dt term)
 * A_a[i][j] = (e_a m0/m_a) E_z sum_q w psi_i d(psi_j)/dz is the E-field advection term on the left of
 * Eq. 4 (charges in e, masses in m0, E_z in the units of Appendix A).  Ez_dev: [nb] device
 * doubles, one field per problem.  vals_dev or F_dev may be NULL.  Same set-up, pair kernel, ordering
 * and determinism as landau_jacobian_batched. */
int landau_implicit_operator_batched(landau_ctx *ctx, int nb, const double *f_dev, const double *Ez_dev,
                                     double shift, double *vals_dev, double *F_dev, void *stream);

/* Per-species batched band LU (section III-G): reverse Cuthill-McKee ordering of the
 * pattern (computed in landau_create; RCM's result depends on its starting node, so it is run from a
 * pseudo-peripheral node, from the unknowns at the corners of the domain and from the one nearest the origin,
 * the plain (z, r) sweep is a candidate too, and among the orders within 10 % of the narrowest band the one with
 * the least envelope work is kept), band storage, Gaussian elimination WITHOUT pivoting in outer-product
 * form (Golub & Van Loan Alg. 4.3.1, the paper's algorithm; blocked), one independent matrix per (problem,
 * species).  Meant for the matrices of landau_implicit_operator_batched (shift M + A - J); like the paper's
 * solver it does not pivot.  Breakdown is REPORTED, not repaired: pivots_dev (NULL, or [nb][S][2] device doubles)
 * receives for every matrix the smallest and the largest |pivot| met; a zero, NaN or infinite pivot gives
 * smallest = 0 (the factors and any solve with them are then meaningless), a tiny ratio smallest / largest
 * tells that elimination without pivoting was unstable for that matrix.
 * landau_band_sizes: per grid the half-bandwidth of the chosen order and the doubles one matrix occupies; the
 * doubles of workspace per problem (all species of all grids); and the flop of the outer-product updates of
 * one factorisation (they are confined to the envelope of the ordered pattern, which elimination without
 * pivoting does not leave: about half of 2 n bw^2 on the refined meshes).  band_dev: caller-owned workspace of
 * nb * workspace_doubles_per_problem doubles, problem-major: problem b owns the doubles
 * [b * workspace_doubles_per_problem, (b + 1) * workspace_doubles_per_problem), so a solve may address the first
 * nb' <= nb problems of an earlier factorisation; the layout inside a problem belongs to the library.
 * landau_band_factor_batched: vals_dev [nb][vals_stride] (CSR values, layout of landau_jacobian_batched)
 *   -> factors in band_dev.
 * landau_band_solve_batched: rhs_dev, x_dev [nb][f_stride] (layout of f); x = A^-1 rhs per species block;
 *   x_dev may equal rhs_dev.  Both are asynchronous on `stream` and deterministic.  The solve keeps the vector of a
 *   matrix in shared memory up to n ~ 28,000 unknowns; beyond that it works in a ctx-owned device scratch of
 *   max_batch * S * n doubles, allocated (synchronously) by the first such call. */
/* Host-only (no CUDA device needed): the band order landau_create chooses for this mesh and order --
 * perm_host[n] (new index -> unknown), the half-bandwidth it gives, the block width the factorisation will
 * use and the flop of its outer-product updates inside the envelope.  Any output may be NULL.
 * Block widths: 16 columns up to a half-bandwidth of 256, 32 up to 384, 16 up to 832, 8 beyond (the panels of a step
 * must fit shared memory); in the 32-column range the FACTORISATION takes 16-column blocks instead when the envelope is
 * jagged and the window of its largest front fits the shared memory of an SM (the slot kernel below), while the solves
 * keep 32: L and U do not depend on the blocking. */
int landau_band_order_host(const landau_mesh *mesh, int order, int32_t *perm_host, int32_t *half_bandwidth,
                           int32_t *block_columns, double *flop_per_factorization);
int landau_band_sizes(const landau_ctx *ctx, int grid, int32_t *half_bandwidth, int64_t *doubles_per_matrix,
                      int64_t *workspace_doubles_per_problem, double *flop_per_factorization);
/* Two kernels factor the band, with the same storage and the same L, U up to rounding order:
 *   LANDAU_BAND_FRONT  gathers, per block step, only the rows / columns inside the ENVELOPE of the ordered pattern (LU
 *                      without pivoting keeps it; on the refined meshes a third of the rows a band step spans) into a
 *                      dense front in shared memory, eliminates there and scatters back (32-column blocks), or keeps the
 *                      front in shared memory for its whole life, every active row in a fixed slot (16-column blocks);
 *   LANDAU_BAND_HULL   updates the whole window of a block step in place (the monotone hull of the envelope).
 * LANDAU_BAND_AUTO (the default) takes the front kernel whenever the largest front fits the shared memory of an SM.
 * landau_band_set_method returns LANDAU_EINVAL for LANDAU_BAND_FRONT when it does not fit; landau_band_method reports
 * the kernel in use for a grid, the longest active list (rows of the largest front beside its block) and the flop of
 * the window updates of one factorisation by that kernel.  Outputs may be NULL. */
#define LANDAU_BAND_AUTO 0
#define LANDAU_BAND_HULL 1
#define LANDAU_BAND_FRONT 2
/* Host-only: for the band order of this mesh, the rows of the largest front beside its block, the flop of the front
 * kernel's window updates (compare landau_band_order_host's flop: the hull kernel's) and whether the largest front
 * fits shared memory.  Any output may be NULL. */
int landau_band_front_host(const landau_mesh *mesh, int order, int32_t *front_rows_max, double *front_flop, int32_t *fits);
int landau_band_set_method(landau_ctx *ctx, int method);
int landau_band_method(const landau_ctx *ctx, int grid, int32_t *method, int32_t *front_rows_max, double *flop_per_factorization);
int landau_band_factor_batched(landau_ctx *ctx, int nb, const double *vals_dev, double *band_dev, double *pivots_dev,
                               void *stream);
int landau_band_solve_batched(landau_ctx *ctx, int nb, const double *band_dev, const double *rhs_dev, double *x_dev,
                              void *stream);

/* landau_band_solve_batched WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (code under CUDA-graph
 * stream capture, tight serving loops, harnesses that forbid it): same arguments, same factors, same solution up to
 * rounding (section III-G: the L and U solves of the band solver).  The permuted vectors of the nb * S matrices
 * live in a scratch that is part of the library image -- a file-scope __device__ array of
 * LANDAU_STATIC_SCRATCH_DOUBLES doubles (32 MiB), held by every GPU that loads the library until the process exits --
 * instead of shared memory or the lazily cudaMalloc'ed scratch of landau_band_solve_batched.  Its device address is taken
 * once per device at landau_create (cudaGetSymbolAddress with that device current); the call itself launches one kernel
 * per grid on `stream` and calls no cudaMalloc, cudaFree, attribute setter or synchronising routine.
 * Limit: nb * S_g * n_g <= LANDAU_STATIC_SCRATCH_DOUBLES for every grid g (S_g species, n_g unknowns), otherwise
 * LANDAU_EINVAL with the sizes in landau_last_cuda_error() and nothing launched; LANDAU_ECUDA when the ctx's device is not
 * the current one.  All ctx and all calls on a device SHARE the array: it keeps the last call's contents (nothing in it
 * has to start at zero: a call writes the part it reads), and two such solves that overlap on the GPU -- different
 * streams, or graphs replayed concurrently -- race; calls on one stream are safe.  x_dev may equal rhs_dev. */
#define LANDAU_STATIC_SCRATCH_DOUBLES (4u << 20)
int landau_band_solve_static(landau_ctx *ctx, int nb, const double *band_dev, const double *rhs_dev, double *x_dev,
                             void *stream);

/* End-to-end variant with HOST buffers (pageable or pinned): copies f to the device, runs
 * landau_jacobian_batched on the ctx's own stream in sub-batches whose device-to-host copies overlap
 * the next sub-batch's build, and synchronises.  Values are bitwise those of the device entry point. */
int landau_jacobian_host(landau_ctx *ctx, int nb, const double *f_host, double *vals_host, double *Cf_host);

/* Number of kernel launches the ctx has enqueued since creation (for bench.py's gpu_launches). */
int landau_launch_count(const landau_ctx *ctx, int64_t *count);

/* Measurement aid: when enabled, the kernels of step a3 are bracketed by CUDA events on their own stream.
 * landau_profile_read synchronises those events and returns, since the last read, the summed device time (ms)
 * and the number of bracketed launches of
 *   [0] the tensor evaluation: per-problem path k_pair_sym (evaluation and accumulation in one kernel),
 *       batch-shared path k_pair_tensor;
 *   [1] the batch-shared path's contraction k_apply_dmma (0 on the per-problem path);
 * ms_total and launches are arrays of 2.  Resets both. */
int landau_profile_enable(landau_ctx *ctx, int on);
int landau_profile_read(landau_ctx *ctx, double *ms_total, int64_t *launches);

/* Measurement aid, not part of the operator: runs a register-resident chain of dependent-free
 * DFMA on every SM for `iters` iterations and returns the achieved FP64 rate in flop/s (the
 * "alu" roofline denominator).  Synchronises. */
int landau_fp64_peak_probe(int iters, double *flops_per_s, double *sm_clock_mhz_est);

/* Measurement aid, not part of the operator: FP64 issue-rate micro-benchmarks (the figures behind the "issue
 * bound" of DESIGN.md).  Register-resident streams on every SM, three warps per SM sub-partition (one for mode 4),
 * timed with clock64() on the SM.  mode: 0 DFMA with two register operands + immediate; 1 DFMA with two distinct
 * registers; 2 DFMA with three distinct registers; 3 DFMA with three registers of which one is shared by
 * consecutive instructions; 4 one dependent DFMA chain (latency); 5 DMMA m8n8k4 with independent accumulators;
 * 6 / 7 as 0 with one / two independent integer multiply-adds beside every DFMA (cycles are still per DFMA: do
 * the other pipes issue in the shadow of the FP64 issue?).
 * Returns SM cycles per (FP64) warp instruction and sub-partition, and (flops_per_s may be NULL) the whole-GPU rate by
 * wall clock (CUDA events).  Synchronises. */
int landau_fp64_issue_probe(int mode, int iters, double *cycles_per_warp_instruction, double *flops_per_s);

const char *landau_strerror(int code);
const char *landau_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LANDAU_H */
