// Launchers of the device kernels (landau_kernels.cu); called by the C-ABI layer only.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <vector>

namespace landau {

constexpr int MAX_SPECIES = 16;

// Device-resident description of one mesh/order/species set (all pointers device memory,
// shared by every problem of a batch).
// First item (weight, source index) of a gather list: read with the list bounds, not after them, so that the
// source value of the (usual) one-item list is two dependent loads away instead of three.
struct GatherHead { double w; int32_t idx; int32_t pad; };

struct DeviceSpace {
    int p, Nq, Nb, S;                            // S = species living on this grid
    int N, Ne, n, nnz;
    // several grids (section III-C): the point-indexed scratch arrays T, G cover the union of
    // all grids' points (Ntot), this grid's points start at poff; f of problem b starts at f + b*fstride
    // (f already offset to this grid's first species)
    int Ntot, poff;
    long long fstride;
    const double *r, *z, *invr, *w_in, *w_out;  // [N]
    const double *invJ;                          // [Ne][2]
    const double *Me, *Ae;                       // Q3 only, [Ne][16][16]: sum_q w_q B_qa B_qb and sum_q w_q (2/hz) B_qa E1_qb (k_element_q3<true>)
    const double *B, *E0, *E1;                   // [Nq][Nb]
    const int32_t *lptr, *ldof; const double *lw;
    const int32_t *rowptr, *colidx;
    const int32_t *gptr, *gidx; const double *gw;
    const int32_t *cptr, *cidx; const double *cw;
    const GatherHead *ghead, *chead, *lhead; // first item of every list, one 16-byte word per output (k_gather) / local node (k_fields_beta)
    double e2[MAX_SPECIES];    // e_b^2
    double m0m[MAX_SPECIES];   // m0/m_b
    double kfac[MAX_SPECIES];  // nu e_a^2 (m0/m_a)
    double dfac[MAX_SPECIES];  // -nu e_a^2 (m0/m_a)^2
    double qm[MAX_SPECIES];    // e_a m0/m_a (E-field advection, Eq. 4)
};

// Scratch for up to max_batch problems (N = points of all grids together).
struct Scratch {
    double *T;      // per-problem path: [nb][3][N]; batch-shared path: [3][Kpad/8][nbpad][8]
    double *G;      // per-problem path: [nb][ntiles][5][N] per source tile partial sums of G_D, G_K;
                    // batch-shared path: [nb][ksplit][5][N]
    double *Gsum;   // [nb][5][N]: G_D (rr,rz,zz), G_K (r,z) after the tile-order sum
    double *U;      // batch-shared path: [5][Kpad/8][Mpad][8] tensor entries of all ordered pairs
};

// each returns the number of kernels launched
int launch_fields_beta(const DeviceSpace &ds, int nb, const double *f, double *T, double *u, cudaStream_t st);

// Batch-shared path (landau_shared.cu): the tensor of every ordered pair is evaluated once per call into
// U[5][Kpad/8][Mpad][8] and applied to all problems by an fp64 tensor-core contraction with T[3][Kpad/8][nbpad][8].
int shared_kpad(int N);      // 16 ceil(N/16): source points padded to whole chunks
int shared_mpad(int N);      // target points padded to whole tiles
int shared_nbpad(int nb);    // problems padded to whole tiles
int shared_ksplit(int N);    // segments of the j range (a function of N only: fixes the summation order)
int launch_fields_beta_tiled(const DeviceSpace &ds, int nb, int nbpad, const double *f, double *T, double *u, cudaStream_t st);
int launch_pair_tensor(int N, const double *r, const double *z, const double *invr, double *U, cudaStream_t st);
// Gpart[b][ksplit][5][N]
int launch_apply(int N, int nb, int nbpad, const double *U, const double *T, double *Gpart, cudaStream_t st);
// pair kernel over the union of points (r, z, invr: [Ntot]); check_all: test every pair for coincidence
// (needed only when points of different grids coincide), else only the diagonal tiles
// latency: the tiling policy of the context (pair_tile_size)
int launch_pair(int Ntot, bool latency, const double *r, const double *z, const double *invr, bool check_all, int nb, const double *T,
                double *Gpart, cudaStream_t st);
// Ez == nullptr: collision Jacobian C_e; else the implicit-step operator shift M + A_E - J (Ez[nb] device)
int launch_element(const DeviceSpace &ds, int nb, int jsplit, const double *f, const double *G, double *Ce,
                   double *ce, const double *Ez, double shift, cudaStream_t st);
// vals / Cf already offset to this grid's first species; ostride = doubles per problem in the output;
// nspecies = 1 with ostride 0 gathers a single matrix (mass)
int launch_gather_vals(const DeviceSpace &ds, int nb, int nspecies, size_t ostride, const double *Ce, double *vals, cudaStream_t st);
int launch_gather_cf(const DeviceSpace &ds, int nb, size_t ostride, const double *ce, double *Cf, cudaStream_t st);
int launch_gather_both(const DeviceSpace &ds, int nb, size_t vstride, size_t fstride, const double *Ce, const double *ce,
                       double *vals, double *Cf, cudaStream_t st);
int launch_mass_element(const DeviceSpace &ds, double shift, double *Ce, cudaStream_t st);
int launch_sum_partials(int Ntot, int nb, int jsplit, bool latency, const double *Gpart, double *G, cudaStream_t st);
int launch_dfma_probe(int blocks, int threads, int iters, double *out, cudaStream_t st);
int launch_issue_probe(int mode, int blocks, int threads, int iters, const double *in, double *out, long long *cycles, cudaStream_t st);

// Band LU (landau_band.cu; section III-G)
struct BandSpace {
    int n, nnz, bw;            // order, CSR entries, half-bandwidth after RCM
    int kb, W;                 // columns per block step of the factorisation (the solves: band_block(bw)); stored half-width
    size_t mat_doubles;        // (2 W + 1) * n doubles per matrix
    const int32_t *perm;       // [n] device: new -> old
    // fill lists per band column (new numbering): the rows of the column inside the region the factorisation and the
    // solves touch (zeroed: zlo = offset of the first one inside the column, zcnt of them), and the CSR entries of the
    // column (fsrc = index into the species' CSR values, foff = offset inside the column), fptr[n + 1]
    const int32_t *zlo, *zcnt, *fptr, *fsrc, *foff;
    // front (envelope) factorisation: per block step the rows / columns that elimination can reach -- the next block's,
    // then every later row whose envelope starts at or before the block (ascending) -- act_ptr[steps + 1], act_idx;
    // na_max = the longest list; front = true when the front of every step fits shared memory
    const int32_t *act_ptr, *act_idx;
    int na_max;
    double front_flop;         // window-update flop of one factorisation by the front kernel (2 KB sum na_s^2)
    bool front;
    // slot kernel (band_slot_lists): slot of every list entry, entering rows per step, load list of the entering rows
    const int32_t *act_slot, *slot_hi, *new_ptr, *new_pos, *ld_ptr, *ld_dst, *ld_csr;   // slot_hi[s]: slots in use at step s are below it
    const int32_t *d0_csr;            // CSR indices of the first diagonal block
    bool slot;
    const int32_t *mlow, *mup; // [ceil(n/kb)] device: rows below / above block step s inside the envelope
    const int32_t *mlow_s, *mup_s;   // the same for the solves' block steps of band_block(bw) columns (= mlow, mup when kb is that)
    const int32_t *first;      // [n] device: first column of row i = first row of column i in the ordered pattern
    double flop_per_matrix;    // 2 KB sum mlow^2: window-update flop of one factorisation
};
// order of the band LU: the cheapest (envelope work) of RCM from several starting nodes and the (z, r) sweep
void rcm_order(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const double *dof_r, const double *dof_z,
               std::vector<int32_t> &perm, int &bw);
// half-bandwidth, per-block-step reach inside the envelope (mlow, mup; may be null) and window-update flop of an order
double band_envelope(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const std::vector<int32_t> &perm,
                     int &bw, std::vector<int32_t> *mlow, std::vector<int32_t> *mup, int KB = 0);     // KB = 0: band_block(bw)
int band_block(int bw);        // columns per block step, a function of bw only: the solves', and the factorisation's unless
                               // band_factor_block() finds that narrower blocks pay
int band_stored_halfwidth(int bw);   // W: the band stores 2 W + 1 diagonals (bw + KB, at least 2 KB - 1, rounded up to even; KB = band_block(bw))
size_t band_factor_smem(int bw, int KB);
// band points at this grid's block of problem 0; matrix (problem b, species s) = band + b pstride + s mat_doubles
// (problem-major workspace: a solve may use a different nb than the factorisation)
void band_fill_lists(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const std::vector<int32_t> &perm,
                     int W, int KB, const std::vector<int32_t> &mlow, const std::vector<int32_t> &mup, int KBs,
                     const std::vector<int32_t> &mlow_s, const std::vector<int32_t> &mup_s, std::vector<int32_t> &zlo,
                     std::vector<int32_t> &zcnt, std::vector<int32_t> &fptr, std::vector<int32_t> &fsrc, std::vector<int32_t> &foff);
// active lists of the front factorisation (see BandSpace); returns the longest list
int band_active_lists(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const std::vector<int32_t> &perm,
                      int KB, std::vector<int32_t> &act_ptr, std::vector<int32_t> &act_idx, double *front_flop);
void band_slot_lists(int n, const std::vector<int32_t> &rowptr, const std::vector<int32_t> &colidx, const std::vector<int32_t> &perm,
                     int KB, int ldp, int ldw, const std::vector<int32_t> &act_ptr, const std::vector<int32_t> &act_idx, int na_max,
                     std::vector<int32_t> &act_slot, std::vector<int32_t> &slot_hi, std::vector<int32_t> &new_ptr, std::vector<int32_t> &new_pos,
                     std::vector<int32_t> &ld_ptr, std::vector<int32_t> &ld_dst, std::vector<int32_t> &ld_csr, std::vector<int32_t> &d0_csr);
int band_front_ldw(int na_max);
int band_front_ldp(int na_max);
size_t band_slot_smem(int KB, int na_max);
size_t band_front_smem(int KB, int na_max);     // dynamic shared memory of the front kernel
cudaError_t launch_band_fill(const BandSpace &bs, int nb, int S, size_t vstride, size_t pstride, const double *vals, double *band,
                             cudaStream_t st);
// pivots: nullptr or (min |pivot|, max |pivot|) of matrix (b, s) at pivots[2 (b pivS + s)]
// vals: this grid's CSR values of problem 0, species s of problem b at vals + b vstride + s nnz (read by the slot kernel)
bool band_needs_fill(const BandSpace &bs);      // false: the factorisation reads the CSR values itself (slot kernel)
cudaError_t launch_band_factor(const BandSpace &bs, int nmat, int S, size_t pstride, const double *vals, size_t vstride, double *band,
                               double *pivots, int pivS, cudaStream_t st);
// xg: nullptr, or scratch of nb * S * n doubles for the permuted vectors when band_solve_smem(n, bw) exceeds an SM
size_t band_solve_smem(int n, int bw);
cudaError_t launch_band_solve(const BandSpace &bs, int nb, int S, size_t xstride, size_t pstride, const double *band, const double *rhs,
                              double *x, double *xg, cudaStream_t st);

// Band solve with its vectors in a scratch that belongs to the library image (file-scope __device__ array in
// landau_band.cu; 32 MiB per GPU that loads the library): nothing is allocated.
constexpr size_t BAND_STATIC_SCRATCH_DOUBLES = size_t(4) << 20;
cudaError_t band_static_scratch(double **ptr);      // its device address on the CURRENT device (cudaGetSymbolAddress, once per device)
cudaError_t launch_band_solve_static(const BandSpace &bs, int nb, int S, size_t xstride, size_t pstride, const double *band,
                                     const double *rhs, double *x, double *scratch, cudaStream_t st);

int pair_tile_size(int N, bool latency);
int pair_tiles(int N, bool latency);

}  // namespace landau
