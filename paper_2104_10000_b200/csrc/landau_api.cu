// C-ABI layer (include/landau.h): context management, argument checking, kernel sequencing.
// Every step of the path runs in landau_kernels.cu; there is no CPU fallback.
//
// A context holds one or several grids (section III-C: species clustered by thermal speed on
// separate meshes).  Species are grouped by grid in ascending order, so the per-problem layouts are
//   f, Cf:  [species][n of its grid]      vals: [species][nnz of its grid]
// i.e. grid-major blocks [S_g][n_g]; with one grid these are the plain [S][n] / [S][nnz].
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <numeric>
#include <string>
#include <vector>

#include "landau.h"
#include "landau_internal.h"
#include "landau_kernels.h"
#include "landau_launch.cuh"

using namespace landau;

namespace {
thread_local std::string g_cuda_err;

int cuda_fail(cudaError_t e, const char *what) {
    g_cuda_err = std::string(what) + ": " + cudaGetErrorString(e);
    return LANDAU_ECUDA;
}
#define CK(call)                                             \
    do {                                                     \
        cudaError_t e_ = (call);                             \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);  \
    } while (0)

// end of a chain of launches: the first failed cudaLaunchKernelEx of the chain, then the sticky error state
int launches_ok() {
    cudaError_t e = take_launch_error();
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(e, "kernel launch"); }
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "kernel launch (cudaGetLastError)");
    return LANDAU_OK;
}

// No exception crosses the C ABI: every entry point that can allocate on the host runs its body through this.
template <class F>
int guarded(F &&body) {
    try {
        return body();
    } catch (const std::bad_alloc &) {
        return LANDAU_ENOMEM;
    } catch (...) {
        g_cuda_err = "unexpected C++ exception";
        return LANDAU_EINVAL;
    }
}

template <class T>
int upload(const std::vector<T> &v, const T **out, std::vector<void *> &owned) {
    void *d = nullptr;
    size_t bytes = v.size() * sizeof(T);
    cudaError_t e = cudaMalloc(&d, bytes ? bytes : sizeof(T));
    if (e != cudaSuccess) { g_cuda_err = std::string("cudaMalloc: ") + cudaGetErrorString(e); return e == cudaErrorMemoryAllocation ? LANDAU_ENOMEM : LANDAU_ECUDA; }
    owned.push_back(d);
    if (bytes) CK(cudaMemcpy(d, v.data(), bytes, cudaMemcpyHostToDevice));
    *out = static_cast<const T *>(d);
    return LANDAU_OK;
}

struct ProfEvent { cudaEvent_t a = nullptr, b = nullptr; int kind = 0; };

struct GridState {
    HostSpace hs;
    DeviceSpace ds;
    int s0 = 0;              // first species of this grid
    size_t foff = 0;         // offset (doubles) of this grid's block inside one problem's f / Cf
    size_t voff = 0;         // ... inside one problem's vals
    size_t moff = 0;         // ... inside mvals
    BandSpace bs;            // band LU of this grid's pattern (RCM order)
    size_t boff = 0;         // offset (doubles) of this grid's matrices inside one problem's band workspace
    double *Ce = nullptr;    // [nb][S_g][Ne][Nb*Nb]
    double *ce = nullptr;    // [nb][S_g][Ne][Nb]
    double *solve_x = nullptr;   // band solve: permuted vectors of orders too large for shared memory (lazy)
    bool front_fits = false;     // the fronts of the envelope factorisation fit shared memory
};
}  // namespace

struct landau_ctx {
    std::vector<GridState> grids;
    int S = 0;                       // all species
    int64_t Ntot = 0;                // integration points of all grids
    size_t fstride = 0, vstride = 0, mstride = 0;   // doubles per problem in f / vals; in mvals
    size_t bstride = 0;                              // doubles per problem in the band-LU workspace
    const double *r = nullptr, *z = nullptr, *invr = nullptr;   // [Ntot] union of the grids' points
    bool check_all = false;          // points of different grids coincide somewhere
    Scratch sc = {};
    std::vector<void *> owned;       // device allocations that live as long as the ctx
    std::vector<void *> pair_owned;  // scratch of the current pair path (T, G, U): replaced by landau_set_pair_path
    int pair_path = LANDAU_PAIR_PER_PROBLEM;   // resolved path (never LANDAU_PAIR_AUTO)
    int nbpad = 0;                   // batch-shared path: problems padded to whole tiles
    int pp_chunk = 1;                // per-problem path: problems per group (their slabs stay in L2)
    bool latency_tiles = false;      // per-problem path: short tiles (context made for single builds, max_batch < LANDAU_SHARED_MIN_BATCH)
    bool tensor_cache = false;       // keep U between calls (the geometry of a ctx never changes)
    bool tensor_valid = false;
    int max_batch = 1;
    int num_sms = 148;
    int64_t launches = 0;
    cudaStream_t own_stream = nullptr, copy_stream = nullptr;
    cudaEvent_t chunk_done = nullptr;
    cudaStream_t side_stream = nullptr;              // batch-shared path: the tensor evaluation runs beside a1 + a2
    cudaEvent_t side_fork = nullptr, side_join = nullptr;
    double *d_f = nullptr, *d_vals = nullptr, *d_Cf = nullptr;  // landau_jacobian_host staging
    int host_nb = 0;
    bool profiling = false;
    std::vector<ProfEvent> prof_events;  // recorded, not yet read
    std::vector<ProfEvent> prof_pool;    // free
    int device = -1;                     // the device current at landau_create
    double *static_scratch = nullptr;    // landau_band_solve_static: address of the library's __device__ scratch on that device
};

namespace {
// launch_pair bracketed by events when profiling is on
// Step a3 bracketed by events when profiling is on.  Per-problem path: the pair kernel; batch-shared path: the
// tensor evaluation (unless cached) and the contraction -- kind 0 / 1 in landau_profile_read.
template <class F>
int timed(landau_ctx *ctx, int kind, cudaStream_t st, F &&go) {
    if (!ctx->profiling) return go();
    ProfEvent ev;
    if (!ctx->prof_pool.empty()) { ev = ctx->prof_pool.back(); ctx->prof_pool.pop_back(); }
    else {
        cudaError_t e = cudaEventCreate(&ev.a);
        if (e == cudaSuccess) e = cudaEventCreate(&ev.b);
        if (e != cudaSuccess) { note_launch_error(e); return go(); }
    }
    ev.kind = kind;
    note_launch_error(cudaEventRecord(ev.a, st));
    const int k = go();
    note_launch_error(cudaEventRecord(ev.b, st));
    ctx->prof_events.push_back(ev);
    return k;
}

// a1-a3 for nb problems.  Per-problem path: fields + beta sums per grid, pair kernel over the union, tile-order
// sum.  Batch-shared path: fields into the tiled T, the tensor of every ordered pair ONCE (reuse_tensor: already
// done by this call for an earlier sub-batch), the fp64 tensor-core contraction, split-order sum.
void inner_integral(landau_ctx *ctx, int nb, const double *f_dev, double *Gsum, cudaStream_t st, bool reuse_tensor = false) {
    const int N = int(ctx->Ntot);
    if (ctx->pair_path == LANDAU_PAIR_SHARED) {
        const bool eval_tensor = !(reuse_tensor || (ctx->tensor_cache && ctx->tensor_valid));
        // The tensor depends on the geometry only and a1 + a2 on f only: for a large batch the two run side by side
        // (fork / join through events, legal under stream capture too); k_fields_beta is latency-bound and leaves
        // the FP64 pipes and the memory system to k_pair_tensor.
        bool forked = false;
        if (eval_tensor && nb > PDL_MAX_NB) {
            if (!ctx->side_stream) {
                cudaError_t e = cudaStreamCreateWithFlags(&ctx->side_stream, cudaStreamNonBlocking);
                if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->side_fork, cudaEventDisableTiming);
                if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->side_join, cudaEventDisableTiming);
                if (e != cudaSuccess) { note_launch_error(e); return; }
            }
            note_launch_error(cudaEventRecord(ctx->side_fork, st));          // after every earlier user of U on st
            note_launch_error(cudaStreamWaitEvent(ctx->side_stream, ctx->side_fork, 0));
            cudaStream_t ss = ctx->side_stream;
            ctx->launches += timed(ctx, 0, ss, [&]() { return launch_pair_tensor(N, ctx->r, ctx->z, ctx->invr, ctx->sc.U, ss); });
            note_launch_error(cudaEventRecord(ctx->side_join, ss));
            ctx->tensor_valid = true;
            forked = true;
        }
        for (auto &g : ctx->grids) ctx->launches += launch_fields_beta_tiled(g.ds, nb, ctx->nbpad, f_dev + g.foff, ctx->sc.T, g.ce, st);
        if (forked) note_launch_error(cudaStreamWaitEvent(st, ctx->side_join, 0));
        else if (eval_tensor) {
            ctx->launches += timed(ctx, 0, st, [&]() { return launch_pair_tensor(N, ctx->r, ctx->z, ctx->invr, ctx->sc.U, st); });
            ctx->tensor_valid = true;
        }
        const int ksplit = shared_ksplit(N);
        ctx->launches += timed(ctx, 1, st, [&]() { return launch_apply(N, nb, ctx->nbpad, ctx->sc.U, ctx->sc.T, ksplit > 1 ? ctx->sc.G : Gsum, st); });
        if (ksplit > 1) ctx->launches += launch_sum_partials(N, nb, ksplit, false, ctx->sc.G, Gsum, st);
        return;
    }
    // Per-problem path: a group of pp_chunk problems at a time, so that the per-source-tile slabs (ntiles * 5 N doubles
    // per problem) do not grow with the batch (at most PP_SLAB_BYTES of scratch; groups are large enough that the
    // last wave of a launch costs < 1 %).  Problems are independent: the grouping changes no value.
    for (int b0 = 0; b0 < nb; b0 += ctx->pp_chunk) {
        const int nbc = std::min(ctx->pp_chunk, nb - b0);
        const double *fc = f_dev + size_t(b0) * ctx->fstride;
        for (auto &g : ctx->grids) ctx->launches += launch_fields_beta(g.ds, nbc, fc + g.foff, ctx->sc.T, g.ce + size_t(b0) * g.ds.S * g.ds.Ne * g.ds.Nb, st);
        ctx->launches += timed(ctx, 0, st, [&]() { return launch_pair(N, ctx->latency_tiles, ctx->r, ctx->z, ctx->invr, ctx->check_all, nbc, ctx->sc.T, ctx->sc.G, st); });
        ctx->launches += launch_sum_partials(N, nbc, pair_tiles(N, ctx->latency_tiles), ctx->latency_tiles, ctx->sc.G, Gsum + size_t(b0) * 5 * N, st);
    }
}

void free_pair_scratch(landau_ctx *ctx) {
    for (void *p : ctx->pair_owned) cudaFree(p);
    ctx->pair_owned.clear();
    ctx->sc.T = ctx->sc.G = ctx->sc.U = nullptr;
    ctx->tensor_valid = false;
}

// Problems per group on the per-problem path: as many as keep the group's slabs within PP_SLAB_BYTES, at least one.
// (Groups small enough for the slabs to stay in L2, 32 MB, were measured: the partial last wave of every pair-kernel
// launch then costs more than the DRAM round trip of the slabs saves.)
constexpr size_t PP_SLAB_BYTES = size_t(1) << 30;
int pp_chunk_size(int max_batch, int64_t N, bool latency) {
    const size_t per_problem = size_t(pair_tiles(int(N), latency)) * 5 * size_t(N) * sizeof(double);
    return int(std::max<size_t>(1, std::min<size_t>(size_t(max_batch), PP_SLAB_BYTES / std::max<size_t>(per_problem, 1))));
}

// Bytes of U, the tensor entries of all ordered pairs (batch-shared path).
size_t tensor_bytes(int64_t N) { return size_t(5) * (shared_kpad(int(N)) / 8) * shared_mpad(int(N)) * 8 * sizeof(double); }

// Scratch of the pair path (sized for max_batch):
//   per problem : T [chunk][3][N], G [chunk][ntiles][5][N] for a group of `chunk` problems (slabs of a group <= 1 GB)
//   batch-shared: T [3][Kpad/8][nbpad][8], U [5][Kpad/8][Mpad][8] (5 N^2 doubles: 0.97 GB for N = 4,928, independent
//                 of the batch), G [nb][ksplit][5][N]; T and U are zeroed once: their padding must stay zero
int alloc_pair_scratch(landau_ctx *ctx, int path) {
    free_pair_scratch(ctx);
    const size_t nbm = size_t(ctx->max_batch), N = size_t(ctx->Ntot);
    struct Alloc { double **p; size_t n; bool zero; };
    std::vector<Alloc> allocs;
    if (path == LANDAU_PAIR_SHARED) {
        ctx->nbpad = shared_nbpad(ctx->max_batch);
        const size_t Kq8 = size_t(shared_kpad(int(N)) / 8);
        allocs = {{&ctx->sc.T, 3 * Kq8 * ctx->nbpad * 8, true},
                  {&ctx->sc.U, tensor_bytes(int64_t(N)) / sizeof(double), true},
                  {&ctx->sc.G, shared_ksplit(int(N)) > 1 ? nbm * shared_ksplit(int(N)) * 5 * N : 0, false}};
    } else {
        ctx->pp_chunk = pp_chunk_size(ctx->max_batch, int64_t(N), ctx->latency_tiles);
        const size_t nbc = size_t(ctx->pp_chunk);
        allocs = {{&ctx->sc.T, nbc * 3 * N, false}, {&ctx->sc.G, nbc * pair_tiles(int(N), ctx->latency_tiles) * 5 * N, false}};
    }
    for (auto &a : allocs) {
        if (!a.n) continue;
        void *d = nullptr;
        cudaError_t e = cudaMalloc(&d, a.n * sizeof(double));
        if (e != cudaSuccess) {
            g_cuda_err = std::string("cudaMalloc(pair scratch): ") + cudaGetErrorString(e);
            cudaGetLastError();
            free_pair_scratch(ctx);
            return e == cudaErrorMemoryAllocation ? LANDAU_ENOMEM : LANDAU_ECUDA;
        }
        ctx->pair_owned.push_back(d);
        *a.p = static_cast<double *>(d);
        if (a.zero) CK(cudaMemset(d, 0, a.n * sizeof(double)));
    }
    ctx->pair_path = path;
    return LANDAU_OK;
}

// LANDAU_PAIR_AUTO: share the tensor across the batch when there is a batch to share it with and U fits easily
int resolve_pair_path(const landau_ctx *ctx, int path) {
    if (path != LANDAU_PAIR_AUTO) return path;
    if (ctx->max_batch < LANDAU_SHARED_MIN_BATCH) return LANDAU_PAIR_PER_PROBLEM;
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { cudaGetLastError(); return LANDAU_PAIR_PER_PROBLEM; }
    return tensor_bytes(ctx->Ntot) <= free_b / 4 ? LANDAU_PAIR_SHARED : LANDAU_PAIR_PER_PROBLEM;
}

// LANDAU_BAND_AUTO: the gather / scatter front kernel when its flops are at most half the hull's (it pays a gather and a
// scatter of its window per block step); the slot kernel -- no fill, no gather, no scatter -- whenever it does not do more
// flops than the hull kernel: measured ahead even on the uniform 8 x 16 Q3 mesh, where front = hull (5.18 against 5.63 ms)
constexpr double FRONT_MAX_WORK_RATIO = 0.5, SLOT_MAX_WORK_RATIO = 1.0;
static bool auto_front(bool front_fits, bool slot, double front_flop, double hull_flop) {
    return front_fits && front_flop <= (slot ? SLOT_MAX_WORK_RATIO : FRONT_MAX_WORK_RATIO) * hull_flop;
}
constexpr size_t FRONT_SMEM_MAX = size_t(225) * 1024;        // + 1 KB the driver reserves per block
// Columns per block step of the FACTORISATION.  band_block(bw) unless that is 32 and the envelope is jagged enough for the
// slot kernel with 16-column blocks: its window must fit the shared memory of an SM (two windows per SM: 256 threads per
// matrix, config 5: fill + factor 14.2 -> 7.4 ms; one window: 512 threads, ten-species 320-cell mesh 20.8 -> 13.6 ms).  The
// solves keep band_block(bw) in either case: L and U do not depend on the blocking, and a 16-column solve of a band
// that wide takes twice as long (config 5: 5.9 against 3.45 ms).
int band_factor_block(const HostSpace &hs, const std::vector<int32_t> &perm, int bw) {
    const int kb = band_block(bw);
    if (kb != 32) return kb;
    std::vector<int32_t> ap, ai;
    double f16 = 0.0;
    const int na16 = band_active_lists(int(hs.n), hs.rowptr, hs.colidx, perm, 16, ap, ai, &f16);
    int bw2 = 0;
    const double hull16 = band_envelope(int(hs.n), hs.rowptr, hs.colidx, perm, bw2, nullptr, nullptr, 16);
    return band_slot_smem(16, na16) <= FRONT_SMEM_MAX && na16 <= 160 && f16 <= FRONT_MAX_WORK_RATIO * hull16 ? 16 : kb;
}

// Small batches are launch-latency bound: both gathers then go in one launch (3-7 us per single build); large
// batches keep the two launches (the merged kernel is 10 % slower there).
constexpr int MERGED_GATHER_MAX_NB = 8;

// a4-a7 for nb problems; Ez == nullptr: collision Jacobian and C(f), else the implicit-step operator
void assemble(landau_ctx *ctx, int nb, const double *f_dev, const double *Ez, double shift, double *vals_dev, double *Cf_dev,
              cudaStream_t st) {
    // (letting k_element add the pair kernel's slabs itself in single-build contexts of Q2 grids -- one launch fewer --
    // was measured slower: config 1 21.8 against 19.5 us per build; the slab sum as a kernel of its own overlaps its
    // neighbours' launch latencies under programmatic dependent launch)
    for (auto &g : ctx->grids) {
        ctx->launches += launch_element(g.ds, nb, 1, f_dev + g.foff, ctx->sc.Gsum, g.Ce, g.ce, Ez, shift, st);
        if (vals_dev && Cf_dev && nb <= MERGED_GATHER_MAX_NB) {
            ctx->launches += launch_gather_both(g.ds, nb, ctx->vstride, ctx->fstride, g.Ce, g.ce, vals_dev + g.voff, Cf_dev + g.foff, st);
            continue;
        }
        if (vals_dev) ctx->launches += launch_gather_vals(g.ds, nb, g.ds.S, ctx->vstride, g.Ce, vals_dev + g.voff, st);
        if (Cf_dev) ctx->launches += launch_gather_cf(g.ds, nb, ctx->fstride, g.ce, Cf_dev + g.foff, st);
    }
}

// Do two points of DIFFERENT grids coincide exactly?  (Then every pair must be tested, reading Q3.)
bool cross_grid_coincidence(const std::vector<GridState> &grids) {
    struct P { double r, z; int g; };
    std::vector<P> pts;
    for (size_t g = 0; g < grids.size(); ++g)
        for (int64_t i = 0; i < grids[g].hs.N; ++i) pts.push_back({grids[g].hs.r[i], grids[g].hs.z[i], int(g)});
    std::sort(pts.begin(), pts.end(), [](const P &a, const P &b) { return a.r != b.r ? a.r < b.r : (a.z != b.z ? a.z < b.z : a.g < b.g); });
    for (size_t i = 1; i < pts.size(); ++i)
        if (pts[i].r == pts[i - 1].r && pts[i].z == pts[i - 1].z) return true;   // within one grid points never coincide
    return false;
}
}  // namespace

extern "C" {

const char *landau_strerror(int code) {
    switch (code) {
        case LANDAU_OK: return "ok";
        case LANDAU_EINVAL: return "invalid argument";
        case LANDAU_ENOMEM: return "out of memory";
        case LANDAU_ECUDA: return "CUDA error";
        default: return "unknown error";
    }
}

const char *landau_last_cuda_error(void) { return g_cuda_err.c_str(); }

int landau_destroy(landau_ctx *ctx) {
    if (!ctx) return LANDAU_OK;
    for (void *p : ctx->owned) cudaFree(p);
    for (void *p : ctx->pair_owned) cudaFree(p);
    if (ctx->d_f) cudaFree(ctx->d_f);
    if (ctx->d_vals) cudaFree(ctx->d_vals);
    if (ctx->d_Cf) cudaFree(ctx->d_Cf);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->chunk_done) cudaEventDestroy(ctx->chunk_done);
    if (ctx->side_stream) cudaStreamDestroy(ctx->side_stream);
    if (ctx->side_fork) cudaEventDestroy(ctx->side_fork);
    if (ctx->side_join) cudaEventDestroy(ctx->side_join);
    for (auto &ev : ctx->prof_events) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
    for (auto &ev : ctx->prof_pool) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
    delete ctx;
    return LANDAU_OK;
}

static int create_impl(const landau_mesh *meshes, int ngrids, const int32_t *species_grid, int order,
                       const landau_species *species, int max_batch, int pair_path, landau_ctx **out) {
    if (!out) return LANDAU_EINVAL;
    *out = nullptr;
    if (!meshes || !species || ngrids < 1 || max_batch < 1 || max_batch > 65535) return LANDAU_EINVAL;
    if (pair_path != LANDAU_PAIR_AUTO && pair_path != LANDAU_PAIR_PER_PROBLEM && pair_path != LANDAU_PAIR_SHARED) return LANDAU_EINVAL;
    if (species->S < 1 || species->S > MAX_SPECIES || !species->mass || !species->charge) return LANDAU_EINVAL;
    if (!(species->m0 > 0.0)) return LANDAU_EINVAL;
    const int S = species->S;
    for (int s = 0; s < S; ++s)
        if (!(species->mass[s] > 0.0)) return LANDAU_EINVAL;
    // species grouped by grid: the map must be non-decreasing and use every grid
    std::vector<int> sgrid(S, 0);
    if (ngrids > 1) {
        if (!species_grid) return LANDAU_EINVAL;
        for (int s = 0; s < S; ++s) {
            sgrid[s] = species_grid[s];
            if (sgrid[s] < 0 || sgrid[s] >= ngrids || (s && sgrid[s] < sgrid[s - 1])) return LANDAU_EINVAL;
        }
        for (int g = 0; g < ngrids; ++g)
            if (std::find(sgrid.begin(), sgrid.end(), g) == sgrid.end()) return LANDAU_EINVAL;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        g_cuda_err = "no CUDA device (this library has no CPU fallback)";
        return LANDAU_ECUDA;
    }
    landau_ctx *ctx = new (std::nothrow) landau_ctx();
    if (!ctx) return LANDAU_ENOMEM;
    struct Guard {                      // an exception (bad_alloc) or an early return destroys the half-built ctx
        landau_ctx *c;
        ~Guard() { if (c) landau_destroy(c); }
    } guard{ctx};
    ctx->grids.resize(ngrids);
    ctx->S = S;
    ctx->max_batch = max_batch;
    {   // set-up of landau_band_solve_static: the device address of the library's static scratch, asked with this device current
        cudaError_t e = cudaGetDevice(&ctx->device);
        if (e == cudaSuccess) e = band_static_scratch(&ctx->static_scratch);
        if (e != cudaSuccess) {
            cudaGetLastError();
            g_cuda_err = std::string("cudaGetSymbolAddress(static band-solve scratch): ") + cudaGetErrorString(e);
            return LANDAU_ECUDA;
        }
    }
    ctx->latency_tiles = max_batch < LANDAU_SHARED_MIN_BATCH;
    int rc = LANDAU_OK;
    for (int g = 0; g < ngrids; ++g) {
        std::string err;
        rc = build_host_space(meshes[g], order, ctx->grids[g].hs, err);
        if (rc != LANDAU_OK) { g_cuda_err = err; return rc; }
    }
    // offsets and sizes
    std::vector<double> r, z, invr;
    for (int g = 0; g < ngrids; ++g) {
        GridState &G = ctx->grids[g];
        const HostSpace &hs = G.hs;
        G.s0 = int(std::find(sgrid.begin(), sgrid.end(), g) - sgrid.begin());
        const int Sg = int(std::count(sgrid.begin(), sgrid.end(), g));
        G.foff = ctx->fstride; G.voff = ctx->vstride; G.moff = ctx->mstride;
        ctx->fstride += size_t(Sg) * hs.n; ctx->vstride += size_t(Sg) * hs.nnz; ctx->mstride += size_t(hs.nnz);
        DeviceSpace &ds = G.ds;
        std::memset(&ds, 0, sizeof(ds));
        ds.p = hs.p; ds.Nq = hs.Nq; ds.Nb = hs.Nb; ds.S = Sg;
        ds.N = int(hs.N); ds.Ne = int(hs.Ne); ds.n = int(hs.n); ds.nnz = int(hs.nnz);
        ds.poff = int(ctx->Ntot);
        ctx->Ntot += hs.N;
        for (int t = 0; t < Sg; ++t) {
            const int s = G.s0 + t;
            const double e2 = species->charge[s] * species->charge[s], mm = species->m0 / species->mass[s];
            ds.e2[t] = e2; ds.m0m[t] = mm;
            ds.kfac[t] = species->nu * e2 * mm;
            ds.dfac[t] = -species->nu * e2 * mm * mm;
            ds.qm[t] = species->charge[s] * mm;
        }
        r.insert(r.end(), hs.r.begin(), hs.r.end());
        z.insert(z.end(), hs.z.begin(), hs.z.end());
        for (int64_t i = 0; i < hs.N; ++i) invr.push_back(1.0 / hs.r[i]);
    }
    if (ctx->Ntot > (int64_t(1) << 30) || ctx->vstride > (size_t(1) << 32)) return LANDAU_EINVAL;
    ctx->check_all = ngrids > 1 && cross_grid_coincidence(ctx->grids);
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, dev);

#define UPC(ptr, vec) \
    if ((rc = upload(vec, &(ptr), ctx->owned)) != LANDAU_OK) return rc;
    UPC(ctx->r, r) UPC(ctx->z, z) UPC(ctx->invr, invr)
    const size_t nbm = size_t(max_batch);
    for (int g = 0; g < ngrids; ++g) {
        GridState &G = ctx->grids[g];
        HostSpace &hs = G.hs;
        DeviceSpace &ds = G.ds;
        ds.Ntot = int(ctx->Ntot);
        ds.fstride = (long long)ctx->fstride;
        ds.r = ctx->r + ds.poff; ds.z = ctx->z + ds.poff; ds.invr = ctx->invr + ds.poff;
        UPC(ds.w_in, hs.w_in) UPC(ds.w_out, hs.w_out) UPC(ds.invJ, hs.invJ)
        UPC(ds.B, hs.B) UPC(ds.E0, hs.E0) UPC(ds.E1, hs.E1)
        ds.Me = ds.Ae = nullptr;
        if (hs.Nb == 16) {     // element mass and advection matrices of the implicit-step operator (k_element_q3<true>)
            std::vector<double> Me(size_t(hs.Ne) * 256), Ae(size_t(hs.Ne) * 256);
            for (int64_t e = 0; e < hs.Ne; ++e)
                for (int a = 0; a < 16; ++a)
                    for (int bb = 0; bb < 16; ++bb) {
                        double m = 0.0, ad = 0.0;
                        for (int q = 0; q < 16; ++q) {
                            const double w = hs.w_out[e * 16 + q], Bqa = hs.B[q * 16 + a];
                            m = std::fma(w * Bqa, hs.B[q * 16 + bb], m);
                            ad = std::fma(w * hs.invJ[2 * e + 1] * Bqa, hs.E1[q * 16 + bb], ad);
                        }
                        Me[(e * 16 + a) * 16 + bb] = m; Ae[(e * 16 + a) * 16 + bb] = ad;
                    }
            UPC(ds.Me, Me) UPC(ds.Ae, Ae)
        }
        UPC(ds.lptr, hs.lptr) UPC(ds.ldof, hs.ldof) UPC(ds.lw, hs.lw)
        UPC(ds.rowptr, hs.rowptr) UPC(ds.colidx, hs.colidx)
        UPC(ds.gptr, hs.gptr) UPC(ds.gidx, hs.gidx) UPC(ds.gw, hs.gw)
        UPC(ds.cptr, hs.cptr) UPC(ds.cidx, hs.cidx) UPC(ds.cw, hs.cw)
        {
            auto heads = [](const std::vector<int32_t> &ptr, const std::vector<int32_t> &idx, const std::vector<double> &w) {
                std::vector<GatherHead> h(ptr.size() - 1, GatherHead{0.0, 0, 0});       // an empty list adds 0 * src[0]
                for (size_t k = 0; k + 1 < ptr.size(); ++k)
                    if (ptr[k + 1] > ptr[k]) h[k] = GatherHead{w[ptr[k]], idx[ptr[k]], 0};
                return h;
            };
            const std::vector<GatherHead> gh = heads(hs.gptr, hs.gidx, hs.gw), ch = heads(hs.cptr, hs.cidx, hs.cw),
                                          lh = heads(hs.lptr, hs.ldof, hs.lw);
            UPC(ds.ghead, gh) UPC(ds.chead, ch) UPC(ds.lhead, lh)
        }
        // band LU: order, half-bandwidth, envelope per block step, fill lists per band column
        std::vector<int32_t> perm;
        int bw = 0;
        rcm_order(int(hs.n), hs.rowptr, hs.colidx, hs.dof_r.data(), hs.dof_z.data(), perm, bw);
        const int64_t Wb = band_stored_halfwidth(bw), LD = 2 * Wb + 1;
        if (LD * hs.n > (int64_t(1) << 31) - 1) return LANDAU_EINVAL;
        const int kb = band_factor_block(hs, perm, bw), kbs = band_block(bw);        // kb <= kbs: the stored width covers both
        G.bs.kb = kb; G.bs.W = int(Wb);
        G.bs.n = int(hs.n); G.bs.nnz = int(hs.nnz); G.bs.bw = bw; G.bs.mat_doubles = (size_t(LD) * hs.n + 1) & ~size_t(1);   // even: every matrix starts 16-byte aligned
        // envelope of the permuted pattern: block step s only reaches mlow[s] rows below and mup[s] rows above its
        // block (<= bw; about half the uniform-band work on the refined meshes)
        {
            std::vector<int32_t> mlow, mup, mlow_s, mup_s, zlo, zcnt, fptr, fsrc, foff;
            int bw2 = 0;
            G.bs.flop_per_matrix = band_envelope(int(hs.n), hs.rowptr, hs.colidx, perm, bw2, &mlow, &mup, kb);
            if (kbs != kb) band_envelope(int(hs.n), hs.rowptr, hs.colidx, perm, bw2, &mlow_s, &mup_s, kbs);
            band_fill_lists(int(hs.n), hs.rowptr, hs.colidx, perm, int(Wb), kb, mlow, mup, kbs, mlow_s, mup_s, zlo, zcnt, fptr, fsrc, foff);
            UPC(G.bs.mlow, mlow) UPC(G.bs.mup, mup)
            if (kbs != kb) { UPC(G.bs.mlow_s, mlow_s) UPC(G.bs.mup_s, mup_s) }
            else { G.bs.mlow_s = G.bs.mlow; G.bs.mup_s = G.bs.mup; }
            {
                std::vector<int32_t> pos(hs.n), first(hs.n);
                for (int64_t i = 0; i < hs.n; ++i) { pos[perm[i]] = int32_t(i); first[i] = int32_t(i); }
                for (int64_t i = 0; i < hs.n; ++i)
                    for (int t = hs.rowptr[i]; t < hs.rowptr[i + 1]; ++t) first[pos[i]] = std::min(first[pos[i]], pos[hs.colidx[t]]);
                UPC(G.bs.first, first)
            }
            UPC(G.bs.zlo, zlo) UPC(G.bs.zcnt, zcnt) UPC(G.bs.fptr, fptr) UPC(G.bs.fsrc, fsrc) UPC(G.bs.foff, foff)
            std::vector<int32_t> act_ptr, act_idx;
            G.bs.na_max = band_active_lists(int(hs.n), hs.rowptr, hs.colidx, perm, kb, act_ptr, act_idx, &G.bs.front_flop);
            if (act_idx.empty()) act_idx.push_back(0);
            {
                std::vector<int32_t> act_slot, slot_hi, new_ptr, new_pos, ld_ptr, ld_dst, ld_csr, d0_csr;
                band_slot_lists(int(hs.n), hs.rowptr, hs.colidx, perm, kb, band_front_ldp(G.bs.na_max), band_front_ldw(G.bs.na_max), act_ptr, act_idx, G.bs.na_max, act_slot,
                                slot_hi, new_ptr, new_pos, ld_ptr, ld_dst, ld_csr, d0_csr);
                if (slot_hi.empty()) slot_hi.push_back(0);
                UPC(G.bs.slot_hi, slot_hi)
                if (act_slot.empty()) act_slot.push_back(0);
                if (new_pos.empty()) new_pos.push_back(0);
                if (ld_dst.empty()) { ld_dst.push_back(0); ld_csr.push_back(-1); }
                UPC(G.bs.act_slot, act_slot) UPC(G.bs.new_ptr, new_ptr) UPC(G.bs.new_pos, new_pos)
                UPC(G.bs.ld_ptr, ld_ptr) UPC(G.bs.ld_dst, ld_dst) UPC(G.bs.ld_csr, ld_csr)
                UPC(G.bs.d0_csr, d0_csr)
                G.bs.slot = kb == 16 && band_slot_smem(kb, G.bs.na_max) <= FRONT_SMEM_MAX;
            }
            UPC(G.bs.act_ptr, act_ptr) UPC(G.bs.act_idx, act_idx)
            G.front_fits = band_front_smem(kb, G.bs.na_max) <= FRONT_SMEM_MAX && G.bs.na_max <= 160 && kb >= 16;   // FRONT_IR rows per lane
            // AUTO: the front kernel pays a gather and a scatter of its window per block step; it wins where the envelope
            // is jagged (refined meshes: a sixth of the hull's flops), not on uniform meshes (front = hull)
            G.bs.front = auto_front(G.front_fits, G.bs.slot, G.bs.front_flop, G.bs.flop_per_matrix);
        }
        UPC(G.bs.perm, perm)
        G.boff = ctx->bstride;
        ctx->bstride += size_t(ds.S) * G.bs.mat_doubles;
    }
#undef UPC
    // scratch arena.  Sizes are validated in 64-bit arithmetic first: an absurd max_batch fails here with
    // LANDAU_ENOMEM instead of overflowing an index later.
    struct Alloc { double **p; size_t n; };
    std::vector<Alloc> allocs = {{&ctx->sc.Gsum, nbm * 5 * ctx->Ntot}};
    for (auto &G : ctx->grids) {
        allocs.push_back({&G.Ce, nbm * G.ds.S * G.hs.Ne * G.hs.Nb * G.hs.Nb});
        allocs.push_back({&G.ce, nbm * G.ds.S * G.hs.Ne * G.hs.Nb});
    }
    for (auto &a : allocs) {
        void *d = nullptr;
        cudaError_t e = cudaMalloc(&d, a.n * sizeof(double));
        if (e != cudaSuccess) {
            g_cuda_err = std::string("cudaMalloc(scratch): ") + cudaGetErrorString(e);
            cudaGetLastError();
            return e == cudaErrorMemoryAllocation ? LANDAU_ENOMEM : LANDAU_ECUDA;
        }
        ctx->owned.push_back(d);
        *a.p = static_cast<double *>(d);
    }
    if ((rc = alloc_pair_scratch(ctx, resolve_pair_path(ctx, pair_path))) != LANDAU_OK) return rc;
    guard.c = nullptr;
    *out = ctx;
    return LANDAU_OK;
}

int landau_create_multigrid(const landau_mesh *meshes, int ngrids, const int32_t *species_grid, int order,
                            const landau_species *species, int max_batch, landau_ctx **out) {
    if (out) *out = nullptr;
    return guarded([&]() { return create_impl(meshes, ngrids, species_grid, order, species, max_batch, LANDAU_PAIR_AUTO, out); });
}

int landau_create(const landau_mesh *mesh, int order, const landau_species *species, int max_batch, landau_ctx **out) {
    return landau_create_multigrid(mesh, 1, nullptr, order, species, max_batch, out);
}

int landau_set_pair_path(landau_ctx *ctx, int path) {
    if (!ctx || (path != LANDAU_PAIR_AUTO && path != LANDAU_PAIR_PER_PROBLEM && path != LANDAU_PAIR_SHARED)) return LANDAU_EINVAL;
    return guarded([&]() {
        CK(cudaDeviceSynchronize());                       // the scratch being replaced may still be in use
        const int want = resolve_pair_path(ctx, path);
        if (want == ctx->pair_path && !ctx->pair_owned.empty()) return int(LANDAU_OK);
        return alloc_pair_scratch(ctx, want);
    });
}

int landau_pair_path(const landau_ctx *ctx, int32_t *path, int64_t *scratch_bytes) {
    if (!ctx) return LANDAU_EINVAL;
    if (path) *path = ctx->pair_path;
    if (scratch_bytes) {
        const size_t N = size_t(ctx->Ntot), nbm = size_t(ctx->max_batch);
        size_t d;
        if (ctx->pair_path == LANDAU_PAIR_SHARED)
            d = 3 * size_t(shared_kpad(int(N)) / 8) * ctx->nbpad * 8 + tensor_bytes(ctx->Ntot) / 8 +
                (shared_ksplit(int(N)) > 1 ? nbm * shared_ksplit(int(N)) * 5 * N : 0);
        else
            d = size_t(ctx->pp_chunk) * (3 * N + pair_tiles(int(N), ctx->latency_tiles) * 5 * N);
        *scratch_bytes = int64_t(d * sizeof(double));
    }
    return LANDAU_OK;
}

int landau_set_tensor_cache(landau_ctx *ctx, int on) {
    if (!ctx) return LANDAU_EINVAL;
    ctx->tensor_cache = on != 0;
    if (!on) ctx->tensor_valid = false;
    return LANDAU_OK;
}

int landau_setup_host(const landau_mesh *mesh, int order, int64_t *n, int64_t *nnz, int64_t *N, int32_t *rowptr_host,
                      int32_t *colidx_host, double *dof_r_host, double *dof_z_host) {
    if (!mesh) return LANDAU_EINVAL;
    return guarded([&]() {
    HostSpace hs;
    std::string err;
    const int rc = build_host_space(*mesh, order, hs, err);
    if (rc != LANDAU_OK) { g_cuda_err = err; return rc; }
    if (n) *n = hs.n;
    if (nnz) *nnz = hs.nnz;
    if (N) *N = hs.N;
    if (rowptr_host) std::memcpy(rowptr_host, hs.rowptr.data(), hs.rowptr.size() * sizeof(int32_t));
    if (colidx_host) std::memcpy(colidx_host, hs.colidx.data(), hs.colidx.size() * sizeof(int32_t));
    if (dof_r_host) std::memcpy(dof_r_host, hs.dof_r.data(), hs.n * sizeof(double));
    if (dof_z_host) std::memcpy(dof_z_host, hs.dof_z.data(), hs.n * sizeof(double));
    return int(LANDAU_OK);
    });
}

int landau_band_order_host(const landau_mesh *mesh, int order, int32_t *perm_host, int32_t *half_bandwidth,
                           int32_t *block_columns, double *flop_per_factorization) {
    if (!mesh) return LANDAU_EINVAL;
    return guarded([&]() {
    HostSpace hs;
    std::string err;
    const int rc = build_host_space(*mesh, order, hs, err);
    if (rc != LANDAU_OK) { g_cuda_err = err; return rc; }
    std::vector<int32_t> perm;
    int bw = 0;
    rcm_order(int(hs.n), hs.rowptr, hs.colidx, hs.dof_r.data(), hs.dof_z.data(), perm, bw);
    if (perm_host) std::memcpy(perm_host, perm.data(), perm.size() * sizeof(int32_t));
    if (half_bandwidth) *half_bandwidth = bw;
    const int kb = band_factor_block(hs, perm, bw);
    if (block_columns) *block_columns = kb;
    if (flop_per_factorization) {      // the envelope work of landau_create, recomputed from the order
        int bw2 = 0;
        *flop_per_factorization = band_envelope(int(hs.n), hs.rowptr, hs.colidx, perm, bw2, nullptr, nullptr, kb);
    }
    return int(LANDAU_OK);
    });
}

int landau_band_front_host(const landau_mesh *mesh, int order, int32_t *front_rows_max, double *front_flop, int32_t *fits) {
    if (!mesh) return LANDAU_EINVAL;
    return guarded([&]() {
        HostSpace hs;
        std::string err;
        const int rc = build_host_space(*mesh, order, hs, err);
        if (rc != LANDAU_OK) { g_cuda_err = err; return rc; }
        std::vector<int32_t> perm, act_ptr, act_idx;
        int bw = 0;
        rcm_order(int(hs.n), hs.rowptr, hs.colidx, hs.dof_r.data(), hs.dof_z.data(), perm, bw);
        double fl = 0.0;
        const int kb = band_factor_block(hs, perm, bw);
        const int na_max = band_active_lists(int(hs.n), hs.rowptr, hs.colidx, perm, kb, act_ptr, act_idx, &fl);
        if (front_rows_max) *front_rows_max = na_max;
        if (front_flop) *front_flop = fl;
        if (fits) *fits = band_front_smem(kb, na_max) <= FRONT_SMEM_MAX && na_max <= 160 && kb >= 16;
        return int(LANDAU_OK);
    });
}

int landau_grid_count(const landau_ctx *ctx, int32_t *ngrids) {
    if (!ctx || !ngrids) return LANDAU_EINVAL;
    *ngrids = int32_t(ctx->grids.size());
    return LANDAU_OK;
}

int landau_grid_sizes(const landau_ctx *ctx, int grid, int32_t *S_g, int32_t *first_species, int64_t *n, int64_t *nnz,
                      int64_t *N, int64_t *Ne) {
    if (!ctx || grid < 0 || grid >= int(ctx->grids.size())) return LANDAU_EINVAL;
    const GridState &G = ctx->grids[grid];
    if (S_g) *S_g = G.ds.S;
    if (first_species) *first_species = G.s0;
    if (n) *n = G.hs.n;
    if (nnz) *nnz = G.hs.nnz;
    if (N) *N = G.hs.N;
    if (Ne) *Ne = G.hs.Ne;
    return LANDAU_OK;
}

int landau_strides(const landau_ctx *ctx, int32_t *S, int64_t *f_stride, int64_t *vals_stride, int64_t *mvals_size, int64_t *N_total) {
    if (!ctx) return LANDAU_EINVAL;
    if (S) *S = ctx->S;
    if (f_stride) *f_stride = int64_t(ctx->fstride);
    if (vals_stride) *vals_stride = int64_t(ctx->vstride);
    if (mvals_size) *mvals_size = int64_t(ctx->mstride);
    if (N_total) *N_total = ctx->Ntot;
    return LANDAU_OK;
}

int landau_sizes(const landau_ctx *ctx, int32_t *S, int64_t *n, int64_t *nnz, int64_t *N, int64_t *Ne) {
    if (!ctx || ctx->grids.size() != 1) return LANDAU_EINVAL;
    const HostSpace &hs = ctx->grids[0].hs;
    if (S) *S = ctx->S;
    if (n) *n = hs.n;
    if (nnz) *nnz = hs.nnz;
    if (N) *N = hs.N;
    if (Ne) *Ne = hs.Ne;
    return LANDAU_OK;
}

int landau_grid_csr_pattern(const landau_ctx *ctx, int grid, const int32_t **rowptr_dev, const int32_t **colidx_dev) {
    if (!ctx || grid < 0 || grid >= int(ctx->grids.size())) return LANDAU_EINVAL;
    if (rowptr_dev) *rowptr_dev = ctx->grids[grid].ds.rowptr;
    if (colidx_dev) *colidx_dev = ctx->grids[grid].ds.colidx;
    return LANDAU_OK;
}

int landau_grid_csr_pattern_host(const landau_ctx *ctx, int grid, int32_t *rowptr_host, int32_t *colidx_host) {
    if (!ctx || grid < 0 || grid >= int(ctx->grids.size())) return LANDAU_EINVAL;
    const HostSpace &hs = ctx->grids[grid].hs;
    if (rowptr_host) std::memcpy(rowptr_host, hs.rowptr.data(), hs.rowptr.size() * sizeof(int32_t));
    if (colidx_host) std::memcpy(colidx_host, hs.colidx.data(), hs.colidx.size() * sizeof(int32_t));
    return LANDAU_OK;
}

int landau_grid_dof_coords(const landau_ctx *ctx, int grid, double *r_host, double *z_host) {
    if (!ctx || grid < 0 || grid >= int(ctx->grids.size())) return LANDAU_EINVAL;
    const HostSpace &hs = ctx->grids[grid].hs;
    if (r_host) std::memcpy(r_host, hs.dof_r.data(), hs.n * sizeof(double));
    if (z_host) std::memcpy(z_host, hs.dof_z.data(), hs.n * sizeof(double));
    return LANDAU_OK;
}

int landau_csr_pattern(const landau_ctx *ctx, const int32_t **rowptr_dev, const int32_t **colidx_dev) {
    if (!ctx || ctx->grids.size() != 1) return LANDAU_EINVAL;
    return landau_grid_csr_pattern(ctx, 0, rowptr_dev, colidx_dev);
}

int landau_csr_pattern_host(const landau_ctx *ctx, int32_t *rowptr_host, int32_t *colidx_host) {
    if (!ctx || ctx->grids.size() != 1) return LANDAU_EINVAL;
    return landau_grid_csr_pattern_host(ctx, 0, rowptr_host, colidx_host);
}

int landau_dof_coords(const landau_ctx *ctx, double *r_host, double *z_host) {
    if (!ctx || ctx->grids.size() != 1) return LANDAU_EINVAL;
    return landau_grid_dof_coords(ctx, 0, r_host, z_host);
}

int landau_points(const landau_ctx *ctx, double *r_host, double *z_host, double *w_host) {
    if (!ctx) return LANDAU_EINVAL;
    size_t off = 0;
    for (const auto &G : ctx->grids) {   // union of the grids' points, grid by grid
        const HostSpace &hs = G.hs;
        if (r_host) std::memcpy(r_host + off, hs.r.data(), hs.N * sizeof(double));
        if (z_host) std::memcpy(z_host + off, hs.z.data(), hs.N * sizeof(double));
        if (w_host) std::memcpy(w_host + off, hs.w_in.data(), hs.N * sizeof(double));
        off += size_t(hs.N);
    }
    return LANDAU_OK;
}

int landau_inner_integral(landau_ctx *ctx, int nb, const double *f_dev, double *G_dev, void *stream) {
    if (!ctx || !f_dev || !G_dev || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    return guarded([&]() {
        inner_integral(ctx, nb, f_dev, G_dev, static_cast<cudaStream_t>(stream));
        return launches_ok();
    });
}

int landau_jacobian_batched(landau_ctx *ctx, int nb, const double *f_dev, double *vals_dev, double *Cf_dev, void *stream) {
    if (!ctx || !f_dev || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return guarded([&]() {
        inner_integral(ctx, nb, f_dev, ctx->sc.Gsum, st);
        assemble(ctx, nb, f_dev, nullptr, 0.0, vals_dev, Cf_dev, st);
        return launches_ok();
    });
}

int landau_implicit_operator_batched(landau_ctx *ctx, int nb, const double *f_dev, const double *Ez_dev, double shift,
                                     double *vals_dev, double *F_dev, void *stream) {
    if (!ctx || !f_dev || !Ez_dev || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return guarded([&]() {
        inner_integral(ctx, nb, f_dev, ctx->sc.Gsum, st);
        assemble(ctx, nb, f_dev, Ez_dev, shift, vals_dev, F_dev, st);
        return launches_ok();
    });
}

int landau_jacobian(landau_ctx *ctx, const double *f_dev, double *vals_dev, double *Cf_dev, void *stream) {
    return landau_jacobian_batched(ctx, 1, f_dev, vals_dev, Cf_dev, stream);
}

int landau_mass(landau_ctx *ctx, double shift, double *mvals_dev, void *stream) {
    if (!ctx || !mvals_dev) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    for (auto &g : ctx->grids) {
        ctx->launches += launch_mass_element(g.ds, shift, g.Ce, st);
        ctx->launches += launch_gather_vals(g.ds, 1, 1, 0, g.Ce, mvals_dev + g.moff, st);
    }
    return launches_ok();
}

int landau_jacobian_host(landau_ctx *ctx, int nb, const double *f_host, double *vals_host, double *Cf_host) {
    if (!ctx || !f_host || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    if (!ctx->own_stream) {
        CK(cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&ctx->chunk_done, cudaEventDisableTiming));
    }
    const size_t fsz = ctx->fstride, vsz = ctx->vstride;
    if (ctx->host_nb < nb) {
        if (ctx->d_f) { cudaFree(ctx->d_f); cudaFree(ctx->d_vals); cudaFree(ctx->d_Cf); ctx->d_f = ctx->d_vals = ctx->d_Cf = nullptr; }
        cudaError_t e = cudaMalloc((void **)&ctx->d_f, size_t(nb) * fsz * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->d_vals, size_t(nb) * vsz * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->d_Cf, size_t(nb) * fsz * sizeof(double));
        if (e != cudaSuccess) { ctx->host_nb = 0; return cuda_fail(e, "cudaMalloc(host staging)"); }
        ctx->host_nb = nb;
    }
    // Pipeline over sub-batches: the device-to-host copy of chunk c overlaps the build of chunk
    // c+1 (the scratch arena is reused in stream order; problems are independent, so the values
    // are bitwise those of one batched call).
    cudaStream_t st = ctx->own_stream, cp = ctx->copy_stream;
    // the body enqueues; whatever it returns, both streams are drained before the caller gets its buffers back
    // (an error half way must not leave device-to-host copies into the caller's memory in flight)
    auto body = [&]() -> int {
        const int nchunks = nb >= 64 ? 8 : (nb >= 8 ? 4 : 1);
        const int cb = (nb + nchunks - 1) / nchunks;
        for (int b0 = 0; b0 < nb; b0 += cb) {
            const int nbc = std::min(cb, nb - b0);
            // inputs chunk by chunk as well: the first results leave for the host after 1/nchunks of the upload
            CK(cudaMemcpyAsync(ctx->d_f + b0 * fsz, f_host + b0 * fsz, size_t(nbc) * fsz * sizeof(double), cudaMemcpyHostToDevice, st));
            // the tensor of the point pairs (batch-shared path) is evaluated by the first sub-batch only
            inner_integral(ctx, nbc, ctx->d_f + b0 * fsz, ctx->sc.Gsum, st, b0 > 0);
            assemble(ctx, nbc, ctx->d_f + b0 * fsz, nullptr, 0.0, vals_host ? ctx->d_vals + b0 * vsz : nullptr,
                     Cf_host ? ctx->d_Cf + b0 * fsz : nullptr, st);
            const int rc = launches_ok();
            if (rc != LANDAU_OK) return rc;
            CK(cudaEventRecord(ctx->chunk_done, st));
            CK(cudaStreamWaitEvent(cp, ctx->chunk_done, 0));
            if (vals_host) CK(cudaMemcpyAsync(vals_host + b0 * vsz, ctx->d_vals + b0 * vsz, size_t(nbc) * vsz * sizeof(double), cudaMemcpyDeviceToHost, cp));
            if (Cf_host) CK(cudaMemcpyAsync(Cf_host + b0 * fsz, ctx->d_Cf + b0 * fsz, size_t(nbc) * fsz * sizeof(double), cudaMemcpyDeviceToHost, cp));
        }
        return LANDAU_OK;
    };
    const int rc = guarded(body);
    const cudaError_t e1 = cudaStreamSynchronize(st), e2 = cudaStreamSynchronize(cp);
    if (rc != LANDAU_OK) return rc;
    if (e1 != cudaSuccess) return cuda_fail(e1, "cudaStreamSynchronize(build stream)");
    if (e2 != cudaSuccess) return cuda_fail(e2, "cudaStreamSynchronize(copy stream)");
    return LANDAU_OK;
}

int landau_band_sizes(const landau_ctx *ctx, int grid, int32_t *half_bandwidth, int64_t *doubles_per_matrix,
                      int64_t *workspace_doubles_per_problem, double *flop_per_factorization) {
    if (!ctx || grid < 0 || grid >= int(ctx->grids.size())) return LANDAU_EINVAL;
    if (flop_per_factorization) *flop_per_factorization = ctx->grids[grid].bs.flop_per_matrix;
    if (half_bandwidth) *half_bandwidth = ctx->grids[grid].bs.bw;
    if (doubles_per_matrix) *doubles_per_matrix = int64_t(ctx->grids[grid].bs.mat_doubles);
    if (workspace_doubles_per_problem) *workspace_doubles_per_problem = int64_t(ctx->bstride);
    return LANDAU_OK;
}

// band workspace layout: [problem][grid][species of the grid][matrix] -- problem-major, so that a solve may
// cover fewer (or other) problems than the factorisation that filled the workspace
int landau_band_factor_batched(landau_ctx *ctx, int nb, const double *vals_dev, double *band_dev, double *pivots_dev, void *stream) {
    if (!ctx || !vals_dev || !band_dev || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    for (auto &g : ctx->grids) {
        if (band_factor_smem(g.bs.bw, g.bs.kb) > 227 * 1024) return LANDAU_EINVAL;
        double *band = band_dev + g.boff;
        const bool fill = band_needs_fill(g.bs);
        if (fill) CK(launch_band_fill(g.bs, nb, g.ds.S, ctx->vstride, ctx->bstride, vals_dev + g.voff, band, st));
        CK(launch_band_factor(g.bs, nb * g.ds.S, g.ds.S, ctx->bstride, vals_dev + g.voff, ctx->vstride, band,
                              pivots_dev ? pivots_dev + 2 * g.s0 : nullptr, ctx->S, st));
        ctx->launches += fill ? 2 : 1;
    }
    return launches_ok();
}

int landau_band_set_method(landau_ctx *ctx, int method) {
    if (!ctx || method < LANDAU_BAND_AUTO || method > LANDAU_BAND_FRONT) return LANDAU_EINVAL;
    for (auto &g : ctx->grids) {
        if (method == LANDAU_BAND_FRONT && !g.front_fits) return LANDAU_EINVAL;
        g.bs.front = method == LANDAU_BAND_HULL ? false
                     : (method == LANDAU_BAND_FRONT ? true : auto_front(g.front_fits, g.bs.slot, g.bs.front_flop, g.bs.flop_per_matrix));
    }
    return LANDAU_OK;
}

int landau_band_method(const landau_ctx *ctx, int grid, int32_t *method, int32_t *front_rows_max, double *flop_per_factorization) {
    if (!ctx || grid < 0 || grid >= int(ctx->grids.size())) return LANDAU_EINVAL;
    const BandSpace &bs = ctx->grids[grid].bs;
    if (method) *method = bs.front ? LANDAU_BAND_FRONT : LANDAU_BAND_HULL;
    if (front_rows_max) *front_rows_max = bs.na_max;
    if (flop_per_factorization) *flop_per_factorization = bs.front ? bs.front_flop : bs.flop_per_matrix;
    return LANDAU_OK;
}

int landau_band_solve_batched(landau_ctx *ctx, int nb, const double *band_dev, const double *rhs_dev, double *x_dev, void *stream) {
    if (!ctx || !band_dev || !rhs_dev || !x_dev || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return guarded([&]() {
    for (auto &g : ctx->grids) {
        // the permuted vector of a matrix is kept in shared memory when it fits (n up to ~28,000), else in a
        // ctx-owned global scratch allocated at the first such call (max_batch * S_g * n doubles)
        double *xg = nullptr;
        if (band_solve_smem(g.bs.n, g.bs.bw) > 227 * 1024) {
            if (!g.solve_x) {
                void *d = nullptr;
                cudaError_t e = cudaMalloc(&d, size_t(ctx->max_batch) * g.ds.S * g.bs.n * sizeof(double));
                if (e != cudaSuccess) { cudaGetLastError(); g_cuda_err = std::string("cudaMalloc(band solve scratch): ") + cudaGetErrorString(e); return int(e == cudaErrorMemoryAllocation ? LANDAU_ENOMEM : LANDAU_ECUDA); }
                ctx->owned.push_back(d);
                g.solve_x = static_cast<double *>(d);
            }
            xg = g.solve_x;
        }
        const double *band = band_dev + g.boff;
        CK(launch_band_solve(g.bs, nb, g.ds.S, ctx->fstride, ctx->bstride, band, rhs_dev + g.foff, x_dev + g.foff, xg, st));
        ctx->launches += 1;
    }
    return launches_ok();
    });
}

int landau_band_solve_static(landau_ctx *ctx, int nb, const double *band_dev, const double *rhs_dev, double *x_dev, void *stream) {
    if (!ctx || !band_dev || !rhs_dev || !x_dev || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device || !ctx->static_scratch) {
        cudaGetLastError();
        g_cuda_err = "landau_band_solve_static: the ctx's device is not current";
        return LANDAU_ECUDA;
    }
    for (auto &g : ctx->grids) {      // checked for every grid before anything is launched
        const size_t need = size_t(nb) * g.ds.S * g.bs.n;
        if (need > BAND_STATIC_SCRATCH_DOUBLES) {
            char msg[192];
            std::snprintf(msg, sizeof msg, "landau_band_solve_static: nb * S * n = %zu doubles exceed the static scratch of %zu doubles (LANDAU_STATIC_SCRATCH_DOUBLES)",
                          need, size_t(BAND_STATIC_SCRATCH_DOUBLES));
            g_cuda_err = msg;
            return LANDAU_EINVAL;
        }
    }
    // the grids' solves follow one another on the stream: each may use the scratch from its start
    for (auto &g : ctx->grids) {
        const cudaError_t e = launch_band_solve_static(g.bs, nb, g.ds.S, ctx->fstride, ctx->bstride, band_dev + g.boff, rhs_dev + g.foff,
                                                       x_dev + g.foff, ctx->static_scratch, st);
        if (e != cudaSuccess) { cudaGetLastError(); g_cuda_err = std::string("landau_band_solve_static: ") + cudaGetErrorString(e); return LANDAU_ECUDA; }
        ctx->launches += 1;
    }
    return LANDAU_OK;
}

int landau_launch_count(const landau_ctx *ctx, int64_t *count) {
    if (!ctx || !count) return LANDAU_EINVAL;
    *count = ctx->launches;
    return LANDAU_OK;
}

int landau_profile_enable(landau_ctx *ctx, int on) {
    if (!ctx) return LANDAU_EINVAL;
    ctx->profiling = on != 0;
    return LANDAU_OK;
}

int landau_profile_read(landau_ctx *ctx, double *ms_total, int64_t *launches) {
    if (!ctx || !ms_total || !launches) return LANDAU_EINVAL;
    return guarded([&]() {
        ms_total[0] = ms_total[1] = 0.0;
        launches[0] = launches[1] = 0;
        for (auto &ev : ctx->prof_events) {
            CK(cudaEventSynchronize(ev.b));
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, ev.a, ev.b));
            ms_total[ev.kind] += ms;
            launches[ev.kind] += 1;
            ctx->prof_pool.push_back(ev);
        }
        ctx->prof_events.clear();
        return int(LANDAU_OK);
    });
}

int landau_fp64_peak_probe(int iters, double *flops_per_s, double *sm_clock_mhz_est) {
    if (iters < 1 || !flops_per_s) return LANDAU_EINVAL;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double *out = nullptr;
    CK(cudaMalloc((void **)&out, sizeof(double)));
    const int blocks = sms * 8, threads = 256;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    launch_dfma_probe(blocks, threads, iters, out, 0);  // warm-up
    CK(cudaEventRecord(e0, 0));
    launch_dfma_probe(blocks, threads, iters, out, 0);
    CK(cudaEventRecord(e1, 0));
    CK(cudaEventSynchronize(e1));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    const double flops = 2.0 * 8.0 * double(iters) * double(blocks) * double(threads);
    *flops_per_s = flops / (double(ms) * 1e-3);
    // 64 DFMA lanes per SM per clock: clock implied by the achieved rate
    if (sm_clock_mhz_est) *sm_clock_mhz_est = *flops_per_s / (2.0 * 64.0 * sms) * 1e-6;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    return LANDAU_OK;
}

int landau_fp64_issue_probe(int mode, int iters, double *cycles_per_warp_instruction, double *flops_per_s) {
    if (iters < 1 || mode < 0 || mode > 7 || !cycles_per_warp_instruction) return LANDAU_EINVAL;
    return guarded([&]() {
        int dev = 0, sms = 0;
        CK(cudaGetDevice(&dev));
        CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        const int warps_per_smsp = mode == 4 ? 1 : 3, threads = 128 * warps_per_smsp;
        double *in = nullptr, *out = nullptr;
        long long *cyc = nullptr;
        CK(cudaMalloc((void **)&in, sizeof(double) * 4096));
        CK(cudaMalloc((void **)&out, sizeof(double)));
        CK(cudaMalloc((void **)&cyc, sizeof(long long) * sms));
        CK(cudaMemset(in, 0, sizeof(double) * 4096));
        cudaEvent_t e0, e1;
        CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
        launch_issue_probe(mode, sms, threads, iters, in, out, cyc, 0);   // warm-up
        CK(cudaEventRecord(e0, 0));
        const int per_iter = launch_issue_probe(mode, sms, threads, iters, in, out, cyc, 0);
        CK(cudaEventRecord(e1, 0));
        CK(cudaEventSynchronize(e1));
        int rc = launches_ok();
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        std::vector<long long> h(sms);
        CK(cudaMemcpy(h.data(), cyc, sizeof(long long) * sms, cudaMemcpyDeviceToHost));
        const double cycles = double(*std::max_element(h.begin(), h.end()));
        // warp instructions per sub-partition = per_iter * iters * warps on it
        *cycles_per_warp_instruction = cycles / (double(per_iter) * iters * warps_per_smsp);
        if (flops_per_s) {
            const double flop_per_inst = mode == 5 ? 512.0 : 64.0;       // DMMA m8n8k4: 256 FMA; DFMA: 32 lanes
            *flops_per_s = flop_per_inst * per_iter * double(iters) * warps_per_smsp * 4 * sms / (double(ms) * 1e-3);
        }
        cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(in); cudaFree(out); cudaFree(cyc);
        return rc;
    });
}

}  // extern "C"
