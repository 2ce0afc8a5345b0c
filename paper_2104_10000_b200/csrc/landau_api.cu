// C-ABI layer (include/landau.h): context management, argument checking, kernel sequencing.
// Every step of the path runs in landau_kernels.cu; there is no CPU fallback.
#include <cuda_runtime.h>

#include <cstdio>
#include <algorithm>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "landau.h"
#include "landau_internal.h"
#include "landau_kernels.h"

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
}  // namespace

struct landau_ctx {
    HostSpace hs;
    DeviceSpace ds;
    Scratch sc;
    std::vector<void *> owned;   // device allocations
    int max_batch = 1;
    int num_sms = 148;
    int64_t launches = 0;
    cudaStream_t own_stream = nullptr, copy_stream = nullptr;
    cudaEvent_t chunk_done = nullptr;
    double *h2d_f = nullptr, *d_f = nullptr, *d_vals = nullptr, *d_Cf = nullptr;  // landau_jacobian_host staging
    int host_nb = 0;
    bool profiling = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_events;  // recorded, not yet read
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_pool;    // free
};

namespace {
// launch_pair bracketed by events when profiling is on
int timed_pair(landau_ctx *ctx, int nb, double *G, cudaStream_t st) {
    if (!ctx->profiling) return launch_pair(ctx->ds, nb, ctx->sc.T, G, st);
    std::pair<cudaEvent_t, cudaEvent_t> ev;
    if (!ctx->prof_pool.empty()) { ev = ctx->prof_pool.back(); ctx->prof_pool.pop_back(); }
    else { cudaEventCreate(&ev.first); cudaEventCreate(&ev.second); }
    cudaEventRecord(ev.first, st);
    int k = launch_pair(ctx->ds, nb, ctx->sc.T, G, st);
    cudaEventRecord(ev.second, st);
    ctx->prof_events.push_back(ev);
    return k;
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
    if (ctx->d_f) cudaFree(ctx->d_f);
    if (ctx->d_vals) cudaFree(ctx->d_vals);
    if (ctx->d_Cf) cudaFree(ctx->d_Cf);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->chunk_done) cudaEventDestroy(ctx->chunk_done);
    for (auto &ev : ctx->prof_events) { cudaEventDestroy(ev.first); cudaEventDestroy(ev.second); }
    for (auto &ev : ctx->prof_pool) { cudaEventDestroy(ev.first); cudaEventDestroy(ev.second); }
    delete ctx;
    return LANDAU_OK;
}

int landau_create(const landau_mesh *mesh, int order, const landau_species *species, int max_batch, landau_ctx **out) {
    if (!out) return LANDAU_EINVAL;
    *out = nullptr;
    if (!mesh || !species || max_batch < 1) return LANDAU_EINVAL;
    if (species->S < 1 || species->S > MAX_SPECIES || !species->mass || !species->charge) return LANDAU_EINVAL;
    if (!(species->m0 > 0.0)) return LANDAU_EINVAL;
    for (int s = 0; s < species->S; ++s)
        if (!(species->mass[s] > 0.0)) return LANDAU_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        g_cuda_err = "no CUDA device (this library has no CPU fallback)";
        return LANDAU_ECUDA;
    }
    landau_ctx *ctx = new (std::nothrow) landau_ctx();
    if (!ctx) return LANDAU_ENOMEM;
    std::string err;
    int rc;
    try {
        rc = build_host_space(*mesh, order, ctx->hs, err);
    } catch (const std::bad_alloc &) {
        delete ctx;
        return LANDAU_ENOMEM;
    }
    if (rc != LANDAU_OK) { g_cuda_err = err; delete ctx; return rc; }
    HostSpace &hs = ctx->hs;
    if (hs.N > (int64_t(1) << 30) || hs.nnz > (int64_t(1) << 30)) { delete ctx; return LANDAU_EINVAL; }
    DeviceSpace &ds = ctx->ds;
    std::memset(&ds, 0, sizeof(ds));
    ds.p = hs.p; ds.Nq = hs.Nq; ds.Nb = hs.Nb; ds.S = species->S;
    ds.N = int(hs.N); ds.Ne = int(hs.Ne); ds.n = int(hs.n); ds.nnz = int(hs.nnz);
    for (int s = 0; s < ds.S; ++s) {
        const double e2 = species->charge[s] * species->charge[s], mm = species->m0 / species->mass[s];
        ds.e2[s] = e2; ds.m0m[s] = mm;
        ds.kfac[s] = species->nu * e2 * mm;
        ds.dfac[s] = -species->nu * e2 * mm * mm;
        ds.qm[s] = species->charge[s] * mm;
    }
    std::vector<double> invr(hs.N);
    for (int64_t i = 0; i < hs.N; ++i) invr[i] = 1.0 / hs.r[i];
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, dev);
    ctx->max_batch = max_batch;

#define UP(field, vec)                                                   \
    if ((rc = upload(vec, &ds.field, ctx->owned)) != LANDAU_OK) { landau_destroy(ctx); return rc; }
    UP(r, hs.r) UP(z, hs.z) UP(invr, invr) UP(w_in, hs.w_in) UP(w_out, hs.w_out) UP(invJ, hs.invJ)
    UP(B, hs.B) UP(E0, hs.E0) UP(E1, hs.E1)
    UP(lptr, hs.lptr) UP(ldof, hs.ldof) UP(lw, hs.lw)
    UP(rowptr, hs.rowptr) UP(colidx, hs.colidx)
    UP(gptr, hs.gptr) UP(gidx, hs.gidx) UP(gw, hs.gw)
    UP(cptr, hs.cptr) UP(cidx, hs.cidx) UP(cw, hs.cw)
#undef UP
    // scratch arena
    const size_t nbm = size_t(max_batch);
    const size_t gsz = nbm * pair_tiles(ds.N) * 5 * hs.N;
    struct { double **p; size_t n; } allocs[] = {
        {&ctx->sc.T, nbm * 3 * hs.N},
        {&ctx->sc.G, gsz},
        {&ctx->sc.Gsum, nbm * 5 * hs.N},
        {&ctx->sc.Ce, nbm * ds.S * hs.Ne * hs.Nb * hs.Nb},
        {&ctx->sc.ce, nbm * ds.S * hs.Ne * hs.Nb},
    };
    for (auto &a : allocs) {
        void *d = nullptr;
        cudaError_t e = cudaMalloc(&d, a.n * sizeof(double));
        if (e != cudaSuccess) {
            g_cuda_err = std::string("cudaMalloc(scratch): ") + cudaGetErrorString(e);
            landau_destroy(ctx);
            return e == cudaErrorMemoryAllocation ? LANDAU_ENOMEM : LANDAU_ECUDA;
        }
        ctx->owned.push_back(d);
        *a.p = static_cast<double *>(d);
    }
    *out = ctx;
    return LANDAU_OK;
}

int landau_setup_host(const landau_mesh *mesh, int order, int64_t *n, int64_t *nnz, int64_t *N, int32_t *rowptr_host,
                      int32_t *colidx_host, double *dof_r_host, double *dof_z_host) {
    if (!mesh) return LANDAU_EINVAL;
    HostSpace hs;
    std::string err;
    int rc;
    try {
        rc = build_host_space(*mesh, order, hs, err);
    } catch (const std::bad_alloc &) {
        return LANDAU_ENOMEM;
    }
    if (rc != LANDAU_OK) { g_cuda_err = err; return rc; }
    if (n) *n = hs.n;
    if (nnz) *nnz = hs.nnz;
    if (N) *N = hs.N;
    if (rowptr_host) std::memcpy(rowptr_host, hs.rowptr.data(), hs.rowptr.size() * sizeof(int32_t));
    if (colidx_host) std::memcpy(colidx_host, hs.colidx.data(), hs.colidx.size() * sizeof(int32_t));
    if (dof_r_host) std::memcpy(dof_r_host, hs.dof_r.data(), hs.n * sizeof(double));
    if (dof_z_host) std::memcpy(dof_z_host, hs.dof_z.data(), hs.n * sizeof(double));
    return LANDAU_OK;
}

int landau_sizes(const landau_ctx *ctx, int32_t *S, int64_t *n, int64_t *nnz, int64_t *N, int64_t *Ne) {
    if (!ctx) return LANDAU_EINVAL;
    if (S) *S = ctx->ds.S;
    if (n) *n = ctx->hs.n;
    if (nnz) *nnz = ctx->hs.nnz;
    if (N) *N = ctx->hs.N;
    if (Ne) *Ne = ctx->hs.Ne;
    return LANDAU_OK;
}

int landau_csr_pattern(const landau_ctx *ctx, const int32_t **rowptr_dev, const int32_t **colidx_dev) {
    if (!ctx) return LANDAU_EINVAL;
    if (rowptr_dev) *rowptr_dev = ctx->ds.rowptr;
    if (colidx_dev) *colidx_dev = ctx->ds.colidx;
    return LANDAU_OK;
}

int landau_csr_pattern_host(const landau_ctx *ctx, int32_t *rowptr_host, int32_t *colidx_host) {
    if (!ctx) return LANDAU_EINVAL;
    if (rowptr_host) std::memcpy(rowptr_host, ctx->hs.rowptr.data(), ctx->hs.rowptr.size() * sizeof(int32_t));
    if (colidx_host) std::memcpy(colidx_host, ctx->hs.colidx.data(), ctx->hs.colidx.size() * sizeof(int32_t));
    return LANDAU_OK;
}

int landau_dof_coords(const landau_ctx *ctx, double *r_host, double *z_host) {
    if (!ctx) return LANDAU_EINVAL;
    if (r_host) std::memcpy(r_host, ctx->hs.dof_r.data(), ctx->hs.n * sizeof(double));
    if (z_host) std::memcpy(z_host, ctx->hs.dof_z.data(), ctx->hs.n * sizeof(double));
    return LANDAU_OK;
}

int landau_points(const landau_ctx *ctx, double *r_host, double *z_host, double *w_host) {
    if (!ctx) return LANDAU_EINVAL;
    if (r_host) std::memcpy(r_host, ctx->hs.r.data(), ctx->hs.N * sizeof(double));
    if (z_host) std::memcpy(z_host, ctx->hs.z.data(), ctx->hs.N * sizeof(double));
    if (w_host) std::memcpy(w_host, ctx->hs.w_in.data(), ctx->hs.N * sizeof(double));
    return LANDAU_OK;
}

int landau_inner_integral(landau_ctx *ctx, int nb, const double *f_dev, double *G_dev, void *stream) {
    if (!ctx || !f_dev || !G_dev || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    ctx->launches += launch_fields_beta(ctx->ds, nb, f_dev, ctx->sc.T, st);
    ctx->launches += timed_pair(ctx, nb, ctx->sc.G, st);
    ctx->launches += launch_sum_partials(ctx->ds, nb, pair_tiles(ctx->ds.N), ctx->sc.G, G_dev, st);
    CK(cudaGetLastError());
    return LANDAU_OK;
}

int landau_jacobian_batched(landau_ctx *ctx, int nb, const double *f_dev, double *vals_dev, double *Cf_dev, void *stream) {
    if (!ctx || !f_dev || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const DeviceSpace &ds = ctx->ds;
    ctx->launches += launch_fields_beta(ds, nb, f_dev, ctx->sc.T, st);
    ctx->launches += timed_pair(ctx, nb, ctx->sc.G, st);
    ctx->launches += launch_sum_partials(ds, nb, pair_tiles(ds.N), ctx->sc.G, ctx->sc.Gsum, st);
    ctx->launches += launch_element(ds, nb, 1, f_dev, ctx->sc.Gsum, ctx->sc.Ce, ctx->sc.ce, nullptr, 0.0, st);
    if (vals_dev) ctx->launches += launch_gather_vals(ds, nb * ds.S, ctx->sc.Ce, vals_dev, st);
    if (Cf_dev) ctx->launches += launch_gather_cf(ds, nb * ds.S, ctx->sc.ce, Cf_dev, st);
    CK(cudaGetLastError());
    return LANDAU_OK;
}

int landau_implicit_operator_batched(landau_ctx *ctx, int nb, const double *f_dev, const double *Ez_dev, double shift,
                                     double *vals_dev, double *F_dev, void *stream) {
    if (!ctx || !f_dev || !Ez_dev || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const DeviceSpace &ds = ctx->ds;
    ctx->launches += launch_fields_beta(ds, nb, f_dev, ctx->sc.T, st);
    ctx->launches += timed_pair(ctx, nb, ctx->sc.G, st);
    ctx->launches += launch_sum_partials(ds, nb, pair_tiles(ds.N), ctx->sc.G, ctx->sc.Gsum, st);
    ctx->launches += launch_element(ds, nb, 1, f_dev, ctx->sc.Gsum, ctx->sc.Ce, ctx->sc.ce, Ez_dev, shift, st);
    if (vals_dev) ctx->launches += launch_gather_vals(ds, nb * ds.S, ctx->sc.Ce, vals_dev, st);
    if (F_dev) ctx->launches += launch_gather_cf(ds, nb * ds.S, ctx->sc.ce, F_dev, st);
    CK(cudaGetLastError());
    return LANDAU_OK;
}

int landau_jacobian(landau_ctx *ctx, const double *f_dev, double *vals_dev, double *Cf_dev, void *stream) {
    return landau_jacobian_batched(ctx, 1, f_dev, vals_dev, Cf_dev, stream);
}

int landau_mass(landau_ctx *ctx, double shift, double *mvals_dev, void *stream) {
    if (!ctx || !mvals_dev) return LANDAU_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    ctx->launches += launch_mass_element(ctx->ds, shift, ctx->sc.Ce, st);
    ctx->launches += launch_gather_vals(ctx->ds, 1, ctx->sc.Ce, mvals_dev, st);
    CK(cudaGetLastError());
    return LANDAU_OK;
}

int landau_jacobian_host(landau_ctx *ctx, int nb, const double *f_host, double *vals_host, double *Cf_host) {
    if (!ctx || !f_host || nb < 1 || nb > ctx->max_batch) return LANDAU_EINVAL;
    const DeviceSpace &ds = ctx->ds;
    if (!ctx->own_stream) {
        CK(cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&ctx->chunk_done, cudaEventDisableTiming));
    }
    if (ctx->host_nb < nb) {
        if (ctx->d_f) { cudaFree(ctx->d_f); cudaFree(ctx->d_vals); cudaFree(ctx->d_Cf); ctx->d_f = ctx->d_vals = ctx->d_Cf = nullptr; }
        cudaError_t e = cudaMalloc((void **)&ctx->d_f, size_t(nb) * ds.S * ds.n * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->d_vals, size_t(nb) * ds.S * ds.nnz * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void **)&ctx->d_Cf, size_t(nb) * ds.S * ds.n * sizeof(double));
        if (e != cudaSuccess) { ctx->host_nb = 0; return cuda_fail(e, "cudaMalloc(host staging)"); }
        ctx->host_nb = nb;
    }
    // Pipeline over sub-batches: the device-to-host copy of chunk c overlaps the build of chunk
    // c+1 (the scratch arena is reused in stream order; problems are independent, so the values
    // are bitwise those of one batched call).
    cudaStream_t st = ctx->own_stream, cp = ctx->copy_stream;
    const size_t fsz = size_t(ds.S) * ds.n, vsz = size_t(ds.S) * ds.nnz;
    CK(cudaMemcpyAsync(ctx->d_f, f_host, size_t(nb) * fsz * sizeof(double), cudaMemcpyHostToDevice, st));
    const int nchunks = nb >= 8 ? 4 : 1;
    const int cb = (nb + nchunks - 1) / nchunks;
    for (int b0 = 0; b0 < nb; b0 += cb) {
        const int nbc = std::min(cb, nb - b0);
        int rc = landau_jacobian_batched(ctx, nbc, ctx->d_f + b0 * fsz, vals_host ? ctx->d_vals + b0 * vsz : nullptr,
                                         Cf_host ? ctx->d_Cf + b0 * fsz : nullptr, st);
        if (rc != LANDAU_OK) return rc;
        CK(cudaEventRecord(ctx->chunk_done, st));
        CK(cudaStreamWaitEvent(cp, ctx->chunk_done, 0));
        if (vals_host) CK(cudaMemcpyAsync(vals_host + b0 * vsz, ctx->d_vals + b0 * vsz, size_t(nbc) * vsz * sizeof(double), cudaMemcpyDeviceToHost, cp));
        if (Cf_host) CK(cudaMemcpyAsync(Cf_host + b0 * fsz, ctx->d_Cf + b0 * fsz, size_t(nbc) * fsz * sizeof(double), cudaMemcpyDeviceToHost, cp));
    }
    CK(cudaStreamSynchronize(st));
    CK(cudaStreamSynchronize(cp));
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

int landau_profile_read(landau_ctx *ctx, double *pair_ms_total, int64_t *pair_launches) {
    if (!ctx || !pair_ms_total || !pair_launches) return LANDAU_EINVAL;
    double total = 0.0;
    for (auto &ev : ctx->prof_events) {
        CK(cudaEventSynchronize(ev.second));
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, ev.first, ev.second));
        total += ms;
        ctx->prof_pool.push_back(ev);
    }
    *pair_ms_total = total;
    *pair_launches = int64_t(ctx->prof_events.size());
    ctx->prof_events.clear();
    return LANDAU_OK;
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

}  // extern "C"
