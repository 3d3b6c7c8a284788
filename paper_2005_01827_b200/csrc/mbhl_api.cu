// mbhl_api.cu - host side of the C ABI declared in include/mbhl.h.
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>
#include <vector>

#include "mbhl.h"
#include "mbhl_kernels.cuh"

using namespace mbhl;

struct mbhl_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int S = 1024;
    uint32_t mode_mask = 0x3F;
    double t0 = 0.0;
    int64_t N = 0;
    double f_min = 0.0, f_max = 0.0, df = 0.0, dd = 0.0;
    // library-owned device data
    double* freqs = nullptr;
    double* tiles = nullptr;               // [n_chunks][10][512] staged layout of f, w, w d (mbhl_kernels.cuh)
    unsigned long long* counters = nullptr;
    // workspace
    void* ws_internal = nullptr;
    size_t ws_internal_bytes = 0;
    void* ws_user = nullptr;
    size_t ws_user_bytes = 0;
    int64_t launches = 0;
    bool timing = false;
    int n_timed = 0;                       // calls recorded since timing was (re-)enabled
    static constexpr int kSlots = 64;      // ring of event sets, one per call
    cudaEvent_t evs[kSlots][6] = {};
    cudaEvent_t* ev = evs[0];
    char err[512] = {0};
};

namespace {

constexpr int64_t kSliceBatch = 32768;   // walkers per pass of the hot path; larger batches are processed in slices

struct WsLayout {
    size_t params, consts, dense, knots, coef, partials, dh, hh, logl, total;
};

// Launch shape of the fused dense kernel: W walkers per CTA tile, G chunks per CTA.  W amortises the staged
// data tile (HBM traffic = data bytes x B / W); both shrink for small problems so the grid still fills 148 SMs.
struct DensePlan {
    int W, G, n_tiles, n_groups;
};

#ifndef MBHL_DENSE_MAXG
#define MBHL_DENSE_MAXG 32
#endif
constexpr int kDenseMaxG = MBHL_DENSE_MAXG;   // chunks per CTA at most: amortises a CTA's start-up over ~0.5 ms of work

DensePlan dense_plan(int64_t B, int n_chunks) {
    DensePlan p;
    int64_t w = B * (int64_t)n_chunks / 4096;
    p.W = (int)(w < 1 ? 1 : (w > kMaxW ? kMaxW : w));
    p.n_tiles = (int)((B + p.W - 1) / p.W);
    int64_t g = (int64_t)p.n_tiles * n_chunks / 8192;
    p.G = (int)(g < 1 ? 1 : (g > kDenseMaxG ? kDenseMaxG : g));
    p.n_groups = (n_chunks + p.G - 1) / p.G;
    return p;
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

int n_chunks_of(int64_t N) { return (int)((N + kChunk - 1) / kChunk); }

// Entries of the partials buffer for any batch b' <= b: b' n_groups(b') is not monotone in b' (G and W grow with the
// batch), so the workspace is sized by a bound that is: b' ceil(n_chunks / G_max) once G has reached its maximum, and
// at most 131072 + 8 b' before that (G >= g/2 for g = n_tiles n_chunks / 8192 >= 1, and b' n_chunks < 65536 for g < 1).
size_t partials_capacity(size_t b, int n_chunks) {
    return b * (size_t)((n_chunks + kDenseMaxG - 1) / kDenseMaxG) + 131072 + 8 * b;
}

WsLayout layout(const mbhl_ctx* c, int64_t B) {
    WsLayout L;
    size_t off = 0;
    if (B > kSliceBatch) B = kSliceBatch;        // larger batches run in slices of kSliceBatch walkers
    const size_t b = (size_t)(B > 0 ? B : 1);
    L.params = off; off += align256(b * MBHL_NPARAM * sizeof(double));
    L.consts = off; off += align256(b * sizeof(WalkerConst));
    L.dense = off; off += align256(b * sizeof(DenseWalker));
    L.knots = off; off += align256(b * MBHL_NMODE * c->S * sizeof(double));
    L.coef = off; off += align256(b * MBHL_NMODE * (size_t)(c->S - 1) * kCoefStride * sizeof(double));
    L.partials = off; off += align256(partials_capacity(b, n_chunks_of(c->N)) * 2 * sizeof(double));
    L.dh = off; off += align256(b * sizeof(double));
    L.hh = off; off += align256(b * sizeof(double));
    L.logl = off; off += align256(b * sizeof(double));
    L.total = off;
    return L;
}

int fail(mbhl_ctx* c, int code, const char* what, cudaError_t e = cudaSuccess) {
    if (c) {
        if (e != cudaSuccess) snprintf(c->err, sizeof(c->err), "%s: %s", what, cudaGetErrorString(e));
        else snprintf(c->err, sizeof(c->err), "%s", what);
    }
    return code;
}

#define CU(call)                                                      \
    do {                                                              \
        cudaError_t e_ = (call);                                      \
        if (e_ != cudaSuccess) return fail(ctx, MBHL_ECUDA, #call, e_); \
    } while (0)

int get_workspace(mbhl_ctx* ctx, int64_t B, char** base) {
    const size_t need = layout(ctx, B).total;
    if (ctx->ws_user) {
        if (ctx->ws_user_bytes < need) return fail(ctx, MBHL_ENOWS, "caller workspace too small for this batch");
        *base = (char*)ctx->ws_user;
        return MBHL_OK;
    }
    if (ctx->ws_internal_bytes < need) {
        if (ctx->ws_internal) {
            CU(cudaStreamSynchronize(ctx->stream));
            cudaFree(ctx->ws_internal);
            ctx->ws_internal = nullptr;
            ctx->ws_internal_bytes = 0;
        }
        cudaError_t e = cudaMalloc(&ctx->ws_internal, need);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return fail(ctx, MBHL_ENOMEM, "cudaMalloc(workspace)", e);
        }
        ctx->ws_internal_bytes = need;
    }
    *base = (char*)ctx->ws_internal;
    return MBHL_OK;
}

bool is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// The fused sparse kernel's dynamic shared memory limit is per function and per device, not per context: keep the
// running maximum so that contexts with different S can coexist (several contexts may be alive at once, mbhl.h).
int ensure_spline_smem(mbhl_ctx* ctx) {
    static size_t granted[64] = {0};
    static std::mutex mu;                                // contexts on different host threads share this table
    std::lock_guard<std::mutex> lock(mu);
    const size_t need = spline_smem_bytes(ctx->S);
    const int d = ctx->device & 63;
    if (granted[d] < need) {
        CU(cudaFuncSetAttribute(k_sparse_spline, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need));
        granted[d] = need;
    }
    return MBHL_OK;
}

// Step a1 + a2 for rows[B][11] on the device, given in the coordinates `coords` (MBHL_COORDS_*).
void run_consts(mbhl_ctx* ctx, const double* rows_dev, int64_t B, int coords, char* base, const WsLayout& L) {
    k_walker_consts<<<(unsigned)((B + kConstsWarps - 1) / kConstsWarps), 32 * kConstsWarps, 0, ctx->stream>>>(
        rows_dev, B, coords, ctx->t0, ctx->f_min, ctx->f_max, ctx->S, ctx->mode_mask, ctx->freqs, (int)ctx->N, ctx->df,
        (WalkerConst*)(base + L.consts), (DenseWalker*)(base + L.dense), (double*)(base + L.params));
    ctx->launches += 1;
}

// Runs the sparse stage (a1-a5) for rows already on the device: the per-walker constants, then (with_coef) the fused
// PhenomHM + response + spline kernel, one cluster of two CTAs per (walker, mode).  y_out: optional export of the knot values.
int run_sparse(mbhl_ctx* ctx, const double* rows_dev, int64_t B, int coords, char* base, const WsLayout& L, bool with_coef,
               double* y_out = nullptr) {
    const int S = ctx->S;
    const bool tm = ctx->timing && with_coef;
    if (tm) ctx->ev = ctx->evs[ctx->n_timed % mbhl_ctx::kSlots];
    if (tm) cudaEventRecord(ctx->ev[0], ctx->stream);
    run_consts(ctx, rows_dev, B, coords, base, L);
    if (tm) cudaEventRecord(ctx->ev[1], ctx->stream);
    if (with_coef) {
        int rc = ensure_spline_smem(ctx);
        if (rc != MBHL_OK) return rc;
        k_sparse_spline<<<(unsigned)(B * MBHL_NMODE * 2), kSplineThreads, spline_smem_bytes(S), ctx->stream>>>(
            (const WalkerConst*)(base + L.consts), S, (double*)(base + L.knots), (double*)(base + L.coef), y_out);
        ctx->launches += 1;
    }
    if (tm) { cudaEventRecord(ctx->ev[2], ctx->stream); cudaEventRecord(ctx->ev[3], ctx->stream); }
    CU(cudaGetLastError());
    return MBHL_OK;
}

// Fused dense kernel + final reduction for the sparse stage results sitting in the workspace.
int run_dense(mbhl_ctx* ctx, int64_t B, char* base, const WsLayout& L, uint32_t mode_mask, double* d_h, double* h_h, double* logL,
              int64_t stride, bool count_work) {
    const DensePlan P = dense_plan(B, n_chunks_of(ctx->N));
    DenseArgs A;
    A.dw = (const DenseWalker*)(base + L.dense);
    A.knots = (const double*)(base + L.knots);
    A.coef = (const double*)(base + L.coef);
    A.tiles = ctx->tiles;
    A.partials = (double*)(base + L.partials);
    A.B = (int)B;
    A.S = ctx->S;
    A.W = P.W;
    A.G = P.G;
    A.n_chunks = n_chunks_of(ctx->N);
    A.n_groups = P.n_groups;
    A.inv_df = 1.0 / ctx->df;
    A.mode_mask = mode_mask;
    if (count_work) CU(cudaMemsetAsync(ctx->counters, 0, 8 * sizeof(unsigned long long), ctx->stream));
    A.work = count_work ? ctx->counters + 2 : nullptr;
    const bool tm = ctx->timing && count_work;
    if (tm) cudaEventRecord(ctx->ev[3], ctx->stream);
    k_dense<<<(unsigned)((int64_t)P.n_groups * P.n_tiles), kDenseThreads, kDenseSmemBytes, ctx->stream>>>(A);
    if (tm) cudaEventRecord(ctx->ev[4], ctx->stream);
    k_final_reduce<<<(unsigned)B, 128, 0, ctx->stream>>>(A.dw, A.partials, A.n_groups, B, ctx->dd, d_h, h_h, logL,
                                                                    count_work ? ctx->counters : nullptr, stride);
    if (tm) { cudaEventRecord(ctx->ev[5], ctx->stream); ctx->n_timed += 1; }
    ctx->launches += 2;
    CU(cudaGetLastError());
    return MBHL_OK;
}

}  // namespace

extern "C" {

const char* mbhl_strerror(int code) {
    switch (code) {
        case MBHL_OK: return "ok";
        case MBHL_EINVAL: return "invalid argument";
        case MBHL_ENOMEM: return "out of memory";
        case MBHL_ECUDA: return "CUDA error";
        case MBHL_ENOWS: return "workspace too small";
        default: return "unknown error";
    }
}

const char* mbhl_last_error(const mbhl_ctx* ctx) { return ctx ? ctx->err : "null context"; }

void mbhl_free(mbhl_ctx* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    cudaFree(ctx->freqs);
    cudaFree(ctx->tiles);
    cudaFree(ctx->counters);
    cudaFree(ctx->ws_internal);
    for (int k = 0; k < mbhl_ctx::kSlots; ++k)
        for (int i = 0; i < 6; ++i)
            if (ctx->evs[k][i]) cudaEventDestroy(ctx->evs[k][i]);
    delete ctx;
}

int mbhl_init(mbhl_ctx** out, const double* freqs, int64_t N, const double* data_AET, const double* psd_AET,
              const mbhl_config* cfg) {
    if (!out) return MBHL_EINVAL;
    *out = nullptr;
    if (!freqs || !data_AET || !psd_AET || N < 4 || N > ((int64_t)1 << 31) - 2 * kChunk) return MBHL_EINVAL;
    mbhl_ctx* ctx = new (std::nothrow) mbhl_ctx();
    if (!ctx) return MBHL_ENOMEM;
    if (cfg) {
        ctx->device = cfg->device;
        ctx->stream = (cudaStream_t)cfg->stream;
        if (cfg->sparse_points) ctx->S = cfg->sparse_points;
        if (cfg->mode_mask) ctx->mode_mask = cfg->mode_mask & 0x3F;
        ctx->t0 = cfg->t0;
    }
    ctx->N = N;
    int rc = MBHL_OK;
    double *d_data = nullptr, *d_psd = nullptr, *d_part = nullptr;
    std::vector<double> host_part;
    auto cleanup = [&](int code) {
        cudaFree(d_data);
        cudaFree(d_psd);
        cudaFree(d_part);
        if (code != MBHL_OK) {
            cudaFree(ctx->freqs); cudaFree(ctx->tiles); cudaFree(ctx->counters);
            delete ctx;
        }
        return code;
    };
    if (ctx->S < 8 || ctx->S > 2048 || !isfinite(ctx->t0)) return cleanup(MBHL_EINVAL);   // mbhl.h: 8 <= S <= 2048
    if (spline_smem_bytes(ctx->S) > 227 * 1024) return cleanup(MBHL_EINVAL);   // S <= ~2170 fits one CTA's shared memory
    if (cudaSetDevice(ctx->device) != cudaSuccess) return cleanup(MBHL_ECUDA);
    if (cudaMemcpyToSymbol(c_table, MBHL_TABLE_HOST, sizeof(double) * MBHL_TABLE_N) != cudaSuccess) return cleanup(MBHL_ECUDA);
    {
        // Table I: ln M_T, q, a1, a2, ln D_L, phi_ref, cos iota, lambda, sin beta, psi, ln t_ref
        const double lo[MBHL_NPARAM] = {log(1e3), 0.05, -0.99, -0.99, log(0.044), 0.0, -1.0, 0.0, -1.0, 0.0, log(1.0)};
        const double hi[MBHL_NPARAM] = {log(1e9), 1.0, 0.99, 0.99, log(1298.00), 2.0 * M_PI, 1.0, 2.0 * M_PI, 1.0, M_PI, log(3.15576e8)};
        if (cudaMemcpyToSymbol(c_prior_lo, lo, sizeof(lo)) != cudaSuccess || cudaMemcpyToSymbol(c_prior_hi, hi, sizeof(hi)) != cudaSuccess)
            return cleanup(MBHL_ECUDA);
    }
    if (cudaFuncSetAttribute(k_sparse_spline, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared) != cudaSuccess ||
        cudaFuncSetAttribute(k_dense, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared) != cudaSuccess)
        return cleanup(MBHL_ECUDA);
    if (cudaFuncSetAttribute(k_dense, cudaFuncAttributeMaxDynamicSharedMemorySize, kDenseSmemBytes) != cudaSuccess)
        return cleanup(MBHL_ECUDA);
    const size_t nb = (size_t)N * sizeof(double);
    const int nblk = (int)((N + 1023) / 1024) > n_chunks_of(N) ? (int)((N + 1023) / 1024) : n_chunks_of(N);
    if (cudaMalloc(&ctx->freqs, nb) != cudaSuccess ||
        cudaMalloc(&ctx->tiles, (size_t)n_chunks_of(N) * kTileBytes) != cudaSuccess ||
        cudaMalloc(&ctx->counters, 8 * sizeof(unsigned long long)) != cudaSuccess ||
        cudaMalloc(&d_part, (size_t)nblk * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        return cleanup(MBHL_ENOMEM);
    }
    cudaStream_t st = ctx->stream;
    // freqs
    if (cudaMemcpyAsync(ctx->freqs, freqs, nb, cudaMemcpyDefault, st) != cudaSuccess) return cleanup(MBHL_ECUDA);
    const double* data_dev = data_AET;
    const double* psd_dev = psd_AET;
    if (!is_device_ptr(data_AET)) {
        if (cudaMalloc(&d_data, 6 * nb) != cudaSuccess) { cudaGetLastError(); return cleanup(MBHL_ENOMEM); }
        if (cudaMemcpyAsync(d_data, data_AET, 6 * nb, cudaMemcpyHostToDevice, st) != cudaSuccess) return cleanup(MBHL_ECUDA);
        data_dev = d_data;
    }
    if (!is_device_ptr(psd_AET)) {
        if (cudaMalloc(&d_psd, 3 * nb) != cudaSuccess) { cudaGetLastError(); return cleanup(MBHL_ENOMEM); }
        if (cudaMemcpyAsync(d_psd, psd_AET, 3 * nb, cudaMemcpyHostToDevice, st) != cudaSuccess) return cleanup(MBHL_ECUDA);
        psd_dev = d_psd;
    }
    // grid: end points, spacing, validation
    double ends[2];
    if (cudaMemcpyAsync(&ends[0], ctx->freqs, sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemcpyAsync(&ends[1], ctx->freqs + (N - 1), sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return cleanup(MBHL_ECUDA);
    ctx->f_min = ends[0];
    ctx->f_max = ends[1];
    ctx->df = (ends[1] - ends[0]) / (double)(N - 1);
    if (!(ctx->f_min > 0.0) || !(ctx->df > 0.0) || !isfinite(ctx->f_max)) return cleanup(MBHL_EINVAL);
    const int ngrid = (int)((N + 1023) / 1024);
    host_part.resize(ngrid);
    k_check_grid<<<ngrid, 256, 0, st>>>(ctx->freqs, N, ctx->df, d_part);
    if (cudaMemcpyAsync(host_part.data(), d_part, (size_t)ngrid * sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return cleanup(MBHL_ECUDA);
    for (int i = 0; i < ngrid; ++i)
        if (!(host_part[i] <= 1e-6)) return cleanup(MBHL_EINVAL);
    // data tiles (weights, weighted data) and <d|d>
    const int nch = n_chunks_of(N);
    host_part.resize(nch);
    k_init_tiles<<<nch, 256, 0, st>>>(ctx->freqs, data_dev, psd_dev, N, ctx->df, ctx->tiles, d_part);
    if (cudaMemcpyAsync(host_part.data(), d_part, (size_t)nch * sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemsetAsync(ctx->counters, 0, 8 * sizeof(unsigned long long), st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return cleanup(MBHL_ECUDA);
    ctx->launches += 2;
    {
        // pairwise (fixed-order) host sum of the per-block partials
        std::vector<double> v(host_part);
        size_t n = v.size();
        while (n > 1) {
            size_t h = (n + 1) / 2;
            for (size_t i = 0; i + h < n; ++i) v[i] += v[i + h];
            n = h;
        }
        ctx->dd = v[0];
    }
    if (cfg && cfg->max_batch > 0) {
        char* base;
        rc = get_workspace(ctx, cfg->max_batch, &base);
        if (rc != MBHL_OK) return cleanup(rc);
    }
    // function attributes now, not in the hot path: with max_batch set, mbhl_loglike* then only enqueues kernels and one
    // memset on the context's stream (no allocation, no synchronisation), so a caller may capture it in a CUDA graph
    rc = ensure_spline_smem(ctx);
    if (rc != MBHL_OK) return cleanup(rc);
    cleanup(MBHL_OK);
    *out = ctx;
    return MBHL_OK;
}

size_t mbhl_workspace_bytes(const mbhl_ctx* ctx, int64_t B) { return ctx ? layout(ctx, B).total : 0; }

int mbhl_set_workspace(mbhl_ctx* ctx, void* dev_ptr, size_t bytes) {
    if (!ctx) return MBHL_EINVAL;
    if (dev_ptr && ((uintptr_t)dev_ptr & 255)) return fail(ctx, MBHL_EINVAL, "workspace must be 256-byte aligned");
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->ws_user = dev_ptr;
    ctx->ws_user_bytes = dev_ptr ? bytes : 0;
    return MBHL_OK;
}

double mbhl_data_norm(const mbhl_ctx* ctx) { return ctx ? ctx->dd : NAN; }
int64_t mbhl_num_bins(const mbhl_ctx* ctx) { return ctx ? ctx->N : 0; }
int32_t mbhl_sparse_points(const mbhl_ctx* ctx) { return ctx ? ctx->S : 0; }
int64_t mbhl_launch_count(const mbhl_ctx* ctx) { return ctx ? ctx->launches : 0; }

}  // extern "C"

namespace {

// The hot path for rows[B][11] given in the coordinates `coords`; batches above kSliceBatch go in slices, so the
// workspace stays that of one slice.
int loglike_impl(mbhl_ctx* ctx, const double* rows, int64_t B, int coords, double* d_h, double* h_h, double* logL) {
    if (!ctx) return MBHL_EINVAL;
    if (B < 0 || (B > 0 && !rows) || coords < 0 || coords > 2) return fail(ctx, MBHL_EINVAL, "bad rows/B/coords");
    if (B == 0) return MBHL_OK;
    CU(cudaSetDevice(ctx->device));
    for (int64_t o = 0; o < B; o += kSliceBatch) {
        const int64_t n = (B - o < kSliceBatch) ? (B - o) : kSliceBatch;
        char* base;
        int rc = get_workspace(ctx, n, &base);
        if (rc != MBHL_OK) return rc;
        const WsLayout L = layout(ctx, n);
        rc = run_sparse(ctx, rows + o * MBHL_NPARAM, n, coords, base, L, true);
        if (rc != MBHL_OK) return rc;
        rc = run_dense(ctx, n, base, L, ctx->mode_mask, d_h ? d_h + o : nullptr, h_h ? h_h + o : nullptr, logL ? logL + o : nullptr, 1, true);
        if (rc != MBHL_OK) return rc;
    }
    return MBHL_OK;
}

}  // namespace

extern "C" {

int mbhl_loglike_parts(mbhl_ctx* ctx, const double* params, int64_t B, double* d_h, double* h_h, double* logL) {
    return loglike_impl(ctx, params, B, MBHL_COORDS_PHYSICAL, d_h, h_h, logL);
}

int mbhl_loglike(mbhl_ctx* ctx, const double* params, int64_t B, double* logL) {
    if (ctx && B > 0 && !logL) return fail(ctx, MBHL_EINVAL, "logL is null");
    return mbhl_loglike_parts(ctx, params, B, nullptr, nullptr, logL);
}

int mbhl_loglike_host(mbhl_ctx* ctx, const double* params_host, int64_t B, double* logL_host) {
    if (!ctx) return MBHL_EINVAL;
    if (B < 0 || (B > 0 && (!params_host || !logL_host))) return fail(ctx, MBHL_EINVAL, "bad host buffers");
    if (B == 0) return MBHL_OK;
    if (B > kSliceBatch) {   // the staging areas live in the workspace of ONE slice: go slice by slice
        for (int64_t o = 0; o < B; o += kSliceBatch) {
            const int rc = mbhl_loglike_host(ctx, params_host + o * MBHL_NPARAM, (B - o < kSliceBatch) ? (B - o) : kSliceBatch, logL_host + o);
            if (rc != MBHL_OK) return rc;
        }
        return MBHL_OK;
    }
    CU(cudaSetDevice(ctx->device));
    char* base;
    int rc = get_workspace(ctx, B, &base);
    if (rc != MBHL_OK) return rc;
    const WsLayout L = layout(ctx, B);
    double* p_dev = (double*)(base + L.params);
    double* l_dev = (double*)(base + L.logl);
    CU(cudaMemcpyAsync(p_dev, params_host, (size_t)B * MBHL_NPARAM * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    rc = loglike_impl(ctx, p_dev, B, MBHL_COORDS_PHYSICAL, nullptr, nullptr, l_dev);
    if (rc != MBHL_OK) return rc;
    CU(cudaMemcpyAsync(logL_host, l_dev, (size_t)B * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MBHL_OK;
}

int mbhl_mode_products(mbhl_ctx* ctx, const double* params, int64_t B, double* d_h, double* h_h) {
    if (!ctx) return MBHL_EINVAL;
    if (B < 0 || (B > 0 && !params)) return fail(ctx, MBHL_EINVAL, "bad params/B");
    if (B == 0) return MBHL_OK;
    CU(cudaSetDevice(ctx->device));
    const bool tm = ctx->timing;
    ctx->timing = false;
    int rc = MBHL_OK;
    for (int64_t o = 0; o < B && rc == MBHL_OK; o += kSliceBatch) {
        const int64_t n = (B - o < kSliceBatch) ? (B - o) : kSliceBatch;
        char* base;
        rc = get_workspace(ctx, n, &base);
        if (rc != MBHL_OK) break;
        const WsLayout L = layout(ctx, n);
        rc = run_sparse(ctx, params + o * MBHL_NPARAM, n, MBHL_COORDS_PHYSICAL, base, L, true);
        for (int mi = 0; mi < MBHL_NMODE && rc == MBHL_OK; ++mi)
            rc = run_dense(ctx, n, base, L, ctx->mode_mask & (1u << mi), d_h ? d_h + o * MBHL_NMODE + mi : nullptr,
                           h_h ? h_h + o * MBHL_NMODE + mi : nullptr, nullptr, MBHL_NMODE, false);
    }
    ctx->timing = tm;
    return rc;
}

int mbhl_loglike_coords(mbhl_ctx* ctx, const double* rows, int64_t B, int32_t coords, double* logL) {
    if (ctx && B > 0 && !logL) return fail(ctx, MBHL_EINVAL, "logL is null");
    return loglike_impl(ctx, rows, B, coords, nullptr, nullptr, logL);
}

int mbhl_loglike_sampled(mbhl_ctx* ctx, const double* theta, int64_t B, double* logL) {
    return mbhl_loglike_coords(ctx, theta, B, MBHL_COORDS_SAMPLED, logL);
}

int mbhl_unpack_coords(mbhl_ctx* ctx, const double* rows, int64_t B, int32_t coords, double* params_out) {
    if (!ctx) return MBHL_EINVAL;
    if (B < 0 || (B > 0 && (!rows || !params_out)) || coords < 0 || coords > 2) return fail(ctx, MBHL_EINVAL, "bad rows/B/coords/params_out");
    CU(cudaSetDevice(ctx->device));
    for (int64_t o = 0; o < B; o += kSliceBatch) {
        const int64_t n = (B - o < kSliceBatch) ? (B - o) : kSliceBatch;
        char* base;
        int rc = get_workspace(ctx, n, &base);
        if (rc != MBHL_OK) return rc;
        const WsLayout L = layout(ctx, n);
        run_consts(ctx, rows + o * MBHL_NPARAM, n, coords, base, L);
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(params_out + o * MBHL_NPARAM, base + L.params, (size_t)n * MBHL_NPARAM * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    }
    return MBHL_OK;
}

// ---------------------------------------------------------------------------------------------
// parallel-tempered stretch-move ensemble driving the likelihood on the device
// ---------------------------------------------------------------------------------------------
struct mbhl_pt {
    mbhl_ctx* ctx = nullptr;
    PtState s = {};
    void* mem = nullptr;
    uint32_t step = 0;
    int coords = MBHL_COORDS_SAMPLED;
};

int mbhl_pt_init(mbhl_ctx* ctx, mbhl_pt** out, const double* theta0, const double* betas_host, int32_t n_temps,
                 int32_t n_walkers, uint64_t seed, double stretch_a, int32_t coords) {
    if (!ctx || !out) return MBHL_EINVAL;
    *out = nullptr;
    if (!theta0 || !betas_host || n_temps < 1 || n_walkers < 2 || (n_walkers & 1) || !(stretch_a > 1.0) ||
        (int64_t)n_temps * n_walkers > 65535 || (coords != MBHL_COORDS_SAMPLED && coords != MBHL_COORDS_SAMPLED_LISA))
        return fail(ctx, MBHL_EINVAL, "mbhl_pt_init: need n_temps >= 1, an even n_walkers >= 2, n_temps * n_walkers <= 65535, a > 1, sampled coords");
    for (int t = 0; t < n_temps; ++t)
        if (!(betas_host[t] >= 0.0) || !isfinite(betas_host[t])) return fail(ctx, MBHL_EINVAL, "mbhl_pt_init: betas must be finite and >= 0");
    CU(cudaSetDevice(ctx->device));
    mbhl_pt* pt = new (std::nothrow) mbhl_pt();
    if (!pt) return MBHL_ENOMEM;
    pt->ctx = ctx;
    pt->coords = coords;
    const size_t T = (size_t)n_temps, K = (size_t)n_walkers, H = K / 2;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align256(bytes); return o; };
    const size_t o_theta = take(T * K * MBHL_NPARAM * 8), o_logl = take(T * K * 8), o_betas = take(T * 8);
    const size_t o_pth = take(T * H * MBHL_NPARAM * 8), o_pl = take(T * H * 8), o_pz = take(T * H * 8);
    const size_t o_acc = take(T * 8), o_swp = take(T * 8);
    if (cudaMalloc(&pt->mem, off) != cudaSuccess) {
        cudaGetLastError();
        delete pt;
        return fail(ctx, MBHL_ENOMEM, "mbhl_pt_init: cudaMalloc");
    }
    char* m = (char*)pt->mem;
    PtState& s = pt->s;
    s.theta = (double*)(m + o_theta); s.logl = (double*)(m + o_logl); s.betas = (double*)(m + o_betas);
    s.prop_theta = (double*)(m + o_pth); s.prop_logl = (double*)(m + o_pl);
    s.prop_z = (double*)(m + o_pz); s.n_accept = (unsigned long long*)(m + o_acc); s.n_swap = (unsigned long long*)(m + o_swp);
    s.T = n_temps; s.K = n_walkers; s.a = stretch_a; s.seed = seed;
    int rc = MBHL_OK;
    auto bail = [&](int code) { cudaFree(pt->mem); delete pt; return code; };
    if (cudaMemcpyAsync(s.theta, theta0, T * K * MBHL_NPARAM * 8, cudaMemcpyDefault, ctx->stream) != cudaSuccess ||
        cudaMemcpyAsync(s.betas, betas_host, T * 8, cudaMemcpyHostToDevice, ctx->stream) != cudaSuccess ||
        cudaMemsetAsync(s.n_accept, 0, 2 * align256(T * 8), ctx->stream) != cudaSuccess)
        return bail(fail(ctx, MBHL_ECUDA, "mbhl_pt_init: copies"));
    // log-likelihood of the starting positions.  Every walker must start inside the prior box of Table I with a finite
    // logL: with beta = 0 on the hottest rung a walker at logL = -inf would give 0 x (-inf) = NaN in the
    // acceptance ratio and could never move; accepted proposals always have a finite logL, so this holds for the whole run.
    rc = loglike_impl(ctx, s.theta, (int64_t)(T * K), coords, nullptr, nullptr, s.logl);
    if (rc != MBHL_OK) return bail(rc);
    std::vector<double> l0(T * K);
    if (cudaMemcpyAsync(l0.data(), s.logl, T * K * 8, cudaMemcpyDeviceToHost, ctx->stream) != cudaSuccess ||
        cudaStreamSynchronize(ctx->stream) != cudaSuccess)
        return bail(fail(ctx, MBHL_ECUDA, "mbhl_pt_init: sync"));
    for (size_t i = 0; i < T * K; ++i)
        if (!isfinite(l0[i])) return bail(fail(ctx, MBHL_EINVAL, "mbhl_pt_init: a starting walker lies outside the prior box or has no finite logL"));
    *out = pt;
    return MBHL_OK;
}

int mbhl_pt_step(mbhl_pt* pt, int32_t n_steps) {
    if (!pt || n_steps < 0) return MBHL_EINVAL;
    mbhl_ctx* ctx = pt->ctx;
    CU(cudaSetDevice(ctx->device));
    const PtState& s = pt->s;
    const int M = s.T * (s.K / 2);
    for (int it = 0; it < n_steps; ++it, ++pt->step) {
        for (int half = 0; half < 2; ++half) {
            k_pt_propose<<<(M + 127) / 128, 128, 0, ctx->stream>>>(s, half, 2u * pt->step + (uint32_t)half);
            int rc = loglike_impl(ctx, s.prop_theta, M, pt->coords, nullptr, nullptr, s.prop_logl);
            if (rc != MBHL_OK) return rc;
            k_pt_accept<<<(M + 127) / 128, 128, 0, ctx->stream>>>(s, half, 2u * pt->step + (uint32_t)half);
            ctx->launches += 2;
        }
        if (s.T > 1) {
            k_pt_swap<<<(s.K + 127) / 128, 128, 0, ctx->stream>>>(s, pt->step);
            ctx->launches += 1;
        }
    }
    CU(cudaGetLastError());
    return MBHL_OK;
}

int mbhl_pt_state(mbhl_pt* pt, double* theta, double* logL, int64_t* n_accept_host, int64_t* n_swap_host) {
    if (!pt) return MBHL_EINVAL;
    mbhl_ctx* ctx = pt->ctx;
    CU(cudaSetDevice(ctx->device));
    const PtState& s = pt->s;
    const size_t n = (size_t)s.T * s.K;
    if (theta) CU(cudaMemcpyAsync(theta, s.theta, n * MBHL_NPARAM * 8, cudaMemcpyDefault, ctx->stream));
    if (logL) CU(cudaMemcpyAsync(logL, s.logl, n * 8, cudaMemcpyDefault, ctx->stream));
    if (n_accept_host) CU(cudaMemcpyAsync(n_accept_host, s.n_accept, (size_t)s.T * 8, cudaMemcpyDeviceToHost, ctx->stream));
    if (n_swap_host && s.T > 1) CU(cudaMemcpyAsync(n_swap_host, s.n_swap, (size_t)(s.T - 1) * 8, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MBHL_OK;
}

void mbhl_pt_free(mbhl_pt* pt) {
    if (!pt) return;
    cudaSetDevice(pt->ctx->device);
    cudaStreamSynchronize(pt->ctx->stream);
    cudaFree(pt->mem);
    delete pt;
}

// ---------------------------------------------------------------------------------------------
// heterodyned (relative-binning) likelihood variant
// ---------------------------------------------------------------------------------------------
struct mbhl_het {
    mbhl_ctx* ctx = nullptr;
    int n_b = 0;
    char* mem = nullptr;            // one allocation: reference records, edges, summary data
    double* partials = nullptr;     // [B][n_groups][2], grown on demand
    size_t partials_bytes = 0;
    HetEvalArgs E = {};
};

void mbhl_het_free(mbhl_het* het) {
    if (!het) return;
    cudaSetDevice(het->ctx->device);
    cudaStreamSynchronize(het->ctx->stream);
    cudaFree(het->mem);
    cudaFree(het->partials);
    delete het;
}

int mbhl_het_init(mbhl_ctx* ctx, mbhl_het** out, const double* params_ref, const int64_t* edges_host, int32_t n_coarse) {
    if (!ctx || !out) return MBHL_EINVAL;
    *out = nullptr;
    if (!params_ref || !edges_host || n_coarse < 1 || edges_host[0] != 0 || edges_host[n_coarse] != ctx->N)
        return fail(ctx, MBHL_EINVAL, "mbhl_het_init: need params_ref, edges[0] = 0, edges[n_coarse] = N");
    for (int b = 0; b < n_coarse; ++b)
        if (edges_host[b + 1] <= edges_host[b]) return fail(ctx, MBHL_EINVAL, "mbhl_het_init: edges must increase strictly");
    CU(cudaSetDevice(ctx->device));
    mbhl_het* het = new (std::nothrow) mbhl_het();
    if (!het) return MBHL_ENOMEM;
    het->ctx = ctx;
    auto bail = [&](int code) { cudaFree(het->mem); delete het; return code; };
    const int S = ctx->S;
    cudaStream_t st = ctx->stream;
    // the reference's sparse stage (a1-a5)
    char* base;
    int rc = get_workspace(ctx, 1, &base);
    if (rc != MBHL_OK) return bail(rc);
    const WsLayout L = layout(ctx, 1);
    const bool tm = ctx->timing;
    ctx->timing = false;
    rc = run_sparse(ctx, params_ref, 1, MBHL_COORDS_PHYSICAL, base, L, true);
    ctx->timing = tm;
    if (rc != MBHL_OK) return bail(rc);
    WalkerConst wc_host;
    DenseWalker dw_host;
    if (cudaMemcpyAsync(&wc_host, base + L.consts, sizeof(WalkerConst), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemcpyAsync(&dw_host, base + L.dense, sizeof(DenseWalker), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return bail(fail(ctx, MBHL_ECUDA, "mbhl_het_init: copies"));
    if (!wc_host.valid) return bail(fail(ctx, MBHL_EINVAL, "mbhl_het_init: the reference parameters are outside the model's domain"));
    // coarse bins actually used: the caller's edges refined by the reference's band edges (reading H1)
    std::vector<long long> ed(edges_host, edges_host + n_coarse + 1);
    for (int i = 0; i < MBHL_NMODE; ++i)
        if (((ctx->mode_mask >> i) & 1u) && dw_host.mode[i].k_hi >= dw_host.mode[i].k_lo) {
            ed.push_back(dw_host.mode[i].k_lo);
            ed.push_back((long long)dw_host.mode[i].k_hi + 1);
        }
    std::sort(ed.begin(), ed.end());
    ed.erase(std::unique(ed.begin(), ed.end()), ed.end());
    n_coarse = (int32_t)ed.size() - 1;
    het->n_b = n_coarse;
    const size_t nb = (size_t)n_coarse;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align256(bytes); return o; };
    const size_t o_wc = take(sizeof(WalkerConst)), o_dw = take(sizeof(DenseWalker)), o_kn = take((size_t)MBHL_NMODE * S * 8);
    const size_t o_cf = take((size_t)MBHL_NMODE * (S - 1) * kCoefStride * 8), o_ed = take((nb + 1) * 8), o_pt = take(nb * 6 * 8), o_rp = take((size_t)MBHL_NMODE * nb * 3 * 8), o_pr = take((size_t)MBHL_NMODE * nb * 4);
    const size_t o_a0 = take(kHetA * nb * 16), o_a1 = take(kHetA * nb * 16), o_a2 = take(kHetA * nb * 16);
    const size_t o_b0 = take(kHetB * nb * 16), o_b1 = take(kHetB * nb * 16), o_b2 = take(kHetB * nb * 16);
    const size_t o_lf = take(MBHL_NMODE * 8), o_id = take(MBHL_NMODE * 8), o_lo = take(MBHL_NMODE * 8), o_hi = take(MBHL_NMODE * 8);
    if (cudaMalloc(&het->mem, off) != cudaSuccess) { cudaGetLastError(); het->mem = nullptr; return bail(fail(ctx, MBHL_ENOMEM, "mbhl_het_init: cudaMalloc")); }
    char* m = het->mem;
    if (cudaMemcpyAsync(m + o_wc, base + L.consts, sizeof(WalkerConst), cudaMemcpyDeviceToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(m + o_dw, base + L.dense, sizeof(DenseWalker), cudaMemcpyDeviceToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(m + o_kn, base + L.knots, (size_t)MBHL_NMODE * S * 8, cudaMemcpyDeviceToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(m + o_cf, base + L.coef, (size_t)MBHL_NMODE * (S - 1) * kCoefStride * 8, cudaMemcpyDeviceToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(m + o_ed, ed.data(), (nb + 1) * 8, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
        return bail(fail(ctx, MBHL_ECUDA, "mbhl_het_init: copies"));
    double lf[MBHL_NMODE], id[MBHL_NMODE], flo[MBHL_NMODE], fhi[MBHL_NMODE];
    for (int i = 0; i < MBHL_NMODE; ++i) {
        lf[i] = wc_host.mode[i].ln_flo; id[i] = wc_host.mode[i].inv_dlog;
        flo[i] = wc_host.mode[i].f_lo; fhi[i] = wc_host.mode[i].f_hi;
    }
    if (cudaMemcpyAsync(m + o_lf, lf, sizeof(lf), cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(m + o_id, id, sizeof(id), cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(m + o_lo, flo, sizeof(flo), cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(m + o_hi, fhi, sizeof(fhi), cudaMemcpyHostToDevice, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess)
        return bail(fail(ctx, MBHL_ECUDA, "mbhl_het_init: copies"));
    HetArgs& H = het->E.H;
    H.tiles = ctx->tiles; H.ref_dw = (const DenseWalker*)(m + o_dw); H.ref_knots = (const double*)(m + o_kn); H.ref_coef = (const double*)(m + o_cf);
    H.edges = (const long long*)(m + o_ed); H.A0 = (double2*)(m + o_a0); H.A1 = (double2*)(m + o_a1); H.A2 = (double2*)(m + o_a2);
    H.B0 = (double2*)(m + o_b0); H.B1 = (double2*)(m + o_b1); H.B2 = (double2*)(m + o_b2);
    H.S = S; H.n_b = n_coarse; H.mode_mask = ctx->mode_mask;
    het->E.pts = (const double*)(m + o_pt); het->E.ref_p4 = (const double*)(m + o_rp); het->E.present = (const int*)(m + o_pr);
    het->E.ref_ln_flo = (const double*)(m + o_lf); het->E.ref_inv_dlog = (const double*)(m + o_id);
    het->E.ref_f_lo = (const double*)(m + o_lo); het->E.ref_f_hi = (const double*)(m + o_hi);
    het->E.n_groups = (n_coarse + kHetEvalThreads - 1) / kHetEvalThreads;
    k_het_bin_points<<<(n_coarse + 127) / 128, 128, 0, st>>>(ctx->freqs, H.edges, n_coarse, H.ref_dw, H.ref_knots, H.ref_coef, S, ctx->mode_mask,
                                                              (double*)(m + o_pt), (double*)(m + o_rp), (int*)(m + o_pr));
    k_het_summary<<<n_coarse, kHetTile, 0, st>>>(H);
    ctx->launches += 2;
    if (cudaGetLastError() != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) return bail(fail(ctx, MBHL_ECUDA, "mbhl_het_init: summary kernel"));
    *out = het;
    return MBHL_OK;
}

int mbhl_het_loglike(mbhl_het* het, const double* params, int64_t B, double* d_h, double* h_h, double* logL) {
    if (!het) return MBHL_EINVAL;
    mbhl_ctx* ctx = het->ctx;
    if (B < 0 || (B > 0 && !params)) return fail(ctx, MBHL_EINVAL, "bad params/B");
    if (B == 0) return MBHL_OK;
    CU(cudaSetDevice(ctx->device));
    const bool tm = ctx->timing;
    for (int64_t o = 0; o < B; o += kSliceBatch) {
        const int64_t n = (B - o < kSliceBatch) ? (B - o) : kSliceBatch;
        char* base;
        int rc = get_workspace(ctx, n, &base);
        if (rc != MBHL_OK) return rc;
        const WsLayout L = layout(ctx, n);
        const size_t need = (size_t)n * het->E.n_groups * 2 * sizeof(double);
        if (het->partials_bytes < need) {
            CU(cudaStreamSynchronize(ctx->stream));
            cudaFree(het->partials);
            het->partials = nullptr;
            het->partials_bytes = 0;
            if (cudaMalloc(&het->partials, need) != cudaSuccess) { cudaGetLastError(); return fail(ctx, MBHL_ENOMEM, "mbhl_het_loglike: cudaMalloc"); }
            het->partials_bytes = need;
        }
        ctx->timing = false;
        rc = run_sparse(ctx, params + o * MBHL_NPARAM, n, MBHL_COORDS_PHYSICAL, base, L, true);
        ctx->timing = tm;
        if (rc != MBHL_OK) return rc;
        HetEvalArgs E = het->E;
        E.wc = (const WalkerConst*)(base + L.consts);
        E.dw = (const DenseWalker*)(base + L.dense);
        E.knots = (const double*)(base + L.knots);
        E.coef = (const double*)(base + L.coef);
        E.partials = het->partials;
        dim3 g((unsigned)((het->n_b + kHetEvalThreads - 1) / kHetEvalThreads), (unsigned)n);
        k_het_eval<<<g, kHetEvalThreads, 0, ctx->stream>>>(E);
        k_final_reduce<<<(unsigned)n, 128, 0, ctx->stream>>>(E.dw, E.partials, E.n_groups, n, ctx->dd, d_h ? d_h + o : nullptr,
                                                                        h_h ? h_h + o : nullptr, logL ? logL + o : nullptr, nullptr, 1);
        ctx->launches += 2;
        CU(cudaGetLastError());
    }
    return MBHL_OK;
}

int mbhl_noise(void* stream, const double* psd_AET, int64_t N, double df, uint64_t seed, double* out_AET) {
    if (!psd_AET || !out_AET || N < 1 || N > ((int64_t)1 << 31) || !(df > 0.0)) return MBHL_EINVAL;
    dim3 g((unsigned)((N + 255) / 256), 3);
    k_noise<<<g, 256, 0, (cudaStream_t)stream>>>(psd_AET, N, df, seed, out_AET);
    return cudaGetLastError() == cudaSuccess ? MBHL_OK : MBHL_ECUDA;
}

int mbhl_last_work(mbhl_ctx* ctx, int64_t* pairs, int64_t* bins) {
    if (!ctx) return MBHL_EINVAL;
    unsigned long long h[2];
    CU(cudaMemcpyAsync(h, ctx->counters, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (pairs) *pairs = (int64_t)h[0];
    if (bins) *bins = (int64_t)h[1];
    return MBHL_OK;
}

int mbhl_last_dense_work(mbhl_ctx* ctx, int64_t counts[5]) {
    if (!ctx || !counts) return MBHL_EINVAL;
    unsigned long long h[8];
    CU(cudaMemcpyAsync(h, ctx->counters, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    for (int i = 0; i < 5; ++i) counts[i] = (int64_t)h[2 + i];
    return MBHL_OK;
}

int mbhl_template(mbhl_ctx* ctx, const double* params, int64_t B, const double* freqs_out, int64_t Nout, double* out_AET,
                  int32_t direct) {
    if (!ctx) return MBHL_EINVAL;
    if (B < 0 || (B > 0 && (!params || !out_AET))) return fail(ctx, MBHL_EINVAL, "bad template arguments");
    if (!freqs_out) { freqs_out = ctx->freqs; Nout = ctx->N; }
    if (Nout < 0) return fail(ctx, MBHL_EINVAL, "bad Nout");
    if (B == 0 || Nout == 0) return MBHL_OK;
    CU(cudaSetDevice(ctx->device));
    for (int64_t o = 0; o < B; o += kSliceBatch) {       // slices, like the likelihood calls
        const int64_t n = (B - o < kSliceBatch) ? (B - o) : kSliceBatch;
        char* base;
        int rc = get_workspace(ctx, n, &base);
        if (rc != MBHL_OK) return rc;
        const WsLayout L = layout(ctx, n);
        rc = run_sparse(ctx, params + o * MBHL_NPARAM, n, MBHL_COORDS_PHYSICAL, base, L, direct == 0);
        if (rc != MBHL_OK) return rc;
        dim3 g((unsigned)((Nout + 127) / 128), (unsigned)n);
        k_template<<<g, 128, 0, ctx->stream>>>((const WalkerConst*)(base + L.consts), (const double*)(base + L.knots),
                                               (const double*)(base + L.coef), ctx->S, freqs_out, Nout, out_AET + o * 6 * Nout, direct ? 1 : 0);
        ctx->launches += 1;
        CU(cudaGetLastError());
    }
    return MBHL_OK;
}

int mbhl_sparse(mbhl_ctx* ctx, const double* params, int64_t B, double* knots, double* y, double* coef) {
    if (!ctx) return MBHL_EINVAL;
    if (B < 0 || B > kSliceBatch || (B > 0 && !params)) return fail(ctx, MBHL_EINVAL, "bad params/B (mbhl_sparse takes B <= 32768)");
    if (B == 0) return MBHL_OK;
    CU(cudaSetDevice(ctx->device));
    char* base;
    int rc = get_workspace(ctx, B, &base);
    if (rc != MBHL_OK) return rc;
    const WsLayout L = layout(ctx, B);
    rc = run_sparse(ctx, params, B, MBHL_COORDS_PHYSICAL, base, L, true, y);      // y lands in the caller's buffer, phase row in cycles
    if (rc != MBHL_OK) return rc;
    if (ctx->timing) {   // stages 3 and 4 (dense, reduce) do not run here: zero-length intervals
        for (int i = 3; i < 6; ++i) cudaEventRecord(ctx->ev[i], ctx->stream);
        ctx->n_timed += 1;
    }
    const size_t nk = (size_t)B * MBHL_NMODE * ctx->S;
    if (knots) CU(cudaMemcpyAsync(knots, base + L.knots, nk * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    if (y) {
        const int64_t rows = B * MBHL_NMODE * MBHL_NQ;
        k_export_y<<<(unsigned)((rows * ctx->S + 255) / 256), 256, 0, ctx->stream>>>(y, rows, ctx->S, y);   // in place: phase row to radians
        ctx->launches += 1;
    }
    if (coef) {
        const int64_t n = B * MBHL_NMODE * (int64_t)(ctx->S - 1) * MBHL_NQ;
        k_export_coef<<<(unsigned)((n + 255) / 256), 256, 0, ctx->stream>>>((const WalkerConst*)(base + L.consts), (const double*)(base + L.knots),
                                                                           (const double*)(base + L.coef), B * MBHL_NMODE, ctx->S, coef);
        ctx->launches += 1;
    }
    CU(cudaGetLastError());
    return MBHL_OK;
}

int mbhl_enable_stage_timing(mbhl_ctx* ctx, int32_t on) {
    if (!ctx) return MBHL_EINVAL;
    CU(cudaSetDevice(ctx->device));
    if (on && !ctx->evs[0][0])
        for (int k = 0; k < mbhl_ctx::kSlots; ++k)
            for (int i = 0; i < 6; ++i) CU(cudaEventCreate(&ctx->evs[k][i]));
    ctx->timing = on != 0;
    ctx->n_timed = 0;
    return MBHL_OK;
}

int mbhl_stage_times(mbhl_ctx* ctx, double ms[5]) {
    if (!ctx || !ms) return MBHL_EINVAL;
    if (!ctx->timing || ctx->n_timed == 0) return fail(ctx, MBHL_EINVAL, "stage timing is off or no call was timed");
    CU(cudaStreamSynchronize(ctx->stream));
    const int n = ctx->n_timed < mbhl_ctx::kSlots ? ctx->n_timed : mbhl_ctx::kSlots;
    for (int i = 0; i < 5; ++i) ms[i] = 0.0;
    for (int k = 0; k < n; ++k)
        for (int i = 0; i < 5; ++i) {
            float t = 0.f;
            CU(cudaEventElapsedTime(&t, ctx->evs[k][i], ctx->evs[k][i + 1]));
            ms[i] += (double)t / n;
        }
    ctx->n_timed = 0;
    return MBHL_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// mbhl_unpack_coords_static: the coordinate conversion with the kernel's scratch records in a fixed array of the
// library image, for callers that must not allocate device memory (who they are and the rules: include/mbhl.h)
// ---------------------------------------------------------------------------------------------
namespace {

constexpr size_t up256(size_t x) { return (x + 255) & ~(size_t)255; }
constexpr size_t kStaticConstsBytes = up256((size_t)MBHL_STATIC_MAX_WALKERS * sizeof(WalkerConst));
constexpr size_t kStaticDenseBytes = up256((size_t)MBHL_STATIC_MAX_WALKERS * sizeof(DenseWalker));
constexpr size_t kStaticScratchBytes = kStaticConstsBytes + kStaticDenseBytes;      // about 2.6 MB
static_assert(kStaticScratchBytes <= ((size_t)4 << 20), "the fixed scratch array is meant to stay small: every GPU holds it until exit");

// [WalkerConst x MBHL_STATIC_MAX_WALKERS][DenseWalker x MBHL_STATIC_MAX_WALKERS], written by k_walker_consts and read by
// nobody.  One copy per device that loads the library, for the process's lifetime.  NOTE for host code: this NAME is only
// a host-side stand-in for the symbol, not a device address - a kernel handed `g_static_scratch` itself would fault (or,
// where the GPU can reach host memory, quietly use the wrong memory).  Host code must go through static_scratch_base().
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_base[kStaticMaxDevices] = {};      // device address of g_static_scratch, per device ordinal; looked up once

// Device address of the array on ctx->device, which must be the current device.  The first call per device asks the
// runtime (cudaGetSymbolAddress resolves the symbol in the CURRENT device's copy of the module); later calls reuse it.
int static_scratch_base(mbhl_ctx* ctx, char** base) {
    const int d = ctx->device;
    if (d < 0 || d >= kStaticMaxDevices) return fail(ctx, MBHL_EINVAL, "mbhl_unpack_coords_static: device ordinal outside 0..63");
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_base[d]) {
        void* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
        if (e != cudaSuccess) return fail(ctx, MBHL_ECUDA, "cudaGetSymbolAddress(g_static_scratch)", e);
        if (!ptr) return fail(ctx, MBHL_ECUDA, "cudaGetSymbolAddress(g_static_scratch) returned a null address");
        g_static_base[d] = ptr;
    }
    *base = (char*)g_static_base[d];
    return MBHL_OK;
}

}  // namespace

extern "C" {

int mbhl_unpack_coords_static(mbhl_ctx* ctx, const double* rows, int64_t B, int32_t coords, double* params_out) {
    if (!ctx) return MBHL_EINVAL;
    if (B < 0 || (B > 0 && (!rows || !params_out)) || coords < 0 || coords > 2)
        return fail(ctx, MBHL_EINVAL, "mbhl_unpack_coords_static: bad rows/B/coords/params_out");
    if (B > MBHL_STATIC_MAX_WALKERS) {
        snprintf(ctx->err, sizeof(ctx->err),
                 "mbhl_unpack_coords_static: B = %lld exceeds MBHL_STATIC_MAX_WALKERS = %d, the size of the fixed scratch array; split the batch",
                 (long long)B, MBHL_STATIC_MAX_WALKERS);
        return MBHL_EINVAL;
    }
    if (B == 0) return MBHL_OK;
    {
        // a warp writes its converted row while other warps may still be reading theirs: fine for distinct buffers (and for
        // the exactly-in-place use inside the library), wrong for buffers that overlap at an offset - refuse any overlap
        const uintptr_t r0 = (uintptr_t)rows, p0 = (uintptr_t)params_out, n = (uintptr_t)B * MBHL_NPARAM * sizeof(double);
        if (r0 < p0 + n && p0 < r0 + n) return fail(ctx, MBHL_EINVAL, "mbhl_unpack_coords_static: rows and params_out overlap");
    }
    CU(cudaSetDevice(ctx->device));
    char* base = nullptr;
    const int rc = static_scratch_base(ctx, &base);
    if (rc != MBHL_OK) return rc;
    // Same launch as run_consts(), with the two record arrays in the fixed array and the converted parameters going
    // straight to the caller's buffer.  Rows 0..B-1 of both record arrays are overwritten in full; nothing is read back.
    k_walker_consts<<<(unsigned)((B + kConstsWarps - 1) / kConstsWarps), 32 * kConstsWarps, 0, ctx->stream>>>(
        rows, B, coords, ctx->t0, ctx->f_min, ctx->f_max, ctx->S, ctx->mode_mask, ctx->freqs, (int)ctx->N, ctx->df,
        (WalkerConst*)base, (DenseWalker*)(base + kStaticConstsBytes), params_out);
    ctx->launches += 1;
    CU(cudaGetLastError());
    return MBHL_OK;
}

int mbhl_dfma_probe(void* stream, int32_t blocks, int32_t threads, int64_t iters, double* sink) {
    if (blocks <= 0 || threads <= 0 || threads > 1024 || iters < 0 || !sink) return MBHL_EINVAL;
    k_dfma_probe<<<blocks, threads, 0, (cudaStream_t)stream>>>(iters, sink);
    return cudaGetLastError() == cudaSuccess ? MBHL_OK : MBHL_ECUDA;
}

}  // extern "C"
