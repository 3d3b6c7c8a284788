// mbhl_kernels.cuh - the hot-path kernels (steps a1-a7 of SURVEY.md section 8(a)).
#pragma once
#include <cuda_runtime.h>

#include "mbhl_model.cuh"
#include "mbhl_sampler.cuh"   // sampler coordinates, LISA frame, stretch move, temperature swaps

namespace mbhl {

constexpr int kCoefStride = MBHL_NQ * 4;   // doubles per (walker, mode, interval) record = 256 B
#ifndef MBHL_DENSE_T
#define MBHL_DENSE_T 128
#endif
constexpr int kDenseThreads = MBHL_DENSE_T;   // 4 warps per CTA
#ifndef MBHL_DENSE_R
#define MBHL_DENSE_R 4
#endif
#ifndef MBHL_DENSE_MINB
#define MBHL_DENSE_MINB 3
#endif
constexpr int kDenseR = MBHL_DENSE_R;      // bins per thread per chunk
constexpr int kWarpTile = 32 * kDenseR;    // 128 consecutive bins per warp
constexpr int kChunk = kDenseThreads * kDenseR;   // 512 bins per CTA step
constexpr int kTileRows = 10;              // rows of a staged data tile: f, w^{A,E,T}, (w Re d, w Im d)^{A,E,T}
constexpr int kTileDoubles = kTileRows * kChunk;
constexpr int kTileBytes = kTileDoubles * 8;      // 40 KB, one bulk copy
#ifndef MBHL_DENSE_W
#define MBHL_DENSE_W 8
#endif
constexpr int kMaxW = MBHL_DENSE_W;                 // walkers per CTA tile (upper bound)
constexpr int kPairs = kMaxW * MBHL_NMODE; // (walker, mode) pairs of a CTA tile: one staged coefficient record each

// ---------------------------------------------------------------------------------------------
// init: data tiles (weights, weighted data), <d|d>, grid validation
// tiles layout [n_chunks][10][512]: row 0 f_k; rows 1-3 w^c = 4 df / S^c; rows 4+2c, 5+2c = w^c Re d^c, w^c Im d^c.
// Bins k >= N of the last chunk are padding: f continues the grid, every weight is 0.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_init_tiles(const double* __restrict__ freqs, const double* __restrict__ data,
                                                    const double* __restrict__ psd, int64_t N, double df,
                                                    double* __restrict__ tiles, double* __restrict__ dd_part) {
    __shared__ double red[256];
    const int64_t k0 = (int64_t)blockIdx.x * kChunk;
    double* tile = tiles + (int64_t)blockIdx.x * kTileDoubles;
    double acc = 0.0;
    for (int i = threadIdx.x; i < kChunk; i += 256) {
        const int64_t k = k0 + i;
        if (k < N) {
            tile[i] = freqs[k];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double s = psd[c * N + k];
                const double ww = (isfinite(s) && s > 0.0) ? 4.0 * df / s : 0.0;
                const double dre = data[(c * N + k) * 2], dim = data[(c * N + k) * 2 + 1];
                tile[(1 + c) * kChunk + i] = ww;
                tile[(4 + 2 * c) * kChunk + i] = ww * dre;
                tile[(5 + 2 * c) * kChunk + i] = ww * dim;
                acc += ww * (dre * dre + dim * dim);
            }
        } else {
            tile[i] = freqs[N - 1] + (double)(k - N + 1) * df;
#pragma unroll
            for (int r = 1; r < kTileRows; ++r) tile[r * kChunk + i] = 0.0;
        }
    }
    red[threadIdx.x] = acc;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) dd_part[blockIdx.x] = red[0];
}

__global__ void k_check_grid(const double* __restrict__ f, int64_t N, double df, double* __restrict__ dev_part) {
    __shared__ double red[256];
    const int64_t k0 = (int64_t)blockIdx.x * 1024;
    double worst = 0.0;
    for (int i = threadIdx.x; i < 1024; i += 256) {
        const int64_t k = k0 + i;
        if (k + 1 < N) {
            const double d = f[k + 1] - f[k];
            double dev = fabs(d / df - 1.0);
            if (!(d > 0.0) || !isfinite(d)) dev = 1e300;
            worst = fmax(worst, dev);
        }
        if (k < N && !(f[k] > 0.0)) worst = 1e300;
    }
    red[threadIdx.x] = worst;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) red[threadIdx.x] = fmax(red[threadIdx.x], red[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) dev_part[blockIdx.x] = red[0];
}

// ---------------------------------------------------------------------------------------------
// a1 + a2: per-walker constants and bands (one thread per walker); also the compact DenseWalker record
// with each band as a bin range of the init grid.
// ---------------------------------------------------------------------------------------------
__device__ inline int first_bin_ge(const double* __restrict__ f, int N, double f0, double inv_df, double x) {
    double e = ceil((x - f0) * inv_df);          // min{k: f_k >= x}, in [0, N]
    int k = (e < 0.0) ? 0 : ((e > (double)N) ? N : (int)e);
    while (k > 0 && f[k - 1] >= x) --k;
    while (k < N && f[k] < x) ++k;
    return k;
}
__device__ inline int last_bin_le(const double* __restrict__ f, int N, double f0, double inv_df, double x) {
    double e = floor((x - f0) * inv_df) + 1.0;   // max{k: f_k <= x} = min{k: f_k > x} - 1, in [-1, N-1]
    int k = (e < 0.0) ? 0 : ((e > (double)N) ? N : (int)e);
    while (k > 0 && f[k - 1] > x) --k;
    while (k < N && f[k] <= x) ++k;
    return k - 1;
}

constexpr int kConstsWarps = 4;      // walkers per CTA of k_walker_consts (one warp each)

// rows [B][11]: the walkers in the coordinates named by `coords` (mbhl.h MBHL_COORDS_*): physical SSB parameters, the
// sampler's coordinates (Table I box :67-81 -> outside it the walker is invalid, logL = -inf), or the
// sampler's coordinates with (lambda, sin beta, psi, ln t) in the LISA frame (reading G20).  The
// conversion runs in registers here, so a sampler hands over raw walker coordinates and no extra kernel runs.
// params_out (may be null): the physical SSB parameters the walker was converted to (NaN row if outside the box).
// rows and params_out carry no __restrict__: mbhl_loglike_host hands over the same buffer for both (a warp reads its own
// row in full, then writes it back after the __syncwarp below; no other warp touches that row).
__global__ void __launch_bounds__(32 * kConstsWarps) k_walker_consts(const double* rows, int64_t B, int coords, double t0, double f_min,
                                                      double f_max, int S, uint32_t mode_mask, const double* __restrict__ freqs,
                                                      int N, double df, WalkerConst* __restrict__ out,
                                                      DenseWalker* __restrict__ dw, double* params_out) {
    __shared__ WalkerConst s_c[kConstsWarps];
    __shared__ DenseWalker s_d[kConstsWarps];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t b = (int64_t)blockIdx.x * kConstsWarps + warp;
    if (b >= B) return;
    WalkerConst& c = s_c[warp];
    DenseWalker& d = s_d[warp];
    double p[MBHL_NPARAM];
#pragma unroll
    for (int i = 0; i < MBHL_NPARAM; ++i) p[i] = rows[b * MBHL_NPARAM + i];
    if (coords != 0) {
        double th[MBHL_NPARAM];
#pragma unroll
        for (int i = 0; i < MBHL_NPARAM; ++i) th[i] = p[i];
        unpack_sampled(th, p);                          // NaN row outside the box of Table I
        if (coords == 2 && isfinite(p[10])) lisa_to_ssb(t0, p[10], p[7], p[8], p[9]);
    }
    __syncwarp();                                       // rows and params_out may be the same buffer: every lane has read its row
    if (params_out != nullptr && lane < MBHL_NPARAM) {
        double v = p[0];
#pragma unroll
        for (int i = 1; i < MBHL_NPARAM; ++i) v = (lane == i) ? p[i] : v;
        params_out[b * MBHL_NPARAM + lane] = v;
    }
    const int mi = lane % MBHL_NMODE;                  // lanes 6.. repeat the work of lanes 0-5 (identical stores)
    build_walker(p, t0, f_min, f_max, S, mode_mask, c, mi, mi + 1);
    __syncwarp();                                      // lanes L, L + 6, ... stored the same mode: all of them are done
    {
        DenseMode m;
        m.k_lo = 1; m.k_hi = 0; m.ln_flo = 0.0; m.inv_dlog = 0.0;
        if (c.valid && c.mode[mi].active) {
            m.k_lo = first_bin_ge(freqs, N, f_min, 1.0 / df, c.mode[mi].f_lo);
            m.k_hi = last_bin_le(freqs, N, f_min, 1.0 / df, c.mode[mi].f_hi);
            m.ln_flo = c.mode[mi].ln_flo;
            m.inv_dlog = c.mode[mi].inv_dlog;
            if (m.k_hi < m.k_lo) { m.k_lo = 1; m.k_hi = 0; }
        }
        d.mode[mi] = m;
    }
    __syncwarp();
    if (lane == 0) {
        d.t_coal = c.valid ? c.t_coal : 0.0;
        d.valid = c.valid;
        d.pad_ = 0;
        long long pairs = 0;
        int lo[MBHL_NMODE], hi[MBHL_NMODE];
        for (int k = 0; k < MBHL_NMODE; ++k) {
            lo[k] = d.mode[k].k_lo; hi[k] = d.mode[k].k_hi;
            if (hi[k] >= lo[k]) pairs += (long long)(hi[k] - lo[k] + 1);
        }
        // bins covered by at least one mode: length of the union of the six ranges
        long long bins = 0;
        int done_to = -1;                               // everything <= done_to is already counted
        for (int it = 0; it < MBHL_NMODE; ++it) {
            int best = -1;
            for (int k = 0; k < MBHL_NMODE; ++k)
                if (hi[k] >= lo[k] && hi[k] > done_to && (best < 0 || lo[k] < lo[best])) best = k;
            if (best < 0) break;
            const int a = max(lo[best], done_to + 1);
            bins += (long long)(hi[best] - a + 1);
            done_to = hi[best];
        }
        d.pairs = pairs;
        d.bins = bins;
    }
    __syncwarp();
    // coalesced copies of the two records to global memory
    static_assert(sizeof(WalkerConst) % 8 == 0 && sizeof(DenseWalker) % 8 == 0, "records are copied as doubles");
    for (int i = lane; i < (int)(sizeof(WalkerConst) / 8); i += 32) reinterpret_cast<double*>(out + b)[i] = reinterpret_cast<const double*>(&c)[i];
    for (int i = lane; i < (int)(sizeof(DenseWalker) / 8); i += 32) reinterpret_cast<double*>(dw + b)[i] = reinterpret_cast<const double*>(&d)[i];
}

// ---------------------------------------------------------------------------------------------
// a3 + a4 + a5: the fused sparse stage (PhenomHM + response at the knots, spline coefficients): mbhl_sparse.cuh
// ---------------------------------------------------------------------------------------------
// frac(f * t) in cycles with the product taken exactly (reading G9): f and t are the supplied doubles.
__device__ __forceinline__ double linear_cycles(double f, double t) {
    const double p = f * t;
    const double e = fma(f, t, -p);
    const double pr = (p + kRoundMagic) - kRoundMagic;
    return (p - pr) + e;
}

}  // namespace mbhl

#include "mbhl_sparse.cuh"

namespace mbhl {

// ---------------------------------------------------------------------------------------------
// a6 + a7: fused dense kernel (mbhl_dense.cuh, which documents the work decomposition): interpolates every
// active mode onto the Fourier bins, sums the modes per bin and accumulates <d|h> and <h|h>
// (eqs. 2, 3, 11); the template is never written to memory.  Here: its arguments and the device functions it
// shares with mbhl_template (quarter-turn sincos, interval lookup, one mode's contribution at one bin).
// ---------------------------------------------------------------------------------------------
struct DenseArgs {
    const DenseWalker* dw;   // [B]
    const double* knots;     // [B][6][S]
    const double* coef;      // [B][6][S-1][8][4]
    const double* tiles;     // [n_chunks][10][512]
    double* partials;        // [B][n_groups][2]
    int B;
    int S;
    int W;                   // walkers per CTA tile (<= kMaxW)
    int G;                   // chunks per CTA
    int n_chunks;
    int n_groups;
    double inv_df;           // 1 / bin spacing of the init grid
    uint32_t mode_mask;      // modes evaluated by this launch (bit i = mode i); the others count as out of band
    unsigned long long* work; // [5] executed-work tallies (may be null): see mbhl_last_dense_work
};

// Locates the spline interval of frequency f (ln f = lf) on the log-spaced knots x[0..S-1]; *x_hi receives x[j + 1].
// The two knots around the guess are loaded together (independent loads: one memory round trip when the guess is right).
__device__ __forceinline__ int find_interval(const double* __restrict__ x, int S, double f, double lf, double ln_flo,
                                             double inv_dlog, double* x_hi = nullptr) {
    int j = (int)((lf - ln_flo) * inv_dlog);
    j = max(0, min(S - 2, j));
    double xl = __ldg(x + j), xh = __ldg(x + j + 1);
    while (j > 0 && f < xl) { --j; xh = xl; xl = __ldg(x + j); }
    while (j < S - 2 && f >= xh) { ++j; xl = xh; xh = __ldg(x + j + 1); }
    if (x_hi) *x_hi = xh;
    return j;
}

// One mode's contribution at one bin from the record `rec` (8 cubics in u = f - f_j): used by the
// per-bin path of the dense kernel and by mbhl_template.  Amplitude scaled by `gate`.
// kGlobal: the record sits in global memory (read-only path); otherwise in shared memory.
template <bool kGlobal = true>
__device__ __forceinline__ void mode_contrib(const double* __restrict__ rec, double u, double gate, double h[6]) {
    double v[MBHL_NQ];
#pragma unroll
    for (int q = 0; q < MBHL_NQ; q += 1) {
        const double2 c01 = kGlobal ? __ldg(reinterpret_cast<const double2*>(rec + q * 4)) : *reinterpret_cast<const double2*>(rec + q * 4);
        const double2 c23 = kGlobal ? __ldg(reinterpret_cast<const double2*>(rec + q * 4 + 2)) : *reinterpret_cast<const double2*>(rec + q * 4 + 2);
        v[q] = fma(fma(fma(c23.y, u, c23.x), u, c01.y), u, c01.x);
    }
    double sn, cs;
    sincos_qturn(v[1], sn, cs);
    const double amp = v[0] * gate;
    const double are = amp * cs, aim = amp * sn;
    h[0] = fma(are, v[2], fma(-aim, v[3], h[0]));
    h[1] = fma(are, v[3], fma(aim, v[2], h[1]));
    h[2] = fma(are, v[4], fma(-aim, v[5], h[2]));
    h[3] = fma(are, v[5], fma(aim, v[4], h[3]));
    h[4] = fma(are, v[6], fma(-aim, v[7], h[4]));
    h[5] = fma(are, v[7], fma(aim, v[6], h[5]));
}

}  // namespace mbhl

#include "mbhl_dense.cuh"   // a6 + a7: the fused dense kernel
#include "mbhl_het.cuh"     // heterodyned likelihood variant

namespace mbhl {

// a7: deterministic final reduction, one CTA (4 warps) per walker; logL = <d|h> - 1/2<h|h> - 1/2<d|d> (eq. 2).
// Fixed order: thread t takes groups t, t + 128, ...; four independent 16-byte loads are in flight per thread and step
// (with few walkers and many groups the loop is a chain of L2 round trips), the running sums are added pairwise, then a
// shuffle tree per warp and the four warp sums in order.
__global__ void __launch_bounds__(128) k_final_reduce(const DenseWalker* __restrict__ dw, const double* __restrict__ partials,
                                                      int n_groups, int64_t B, double dd, double* __restrict__ d_h,
                                                      double* __restrict__ h_h, double* __restrict__ logL,
                                                      unsigned long long* __restrict__ counters, int64_t stride) {
    __shared__ double s_w[4][2];
    const int64_t b = blockIdx.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const double2* p2 = reinterpret_cast<const double2*>(partials + b * n_groups * 2);
    double2 acc[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) acc[k] = make_double2(0.0, 0.0);
    int i = tid;
    for (; i + 384 < n_groups; i += 512) {
        double2 v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = p2[i + 128 * k];
#pragma unroll
        for (int k = 0; k < 4; ++k) { acc[k].x += v[k].x; acc[k].y += v[k].y; }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k)
        if (i + 128 * k < n_groups) { const double2 v = p2[i + 128 * k]; acc[k].x += v.x; acc[k].y += v.y; }
    double sdh = (acc[0].x + acc[1].x) + (acc[2].x + acc[3].x);
    double shh = (acc[0].y + acc[1].y) + (acc[2].y + acc[3].y);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sdh += __shfl_down_sync(0xffffffffu, sdh, o);
        shh += __shfl_down_sync(0xffffffffu, shh, o);
    }
    if (lane == 0) { s_w[warp][0] = sdh; s_w[warp][1] = shh; }
    __syncthreads();
    if (tid == 0) {
        sdh = (s_w[0][0] + s_w[1][0]) + (s_w[2][0] + s_w[3][0]);
        shh = (s_w[0][1] + s_w[1][1]) + (s_w[2][1] + s_w[3][1]);
        const bool valid = dw[b].valid != 0;
        if (!valid) { sdh = 0.0; shh = 0.0; }
        if (d_h) d_h[b * stride] = sdh;
        if (h_h) h_h[b * stride] = shh;
        if (logL) logL[b * stride] = valid ? (sdh - 0.5 * shh - 0.5 * dd) : -INFINITY;
        if (counters && valid && dw[b].pairs) {
            atomicAdd(counters, (unsigned long long)dw[b].pairs);
            atomicAdd(counters + 1, (unsigned long long)dw[b].bins);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// mbhl_template: materialised template for tests / injections (spline path or direct evaluation)
// out layout [B][3][Nout][2]
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_template(const WalkerConst* __restrict__ wc, const double* __restrict__ knots,
                                                  const double* __restrict__ coef, int S, const double* __restrict__ freqs,
                                                  int64_t Nout, double* __restrict__ out, int direct) {
    const int64_t b = blockIdx.y;
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= Nout) return;
    const WalkerConst& c = wc[b];
    double h[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if (c.valid) {
        const double f = freqs[k];
        const double lf = log(f);
        for (int mi = 0; mi < MBHL_NMODE; ++mi) {
            const ModeConst& mc = c.mode[mi];
            if (!mc.active || !(f >= mc.f_lo) || !(f <= mc.f_hi)) continue;
            if (direct) {
                double q[MBHL_NQ];
                smooth_quantities(c, mi, f, q);
                double sn, cs;
                sincos_qturn(fma(q[1] - rint(q[1]), 4.0, -4.0 * linear_cycles(f, c.t_coal)), sn, cs);
                const double are = q[0] * cs, aim = q[0] * sn;
                h[0] += are * q[2] - aim * q[3];
                h[1] += are * q[3] + aim * q[2];
                h[2] += are * q[4] - aim * q[5];
                h[3] += are * q[5] + aim * q[4];
                h[4] += are * q[6] - aim * q[7];
                h[5] += are * q[7] + aim * q[6];
            } else {
                const double* x = knots + (b * MBHL_NMODE + mi) * S;
                const int j = find_interval(x, S, f, lf, mc.ln_flo, mc.inv_dlog);
                const double u = f - x[j];
                mode_contrib(coef + ((b * MBHL_NMODE + mi) * (int64_t)(S - 1) + j) * kCoefStride, u, 1.0, h);
            }
        }
    }
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
        double2* o = reinterpret_cast<double2*>(out + ((b * 3 + ch) * Nout + k) * 2);
        *o = make_double2(h[2 * ch], h[2 * ch + 1]);
    }
}

// mbhl_sparse: copy of the y rows with the phase row converted to radians
__global__ void k_export_y(const double* y, int64_t n_rows, int S, double* out) {   // out may alias y
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_rows * S) return;
    const int64_t row = i / S;
    const double v = y[i];
    out[i] = ((row % MBHL_NQ) == 1) ? v * kTwoPi : v;
}

// mbhl_sparse: coefficient records with the phase row converted back to the documented form (cycles, y_j in
// [-1/2, 1/2], no linear term): one thread per (walker, mode, interval, quantity)
__global__ void k_export_coef(const WalkerConst* __restrict__ wc, const double* __restrict__ knots, const double* __restrict__ coef,
                              int64_t n_bm, int S, double* __restrict__ out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_bm * (S - 1) * MBHL_NQ) return;
    const int q = (int)(i % MBHL_NQ);
    const int64_t ij = i / MBHL_NQ;
    const int64_t bm = ij / (S - 1);
    const int j = (int)(ij - bm * (S - 1));
    double2 a = reinterpret_cast<const double2*>(coef)[2 * i], c = reinterpret_cast<const double2*>(coef)[2 * i + 1];
    const WalkerConst& w = wc[bm / MBHL_NMODE];
    if (q == 1 && w.valid && w.mode[bm % MBHL_NMODE].active) {
        const double t = w.t_coal;
        double y = 0.25 * a.x + linear_cycles(knots[bm * S + j], t);
        y -= rint(y);
        a = make_double2(y, 0.25 * a.y + t);
        c = make_double2(0.25 * c.x, 0.25 * c.y);
    }
    reinterpret_cast<double2*>(out)[2 * i] = a;
    reinterpret_cast<double2*>(out)[2 * i + 1] = c;
}

// FP64 peak probe: 8 independent DFMA chains per thread
__global__ void k_dfma_probe(int64_t iters, double* __restrict__ sink) {
    double a0 = 1.0 + threadIdx.x * 1e-9, a1 = 1.1, a2 = 1.2, a3 = 1.3, a4 = 1.4, a5 = 1.5, a6 = 1.6, a7 = 1.7;
    const double m = 0.999999, c = 1e-6;
    for (int64_t i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 12345.678) sink[0] = s;   // never true; keeps the chains alive
}

}  // namespace mbhl
