// mbhl_kernels.cuh - the hot-path kernels (steps a1-a7 of SURVEY.md section 8(a)).
#pragma once
#include <cuda_runtime.h>

#include "mbhl_model.cuh"

namespace mbhl {

constexpr int kCoefStride = MBHL_NQ * 4;   // doubles per (walker, mode, interval) record = 256 B
constexpr int kSplineHalo = 32;            // overlap rows of the block-parallel tridiagonal solve
constexpr int kDenseThreads = 128;
constexpr int kDenseR = 4;                 // bins per thread per chunk
constexpr int kChunk = kDenseThreads * kDenseR;

// ---------------------------------------------------------------------------------------------
// init: weights, weighted data, <d|d>, grid validation
// ---------------------------------------------------------------------------------------------
__global__ void k_init_weights(const double* __restrict__ data, const double* __restrict__ psd, int64_t N, double df,
                               double* __restrict__ w, double* __restrict__ wdre, double* __restrict__ wdim,
                               double* __restrict__ dd_part) {
    // one block handles 1024 consecutive bins of all three channels; fixed-order reduction
    __shared__ double red[256];
    const int64_t k0 = (int64_t)blockIdx.x * 1024;
    double acc = 0.0;
    for (int c = 0; c < 3; ++c) {
        for (int i = threadIdx.x; i < 1024; i += 256) {
            const int64_t k = k0 + i;
            if (k < N) {
                const double s = psd[c * N + k];
                const double ww = (isfinite(s) && s > 0.0) ? 4.0 * df / s : 0.0;
                const double dre = data[(c * N + k) * 2], dim = data[(c * N + k) * 2 + 1];
                w[c * N + k] = ww;
                wdre[c * N + k] = ww * dre;
                wdim[c * N + k] = ww * dim;
                acc += ww * (dre * dre + dim * dim);
            }
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
// a1 + a2: per-walker constants and bands (one thread per walker)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(64) k_walker_consts(const double* __restrict__ params, int64_t B, double t0, double f_min,
                                                      double f_max, int S, uint32_t mode_mask, WalkerConst* __restrict__ out) {
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    WalkerConst c;
    build_walker(params + b * 11, t0, f_min, f_max, S, mode_mask, c);
    out[b] = c;
}

// ---------------------------------------------------------------------------------------------
// a3 + a4: PhenomHM + response at the sparse knots, one thread per (walker, mode, knot)
// y layout [walker][mode][q][S], phase row in cycles; knots [walker][mode][S]
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_sparse_eval(const WalkerConst* __restrict__ wc, int S, double* __restrict__ knots,
                                                     double* __restrict__ y) {
    const int64_t bm = blockIdx.x;                  // walker * 6 + mode
    const int64_t b = bm / MBHL_NMODE;
    const int mi = (int)(bm - b * MBHL_NMODE);
    const int s = blockIdx.y * blockDim.x + threadIdx.x;
    if (s >= S) return;
    const WalkerConst& c = wc[b];
    double q[MBHL_NQ];
    double f = 0.0;
    if (c.valid && c.mode[mi].active) {
        const ModeConst& mc = c.mode[mi];
        f = (s == 0) ? mc.f_lo : ((s == S - 1) ? mc.f_hi : mc.f_lo * exp(s * mc.dlog));
        smooth_quantities(c, mi, f, q);
    } else {
#pragma unroll
        for (int i = 0; i < MBHL_NQ; ++i) q[i] = 0.0;
    }
    knots[bm * S + s] = f;
#pragma unroll
    for (int i = 0; i < MBHL_NQ; ++i) y[(bm * MBHL_NQ + i) * S + s] = q[i];
}

// ---------------------------------------------------------------------------------------------
// a5: not-a-knot cubic spline coefficients.  One CTA of 4 warps per (walker, mode);
// warp w solves quantities 2w and 2w+1 (the matrix is shared).  Each lane owns a block of consecutive
// rows of the tridiagonal slope system.  It runs the forward (LU) recurrence from kSplineHalo rows
// before its block and the backward (UL) recurrence from kSplineHalo rows after it, then combines the
// two at every owned row (twisted factorisation).  The system is strictly diagonally dominant, so the
// influence of the cut decays like 0.27^halo for log-spaced knots - below fp64 rounding; blocks that
// reach row 0 / S-1 use the true not-a-knot rows, so systems with S <= halo are solved exactly.
// coef layout [walker][mode][interval][q][4] = (y_j, s_j, c_j, d_j); phase row: y_j reduced mod 1 cycle.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int pad_idx(int r) { return r + (r >> 5); }

__host__ __device__ inline size_t spline_smem_bytes(int S) {
    const int SP = S + (S >> 5) + 1;
    return (size_t)(2 + 2 * MBHL_NQ) * SP * sizeof(double);
}

__global__ void __launch_bounds__(128) k_spline(const WalkerConst* __restrict__ wc, int S, const double* __restrict__ knots,
                                                const double* __restrict__ y, double* __restrict__ coef) {
    extern __shared__ double sm[];
    const int SP = S + (S >> 5) + 1;
    double* xk = sm;                     // knots                         [SP]
    double* cps = sm + SP;               // forward pivots c'_r           [SP]
    double* rhs = cps + SP;              // right-hand sides              [8][SP]
    double* wk = rhs + MBHL_NQ * SP;     // forward d'_r, then the slopes [8][SP]
    const int64_t bm = blockIdx.x;
    const int64_t b = bm / MBHL_NMODE;
    const int mi = (int)(bm - b * MBHL_NMODE);
    double* cout = coef + bm * (int64_t)(S - 1) * kCoefStride;
    const bool active = wc[b].valid && wc[b].mode[mi].active;
    if (!active) {
        for (int64_t i = threadIdx.x; i < (int64_t)(S - 1) * kCoefStride; i += blockDim.x) cout[i] = 0.0;
        return;
    }
    const double* xg = knots + bm * S;
    const double* yg = y + bm * MBHL_NQ * S;
    for (int i = threadIdx.x; i < S; i += blockDim.x) xk[pad_idx(i)] = xg[i];
    __syncthreads();
    // right-hand sides of the slope system, all rows in parallel
    for (int idx = threadIdx.x; idx < MBHL_NQ * S; idx += blockDim.x) {
        const int q = idx / S, r = idx - q * S;
        const double* yq = yg + q * S;
        double v;
        if (r == 0) {
            const double h0 = xk[pad_idx(1)] - xk[pad_idx(0)], h1 = xk[pad_idx(2)] - xk[pad_idx(1)];
            const double d0 = (yq[1] - yq[0]) / h0, d1 = (yq[2] - yq[1]) / h1;
            v = ((3.0 * h0 + 2.0 * h1) * h1 * d0 + h0 * h0 * d1) / (h0 + h1);
        } else if (r == S - 1) {
            const double hm = xk[pad_idx(S - 1)] - xk[pad_idx(S - 2)], hn = xk[pad_idx(S - 2)] - xk[pad_idx(S - 3)];
            const double dm = (yq[S - 1] - yq[S - 2]) / hm, dn = (yq[S - 2] - yq[S - 3]) / hn;
            v = (hm * hm * dn + (2.0 * hn + 3.0 * hm) * hn * dm) / (hn + hm);
        } else {
            const double hl = xk[pad_idx(r)] - xk[pad_idx(r - 1)], hr = xk[pad_idx(r + 1)] - xk[pad_idx(r)];
            v = 3.0 * (hr * ((yq[r] - yq[r - 1]) / hl) + hl * ((yq[r + 1] - yq[r]) / hr));
        }
        rhs[q * SP + pad_idx(r)] = v;
    }
    __syncthreads();

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int qa = 2 * warp, qb = 2 * warp + 1;
    const int m = (S + 31) / 32;                       // rows per lane
    const int own0 = lane * m, own1 = min(S, own0 + m);
    if (own0 < own1) {
        const int r0 = max(0, own0 - kSplineHalo), r1 = min(S, own1 + kSplineHalo);
        // matrix row r: (lower a, diag d, upper u)
        auto mat = [&](int r, double& a, double& d, double& u) {
            if (r == 0) {
                const double h0 = xk[pad_idx(1)] - xk[pad_idx(0)], h1 = xk[pad_idx(2)] - xk[pad_idx(1)];
                a = 0.0; d = h1; u = h0 + h1;
            } else if (r == S - 1) {
                const double hm = xk[pad_idx(S - 1)] - xk[pad_idx(S - 2)], hn = xk[pad_idx(S - 2)] - xk[pad_idx(S - 3)];
                a = hm + hn; d = hn; u = 0.0;
            } else {
                const double hl = xk[pad_idx(r)] - xk[pad_idx(r - 1)], hr = xk[pad_idx(r + 1)] - xk[pad_idx(r)];
                a = hr; d = 2.0 * (hl + hr); u = hl;
            }
        };
        // forward recurrence: s_r + cp_r s_{r+1} = dp_r
        double cp = 0.0, gA = 0.0, gB = 0.0;           // values at row r-1
        double cp_e = 0.0, gA_e = 0.0, gB_e = 0.0;     // values at row own0-1 (kept in registers)
        for (int r = r0; r < own1 - 1; ++r) {
            double a, d, u;
            mat(r, a, d, u);
            const double inv = 1.0 / (d - a * cp);
            cp = u * inv;
            gA = (rhs[qa * SP + pad_idx(r)] - a * gA) * inv;
            gB = (rhs[qb * SP + pad_idx(r)] - a * gB) * inv;
            if (r == own0 - 1) { cp_e = cp; gA_e = gA; gB_e = gB; }
            if (r >= own0) {
                cps[pad_idx(r)] = cp;                   // all four warps write identical values
                wk[qa * SP + pad_idx(r)] = gA;
                wk[qb * SP + pad_idx(r)] = gB;
            }
        }
        // backward recurrence: s_r + bp_r s_{r-1} = ep_r, combined with the forward one at owned rows
        double bp = 0.0, eA = 0.0, eB = 0.0;           // values at row r+1
        for (int r = r1 - 1; r >= own0; --r) {
            double a, d, u;
            mat(r, a, d, u);
            const double rA = rhs[qa * SP + pad_idx(r)], rB = rhs[qb * SP + pad_idx(r)];
            if (r < own1) {
                double fc, fA, fB;                      // forward quantities of row r-1
                if (r == own0) { fc = cp_e; fA = gA_e; fB = gB_e; }
                else { fc = cps[pad_idx(r - 1)]; fA = wk[qa * SP + pad_idx(r - 1)]; fB = wk[qb * SP + pad_idx(r - 1)]; }
                const double invD = 1.0 / (d - a * fc - u * bp);
                const double sA = (rA - a * fA - u * eA) * invD;
                const double sB = (rB - a * fB - u * eB) * invD;
                wk[qa * SP + pad_idx(r)] = sA;          // d'_r of this row is no longer needed
                wk[qb * SP + pad_idx(r)] = sB;
            }
            const double inv = 1.0 / (d - u * bp);
            bp = a * inv;
            eA = (rA - u * eA) * inv;
            eB = (rB - u * eB) * inv;
        }
    }
    __syncthreads();
    // coefficients: one (interval, quantity) per thread, 32 B each, consecutive threads -> consecutive records
    for (int idx = threadIdx.x; idx < (S - 1) * MBHL_NQ; idx += blockDim.x) {
        const int j = idx / MBHL_NQ, q = idx - j * MBHL_NQ;
        const double h = xk[pad_idx(j + 1)] - xk[pad_idx(j)];
        double y0 = yg[q * S + j];
        const double y1 = yg[q * S + j + 1];
        const double s0 = wk[q * SP + pad_idx(j)], s1 = wk[q * SP + pad_idx(j + 1)];
        const double dl = (y1 - y0) / h;
        const double cc = (3.0 * dl - 2.0 * s0 - s1) / h;
        const double dd = (s0 + s1 - 2.0 * dl) / (h * h);
        if (q == 1) y0 -= rint(y0);
        double2* o = reinterpret_cast<double2*>(cout + (int64_t)j * kCoefStride + q * 4);
        o[0] = make_double2(y0, s0);
        o[1] = make_double2(cc, dd);
    }
}

// ---------------------------------------------------------------------------------------------
// a6 + a7: fused dense kernel.  Interpolates every active mode onto the Fourier bins of one chunk,
// sums the modes per bin, and accumulates <d|h> and <h|h> (eqs. 2, 3, 11); the template
// is never written to memory.  One CTA per (chunk, walker); thread t owns bins k0 + t + 128 r.
// ---------------------------------------------------------------------------------------------
struct DenseArgs {
    const WalkerConst* wc;
    const double* knots;     // [B][6][S]
    const double* coef;      // [B][6][S-1][8][4]
    const double* freqs;     // [N]
    const double* w;         // [3][N]
    const double* wdre;      // [3][N]
    const double* wdim;      // [3][N]
    double* partials;        // [B][n_chunks][2]
    unsigned long long* counters;   // [2]: in-band (bin, mode) pairs, bins covered by >= 1 mode
    int64_t N;
    int S;
    int n_chunks;
};

// Locates the spline interval of frequency f (ln f = lf) on the log-spaced knots x[0..S-1].
__device__ __forceinline__ int find_interval(const double* __restrict__ x, int S, double f, double lf, const ModeConst& mc) {
    int j = (int)((lf - mc.ln_flo) * mc.inv_dlog);
    j = max(0, min(S - 2, j));
    while (j > 0 && f < __ldg(x + j)) --j;
    while (j < S - 2 && f >= __ldg(x + j + 1)) ++j;
    return j;
}

// One mode's contribution at one bin: 8 Horner cubics, phase in cycles, sincospi, complex MACs.
__device__ __forceinline__ void mode_contrib(const double* __restrict__ rec, double u, double lin, double h[6]) {
    double v[MBHL_NQ];
#pragma unroll
    for (int q = 0; q < MBHL_NQ; q += 1) {
        const double2 c01 = __ldg(reinterpret_cast<const double2*>(rec + q * 4));
        const double2 c23 = __ldg(reinterpret_cast<const double2*>(rec + q * 4 + 2));
        v[q] = fma(fma(fma(c23.y, u, c23.x), u, c01.y), u, c01.x);
    }
    double cyc = v[1] - lin;
    cyc -= rint(cyc);
    double sn, cs;
    sincospi(2.0 * cyc, &sn, &cs);
    const double are = v[0] * cs, aim = v[0] * sn;
    h[0] = fma(are, v[2], fma(-aim, v[3], h[0]));
    h[1] = fma(are, v[3], fma(aim, v[2], h[1]));
    h[2] = fma(are, v[4], fma(-aim, v[5], h[2]));
    h[3] = fma(are, v[5], fma(aim, v[4], h[3]));
    h[4] = fma(are, v[6], fma(-aim, v[7], h[4]));
    h[5] = fma(are, v[7], fma(aim, v[6], h[5]));
}

// frac(f * t) with the product taken exactly (reading G9): f and t are the supplied doubles.
__device__ __forceinline__ double linear_cycles(double f, double t) {
    const double p = f * t;
    const double e = fma(f, t, -p);
    return (p - rint(p)) + e;
}

__global__ void __launch_bounds__(kDenseThreads) k_dense(DenseArgs A) {
    const int chunk = blockIdx.x;
    const int64_t b = blockIdx.y;
    const int64_t k0 = (int64_t)chunk * kChunk;
    const WalkerConst& c = A.wc[b];
    double* part = A.partials + (b * A.n_chunks + chunk) * 2;
    // chunk-level early exit: no active mode overlaps [fa, fb]
    const double fa = A.freqs[k0];
    const double fb = A.freqs[min(k0 + kChunk, A.N) - 1];
    bool any = false;
    if (c.valid) {
#pragma unroll
        for (int mi = 0; mi < MBHL_NMODE; ++mi)
            any = any || (c.mode[mi].active && fb >= c.mode[mi].f_lo && fa <= c.mode[mi].f_hi);
    }
    if (!any) {
        if (threadIdx.x == 0) { part[0] = 0.0; part[1] = 0.0; }
        return;
    }
    const double t_coal = c.t_coal;
    double dh = 0.0, hh = 0.0;
    unsigned int npairs = 0, nbins = 0;
#pragma unroll 1
    for (int r = 0; r < kDenseR; ++r) {
        const int64_t k = k0 + threadIdx.x + r * kDenseThreads;
        if (k >= A.N) break;
        const double f = A.freqs[k];
        const double lf = log(f);
        const double lin = linear_cycles(f, t_coal);
        double h[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        unsigned int hit = 0;
#pragma unroll 1
        for (int mi = 0; mi < MBHL_NMODE; ++mi) {
            const ModeConst& mc = c.mode[mi];
            if (!mc.active || f < mc.f_lo || f > mc.f_hi) continue;
            const double* x = A.knots + (b * MBHL_NMODE + mi) * A.S;
            const int j = find_interval(x, A.S, f, lf, mc);
            const double u = f - __ldg(x + j);
            const double* rec = A.coef + ((b * MBHL_NMODE + mi) * (int64_t)(A.S - 1) + j) * kCoefStride;
            mode_contrib(rec, u, lin, h);
            ++hit;
        }
        if (hit) {
            npairs += hit;
            ++nbins;
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                const double wre = A.wdre[ch * A.N + k], wim = A.wdim[ch * A.N + k], ww = A.w[ch * A.N + k];
                dh = fma(wre, h[2 * ch], fma(wim, h[2 * ch + 1], dh));
                hh = fma(ww, fma(h[2 * ch], h[2 * ch], h[2 * ch + 1] * h[2 * ch + 1]), hh);
            }
        }
    }
    // block reduction (fixed order): warp shuffles, then the four warp sums
    __shared__ double red[2][kDenseThreads / 32];
    __shared__ unsigned int redc[2][kDenseThreads / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dh += __shfl_down_sync(0xffffffffu, dh, o);
        hh += __shfl_down_sync(0xffffffffu, hh, o);
        npairs += __shfl_down_sync(0xffffffffu, npairs, o);
        nbins += __shfl_down_sync(0xffffffffu, nbins, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { red[0][warp] = dh; red[1][warp] = hh; redc[0][warp] = npairs; redc[1][warp] = nbins; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double sdh = 0.0, shh = 0.0;
        unsigned int sp = 0, sb = 0;
        for (int i = 0; i < kDenseThreads / 32; ++i) { sdh += red[0][i]; shh += red[1][i]; sp += redc[0][i]; sb += redc[1][i]; }
        part[0] = sdh;
        part[1] = shh;
        if (sp) { atomicAdd(A.counters, (unsigned long long)sp); atomicAdd(A.counters + 1, (unsigned long long)sb); }
    }
}

// a7: deterministic final reduction, one warp per walker; logL = <d|h> - 1/2<h|h> - 1/2<d|d> (eq. 2)
__global__ void __launch_bounds__(128) k_final_reduce(const WalkerConst* __restrict__ wc, const double* __restrict__ partials,
                                                      int n_chunks, int64_t B, double dd, double* __restrict__ d_h,
                                                      double* __restrict__ h_h, double* __restrict__ logL) {
    const int64_t b = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (b >= B) return;
    const int lane = threadIdx.x & 31;
    const double* p = partials + b * n_chunks * 2;
    double sdh = 0.0, shh = 0.0;
    for (int i = lane; i < n_chunks; i += 32) { sdh += p[2 * i]; shh += p[2 * i + 1]; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sdh += __shfl_down_sync(0xffffffffu, sdh, o);
        shh += __shfl_down_sync(0xffffffffu, shh, o);
    }
    if (lane == 0) {
        const bool valid = wc[b].valid != 0;
        if (!valid) { sdh = 0.0; shh = 0.0; }
        if (d_h) d_h[b] = sdh;
        if (h_h) h_h[b] = shh;
        if (logL) logL[b] = valid ? (sdh - 0.5 * shh - 0.5 * dd) : -INFINITY;
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
        const double lin = linear_cycles(f, c.t_coal);
        for (int mi = 0; mi < MBHL_NMODE; ++mi) {
            const ModeConst& mc = c.mode[mi];
            if (!mc.active || !(f >= mc.f_lo) || !(f <= mc.f_hi)) continue;
            if (direct) {
                double q[MBHL_NQ];
                smooth_quantities(c, mi, f, q);
                double cyc = q[1] - rint(q[1]) - lin;
                cyc -= rint(cyc);
                double sn, cs;
                sincospi(2.0 * cyc, &sn, &cs);
                const double are = q[0] * cs, aim = q[0] * sn;
                h[0] += are * q[2] - aim * q[3];
                h[1] += are * q[3] + aim * q[2];
                h[2] += are * q[4] - aim * q[5];
                h[3] += are * q[5] + aim * q[4];
                h[4] += are * q[6] - aim * q[7];
                h[5] += are * q[7] + aim * q[6];
            } else {
                const double* x = knots + (b * MBHL_NMODE + mi) * S;
                const int j = find_interval(x, S, f, lf, mc);
                const double u = f - x[j];
                mode_contrib(coef + ((b * MBHL_NMODE + mi) * (int64_t)(S - 1) + j) * kCoefStride, u, lin, h);
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
__global__ void k_export_y(const double* __restrict__ y, int64_t n_rows, int S, double* __restrict__ out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_rows * S) return;
    const int64_t row = i / S;
    const double v = y[i];
    out[i] = ((row % MBHL_NQ) == 1) ? v * kTwoPi : v;
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
