// mbhl_het.cuh - heterodyned ("relative binning") likelihood, an accuracy-controlled variant of the hot path
// ("we may test different approximations").  Definition: DESIGN.md section 10, reading H1.
//
// A reference parameter set gives per-mode reference phasors E0_m(k) = exp(i theta0_m(f_k)) on the fine grid (the total
// phase of its spline template; 0 outside the reference band of the mode).  A walker's template is
// h^c(f_k) = sum_m r_{c,m}(f_k) E0_m(k) with the slowly varying envelope
//     r_{c,m}(f) = A_m(f) That^c_m(f) exp(i [theta_m(f) - theta0_m(f)]),
// replaced on every coarse bin b = [e_b, e_{b+1}) by the parabola r0 + r1 x + r2 x^2 (x = f - fbar_b) through its values at
// the bin's first, centre and last frequency.  Then <d|h> and <h|h> are contractions of (r0, r1, r2) with the moments
//     A_n[c][m][b]     = sum_{k in b} w_c conj(d_c) E0_m x_k^n,   B_n[c][m][m'][b] = sum_{k in b} w_c E0_m conj(E0_m') x_k^n,
// n = 0, 1, 2, computed ONCE per reference:
//   k_het_summary   one CTA per coarse bin: a thread per fine bin forms the 6 phasors, then a thread per summary
//                   entry accumulates it over the tile from shared memory (fixed order: reproducible)
//   k_het_eval      one thread per (walker, coarse bin): envelope at f_L and f_R (each moved to the nearest
//                   frequency inside the band common to walker and reference: no spline is extrapolated) for the 6 modes
//                   from the walker's spline records and the reference's phase records, contraction with A and B, block reduction -> one partial per (walker, block);
//                   k_final_reduce adds them in fixed order.
#pragma once
#include <cuda_runtime.h>

namespace mbhl {

constexpr int kHetTile = 256;                 // fine bins per pass of k_het_summary
constexpr int kHetRow = 23;                   // doubles per fine bin in shared memory: 12 phasor + 3 w + 6 w d + 1 (f - fbar), padded odd
constexpr int kHetA = 3 * MBHL_NMODE;         // (c, m) entries
constexpr int kHetB = 3 * MBHL_NMODE * MBHL_NMODE;   // (c, m, m') entries
constexpr int kHetEvalThreads = 128;

struct HetArgs {
    const double* tiles;        // the context's data tiles [n_chunks][10][512]
    const DenseWalker* ref_dw;  // [1] bin ranges of the reference's modes
    const double* ref_knots;    // [6][S]
    const double* ref_coef;     // [6][S-1][8][4]
    const long long* edges;     // [n_b + 1]
    double2* A0; double2* A1; double2* A2;   // [3][6][n_b]
    double2* B0; double2* B1; double2* B2;   // [3][6][6][n_b]
    int S, n_b;
    uint32_t mode_mask;
};

// total phase of the reference's mode mi at frequency f in quarter turns (the record's phase cubic carries the linear term)
__device__ __forceinline__ double het_ref_phase(const double* __restrict__ x, const double* __restrict__ coef, int S, double f,
                                                double ln_flo, double inv_dlog) {
    const int j = find_interval(x, S, f, log(f), ln_flo, inv_dlog);
    const double u = f - __ldg(x + j);
    const double* rec = coef + (int64_t)j * kCoefStride + 4;
    const double2 p01 = __ldg(reinterpret_cast<const double2*>(rec)), p23 = __ldg(reinterpret_cast<const double2*>(rec + 2));
    return fma(fma(fma(p23.y, u, p23.x), u, p01.y), u, p01.x);
}

// Per coarse bin b, once per reference: the three evaluation frequencies f_p (first, centre, last), their logarithms, and
// for every mode present in the bin (the bins are refined by the reference's band edges: present throughout or absent)
// the reference's phase at the three frequencies in quarter turns.  pts [n_b][3][2] = (f, ln f); ref_p4 [6][n_b][3];
// present [6][n_b].
__global__ void k_het_bin_points(const double* __restrict__ freqs, const long long* __restrict__ edges, int n_b, const DenseWalker* __restrict__ ref_dw,
                                 const double* __restrict__ ref_knots, const double* __restrict__ ref_coef, int S, uint32_t mode_mask,
                                 double* __restrict__ pts, double* __restrict__ ref_p4, int* __restrict__ present) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_b) return;
    const long long k0 = edges[b], k1 = edges[b + 1] - 1;
    const double fl = freqs[k0], fr = freqs[k1];
    const double f3[3] = {fl, 0.5 * (fl + fr), fr};
#pragma unroll
    for (int p = 0; p < 3; ++p) { pts[(b * 3 + p) * 2] = f3[p]; pts[(b * 3 + p) * 2 + 1] = log(f3[p]); }
    for (int mi = 0; mi < MBHL_NMODE; ++mi) {
        const DenseMode dm = ref_dw->mode[mi];
        const int in = ref_dw->valid && ((mode_mask >> mi) & 1u) && k0 >= dm.k_lo && k1 <= dm.k_hi;
        present[mi * n_b + b] = in;
#pragma unroll
        for (int p = 0; p < 3; ++p)
            ref_p4[((int64_t)mi * n_b + b) * 3 + p] =
                in ? het_ref_phase(ref_knots + mi * S, ref_coef + (int64_t)mi * (S - 1) * kCoefStride, S, f3[p], dm.ln_flo, dm.inv_dlog) : 0.0;
    }
}

__global__ void __launch_bounds__(kHetTile) k_het_summary(HetArgs H) {
    __shared__ double s_bin[kHetTile * kHetRow];
    const int b = blockIdx.x, tid = threadIdx.x;
    const long long k0 = H.edges[b], k1 = H.edges[b + 1];       // fine bins [k0, k1)
    auto freq = [&](long long k) { return H.tiles[(k / kChunk) * kTileDoubles + (k % kChunk)]; };
    const double fbar = 0.5 * (freq(k0) + freq(k1 - 1));
    // this thread's summary entry: tid < 18 -> A[c][m]; 18 <= tid < 18 + 108 -> B[c][m][m']
    double a0r = 0.0, a0i = 0.0, a1r = 0.0, a1i = 0.0, a2r = 0.0, a2i = 0.0;
    const bool isA = tid < kHetA, isB = tid >= kHetA && tid < kHetA + kHetB;
    int c = 0, m = 0, mp = 0;
    if (isA) { c = tid / MBHL_NMODE; m = tid % MBHL_NMODE; }
    if (isB) { const int e = tid - kHetA; c = e / (MBHL_NMODE * MBHL_NMODE); m = (e / MBHL_NMODE) % MBHL_NMODE; mp = e % MBHL_NMODE; }
    for (long long t0 = k0; t0 < k1; t0 += kHetTile) {
        const long long k = t0 + tid;
        double* row = s_bin + tid * kHetRow;
        if (k < k1) {
            const double* tile = H.tiles + (k / kChunk) * kTileDoubles;
            const int i = (int)(k % kChunk);
            const double f = tile[i];
#pragma unroll
            for (int mi = 0; mi < MBHL_NMODE; ++mi) {
                const DenseMode dm = H.ref_dw->mode[mi];
                double cs = 0.0, sn = 0.0;
                if (H.ref_dw->valid && ((H.mode_mask >> mi) & 1u) && k >= dm.k_lo && k <= dm.k_hi)
                    sincos_qturn(het_ref_phase(H.ref_knots + mi * H.S, H.ref_coef + (int64_t)mi * (H.S - 1) * kCoefStride, H.S, f,
                                               dm.ln_flo, dm.inv_dlog), sn, cs);
                row[2 * mi] = cs;
                row[2 * mi + 1] = sn;
            }
#pragma unroll
            for (int r = 0; r < 9; ++r) row[12 + r] = tile[(1 + r) * kChunk + i];      // w^A,E,T then (w Re d, w Im d)^A,E,T
            row[21] = f - fbar;
        }
        __syncthreads();
        const int n = (int)((k1 - t0 < kHetTile) ? (k1 - t0) : kHetTile);
        if (isA) {
            for (int i = 0; i < n; ++i) {
                const double* r = s_bin + i * kHetRow;
                const double ec = r[2 * m], es = r[2 * m + 1], wr = r[15 + 2 * c], wi = r[16 + 2 * c], d = r[21];
                const double re = wr * ec + wi * es, im = wr * es - wi * ec;       // w conj(d) E0
                a0r += re; a0i += im;
                a1r = fma(re, d, a1r); a1i = fma(im, d, a1i);
                a2r = fma(re * d, d, a2r); a2i = fma(im * d, d, a2i);
            }
        } else if (isB) {
            for (int i = 0; i < n; ++i) {
                const double* r = s_bin + i * kHetRow;
                const double ec = r[2 * m], es = r[2 * m + 1], fc = r[2 * mp], fs = r[2 * mp + 1], w = r[12 + c], d = r[21];
                const double re = w * (ec * fc + es * fs), im = w * (es * fc - ec * fs);   // w E0_m conj(E0_m')
                a0r += re; a0i += im;
                a1r = fma(re, d, a1r); a1i = fma(im, d, a1i);
                a2r = fma(re * d, d, a2r); a2i = fma(im * d, d, a2i);
            }
        }
        __syncthreads();
    }
    if (isA) {
        H.A0[(c * MBHL_NMODE + m) * (int64_t)H.n_b + b] = make_double2(a0r, a0i);
        H.A1[(c * MBHL_NMODE + m) * (int64_t)H.n_b + b] = make_double2(a1r, a1i);
        H.A2[(c * MBHL_NMODE + m) * (int64_t)H.n_b + b] = make_double2(a2r, a2i);
    } else if (isB) {
        H.B0[((c * MBHL_NMODE + m) * MBHL_NMODE + mp) * (int64_t)H.n_b + b] = make_double2(a0r, a0i);
        H.B1[((c * MBHL_NMODE + m) * MBHL_NMODE + mp) * (int64_t)H.n_b + b] = make_double2(a1r, a1i);
        H.B2[((c * MBHL_NMODE + m) * MBHL_NMODE + mp) * (int64_t)H.n_b + b] = make_double2(a2r, a2i);
    }
}

struct HetEvalArgs {
    HetArgs H;
    const WalkerConst* wc;      // [B] (valid flag, mode activity, knot-grid constants)
    const DenseWalker* dw;      // [B]
    const double* knots;        // [B][6][S]
    const double* coef;         // [B][6][S-1][8][4]
    const double* pts;          // [n_b][3][2] (f, ln f) at the first, centre and last frequency of every coarse bin
    const double* ref_p4;       // [6][n_b][3] the reference's phase there (quarter turns)
    const int* present;         // [6][n_b] mode in band throughout the coarse bin (else absent: contributes nothing)
    const double* ref_ln_flo; const double* ref_inv_dlog;   // [6]
    const double* ref_f_lo; const double* ref_f_hi;                               // [6] the reference's bands
    double* partials;           // [B][n_groups][2]
    int n_groups;               // ceil(n_b / kHetEvalThreads)
};

// grid (ceil(n_b / 128), B): thread = coarse bin, blockIdx.y = walker.  Per mode and evaluation point (first, centre, last
// frequency of the bin, each moved into the band common to walker and reference; a bin the walker's band does not reach is skipped) the channel-independent part
// A exp(i [theta - theta0]) is formed once; the three channels then differ by their transfer cubics only.
__global__ void __launch_bounds__(kHetEvalThreads) k_het_eval(HetEvalArgs E) {
    __shared__ double s_red[2][kHetEvalThreads / 32];
    const int b = blockIdx.x * kHetEvalThreads + threadIdx.x;
    const int64_t wkr = blockIdx.y;
    const int n_b = E.H.n_b, S = E.H.S;
    double dh = 0.0, hh = 0.0;
    if (b < n_b && E.wc[wkr].valid) {
        const double* pt = E.pts + (int64_t)b * 6;
        const double f3[3] = {pt[0], pt[2], pt[4]}, lf3[3] = {pt[1], pt[3], pt[5]};
        const double s = 0.5 * (f3[2] - f3[0]);
        const double i1 = s > 0.0 ? 0.5 / s : 0.0, i2 = s > 0.0 ? 0.5 / (s * s) : 0.0;
        double er[MBHL_NMODE][3], ei[MBHL_NMODE][3], uu[MBHL_NMODE][3];     // A exp(i dtheta) and u = f - x_j at the three points
        int jj[MBHL_NMODE][3];                                              // walker interval of each point; -1: mode absent
#pragma unroll
        for (int mi = 0; mi < MBHL_NMODE; ++mi) {
#pragma unroll
            for (int p = 0; p < 3; ++p) { er[mi][p] = ei[mi][p] = uu[mi][p] = 0.0; jj[mi][p] = -1; }
            if (!E.present[mi * n_b + b] || !E.wc[wkr].mode[mi].active) continue;
            const ModeConst& mc = E.wc[wkr].mode[mi];
            if (!(fmax(mc.f_lo, E.ref_f_lo[mi]) <= fmin(mc.f_hi, E.ref_f_hi[mi]))) continue;
            if (f3[2] < mc.f_lo || f3[0] > mc.f_hi) continue;     // the walker's own band does not reach this coarse bin: no signal here (H1, amended)
            const double* x = E.knots + (wkr * MBHL_NMODE + mi) * S;
            const double* cbase = E.coef + (wkr * MBHL_NMODE + mi) * (int64_t)(S - 1) * kCoefStride;
#pragma unroll
            for (int p = 0; p < 3; ++p) {
                // inside the reference's band by construction; moved into the walker's band if it lies outside it
                const double f = fmin(fmax(f3[p], mc.f_lo), mc.f_hi);
                const bool moved = f != f3[p];
                const double lf = moved ? log(f) : lf3[p];
                const int j = find_interval(x, S, f, lf, mc.ln_flo, mc.inv_dlog);
                const double u = f - __ldg(x + j);
                const double* rec = cbase + (int64_t)j * kCoefStride;
                const double2 a01 = __ldg(reinterpret_cast<const double2*>(rec)), a23 = __ldg(reinterpret_cast<const double2*>(rec + 2));
                const double2 p01 = __ldg(reinterpret_cast<const double2*>(rec + 4)), p23 = __ldg(reinterpret_cast<const double2*>(rec + 6));
                const double amp = fma(fma(fma(a23.y, u, a23.x), u, a01.y), u, a01.x);
                const double p4w = fma(fma(fma(p23.y, u, p23.x), u, p01.y), u, p01.x);
                const double p4r = moved ? het_ref_phase(E.H.ref_knots + mi * S, E.H.ref_coef + (int64_t)mi * (S - 1) * kCoefStride, S, f, E.ref_ln_flo[mi],
                                                         E.ref_inv_dlog[mi])
                                         : E.ref_p4[((int64_t)mi * n_b + b) * 3 + p];
                double sn, cs;
                sincos_qturn(p4w - p4r, sn, cs);
                er[mi][p] = amp * cs;
                ei[mi][p] = amp * sn;
                uu[mi][p] = u;
                jj[mi][p] = j;
            }
        }
        // Re(x conj(y)) and Im(x conj(y))
        auto cre = [](double xr, double xi, double yr, double yi) { return xr * yr + xi * yi; };
        auto cim = [](double xr, double xi, double yr, double yi) { return xi * yr - xr * yi; };
        for (int c = 0; c < 3; ++c) {
            double r0r[MBHL_NMODE], r0i[MBHL_NMODE], r1r[MBHL_NMODE], r1i[MBHL_NMODE], r2r[MBHL_NMODE], r2i[MBHL_NMODE];
#pragma unroll
            for (int mi = 0; mi < MBHL_NMODE; ++mi) {
                double vr[3], vi[3];
#pragma unroll
                for (int p = 0; p < 3; ++p) {
                    vr[p] = vi[p] = 0.0;
                    if (jj[mi][p] < 0) continue;
                    const double* rec = E.coef + ((wkr * MBHL_NMODE + mi) * (int64_t)(S - 1) + jj[mi][p]) * kCoefStride + 8 + 8 * c;
                    const double u = uu[mi][p];
                    const double2 t01 = __ldg(reinterpret_cast<const double2*>(rec)), t23 = __ldg(reinterpret_cast<const double2*>(rec + 2));
                    const double2 s01 = __ldg(reinterpret_cast<const double2*>(rec + 4)), s23 = __ldg(reinterpret_cast<const double2*>(rec + 6));
                    const double tr = fma(fma(fma(t23.y, u, t23.x), u, t01.y), u, t01.x);
                    const double ti = fma(fma(fma(s23.y, u, s23.x), u, s01.y), u, s01.x);
                    vr[p] = er[mi][p] * tr - ei[mi][p] * ti;
                    vi[p] = er[mi][p] * ti + ei[mi][p] * tr;
                }
                r0r[mi] = vr[1]; r0i[mi] = vi[1];
                r1r[mi] = (vr[2] - vr[0]) * i1; r1i[mi] = (vi[2] - vi[0]) * i1;
                r2r[mi] = (vr[2] - 2.0 * vr[1] + vr[0]) * i2; r2i[mi] = (vi[2] - 2.0 * vi[1] + vi[0]) * i2;
            }
#pragma unroll
            for (int mi = 0; mi < MBHL_NMODE; ++mi) {
                const int64_t ia = (c * MBHL_NMODE + mi) * (int64_t)n_b + b;
                const double2 a0 = E.H.A0[ia], a1 = E.H.A1[ia], a2 = E.H.A2[ia];
                dh += (a0.x * r0r[mi] - a0.y * r0i[mi]) + (a1.x * r1r[mi] - a1.y * r1i[mi]) + (a2.x * r2r[mi] - a2.y * r2i[mi]);
                // B_n(m', m) = conj B_n(m, m') and the envelope products are Hermitian too: pairs m' > m count twice
#pragma unroll
                for (int mp = mi; mp < MBHL_NMODE; ++mp) {
                    const int64_t ib = ((c * MBHL_NMODE + mi) * MBHL_NMODE + mp) * (int64_t)n_b + b;
                    const double2 b0 = E.H.B0[ib], b1 = E.H.B1[ib], b2 = E.H.B2[ib];
                    const double pr = cre(r0r[mi], r0i[mi], r0r[mp], r0i[mp]), pi = cim(r0r[mi], r0i[mi], r0r[mp], r0i[mp]);
                    const double qr = cre(r1r[mi], r1i[mi], r0r[mp], r0i[mp]) + cre(r0r[mi], r0i[mi], r1r[mp], r1i[mp]);
                    const double qi = cim(r1r[mi], r1i[mi], r0r[mp], r0i[mp]) + cim(r0r[mi], r0i[mi], r1r[mp], r1i[mp]);
                    const double sr = cre(r2r[mi], r2i[mi], r0r[mp], r0i[mp]) + cre(r1r[mi], r1i[mi], r1r[mp], r1i[mp]) + cre(r0r[mi], r0i[mi], r2r[mp], r2i[mp]);
                    const double si = cim(r2r[mi], r2i[mi], r0r[mp], r0i[mp]) + cim(r1r[mi], r1i[mi], r1r[mp], r1i[mp]) + cim(r0r[mi], r0i[mi], r2r[mp], r2i[mp]);
                    hh += (mp == mi ? 1.0 : 2.0) * ((b0.x * pr - b0.y * pi) + (b1.x * qr - b1.y * qi) + (b2.x * sr - b2.y * si));
                }
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dh += __shfl_down_sync(0xffffffffu, dh, o);
        hh += __shfl_down_sync(0xffffffffu, hh, o);
    }
    if ((threadIdx.x & 31) == 0) { s_red[0][threadIdx.x >> 5] = dh; s_red[1][threadIdx.x >> 5] = hh; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, h = 0.0;
#pragma unroll
        for (int i = 0; i < kHetEvalThreads / 32; ++i) { a += s_red[0][i]; h += s_red[1][i]; }
        double* part = E.partials + (wkr * E.n_groups + blockIdx.x) * 2;
        part[0] = a;
        part[1] = h;
    }
}

}  // namespace mbhl
