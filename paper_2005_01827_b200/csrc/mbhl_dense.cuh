// mbhl_dense.cuh - steps a6 + a7: the fused dense kernel, version 3.
//
// Interpolates every active mode onto the Fourier bins, sums the modes per bin and accumulates
// <d|h> and <h|h> (eqs. 2, 3, 11).  The template is never written to memory (the paper
// stores it and calls cuBLAS).
//
// Work decomposition.  A CTA (4 warps) owns a tile of W <= 8 consecutive walkers and G consecutive 512-bin
// chunks.  Per chunk:
//   1. the 40 KB data tile (f, w, w d) is staged in shared memory by ONE bulk asynchronous copy (TMA,
//      cp.async.bulk + mbarrier) and reused by all W walkers;
//   2. "prepare": thread p < 6 W owns the (walker, mode) pair p for the CTA's whole life.  It checks whether the
//      chunk's in-band bins of its pair lie in ONE spline interval (true for ~93 % of the chunks of config 2:
//      above ~2 mHz an interval of the 1024-knot log grid is wider than a chunk).  If so the 256-byte
//      coefficient record of that interval is staged in shared memory with 16-byte cp.async copies - only
//      when the interval changed since the previous chunk (the thread keeps the staged interval and its
//      bounds in registers) - and every warp whose 128 bins are all in band is marked "fast";
//   3. every warp loops over the walkers.  A warp owns 128 consecutive bins, a lane 4 of them (stride 32) and
//      advances the 4 bins in lockstep (4 independent dependency chains: DFMA latency is 8.4 cycles at an
//      issue rate of one warp-DFMA per 2 cycles per SM sub-partition, measured).  Fast modes read the staged
//      record with warp-uniform 16-byte shared-memory loads; the rest (chunks that straddle a knot, band
//      edges, the lowest ~1e5 bins where intervals are narrower than a chunk) go through the general path:
//      per-warp interval check with warp-uniform global loads, else a per-bin lookup;
//   4. per (walker, bin): <d|h> and <h|h> terms, warp shuffle tree, one shared-memory slot per (warp, walker).
// One partial per (walker, CTA) leaves the kernel; k_final_reduce adds them in fixed order (bitwise
// reproducible, no atomics on values).
//
// The loop body is FP64-pipe bound: per (bin, mode) 8 Horner cubics (24 DFMA), the exact linear phase term
// (reading G9), a quarter-turn sincos (19) and 3 complex multiply-adds (12).
#pragma once
#include <cuda_runtime.h>

namespace mbhl {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// sin and cos of p4[r] quarter turns for the kDenseR bins of a lane, advanced in lockstep so that the
// kDenseR polynomial chains interleave (same arithmetic as sincos_qturn).
__device__ __forceinline__ void sincos_qturn_x(const double (&p4)[kDenseR], double (&sn)[kDenseR], double (&cs)[kDenseR]) {
    double y[kDenseR], z[kDenseR], ps[kDenseR], pc[kDenseR];
    int n[kDenseR];
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) {
        const double t = p4[r] + kRoundMagic;
        n[r] = __double2loint(t);
        y[r] = p4[r] - (t - kRoundMagic);
    }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) z[r] = y[r] * y[r];
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], kS6, kS5); pc[r] = fma(z[r], kC6, kC5); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], ps[r], kS4); pc[r] = fma(z[r], pc[r], kC4); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], ps[r], kS3); pc[r] = fma(z[r], pc[r], kC3); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], ps[r], kS2); pc[r] = fma(z[r], pc[r], kC2); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], ps[r], kS1); pc[r] = fma(z[r], pc[r], kC1); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], ps[r], kS0); pc[r] = fma(z[r], pc[r], 1.0); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) {
        ps[r] *= y[r];
        const bool odd = (n[r] & 1) != 0;
        const double a = odd ? pc[r] : ps[r];      // sin(angle) up to sign
        const double b = odd ? ps[r] : pc[r];      // cos(angle) up to sign
        sn[r] = __hiloint2double(__double2hiint(a) ^ ((n[r] & 2) << 30), __double2loint(a));
        cs[r] = __hiloint2double(__double2hiint(b) ^ (((n[r] + 1) & 2) << 30), __double2loint(b));
    }
}

// One mode's contribution to the kDenseR bins of a lane when all of them lie in one spline interval and in
// band: `rec` is that interval's record (shared or global memory, same address for every lane), xj its knot.
__device__ __forceinline__ void mode_uniform(const double* __restrict__ rec, double xj, const double (&f)[kDenseR],
                                             const double (&lin4)[kDenseR], double (&h)[kDenseR][6]) {
    double u[kDenseR], are[kDenseR], aim[kDenseR];
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) u[r] = f[r] - xj;
    {
        const double2 p01 = *reinterpret_cast<const double2*>(rec + 4);
        const double2 p23 = *reinterpret_cast<const double2*>(rec + 6);
        double p4[kDenseR], sn[kDenseR], cs[kDenseR];
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) p4[r] = fma(p23.y, u[r], p23.x);
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) p4[r] = fma(p4[r], u[r], p01.y);
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) p4[r] = fma(p4[r], u[r], p01.x);
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) p4[r] = fma(p4[r], 4.0, -lin4[r]);
        sincos_qturn_x(p4, sn, cs);
        const double2 a01 = *reinterpret_cast<const double2*>(rec);
        const double2 a23 = *reinterpret_cast<const double2*>(rec + 2);
        double amp[kDenseR];
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) amp[r] = fma(a23.y, u[r], a23.x);
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) amp[r] = fma(amp[r], u[r], a01.y);
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) amp[r] = fma(amp[r], u[r], a01.x);
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) { are[r] = amp[r] * cs[r]; aim[r] = amp[r] * sn[r]; }
    }
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
        const double2 r01 = *reinterpret_cast<const double2*>(rec + 8 + 8 * ch);
        const double2 r23 = *reinterpret_cast<const double2*>(rec + 10 + 8 * ch);
        const double2 i01 = *reinterpret_cast<const double2*>(rec + 12 + 8 * ch);
        const double2 i23 = *reinterpret_cast<const double2*>(rec + 14 + 8 * ch);
        double tre[kDenseR], tim[kDenseR];
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) { tre[r] = fma(r23.y, u[r], r23.x); tim[r] = fma(i23.y, u[r], i23.x); }
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) { tre[r] = fma(tre[r], u[r], r01.y); tim[r] = fma(tim[r], u[r], i01.y); }
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) { tre[r] = fma(tre[r], u[r], r01.x); tim[r] = fma(tim[r], u[r], i01.x); }
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) {
            h[r][2 * ch] = fma(are[r], tre[r], fma(-aim[r], tim[r], h[r][2 * ch]));
            h[r][2 * ch + 1] = fma(are[r], tim[r], fma(aim[r], tre[r], h[r][2 * ch + 1]));
        }
    }
}

constexpr int kDenseSmemBytes = kTileBytes + kPairs * kCoefStride * (int)sizeof(double);   // 40 KB tile + 12 KB records

// Grid: 1-D, block id = group * n_tiles + tile (walker tiles vary fastest, so the CTAs resident at one time
// share a few chunk groups and the data tiles are served by L2).
__global__ void __launch_bounds__(kDenseThreads, 4) k_dense(DenseArgs A) {
    extern __shared__ __align__(128) double s_dyn[];
    double* const s_tile = s_dyn;                                   // [10][512] staged data tile
    double* const s_rec = s_dyn + kTileDoubles;                     // [kPairs][32] staged coefficient records
    __shared__ DenseWalker s_dw[kMaxW];
    __shared__ double s_xj[kPairs];                                 // knot x_j of the staged record
    __shared__ unsigned s_desc[kPairs];                             // 2 bits per warp: 0 none, 1 fast, 2 general
    __shared__ double s_acc[kDenseThreads / 32][kMaxW][2];
    __shared__ __align__(8) unsigned long long s_bar;
    __shared__ int s_range[2];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int n_tiles = (A.B + A.W - 1) / A.W;
    const int tile_id = blockIdx.x % n_tiles, group = blockIdx.x / n_tiles;
    const int b0 = tile_id * A.W;
    const int nb = min(A.W, A.B - b0);
    // stage the tile's walker records, find the bin range any of them touches
    if (tid == 0) { s_range[0] = 0x7fffffff; s_range[1] = -1; }
    for (int i = tid; i < nb * (int)(sizeof(DenseWalker) / 8); i += kDenseThreads)
        reinterpret_cast<double*>(s_dw)[i] = reinterpret_cast<const double*>(A.dw + b0)[i];
    for (int i = tid; i < (kDenseThreads / 32) * kMaxW * 2; i += kDenseThreads) (&s_acc[0][0][0])[i] = 0.0;
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&s_bar)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // pair owned by this thread in the prepare step
    const int p_wi = tid / MBHL_NMODE, p_mi = tid - p_wi * MBHL_NMODE;
    const bool p_own = tid < nb * MBHL_NMODE;
    DenseMode p_m;
    p_m.k_lo = 1; p_m.k_hi = 0; p_m.ln_flo = 0.0; p_m.inv_dlog = 0.0;
    if (p_own && s_dw[p_wi].valid) p_m = s_dw[p_wi].mode[p_mi];
    if (p_m.k_hi >= p_m.k_lo) { atomicMin(&s_range[0], p_m.k_lo); atomicMax(&s_range[1], p_m.k_hi); }
    const double* const p_x = A.knots + ((int64_t)(b0 + p_wi) * MBHL_NMODE + p_mi) * A.S;
    const double* const p_coef = A.coef + ((int64_t)(b0 + p_wi) * MBHL_NMODE + p_mi) * (int64_t)(A.S - 1) * kCoefStride;
    int c_j = -1;                                                   // interval whose record is staged in s_rec[tid]
    double c_lo = 0.0, c_hi = 0.0;                                  // it serves f in [c_lo, c_hi)
    __syncthreads();
    const int c_first = max(group * A.G, s_range[0] / kChunk);
    const int c_last = min(min((group + 1) * A.G, A.n_chunks) - 1, s_range[1] >= 0 ? s_range[1] / kChunk : -1);

    const uint32_t bar = smem_u32(&s_bar);
    uint32_t parity = 0;
    for (int chunk = c_first; chunk <= c_last; ++chunk) {
        __syncthreads();                                            // every reader of the previous tile / records is done
        if (tid == 0) {
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(kTileBytes) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(smem_u32(s_tile)), "l"(A.tiles + (int64_t)chunk * kTileDoubles), "r"(kTileBytes), "r"(bar)
                         : "memory");
        }
        mbar_wait(bar, parity);
        parity ^= 1u;

        // ---- prepare: one thread per (walker, mode) pair ----
        const int kc0 = chunk * kChunk;
        if (p_own) {
            unsigned desc = 0;
            const int a = max(kc0, p_m.k_lo), b = min(kc0 + kChunk - 1, p_m.k_hi);
            if (a <= b) {
                const double fa = s_tile[a - kc0], fb = s_tile[b - kc0];
                bool uni = c_j >= 0 && fa >= c_lo && fb < c_hi;
                if (!uni) {
                    const int j = find_interval(p_x, A.S, fa, log(fa), p_m.ln_flo, p_m.inv_dlog);
                    const double xlo = __ldg(p_x + j), xhi = __ldg(p_x + j + 1);
                    if (fb < xhi || j == A.S - 2) {
                        uni = true;
                        c_j = j;
                        c_lo = (j == 0) ? -1.0 : xlo;
                        c_hi = (j == A.S - 2) ? 1e300 : xhi;
                        s_xj[tid] = xlo;
                        const double* src = p_coef + (int64_t)j * kCoefStride;
                        double* dst = s_rec + tid * kCoefStride;
#pragma unroll
                        for (int i = 0; i < kCoefStride; i += 2) cp_async16(dst + i, src + i);
                    } else {
                        c_j = -1;
                    }
                }
#pragma unroll
                for (int w4 = 0; w4 < kDenseThreads / 32; ++w4) {
                    const int t0 = kc0 + w4 * kWarpTile, t1 = t0 + kWarpTile - 1;
                    const unsigned kind = (t1 < a || t0 > b) ? 0u : ((uni && t0 >= a && t1 <= b) ? 1u : 2u);
                    desc |= kind << (2 * w4);
                }
            }
            s_desc[tid] = desc;
        }
        cp_async_wait_all();
        __syncthreads();

        // ---- evaluate: every warp loops over the walkers of the tile ----
        const int kt0 = kc0 + warp * kWarpTile;                     // first bin of this warp's 128
        const double* sf = s_tile + warp * kWarpTile;
        double f[kDenseR];
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) f[r] = sf[lane + 32 * r];

        for (int wi = 0; wi < nb; ++wi) {
            const unsigned kind = (lane < MBHL_NMODE) ? ((s_desc[wi * MBHL_NMODE + lane] >> (2 * warp)) & 3u) : 0u;
            unsigned m_fast = __ballot_sync(0xffffffffu, kind == 1u);
            unsigned m_gen = __ballot_sync(0xffffffffu, kind == 2u);
            if (!(m_fast | m_gen)) continue;
            const double t_coal = s_dw[wi].t_coal;

            double lin4[kDenseR], h[kDenseR][6];
#pragma unroll
            for (int r = 0; r < kDenseR; ++r) {
                lin4[r] = 4.0 * linear_cycles(f[r], t_coal);
#pragma unroll
                for (int i = 0; i < 6; ++i) h[r][i] = 0.0;
            }
            while (m_fast) {
                const int mi = __ffs(m_fast) - 1;
                m_fast &= m_fast - 1;
                const int p = wi * MBHL_NMODE + mi;
                mode_uniform(s_rec + p * kCoefStride, s_xj[p], f, lin4, h);
            }
            if (m_gen) {
                // general path: lanes 0..5 find, for mode `lane`, the in-band part of the warp tile and the
                // spline intervals of its two ends
                const DenseWalker& w = s_dw[wi];
                const double* xk = A.knots + ((int64_t)(b0 + wi) * MBHL_NMODE) * A.S;
                int ja = 0, jb = -1, full = 0;
                if (kind == 2u) {
                    const DenseMode m = w.mode[lane];
                    const int a = max(kt0, m.k_lo), b = min(kt0 + kWarpTile - 1, m.k_hi);
                    const double* x = xk + lane * A.S;
                    const double fa = sf[a - kt0], fb = sf[b - kt0];
                    ja = find_interval(x, A.S, fa, log(fa), m.ln_flo, m.inv_dlog);
                    jb = (fb < __ldg(x + ja + 1)) ? ja : find_interval(x, A.S, fb, log(fb), m.ln_flo, m.inv_dlog);
                    full = (a == kt0 && b == kt0 + kWarpTile - 1) ? 1 : 0;
                }
                while (m_gen) {
                    const int mi = __ffs(m_gen) - 1;
                    m_gen &= m_gen - 1;
                    const int ja_m = __shfl_sync(0xffffffffu, ja, mi), jb_m = __shfl_sync(0xffffffffu, jb, mi);
                    const int full_m = __shfl_sync(0xffffffffu, full, mi);
                    const double* x = xk + mi * A.S;
                    const double* cbase = A.coef + ((int64_t)(b0 + wi) * MBHL_NMODE + mi) * (int64_t)(A.S - 1) * kCoefStride;
                    if (ja_m == jb_m && full_m) {
                        mode_uniform(cbase + (int64_t)ja_m * kCoefStride, __ldg(x + ja_m), f, lin4, h);
                    } else {
                        const int k_lo = w.mode[mi].k_lo, k_hi = w.mode[mi].k_hi;
#pragma unroll
                        for (int r = 0; r < kDenseR; ++r) {
                            const int k = kt0 + lane + 32 * r;
                            if (k < k_lo || k > k_hi) continue;
                            int j = ja_m + ((jb_m - ja_m) * (lane + 32 * r)) / kWarpTile;
                            while (j > ja_m && f[r] < __ldg(x + j)) --j;
                            while (j < jb_m && f[r] >= __ldg(x + j + 1)) ++j;
                            mode_contrib(cbase + (int64_t)j * kCoefStride, f[r] - __ldg(x + j), lin4[r], 1.0, h[r]);
                        }
                    }
                }
            }
            // inner products of this walker over the warp's 128 bins
            double dh = 0.0, hh = 0.0;
#pragma unroll
            for (int r = 0; r < kDenseR; ++r) {
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    const double ww = sf[(1 + ch) * kChunk + lane + 32 * r];
                    const double wre = sf[(4 + 2 * ch) * kChunk + lane + 32 * r];
                    const double wim = sf[(5 + 2 * ch) * kChunk + lane + 32 * r];
                    dh = fma(wre, h[r][2 * ch], fma(wim, h[r][2 * ch + 1], dh));
                    hh = fma(ww, fma(h[r][2 * ch], h[r][2 * ch], h[r][2 * ch + 1] * h[r][2 * ch + 1]), hh);
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                dh += __shfl_down_sync(0xffffffffu, dh, o);
                hh += __shfl_down_sync(0xffffffffu, hh, o);
            }
            if (lane == 0) { s_acc[warp][wi][0] += dh; s_acc[warp][wi][1] += hh; }
        }
    }
    __syncthreads();
    if (tid < nb) {
        double sdh = 0.0, shh = 0.0;
#pragma unroll
        for (int i = 0; i < kDenseThreads / 32; ++i) { sdh += s_acc[i][tid][0]; shh += s_acc[i][tid][1]; }
        double* part = A.partials + ((int64_t)(b0 + tid) * A.n_groups + group) * 2;
        part[0] = sdh;
        part[1] = shh;
    }
}

}  // namespace mbhl
