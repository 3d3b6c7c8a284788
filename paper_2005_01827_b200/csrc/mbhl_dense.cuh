// mbhl_dense.cuh - steps a6 + a7: the fused dense kernel, version 4.
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
//      record with warp-uniform 16-byte shared-memory loads; a knot inside the warp tile is one pass in which
//      every bin reads the staged record of its side; a band edge is one gated pass; chunks with three or more
//      intervals (the lowest ~1e5 bins) go through the general path: the records and knots of up to 6
//      consecutive intervals of the warp tile are copied to a per-warp scratch, then looked up per bin;
//   4. per (walker, bin): <d|h> and <h|h> terms, warp shuffle tree, one shared-memory slot per (warp, walker).
// One partial per (walker, CTA) leaves the kernel; k_final_reduce adds them in fixed order (bitwise
// reproducible, no atomics on values).
//
// The loop body is bound by instruction issue (an FP64 instruction takes 2 cycles of a sub-partition, 3 with
// three fresh register operands, and every other instruction 1): per (bin, mode) 8 Horner cubics (24 DFMA), a quarter-turn
// sincos (14) and 3 complex multiply-adds (12).  The linear term -2 pi f t_coal of the phase (reading G9) costs nothing here:
// k_spline folds it into the phase record of every interval (exact reduction of x_j t_coal, slope minus
// t_coal), so the total phase of a bin in quarter turns is one cubic in u = f - x_j.
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
// kDenseR polynomial chains interleave.  Same reduction as sincos_qturn, with the shorter polynomial pair c_scd (sine of
// degree 4, cosine of degree 5 in y^2: errors 3.4e-12 / 5.6e-14) - every instruction of this loop costs FP64 issue time.
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
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], c_scd[4], c_scd[3]); pc[r] = fma(z[r], c_scd[10], c_scd[9]); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], ps[r], c_scd[2]); pc[r] = fma(z[r], pc[r], c_scd[8]); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], ps[r], c_scd[1]); pc[r] = fma(z[r], pc[r], c_scd[7]); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) { ps[r] = fma(z[r], ps[r], c_scd[0]); pc[r] = fma(z[r], pc[r], c_scd[6]); }
#pragma unroll
    for (int r = 0; r < kDenseR; ++r) pc[r] = fma(z[r], pc[r], c_scd[5]);
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
// kGated: the amplitude of bin r is multiplied by gate[r] (1 inside the segment served by `rec`, else 0).
template <bool kGated>
__device__ __forceinline__ void mode_uniform(const double* __restrict__ rec, double xj, const double (&f)[kDenseR],
                                             const double (&gate)[kDenseR],
                                             double (&h)[kDenseR][6]) {
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
        if (kGated) {
#pragma unroll
            for (int r = 0; r < kDenseR; ++r) amp[r] *= gate[r];
        }
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

// One mode's contribution when the kDenseR bins of a lane lie in different spline intervals whose records sit in
// shared memory: bin r reads its own record rec[r] at u[r] = f - x_j, amplitude gated by gate[r] (0 for bins out of
// band, whose rec[r] is any valid record).  Same lockstep arithmetic as mode_uniform.
__device__ __forceinline__ void mode_perbin(const double* const (&rec)[kDenseR], const double (&u)[kDenseR],
                                            const double (&gate)[kDenseR], double (&h)[kDenseR][6]) {
    double are[kDenseR], aim[kDenseR];
    {
        double p4[kDenseR], sn[kDenseR], cs[kDenseR], amp[kDenseR];
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) {
            const double2 p01 = *reinterpret_cast<const double2*>(rec[r] + 4);
            const double2 p23 = *reinterpret_cast<const double2*>(rec[r] + 6);
            p4[r] = fma(fma(fma(p23.y, u[r], p23.x), u[r], p01.y), u[r], p01.x);
        }
        sincos_qturn_x(p4, sn, cs);
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) {
            const double2 a01 = *reinterpret_cast<const double2*>(rec[r]);
            const double2 a23 = *reinterpret_cast<const double2*>(rec[r] + 2);
            amp[r] = fma(fma(fma(a23.y, u[r], a23.x), u[r], a01.y), u[r], a01.x) * gate[r];
        }
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) { are[r] = amp[r] * cs[r]; aim[r] = amp[r] * sn[r]; }
    }
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
        double tre[kDenseR], tim[kDenseR];
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) {
            const double2 r01 = *reinterpret_cast<const double2*>(rec[r] + 8 + 8 * ch);
            const double2 r23 = *reinterpret_cast<const double2*>(rec[r] + 10 + 8 * ch);
            const double2 i01 = *reinterpret_cast<const double2*>(rec[r] + 12 + 8 * ch);
            const double2 i23 = *reinterpret_cast<const double2*>(rec[r] + 14 + 8 * ch);
            tre[r] = fma(fma(fma(r23.y, u[r], r23.x), u[r], r01.y), u[r], r01.x);
            tim[r] = fma(fma(fma(i23.y, u[r], i23.x), u[r], i01.y), u[r], i01.x);
        }
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) {
            h[r][2 * ch] = fma(are[r], tre[r], fma(-aim[r], tim[r], h[r][2 * ch]));
            h[r][2 * ch + 1] = fma(are[r], tim[r], fma(aim[r], tre[r], h[r][2 * ch + 1]));
        }
    }
}

// What the prepare step found for one (walker, mode) pair in the current chunk; offsets are bins within the chunk.
struct PairDesc {
    short a, b;      // in-band bins [a, b]
    short ks;        // first bin of the second staged interval (b + 1 when the pair stays in one interval)
    short kind;      // 0: no in-band bin, 1: one or two staged records (slots 2p, 2p+1), 2: three or more intervals
};

constexpr int kRecSlots = 2 * kPairs;                                                       // two records per pair
// per-warp scratch of the general path: the records and knots of up to kGenSlots consecutive intervals
constexpr int kGenSlots = 6;
constexpr int kGenDoubles = kGenSlots * kCoefStride + 8;
constexpr int kDenseSmemBytes = (kTileDoubles + kRecSlots * kCoefStride + (kDenseThreads / 32) * kGenDoubles) * (int)sizeof(double);   // 40 KB tile + 24 KB records + 6.2 KB scratch

__device__ __forceinline__ void stage_record(double* dst, const double* __restrict__ src) {
#pragma unroll
    for (int i = 0; i < kCoefStride; i += 2) cp_async16(dst + i, src + i);
}

// Grid: 1-D, block id = group * n_tiles + tile (walker tiles vary fastest, so the CTAs resident at one time
// share a few chunk groups and the data tiles are served by L2).
__global__ void __launch_bounds__(kDenseThreads, MBHL_DENSE_MINB) k_dense(DenseArgs A) {
    extern __shared__ __align__(128) double s_dyn[];
    double* const s_tile = s_dyn;                                   // [10][512] staged data tile
    double* const s_rec = s_dyn + kTileDoubles;                     // [kRecSlots][32] staged coefficient records
    double* const s_gen = s_rec + kRecSlots * kCoefStride + (threadIdx.x >> 5) * kGenDoubles;   // this warp's general-path scratch
    __shared__ DenseWalker s_dw[kMaxW];
    __shared__ double s_xj[kRecSlots];                              // knot x_j of each staged record
    __shared__ PairDesc s_desc[kPairs];
    __shared__ unsigned s_cls[kPairs];                              // per pair: 8 class bits for each of the CTA's warp tiles (prepare step)
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
    if (p_own && s_dw[p_wi].valid && ((A.mode_mask >> p_mi) & 1u)) p_m = s_dw[p_wi].mode[p_mi];
    if (p_m.k_hi >= p_m.k_lo) { atomicMin(&s_range[0], p_m.k_lo); atomicMax(&s_range[1], p_m.k_hi); }
    const double* const p_x = A.knots + ((int64_t)(b0 + p_wi) * MBHL_NMODE + p_mi) * A.S;
    const double* const p_coef = A.coef + ((int64_t)(b0 + p_wi) * MBHL_NMODE + p_mi) * (int64_t)(A.S - 1) * kCoefStride;
    // staged intervals, kept in registers across chunks: slot 2p holds interval c_j, serving f in [c_lo, c_hi);
    // slot 2p+1 holds interval c_j + 1 when c_b is set, serving [c_hi, c_hi2)
    int c_j = -1;
    bool c_b = false;
    double c_lo = 0.0, c_hi = 0.0, c_hi2 = 0.0;
    __syncthreads();
    const int c_first = max(group * A.G, s_range[0] / kChunk);
    const int c_last = min(min((group + 1) * A.G, A.n_chunks) - 1, s_range[1] >= 0 ? s_range[1] / kChunk : -1);

    const uint32_t bar = smem_u32(&s_bar);
    uint32_t parity = 0;
    // executed-work tallies of this warp (warp-uniform; mbhl_last_dense_work): calls of the uniform / gated / per-bin-record
    // evaluators (each evaluates kDenseR bins on all 32 lanes), lane evaluations of the global per-bin path, epilogues
    unsigned n_uni = 0, n_gat = 0, n_rec = 0, n_lane = 0, n_epi = 0;
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
            PairDesc d;
            d.a = 0; d.b = -1; d.ks = 0; d.kind = 0;
            const int a = max(kc0, p_m.k_lo) - kc0, b = min(kc0 + kChunk - 1, p_m.k_hi) - kc0;
            if (a <= b) {
                const double fa = s_tile[a], fb = s_tile[b];
                if (!(c_j >= 0 && fa >= c_lo && fa < c_hi)) {
                    // the first in-band bin left the staged interval: usually into the next one
                    int j;
                    if (c_j >= 0 && fa >= c_hi && fa < c_hi2) j = c_j + 1;
                    else j = find_interval(p_x, A.S, fa, log(fa), p_m.ln_flo, p_m.inv_dlog);
                    c_j = j;
                    c_b = false;
                    const double xlo = __ldg(p_x + j);
                    c_lo = (j == 0) ? -1.0 : xlo;
                    c_hi = (j >= A.S - 2) ? 1e300 : __ldg(p_x + j + 1);
                    c_hi2 = (j >= A.S - 3) ? 1e300 : __ldg(p_x + j + 2);
                    s_xj[2 * tid] = xlo;
                    stage_record(s_rec + (2 * tid) * kCoefStride, p_coef + (int64_t)j * kCoefStride);
                }
                d.a = (short)a; d.b = (short)b;
                if (fb < c_hi) {
                    d.ks = (short)(b + 1);
                    d.kind = 1;
                } else if (fb < c_hi2) {
                    if (!c_b) {
                        c_b = true;
                        s_xj[2 * tid + 1] = c_hi;
                        stage_record(s_rec + (2 * tid + 1) * kCoefStride, p_coef + (int64_t)(c_j + 1) * kCoefStride);
                    }
                    // first bin with f >= c_hi: fa < c_hi <= fb, so it lies in (a, b]
                    int i = a + (int)ceil((c_hi - fa) * A.inv_df);
                    i = max(a + 1, min(b, i));
                    while (i > a + 1 && s_tile[i - 1] >= c_hi) --i;
                    while (i < b && s_tile[i] < c_hi) ++i;
                    d.ks = (short)i;
                    d.kind = 1;
                } else {
                    d.kind = 2;
                }
            }
            s_desc[tid] = d;
            // class of the pair in each warp tile: 1 = the whole tile lies in the segment served by slot 2p, 2 = by slot 2p + 1,
            // 4 = partly covered (knot or band edge inside the tile), 8 = three or more intervals in the chunk (general path)
            unsigned cw = 0;
#pragma unroll
            for (int w = 0; w < kDenseThreads / 32; ++w) {
                const int t0 = w * kWarpTile, t1 = t0 + kWarpTile - 1;
                unsigned c = 0;
                if (d.kind == 1) {
                    const int loA = max((int)d.a, t0), hiA = min((int)d.ks - 1, t1);
                    const int loB = max((int)d.ks, t0), hiB = min((int)d.b, t1);
                    if (loA == t0 && hiA == t1) c = 1u;
                    else if (loB == t0 && hiB == t1) c = 2u;
                    else if (loA <= hiA || loB <= hiB) c = 4u;
                } else if (d.kind == 2) {
                    if (max((int)d.a, t0) <= min((int)d.b, t1)) c = 8u;
                }
                cw |= c << (8 * w);
            }
            s_cls[tid] = cw;
        }
        cp_async_wait_all();
        __syncthreads();

        // ---- evaluate: every warp loops over the walkers of the tile ----
        const int t0 = warp * kWarpTile, t1 = t0 + kWarpTile - 1;   // this warp's bins, as offsets in the chunk
        const int kt0 = kc0 + t0;
        const double* sf = s_tile + t0;
        double f[kDenseR];
#pragma unroll
        for (int r = 0; r < kDenseR; ++r) f[r] = sf[lane + 32 * r];

        for (int wi = 0; wi < nb; ++wi) {
            // lanes 0..5 read the class of mode `lane` in this warp tile (set by the prepare step)
            unsigned cls = 0;
            if (lane < MBHL_NMODE) cls = (s_cls[wi * MBHL_NMODE + lane] >> (8 * warp)) & 0xffu;
            const bool gen = (cls & 8u) != 0;
            unsigned m_full = __ballot_sync(0xffffffffu, (cls & 3u) != 0);
            const unsigned m_selB = __ballot_sync(0xffffffffu, (cls & 2u) != 0);
            unsigned m_part = __ballot_sync(0xffffffffu, (cls & 4u) != 0);
            unsigned m_gen = __ballot_sync(0xffffffffu, gen);
            if (!(m_full | m_part | m_gen)) continue;

            double h[kDenseR][6];
#pragma unroll
            for (int r = 0; r < kDenseR; ++r) {
#pragma unroll
                for (int i = 0; i < 6; ++i) h[r][i] = 0.0;
            }
            while (m_full) {
                const int mi = __ffs(m_full) - 1;
                m_full &= m_full - 1;
                const int slot = 2 * (wi * MBHL_NMODE + mi) + ((m_selB >> mi) & 1u);
                mode_uniform<false>(s_rec + slot * kCoefStride, s_xj[slot], f, f, h);
                ++n_uni;
            }
            while (m_part) {
                                const int mi = __ffs(m_part) - 1;
                m_part &= m_part - 1;
                const PairDesc d = s_desc[wi * MBHL_NMODE + mi];
                const int lo0 = max((int)d.a, t0), hi0 = min((int)d.ks - 1, t1);     // segment served by slot 2p
                const int lo1 = max((int)d.ks, t0), hi1 = min((int)d.b, t1);         // segment served by slot 2p + 1
                const int slot0 = 2 * (wi * MBHL_NMODE + mi);
                if (lo0 <= hi0 && lo1 <= hi1) {
                    // a knot inside the warp tile: every bin reads the staged record of its own side, one pass
                    const double* rec[kDenseR];
                    double u[kDenseR], gate[kDenseR];
                    const double xa = s_xj[slot0], xb = s_xj[slot0 + 1];
#pragma unroll
                    for (int r = 0; r < kDenseR; ++r) {
                        const int o = t0 + lane + 32 * r;
                        const bool inB = o >= lo1;
                        rec[r] = s_rec + (slot0 + (inB ? 1 : 0)) * kCoefStride;
                        u[r] = f[r] - (inB ? xb : xa);
                        gate[r] = (o >= lo0 && o <= hi1) ? 1.0 : 0.0;
                    }
                    mode_perbin(rec, u, gate, h);
                    ++n_rec;
                } else {
                    // band edge: the one staged segment is evaluated on all bins with the amplitude gated
                    const int seg = (lo1 <= hi1) ? 1 : 0;
                    const int lo = seg ? lo1 : lo0, hi = seg ? hi1 : hi0;
                    double gate[kDenseR];
#pragma unroll
                    for (int r = 0; r < kDenseR; ++r) {
                        const int o = t0 + lane + 32 * r;
                        gate[r] = (o >= lo && o <= hi) ? 1.0 : 0.0;
                    }
                    mode_uniform<true>(s_rec + (slot0 + seg) * kCoefStride, s_xj[slot0 + seg], f, gate, h);
                    ++n_gat;
                }
            }
            if (m_gen) {
                // three or more intervals in the chunk (below ~2 mHz): lanes 0..5 find, for mode `lane`, the
                // in-band part of the warp tile and the spline intervals of its two ends
                const DenseWalker& w = s_dw[wi];
                const double* xk = A.knots + ((int64_t)(b0 + wi) * MBHL_NMODE) * A.S;
                int ja = 0, jb = -1, full = 0;
                if (gen) {
                    const DenseMode m = w.mode[lane];
                    const int a = max(kt0, m.k_lo), b = min(kt0 + kWarpTile - 1, m.k_hi);
                    const double* x = xk + lane * A.S;
                    const double fa = sf[a - kt0], fb = sf[b - kt0];
                    double xh;
                    ja = find_interval(x, A.S, fa, log(fa), m.ln_flo, m.inv_dlog, &xh);
                    jb = (fb < xh) ? ja : find_interval(x, A.S, fb, log(fb), m.ln_flo, m.inv_dlog);
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
                        mode_uniform<false>(cbase + (int64_t)ja_m * kCoefStride, __ldg(x + ja_m), f, f, h);
                        ++n_uni;
                    } else if (jb_m - ja_m < kGenSlots) {
                        // a few intervals in the warp tile: their records and knots are copied to this warp's scratch with
                        // independent loads (one L2 round trip), then every bin looks its interval up in shared memory
                        const int k_lo = w.mode[mi].k_lo, k_hi = w.mode[mi].k_hi;
                        const int nrec = jb_m - ja_m + 1;
                        __syncwarp();
                        for (int i = lane; i < nrec * (kCoefStride / 2); i += 32)
                            reinterpret_cast<double2*>(s_gen)[i] = __ldg(reinterpret_cast<const double2*>(cbase + (int64_t)ja_m * kCoefStride) + i);
                        double* const gx = s_gen + kGenSlots * kCoefStride;
                        if (lane <= nrec) gx[lane] = __ldg(x + ja_m + lane);
                        __syncwarp();
                        const double* rec[kDenseR];
                        double u[kDenseR], gate[kDenseR];
#pragma unroll
                        for (int r = 0; r < kDenseR; ++r) {
                            const int k = kt0 + lane + 32 * r;
                            int j = 0;                               // interval of the bin: how many of the staged knots lie at or below it
#pragma unroll
                            for (int i = 1; i < kGenSlots; ++i) j += (i < nrec && f[r] >= gx[i]) ? 1 : 0;
                            rec[r] = s_gen + j * kCoefStride;
                            u[r] = f[r] - gx[j];
                            gate[r] = (k >= k_lo && k <= k_hi) ? 1.0 : 0.0;
                        }
                        mode_perbin(rec, u, gate, h);
                        ++n_rec;
                    } else {
                        // every bin reads its own record from global memory.  Latency-bound, so the 4 bins of a lane advance in
                        // phases: the two knots around every bin's guess first (8 independent loads), then the records
                        const int k_lo = w.mode[mi].k_lo, k_hi = w.mode[mi].k_hi;
                        int jj[kDenseR];
                        bool in[kDenseR];
                        double xl[kDenseR], xh[kDenseR];
#pragma unroll
                        for (int r = 0; r < kDenseR; ++r) {
                            const int k = kt0 + lane + 32 * r;
                            in[r] = k >= k_lo && k <= k_hi;
                            n_lane += __popc(__ballot_sync(0xffffffffu, in[r]));
                            jj[r] = ja_m + ((jb_m - ja_m) * (lane + 32 * r)) / kWarpTile;
                            xl[r] = in[r] ? __ldg(x + jj[r]) : 0.0;
                            xh[r] = in[r] ? __ldg(x + jj[r] + 1) : 1e300;
                        }
#pragma unroll
                        for (int r = 0; r < kDenseR; ++r) {
                            if (!in[r]) continue;
                            while (jj[r] > ja_m && f[r] < xl[r]) { --jj[r]; xh[r] = xl[r]; xl[r] = __ldg(x + jj[r]); }
                            while (jj[r] < jb_m && f[r] >= xh[r]) { ++jj[r]; xl[r] = xh[r]; xh[r] = __ldg(x + jj[r] + 1); }
                        }
#pragma unroll
                        for (int r = 0; r < kDenseR; ++r)
                            if (in[r]) mode_contrib(cbase + (int64_t)jj[r] * kCoefStride, f[r] - xl[r], 1.0, h[r]);
                    }
                }
            }
            // inner products of this walker over the warp's 128 bins (one accumulator pair per bin: independent chains)
            double dhr[kDenseR], hhr[kDenseR];
#pragma unroll
            for (int r = 0; r < kDenseR; ++r) { dhr[r] = 0.0; hhr[r] = 0.0; }
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                double ww[kDenseR], wre[kDenseR], wim[kDenseR], n2[kDenseR];
#pragma unroll
                for (int r = 0; r < kDenseR; ++r) {
                    ww[r] = sf[(1 + ch) * kChunk + lane + 32 * r];
                    wre[r] = sf[(4 + 2 * ch) * kChunk + lane + 32 * r];
                    wim[r] = sf[(5 + 2 * ch) * kChunk + lane + 32 * r];
                }
#pragma unroll
                for (int r = 0; r < kDenseR; ++r) n2[r] = h[r][2 * ch] * h[r][2 * ch];
#pragma unroll
                for (int r = 0; r < kDenseR; ++r) dhr[r] = fma(wre[r], h[r][2 * ch], dhr[r]);
#pragma unroll
                for (int r = 0; r < kDenseR; ++r) n2[r] = fma(h[r][2 * ch + 1], h[r][2 * ch + 1], n2[r]);
#pragma unroll
                for (int r = 0; r < kDenseR; ++r) dhr[r] = fma(wim[r], h[r][2 * ch + 1], dhr[r]);
#pragma unroll
                for (int r = 0; r < kDenseR; ++r) hhr[r] = fma(ww[r], n2[r], hhr[r]);
            }
            double dh = 0.0, hh = 0.0;
#pragma unroll
            for (int r = 0; r < kDenseR; ++r) { dh += dhr[r]; hh += hhr[r]; }
            // lanes 0-15 collect <d|h>, lanes 16-31 collect <h|h>: one exchange, then a 4-step tree per half
            const bool upper = lane >= 16;
            double v = (upper ? hh : dh) + __shfl_xor_sync(0xffffffffu, upper ? dh : hh, 16);
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if ((lane & 15) == 0) s_acc[warp][wi][lane >> 4] += v;
            ++n_epi;
        }
    }
    if (A.work != nullptr && lane == 0) {
        if (n_uni) atomicAdd(A.work + 0, (unsigned long long)n_uni);
        if (n_gat) atomicAdd(A.work + 1, (unsigned long long)n_gat);
        if (n_rec) atomicAdd(A.work + 2, (unsigned long long)n_rec);
        if (n_lane) atomicAdd(A.work + 3, (unsigned long long)n_lane);
        if (n_epi) atomicAdd(A.work + 4, (unsigned long long)n_epi);
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
