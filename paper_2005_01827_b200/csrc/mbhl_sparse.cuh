// mbhl_sparse.cuh - steps a3 + a4 + a5 in ONE kernel: PhenomHM amplitude / phase / t(f) and the
// LISA response at the sparse knots (eqs. 5-10), then the not-a-knot cubic-spline coefficients of the
// Q = 8 smooth functions.  The knot values y never touch HBM.
//
// Decomposition.  A thread-block CLUSTER of two CTAs owns one (walker, mode).  CTA r of the pair
//   1. computes all S knots (cheap) and evaluates the smooth functions at ITS half of them, one thread per knot;
//      of the 8 values it keeps quantities 4r..4r+3 in its own shared memory and stores the other four into the
//      PEER's shared memory (distributed shared memory, a plain store through cluster.map_shared_rank);
//   2. after one cluster barrier holds the S values of its 4 quantities and solves their slope systems as before:
//      the matrix of a (walker, mode) is tridiagonal, strictly diagonally dominant and shared by the quantities.
//      Every recurrence of the Thomas algorithm is contractive here (factors 0.07 for the pivots, 0.27 for both
//      sweeps on log-spaced knots), so each is cut into blocks that start a few rows early ("halo"): the sweeps 32 rows
//      early from a zero state (the influence of the cut is below fp64 rounding by then), the pivots 3 rows early from the
//      fixed point of the recurrence on a geometric grid (the true pivots differ from it by the rounding of the knots
//      only); blocks that reach row 0 / S-1 use the true not-a-knot rows.
//        A. 1/h_r; pivots: thread t owns ceil(S/256) rows: c'_r = u_r / (d_r - a_r c'_{r-1}), 1 division per row
//        B. b_r = rhs_r / (d_r - a_r c'_{r-1}) for 4 quantities, all rows in parallel
//        C. forward sweep g_r = b_r - m_r g_{r-1}   (warp = quantity, lane = block of 32 rows addressed with compile-time
//           offsets when S is a multiple of 32 up to 1024; operands of 8 steps are loaded before the 8 dependent multiply-adds)
//        D. backward sweep s_r = g_r - c'_r s_{r+1}
//        E. c_j, d_j of every interval; each thread writes the 32 bytes of one (interval, quantity) with ONE 256-bit
//           store, a warp 8 full 128-byte lines.
// Two CTAs (of different clusters) share an SM, so one pair's evaluation (FP64 pipe) overlaps another's solve and
// stores (latency / HBM).  coef layout [walker][mode][interval][q][4] = (y_j, s_j, c_j, d_j); CTA r writes the half
// record of its 4 quantities.  Phase row (q = 1) as the dense kernel wants it: quarter turns, linear term folded in:
// 4 [(y_j mod 1) - frac(x_j t_coal)], 4 (s_j - t_coal), 4 c_j, 4 d_j, so that the total phase of a bin is ONE cubic in
// u = f - x_j (mbhl_sparse converts back to cycles on export; reading G9).
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>

namespace mbhl {

namespace cg = cooperative_groups;

__device__ __forceinline__ int pad_idx(int r) { return r + (r >> 5); }

constexpr int kSplineQ = 4;              // quantities per CTA
constexpr int kSplineThreads = 256;      // 8 warps: evaluation and row-parallel phases; 4 of them run the sweeps (one quantity each)
constexpr int kSplineHaloPivot = 16;
constexpr int kSplineHaloSweep = 32;
#ifndef MBHL_SWEEP_BLOCKS
#define MBHL_SWEEP_BLOCKS 32            // blocks of rows per quantity in the sweeps, one thread each (measured at config 3:
                                        // 64 blocks 16.9 ms, 32 blocks 16.0 ms, 16 blocks 16.9 ms, 8 blocks 19.2 ms)
#endif

// Row strides (in doubles) congruent to 4 mod 16: the last phase reads rows q = 0..3 at intervals j..j+3 from one
// half-warp, and 4 q + j then covers the 16 bank pairs once (a stride of S or S + S/32 + 1 gives 4-way conflicts).
__host__ __device__ inline int spline_stride(int n) { return n + ((4 - n % 16) + 16) % 16; }
__host__ __device__ inline int spline_sp(int S) { return spline_stride(S + (S >> 5) + 1); }

__host__ __device__ inline size_t spline_smem_bytes(int S) {
    return (size_t)(5 + kSplineQ) * spline_sp(S) * sizeof(double) + (size_t)kSplineQ * spline_stride(S) * sizeof(double);
}

// one 256-bit store (sm_100: st.global.v4.f64), 32-byte aligned
__device__ __forceinline__ void store_v4(double* p, double a, double b, double c, double d) {
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// y_out (may be null): the knot values [walker][mode][q][S] for mbhl_sparse's export, phase row in cycles.
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kSplineThreads, 2)
k_sparse_spline(const WalkerConst* __restrict__ wc, int S, double* __restrict__ knots, double* __restrict__ coef,
                double* __restrict__ y_out) {
    extern __shared__ double sm[];
    __shared__ WalkerConst s_c;
    __shared__ double s_cstar;
    const int SP = spline_sp(S), SY = spline_stride(S);
    double* xk = sm;                     // knots                                  [SP]
    double* ih = xk + SP;                // 1 / h_r, h_r = x_{r+1} - x_r          [SP]
    double* cps = ih + SP;               // pivots c'_r                            [SP]
    double* ivs = cps + SP;              // 1 / (d_r - a_r c'_{r-1})               [SP]
    double* mls = ivs + SP;              // a_r / (d_r - a_r c'_{r-1})             [SP]
    double* A1 = mls + SP;               // b, then g, then the slopes s (in place) [4][SP]
    double* Y = A1 + kSplineQ * SP;      // y values of this CTA's 4 quantities    [4][SY]
    cg::cluster_group cluster = cg::this_cluster();
    const int half = (int)cluster.block_rank();          // = blockIdx.x & 1
    const int64_t bm = blockIdx.x >> 1;                  // walker * 6 + mode
    const int64_t b = bm / MBHL_NMODE;
    const int mi = (int)(bm - b * MBHL_NMODE);
    const int tid = threadIdx.x;
    double* cout = coef + bm * (int64_t)(S - 1) * kCoefStride + half * (kSplineQ * 4);
    for (int i = tid; i < (int)(sizeof(WalkerConst) / 8); i += kSplineThreads)
        reinterpret_cast<double*>(&s_c)[i] = reinterpret_cast<const double*>(wc + b)[i];
    __syncthreads();
    const WalkerConst& c = s_c;
    const bool active = c.valid && c.mode[mi].active;
    if (!active) {                                       // both CTAs of the pair take this branch: no cluster barrier is skipped by one only
        for (int idx = tid; idx < (S - 1) * kSplineQ; idx += kSplineThreads)
            store_v4(cout + (int64_t)(idx >> 2) * kCoefStride + (idx & 3) * 4, 0.0, 0.0, 0.0, 0.0);
        if (half == 0)
            for (int i = tid; i < S; i += kSplineThreads) knots[bm * S + i] = 0.0;
        if (y_out != nullptr)
            for (int i = tid; i < kSplineQ * S; i += kSplineThreads) y_out[(bm * MBHL_NQ + half * kSplineQ) * S + i] = 0.0;
        return;
    }
    // The evaluation loop below stores into the PEER CTA's shared memory.  Distributed shared memory may only be touched once
    // the peer is known to have started: arrive here, wait just before the first remote store, with the knot set-up in between
    // to cover the latency.  (The `!active` return above is taken by both CTAs of a pair or by neither, so the pair always
    // agrees on whether this barrier exists.)
    cluster.barrier_arrive();
    const double t_coal = c.t_coal;
    // 1. knots (both CTAs, identical arithmetic), then the smooth functions at this CTA's half of them
    {
        const ModeConst& mc = c.mode[mi];
        for (int s = tid; s < S; s += kSplineThreads) {
            const double f = (s == 0) ? mc.f_lo : ((s == S - 1) ? mc.f_hi : mc.f_lo * exp(s * mc.dlog));
            xk[pad_idx(s)] = f;
            if (half == 0) knots[bm * S + s] = f;
        }
        if (tid == 0) {
            // fixed point of the pivot recurrence on an exactly geometric grid of ratio rho = exp(dlog): c = 1 / (2 (1 + rho) - rho c)
            const double rho = exp(mc.dlog), b = 1.0 + rho;
            s_cstar = (b - sqrt(b * b - rho)) / rho;
        }
        __syncthreads();
        const int S0 = (S + 1) >> 1;
        const int s_lo = half ? S0 : 0, s_hi = half ? S : S0;
        double* Ypeer = cluster.map_shared_rank(Y, half ^ 1);
        cluster.barrier_wait();                          // the peer CTA is running: its shared memory exists
        for (int s = s_lo + tid; s < s_hi; s += kSplineThreads) {
            double q[MBHL_NQ];
            smooth_quantities(c, mi, xk[pad_idx(s)], q);
#pragma unroll
            for (int i = 0; i < kSplineQ; ++i) {
                Y[i * SY + s] = half ? q[kSplineQ + i] : q[i];               // selects, not dynamic register indexing
                Ypeer[i * SY + s] = half ? q[i] : q[kSplineQ + i];
            }
            if (y_out != nullptr) {
#pragma unroll
                for (int i = 0; i < MBHL_NQ; ++i) y_out[(bm * MBHL_NQ + i) * S + s] = q[i];
            }
        }
    }
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
    // A. reciprocal spacings and pivots
    for (int r = tid; r < S - 1; r += kSplineThreads) ih[pad_idx(r)] = 1.0 / (xk[pad_idx(r + 1)] - xk[pad_idx(r)]);
    {
        const int m = (S + (int)kSplineThreads - 1) / (int)kSplineThreads;
        const int own0 = tid * m, own1 = min(S, own0 + m);
        if (own0 < own1) {
            // The recurrence contracts by 0.07 per row towards the fixed point of the geometric grid, from which the true pivots
            // differ by the rounding of the knots only (1e-13 relative): three rows from there are exact to fp64.  The first
            // rows, where the not-a-knot row 0 is still felt, run the chain from row 0.
            double cp = 0.0;
            int r = 0;
            if (own0 >= kSplineHaloPivot + 3) { r = own0 - 3; cp = s_cstar; }
            // three consecutive knots roll through registers: one shared-memory load per row
            double xa = (r > 0) ? xk[pad_idx(r - 1)] : 0.0, xb = xk[pad_idx(r)], xc = (r + 1 < S) ? xk[pad_idx(r + 1)] : 0.0;
            for (; r < own1; ++r) {
                double a, d, u;
                if (r == 0 || r == S - 1) {
                    mat(r, a, d, u);                                 // the not-a-knot rows
                } else {
                    const double hl = xb - xa, hr = xc - xb;
                    a = hr; d = 2.0 * (hl + hr); u = hl;
                }
                const double inv = 1.0 / (d - a * cp);
                cp = u * inv;
                if (r >= own0) { cps[pad_idx(r)] = cp; ivs[pad_idx(r)] = inv; mls[pad_idx(r)] = a * inv; }
                xa = xb; xb = xc; xc = (r + 2 < S) ? xk[pad_idx(r + 2)] : 0.0;
            }
        }
    }
    cluster.sync();                                      // both halves of every quantity have landed; no remote access after this
    // B. scaled right-hand sides of the slope system, all rows in parallel; a thread takes one row of all 4 quantities
    // (the spacings and the pivot factor of the row are read once, the 4 right-hand sides are independent chains)
    for (int r = tid; r < S; r += kSplineThreads) {
        const double piv = ivs[pad_idx(r)];
        if (r == 0 || r == S - 1) {
            const int r0 = (r == 0) ? 0 : S - 3;          // the three knots of the not-a-knot row
            const double h0 = xk[pad_idx(r0 + 1)] - xk[pad_idx(r0)], h1 = xk[pad_idx(r0 + 2)] - xk[pad_idx(r0 + 1)];
            const double i0 = ih[pad_idx(r0)], i1 = ih[pad_idx(r0 + 1)];
#pragma unroll
            for (int q = 0; q < kSplineQ; ++q) {
                const double* yq = Y + q * SY;
                const double d0 = (yq[r0 + 1] - yq[r0]) * i0, d1 = (yq[r0 + 2] - yq[r0 + 1]) * i1;
                const double v = (r == 0) ? ((3.0 * h0 + 2.0 * h1) * h1 * d0 + h0 * h0 * d1) / (h0 + h1)
                                          : (h1 * h1 * d0 + (2.0 * h0 + 3.0 * h1) * h0 * d1) / (h0 + h1);
                A1[q * SP + pad_idx(r)] = v * piv;
            }
        } else {
            const double hl = xk[pad_idx(r)] - xk[pad_idx(r - 1)], hr = xk[pad_idx(r + 1)] - xk[pad_idx(r)];
            const double wl = 3.0 * hr * ih[pad_idx(r - 1)] * piv, wr = 3.0 * hl * ih[pad_idx(r)] * piv;
#pragma unroll
            for (int q = 0; q < kSplineQ; ++q) {
                const double* yq = Y + q * SY;
                const double yr = yq[r];
                A1[q * SP + pad_idx(r)] = wl * (yr - yq[r - 1]) + wr * (yq[r + 1] - yr);
            }
        }
    }
    __syncthreads();
    // C, D. sweeps in place.  A thread owns a block of consecutive rows and first copies the halo rows it needs from its
    // neighbour's block into registers, so the neighbour may overwrite them afterwards.  The recurrences are latency chains:
    // the shared-memory operands of 8 steps are loaded first (independent loads), then the 8 dependent multiply-adds run back
    // to back.
    if ((S & 31) == 0 && S <= 1024) {
        // The usual case (S = 256, 512, 1024): blocks of exactly 32 rows, warp = quantity, lane = block.  Row 32 blk + k sits
        // at padded index 33 blk + k, so a block and its neighbours are addressed with compile-time offsets from one base
        // and nothing is bounds-checked: this phase was a fifth of the kernel's instructions, none of them FP64.
        const int nblk = S >> 5;
        const int q = tid >> 5, blk = tid & 31;
        const bool on = q < kSplineQ && blk < nblk;
        double* const aq = A1 + min(q, kSplineQ - 1) * SP + min(blk, nblk - 1) * 33;
        const double* const mq = mls + min(blk, nblk - 1) * 33;
        const double* const cq = cps + min(blk, nblk - 1) * 33;
        const bool has_prev = on && blk > 0, has_next = on && blk + 1 < nblk;
        double halo[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) halo[k] = has_prev ? aq[k - 33] : 0.0;
        __syncthreads();
        if (on) {
            double g = 0.0;
            if (has_prev) {
#pragma unroll
                for (int i0 = 0; i0 < 32; i0 += 8) {
                    double mm[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) mm[k] = mq[i0 + k - 33];
#pragma unroll
                    for (int k = 0; k < 8; ++k) g = fma(-mm[k], g, halo[i0 + k]);
                }
            }
#pragma unroll
            for (int r0 = 0; r0 < 32; r0 += 8) {
                double mm[8], bb[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) { mm[k] = mq[r0 + k]; bb[k] = aq[r0 + k]; }
#pragma unroll
                for (int k = 0; k < 8; ++k) { g = fma(-mm[k], g, bb[k]); aq[r0 + k] = g; }
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 32; ++k) halo[k] = has_next ? aq[k + 33] : 0.0;
        __syncthreads();
        if (on) {
            double sl = 0.0;
            if (has_next) {
#pragma unroll
                for (int i0 = 24; i0 >= 0; i0 -= 8) {
                    double cc[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) cc[k] = cq[i0 + k + 33];
#pragma unroll
                    for (int k = 7; k >= 0; --k) sl = fma(-cc[k], sl, halo[i0 + k]);
                }
            }
#pragma unroll
            for (int r0 = 31; r0 >= 0; r0 -= 8) {
                double cc[8], gg[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) { cc[k] = cq[r0 - k]; gg[k] = aq[r0 - k]; }
#pragma unroll
                for (int k = 0; k < 8; ++k) { sl = fma(-cc[k], sl, gg[k]); aq[r0 - k] = sl; }
            }
        }
    } else {
        // any other S: MBHL_SWEEP_BLOCKS blocks of ceil(S / MBHL_SWEEP_BLOCKS) rows per quantity, rows outside the matrix enter
        // with coefficient 0
        // MBHL_SWEEP_BLOCKS blocks of rows per quantity: fewer blocks mean fewer redundant halo rows (instructions), more
        // blocks a shorter dependent chain
        constexpr int NB = MBHL_SWEEP_BLOCKS;
        const int q = tid / NB, blk = tid % NB;
        const int m = (S + NB - 1) / NB;
        const int own0 = (tid < kSplineQ * NB) ? min(S, blk * m) : S, own1 = min(S, own0 + m);
        double* aq = A1 + min(q, kSplineQ - 1) * SP;
        double halo[kSplineHaloSweep];
#pragma unroll
        for (int i = 0; i < kSplineHaloSweep; ++i) {
            const int r = own0 - kSplineHaloSweep + i;
            halo[i] = (r >= 0 && r < S) ? aq[pad_idx(r)] : 0.0;
        }
        __syncthreads();
        {
            double g = 0.0;
#pragma unroll
            for (int i0 = 0; i0 < kSplineHaloSweep; i0 += 8) {
                double mm[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int r = own0 - kSplineHaloSweep + i0 + k;
                    mm[k] = (r >= 0 && r < S) ? mls[pad_idx(r)] : 0.0;
                }
#pragma unroll
                for (int k = 0; k < 8; ++k) g = fma(-mm[k], g, halo[i0 + k]);
            }
            for (int r0 = own0; r0 < own1; r0 += 8) {
                double mm[8], bb[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int r = min(r0 + k, own1 - 1);     // stay inside this thread's own rows: the rows past own1 are a
                    mm[k] = mls[pad_idx(r)];                 // neighbour's, who may be writing them (the values were never used)
                    bb[k] = aq[pad_idx(r)];
                }
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    g = fma(-mm[k], g, bb[k]);
                    if (r0 + k < own1) aq[pad_idx(r0 + k)] = g;
                }
            }
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < kSplineHaloSweep; ++i) {
            const int r = own1 + i;
            halo[i] = (r < S) ? aq[pad_idx(r)] : 0.0;
        }
        __syncthreads();
        {
            double sl = 0.0;
#pragma unroll
            for (int i0 = kSplineHaloSweep - 8; i0 >= 0; i0 -= 8) {
                double cc[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int r = own1 + i0 + k;
                    cc[k] = (r < S) ? cps[pad_idx(r)] : 0.0;
                }
#pragma unroll
                for (int k = 7; k >= 0; --k) sl = fma(-cc[k], sl, halo[i0 + k]);
            }
            for (int r0 = own1 - 1; r0 >= own0; r0 -= 8) {
                double cc[8], gg[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int r = max(r0 - k, own0);         // likewise: never read below this thread's first row
                    cc[k] = cps[pad_idx(r)];
                    gg[k] = aq[pad_idx(r)];
                }
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    sl = fma(-cc[k], sl, gg[k]);
                    if (r0 - k >= own0) aq[pad_idx(r0 - k)] = sl;
                }
            }
        }
    }
    __syncthreads();
    // E. coefficients: one (interval, quantity) per thread, one 256-bit store each; 4 consecutive threads write a 128-byte
    // half record, a warp 8 full lines (a thread per interval writing its whole half record touches 32 lines per store
    // instruction and was measured slower)
    for (int idx = tid; idx < (S - 1) * kSplineQ; idx += kSplineThreads) {
        const int j = idx >> 2, q = idx & 3;
        const double hinv = ih[pad_idx(j)];
        double y0 = Y[q * SY + j];
        const double y1 = Y[q * SY + j + 1];
        const double s0 = A1[q * SP + pad_idx(j)], s1 = A1[q * SP + pad_idx(j + 1)];
        const double dl = (y1 - y0) * hinv;
        const double cc = (3.0 * dl - 2.0 * s0 - s1) * hinv;
        const double dd = (s0 + s1 - 2.0 * dl) * (hinv * hinv);
        double s0w = s0, ccw = cc, ddw = dd;
        if (half == 0 && q == 1) {
            // phase row: quarter turns, with the linear term -f t_coal of the total phase (reading G9) folded in.
            // f t_coal = x_j t_coal + u t_coal: the first product is reduced mod 1 exactly, the second joins the slope.
            y0 = 4.0 * ((y0 - rint(y0)) - linear_cycles(xk[pad_idx(j)], t_coal));
            s0w = 4.0 * (s0 - t_coal);
            ccw = 4.0 * cc;
            ddw = 4.0 * dd;
        }
        store_v4(cout + (int64_t)j * kCoefStride + q * 4, y0, s0w, ccw, ddw);
    }
}

}  // namespace mbhl
