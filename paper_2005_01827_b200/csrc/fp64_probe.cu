// fp64_probe.cu - MEASUREMENT AID (not part of the method, not linked into libmbhl.so): how fast one SM sub-partition of
// the B200 issues FP64 instructions as a function of where their source operands come from.
// uses the table this prints (profiles/r02_fp64_operand_probe.txt) to bound the fused dense kernel's inner loop.
//
//   build: python -m paper_2005_01827_b200.build --probe      run: paper_2005_01827_b200/fp64_probe
//
// Part 1 (operand sources), part 2 (what an instruction of another pipe between two DFMAs costs, and multiply-add chains
// that share operands) and part 3 (the fast-path body of k_dense, mode_uniform of mbhl_dense.cuh, alone on every SM at the
// kernel's own occupancy).
// One CTA on one SM; every warp runs `iters` passes over CH independent dependency chains; the cycle count comes from
// clock64 around the loop, so the figure is cycles per warp-level instruction per sub-partition (4 per SM).
#include <cstdio>
#include <cuda_runtime.h>
#include "mbhl.h"
#include "mbhl_kernels.cuh"   // for part 3: the fast-path body of k_dense (mode_uniform) timed in isolation

enum Mode {
    kConst2 = 0,     // x = fma(x, m, e)        m, e loop constants (kept in registers, reused by every instruction)
    kReg2 = 1,       // x = fma(x, y, e)        two per-chain registers + one constant
    kReg3 = 2,       // x = fma(x, y, z)        three per-chain registers
    kAcc3 = 3,       // x = fma(y, z, x)        three per-chain registers, accumulator form (the complex multiply-adds of k_dense)
    kShared2of3 = 4, // x = fma(x, y0, z1)      one per-chain register, two registers shared by consecutive instructions
    kHorner = 5,     // p = fma(p, u, c_k)      per-chain p and u, coefficient c_k shared by the CH chains (Horner step of k_dense)
    kMacPair = 6,    // hr = fma(a, tr, hr); hi = fma(a, ti, hi)   a shared by the pair (ordering the multiply-adds for reuse)
    kDmma = 7,       // mma.sync.m8n8k4.f64 alone (FLOPs per cycle reported as DFMA-equivalents)
    kDmmaDfma = 8,   // mma.sync.m8n8k4.f64 interleaved 1:1 with independent DFMA chains
    kAdd2 = 9,       // x = x + y               DADD, two per-chain registers
    kNumModes = 10
};

template <int MODE, int CH>
__global__ void k_probe(long iters, const double* __restrict__ in, double* sink, long long* cyc) {
    double x[CH], y[CH], z[CH], w[CH];
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        x[i] = in[threadIdx.x % 32 + 32 * i]; y[i] = in[1024 + threadIdx.x % 32 + 32 * i];
        z[i] = in[2048 + threadIdx.x % 32 + 32 * i]; w[i] = in[3072 + threadIdx.x % 32 + 32 * i];
    }
    const double m = 0.999999, e = 1e-6;
    double c0 = in[7], c1 = in[8], c2 = in[9];
    double acc0 = 0.0, acc1 = 0.0;           // DMMA accumulators
    __syncthreads();
    const long long t0 = clock64();
    for (long it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            if (MODE == kConst2) x[i] = fma(x[i], m, e);
            if (MODE == kReg2) x[i] = fma(x[i], y[i], e);
            if (MODE == kReg3) x[i] = fma(x[i], y[i], z[i]);
            if (MODE == kAcc3) x[i] = fma(y[i], z[i], x[i]);
            if (MODE == kShared2of3) x[i] = fma(x[i], y[0], z[1]);
            if (MODE == kAdd2) x[i] = x[i] + y[i];
        }
        if (MODE == kHorner) {
#pragma unroll
            for (int i = 0; i < CH; ++i) x[i] = fma(x[i], y[i], c0);
#pragma unroll
            for (int i = 0; i < CH; ++i) x[i] = fma(x[i], y[i], c1);
#pragma unroll
            for (int i = 0; i < CH; ++i) x[i] = fma(x[i], y[i], c2);
        }
        if (MODE == kMacPair) {
#pragma unroll
            for (int i = 0; i < CH; ++i) { x[i] = fma(y[i], z[i], x[i]); w[i] = fma(y[i], z[(i + 1) % CH], w[i]); }
        }
        if (MODE == kDmma || MODE == kDmmaDfma) {
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                             : "+d"(acc0), "+d"(acc1) : "d"(y[i]), "d"(z[i]));
                if (MODE == kDmmaDfma) x[i] = fma(x[i], m, e);
            }
        }
    }
    const long long t1 = clock64();
    double s = acc0 + acc1 + c0;
#pragma unroll
    for (int i = 0; i < CH; ++i) s += x[i] + w[i];
    if (s == 12345.678) sink[0] = s;
    if ((threadIdx.x & 31) == 0) cyc[threadIdx.x >> 5] = t1 - t0;
}

static const char* kNames[kNumModes] = {
    "DFMA x = fma(x, m, e)       1 fresh register operand, 2 loop constants",
    "DFMA x = fma(x, y, e)       2 fresh register operands, 1 loop constant",
    "DFMA x = fma(x, y, z)       3 fresh register operands",
    "DFMA x = fma(y, z, x)       3 fresh register operands, accumulator form",
    "DFMA x = fma(x, y0, z1)     1 fresh, 2 shared by consecutive instructions",
    "DFMA p = fma(p, u, c_k)     Horner step: p, u per chain, coefficient shared by the 8 chains",
    "DFMA multiply-add pair      hr += a tr; hi += a ti (a shared by the pair)",
    "DMMA m8n8k4 alone           (256 FMA per warp instruction)",
    "DMMA m8n8k4 + DFMA 1:1      interleaved, independent chains",
    "DADD x = x + y              2 fresh register operands",
};

template <int MODE, int CH>
static void run(int warps, const double* in) {
    double* sink; long long* cyc;
    cudaMalloc(&sink, 64); cudaMalloc(&cyc, 8 * 64);
    const long iters = 40000;
    for (int rep = 0; rep < 2; ++rep) { k_probe<MODE, CH><<<1, warps * 32>>>(iters, in, sink, cyc); cudaDeviceSynchronize(); }
    long long h[64];
    cudaMemcpy(h, cyc, 8 * warps, cudaMemcpyDeviceToHost);
    long long mx = 0;
    for (int i = 0; i < warps; ++i) if (h[i] > mx) mx = h[i];
    int per_iter = CH;                                   // FP64-pipe warp instructions per pass
    if (MODE == kHorner) per_iter = 3 * CH;
    if (MODE == kMacPair || MODE == kDmmaDfma) per_iter = 2 * CH;
    const double per = (double)mx / ((double)iters * per_iter * (warps / 4.0));
    printf("  %-82s %2d warps/SM: %.3f cycles per warp instruction per sub-partition\n", kNames[MODE], warps, per);
    if (MODE == kDmma || MODE == kDmmaDfma) {
        // FMA lanes per cycle per SM: a DMMA is 8x8x4 = 256 FMA, a DFMA 32
        const double fma_per_pass = (MODE == kDmma ? 256.0 : 288.0) * CH * warps;
        printf("  %-82s              -> %.1f FMA per cycle per SM (64 = the DFMA rate)\n", "", fma_per_pass * iters / (double)mx);
    }
    cudaFree(sink); cudaFree(cyc);
}

// ---- part 2: instruction mix.  12 warps on one SM; every pass issues 8 DFMAs (2 fresh registers + 1 constant: 2.0 cycles
// each when alone) and, per DFMA, the extra instructions of the mode.  The figure is cycles per DFMA per sub-partition.
enum Mix { kMixNone = 0, kMixImad = 1, kMixLop3 = 2, kMixFfma = 3, kMix3 = 4, kMac4Shared = 5, kMac4Distinct = 6, kNumMix = 7 };

template <int MODE>
__global__ void __launch_bounds__(384, 1) k_mix(long iters, const double* __restrict__ in, double* sink, long long* cyc) {
    double x[8], y[8];
    unsigned a[8], b[8];
    float fa[8], fb[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        x[i] = in[threadIdx.x % 32 + 32 * i]; y[i] = in[1024 + threadIdx.x % 32 + 32 * i];
        a[i] = threadIdx.x * 7 + i; b[i] = threadIdx.x * 13 + i * 5; fa[i] = a[i]; fb[i] = b[i];
    }
    const double e = 1e-6;
    const unsigned pred = threadIdx.x & 1;
    __syncthreads();
    const long long t0 = clock64();
    for (long it = 0; it < iters; ++it) {
        if (MODE == kMac4Shared) {       // the 4 multiply-adds of a complex product on ONE bin: consecutive instructions share an operand
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                x[0] = fma(y[0], y[2], x[0]); x[1] = fma(y[0], y[3], x[1]); x[0] = fma(-y[1], y[3], x[0]); x[1] = fma(y[1], y[2], x[1]);
            }
        } else if (MODE == kMac4Distinct) {   // same dependency structure, no operand shared with the previous instruction
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                x[0] = fma(y[0], y[2], x[0]); x[1] = fma(y[1], y[3], x[1]); x[0] = fma(-y[4], y[5], x[0]); x[1] = fma(y[6], y[7], x[1]);
            }
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                x[i] = fma(x[i], y[i], e);
                if (MODE == kMixImad) a[i] = a[i] * 3 + b[i];
                if (MODE == kMixLop3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(b[i]), "r"(pred));
                if (MODE == kMixFfma) fa[i] = fmaf(fa[i], fb[i], 1.0f);
                if (MODE == kMix3) { fa[i] = fmaf(fa[i], fb[i], 1.0f); fb[i] = fmaf(fb[i], 0.5f, fa[i]); a[i] = a[i] * 3 + b[i]; }
            }
        }
    }
    const long long t1 = clock64();
    double r = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) r += x[i] + a[i] + b[i] + fa[i] + fb[i];
    if (r == 12345.678) sink[0] = r;
    if ((threadIdx.x & 31) == 0) cyc[threadIdx.x >> 5] = t1 - t0;
}

static const char* kMixNames[kNumMix] = {
    "DFMA alone (x = fma(x, y, e))",
    "DFMA + 1 IMAD (2 register reads)",
    "DFMA + 1 LOP3 (3 register reads)",
    "DFMA + 1 FFMA (2 register reads)",
    "DFMA + 2 FFMA + 1 IMAD",
    "complex multiply-add, 4-chain on one bin, every instruction shares an operand with the previous one",
    "complex multiply-add, 4-chain on one bin, no shared operand",
};

template <int MODE>
static void run_mix(const double* in) {
    double* sink; long long* cyc;
    cudaMalloc(&sink, 64); cudaMalloc(&cyc, 8 * 64);
    const long iters = 20000;
    for (int rep = 0; rep < 2; ++rep) { k_mix<MODE><<<1, 384>>>(iters, in, sink, cyc); cudaDeviceSynchronize(); }
    long long h[12]; cudaMemcpy(h, cyc, 8 * 12, cudaMemcpyDeviceToHost);
    long long mx = 0; for (int i = 0; i < 12; ++i) if (h[i] > mx) mx = h[i];
    const int dfma_per_pass = (MODE == kMac4Shared || MODE == kMac4Distinct) ? 32 : 8;
    printf("  %-100s %.3f cycles per DFMA per sub-partition\n", kMixNames[MODE], (double)mx / ((double)iters * dfma_per_pass * 3));
    cudaFree(sink); cudaFree(cyc);
}

// ---- part 3: the fast-path body of k_dense (one mode at the 4 bins of every lane, record in shared memory) alone on the
// whole GPU at the kernel's occupancy (3 CTAs x 4 warps per SM).  220 FP64 warp instructions per call (u = f - x_j is loop
// invariant here); 440 cycles per call per sub-partition would be the FP64 pipe's own limit.
__global__ void __launch_bounds__(128, 3) k_body(int iters, const double* __restrict__ in, double* out, long long* cyc) {
    extern __shared__ __align__(128) double s_dyn[];
    double* s_rec = s_dyn;     // 96 records
    for (int i = threadIdx.x; i < 96 * mbhl::kCoefStride; i += 128) s_rec[i] = in[i % 4096] * 1e-3;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    double f[mbhl::kDenseR], h[mbhl::kDenseR][6];
#pragma unroll
    for (int r = 0; r < mbhl::kDenseR; ++r) {
        f[r] = 1e-3 + 1e-6 * (lane + 32 * r);
#pragma unroll
        for (int i = 0; i < 6; ++i) h[r][i] = 0.0;
    }
    const long long t0 = clock64();
    int slot = threadIdx.x >> 5;
    for (int it = 0; it < iters; ++it)
        for (int m = 0; m < 6; ++m) {
            slot = (slot + 7) % 96;
            mbhl::mode_uniform<false>(s_rec + slot * mbhl::kCoefStride, 1e-3, f, f, h);
        }
    const long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int r = 0; r < mbhl::kDenseR; ++r)
#pragma unroll
        for (int i = 0; i < 6; ++i) s += h[r][i];
    out[blockIdx.x * 128 + threadIdx.x] = s;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

static void run_body(const double* in, int sms) {
    const int nb = sms * 3, iters = 20000, smem = 72 * 1024;
    double* out; long long* cyc;
    cudaMalloc(&out, 8 * nb * 128); cudaMalloc(&cyc, 8 * nb);
    cudaFuncSetAttribute(k_body, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    long long mx = 0;
    for (int rep = 0; rep < 2; ++rep) {
        k_body<<<nb, 128, smem>>>(iters, in, out, cyc);
        cudaDeviceSynchronize();
        long long* hc = new long long[nb];
        cudaMemcpy(hc, cyc, 8 * nb, cudaMemcpyDeviceToHost);
        mx = 0;
        for (int i = 0; i < nb; ++i) if (hc[i] > mx) mx = hc[i];
        delete[] hc;
    }
    printf("  mode_uniform<false> alone, 3 CTAs x 4 warps per SM: %.1f cycles per call per sub-partition (%s)\n",
           (double)mx / (3.0 * iters * 6), cudaGetErrorString(cudaGetLastError()));
    cudaFree(out); cudaFree(cyc);
}

int main() {
    cudaDeviceProp p;
    cudaGetDeviceProperties(&p, 0);
    printf("fp64_probe on %s (%d SMs), one CTA on one SM, 8 independent chains per thread\n", p.name, p.multiProcessorCount);
    double* in;
    cudaMalloc(&in, 8 * 4096);
    static double h[4096];
    for (int i = 0; i < 4096; ++i) h[i] = 0.9999 + 1e-7 * (i % 97);
    cudaMemcpy(in, h, sizeof(h), cudaMemcpyHostToDevice);
    for (int w : {4, 12}) {
        run<kConst2, 8>(w, in); run<kReg2, 8>(w, in); run<kReg3, 8>(w, in); run<kAcc3, 8>(w, in); run<kShared2of3, 8>(w, in);
        run<kHorner, 8>(w, in); run<kMacPair, 8>(w, in); run<kAdd2, 8>(w, in); run<kDmma, 8>(w, in); run<kDmmaDfma, 8>(w, in);
        printf("\n");
    }
    printf("part 2: instruction mix, 12 warps on one SM\n");
    run_mix<kMixNone>(in); run_mix<kMixImad>(in); run_mix<kMixLop3>(in); run_mix<kMixFfma>(in); run_mix<kMix3>(in);
    run_mix<kMac4Shared>(in); run_mix<kMac4Distinct>(in);
    printf("\npart 3: the fast-path body of k_dense in isolation\n");
    run_body(in, p.multiProcessorCount);
    return 0;
}
