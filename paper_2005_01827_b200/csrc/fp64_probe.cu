// fp64_probe.cu - MEASUREMENT AID (not part of the method, not linked into libmbhl.so): how fast one SM sub-partition of
// the B200 issues FP64 instructions as a function of where their source operands come from.
// uses the table this prints (profiles/r02_fp64_operand_probe.txt) to bound the fused dense kernel's inner loop.
//
//   build: python -m paper_2005_01827_b200.build --probe      run: paper_2005_01827_b200/fp64_probe
//
// One CTA on one SM; every warp runs `iters` passes over CH independent dependency chains; the cycle count comes from
// clock64 around the loop, so the figure is cycles per warp-level instruction per sub-partition (4 per SM).
#include <cstdio>
#include <cuda_runtime.h>

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
    return 0;
}
