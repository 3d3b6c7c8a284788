// mbhl_sampler.cuh - sampler-side steps next to the likelihood (section II.B).
//
//   unpack_sampled     sampler coordinates (Table I :67-81) -> physical parameters;
//                      a walker outside the prior box becomes a NaN row, which the hot path maps to logL = -inf
//   lisa_to_ssb        LISA-frame (lambda, beta, psi, t) -> SSB (reading G20)
//                      (both run inside k_walker_consts, in registers: no separate kernel)
//   k_pt_propose       stretch move, eqs. 14-15, a = 1.15 (:222): one thread per moving walker
//   k_pt_accept        eq. 16 on the tempered density prior x L^beta (:211)
//   k_pt_swap          eq. 17: swaps between adjacent temperatures, hottest pair first
// Random numbers come from Philox4x32-10 (Salmon et al. 2011) keyed by the seed and counted by (walker, step,
// stream), so a run is reproducible and independent of the launch shape.  Written from the paper and the
// generator's published definition; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mbhl {

// Table I; filled by mbhl_init from the host's log() of the printed bounds
__constant__ double c_prior_lo[MBHL_NPARAM];
__constant__ double c_prior_hi[MBHL_NPARAM];

__device__ __forceinline__ bool in_prior_box(const double* th) {
    bool ok = true;
#pragma unroll
    for (int i = 0; i < MBHL_NPARAM; ++i) ok = ok && isfinite(th[i]) && th[i] >= c_prior_lo[i] && th[i] <= c_prior_hi[i];
    return ok;
}

// theta = (ln M_T, q, a1, a2, ln D_L, phi_ref, cos iota, lambda, sin beta, psi, ln t_ref)
__device__ __forceinline__ void unpack_sampled(const double* th, double* p) {
    if (!in_prior_box(th)) {
#pragma unroll
        for (int i = 0; i < MBHL_NPARAM; ++i) p[i] = NAN;
        return;
    }
    p[0] = exp(th[0]); p[1] = th[1]; p[2] = th[2]; p[3] = th[3]; p[4] = exp(th[4]); p[5] = th[5];
    p[6] = acos(th[6]); p[7] = th[7]; p[8] = asin(th[8]); p[9] = th[9]; p[10] = exp(th[10]);
}

// LISA-frame coordinates -> SSB (reading G20).  The frame is that of the constellation at the
// orbital phase alpha = Omega_0 (t0 + t_L): R = R_z(alpha) R_y(-pi/3) R_z(-alpha), written out entry by entry (the three
// spacecraft are at rest in it).  Sky direction and polarisation basis rotate as vectors; t_L is the arrival time of the
// wavefront at the constellation centre: t_ref = t_L - k.p_0/c = t_L + n.p_0/c.  lambda wraps mod 2 pi, psi mod pi.
__device__ __forceinline__ void lisa_to_ssb(double t0, double& t, double& lam, double& beta, double& psi) {
    double sa, ca;
    sincos(kOmega0 * (t0 + t), &sa, &ca);
    const double ct = 0.5, st = -0.86602540378443864676;        // cos, sin of the tilt -pi/3
    const double R00 = ct * ca * ca + sa * sa, R01 = ca * sa * (ct - 1.0), R02 = ca * st;
    const double R10 = R01, R11 = ct * sa * sa + ca * ca, R12 = sa * st;
    const double R20 = -st * ca, R21 = -st * sa, R22 = ct;
    double sl, cl, sb, cb;
    sincos(lam, &sl, &cl);
    sincos(beta, &sb, &cb);
    const double nL[3] = {cb * cl, cb * sl, sb}, uL[3] = {sl, -cl, 0.0};
    const double n0 = R00 * nL[0] + R01 * nL[1] + R02 * nL[2];
    const double n1 = R10 * nL[0] + R11 * nL[1] + R12 * nL[2];
    const double n2 = R20 * nL[0] + R21 * nL[1] + R22 * nL[2];
    const double u0 = R00 * uL[0] + R01 * uL[1], u1 = R10 * uL[0] + R11 * uL[1], u2 = R20 * uL[0] + R21 * uL[1];
    const double beta_s = asin(fmax(-1.0, fmin(1.0, n2)));
    double lam_s = atan2(n1, n0);
    if (lam_s < 0.0) lam_s += kTwoPi;
    if (lam_s >= kTwoPi) lam_s -= kTwoPi;
    double sls, cls, sbs, cbs;
    sincos(lam_s, &sls, &cls);
    sincos(beta_s, &sbs, &cbs);
    // SSB polarisation basis at (lam_s, beta_s): u = (sin, -cos, 0), v = (-sin b cos l, -sin b sin l, cos b)
    const double uu = u0 * sls - u1 * cls;
    const double uv = -u0 * sbs * cls - u1 * sbs * sls + u2 * cbs;
    double ps = psi + atan2(uv, uu);
    ps -= floor(ps / kPi) * kPi;
    if (ps >= kPi) ps -= kPi;
    if (ps < 0.0) ps += kPi;
    t = t + kAuS * (n0 * ca + n1 * sa);
    lam = lam_s;
    beta = beta_s;
    psi = ps;
}

// Philox4x32-10: counter c[4], key k[2]
__device__ __forceinline__ void philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c[0]), lo0 = 0xD2511F53u * c[0];
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c[2]), lo1 = 0xCD9E8D57u * c[2];
        const uint32_t n0 = hi1 ^ c[1] ^ k0, n2 = hi0 ^ c[3] ^ k1;
        c[0] = n0; c[1] = lo1; c[2] = n2; c[3] = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
}

// two uniforms in (0, 1), 52 random bits each: counter = (index, step, stream, 0), key = seed
__device__ __forceinline__ void uniforms2(uint64_t seed, uint32_t step, uint32_t stream, uint32_t index, double& u0, double& u1) {
    uint32_t c[4] = {index, step, stream, 0u};
    philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
    const uint64_t a = ((uint64_t)c[0] << 20) | (c[1] >> 12), b = ((uint64_t)c[2] << 20) | (c[3] >> 12);
    u0 = ((double)a + 0.5) * 0x1p-52;
    u1 = ((double)b + 0.5) * 0x1p-52;
}

// Noise realisation of eq. 12 (reading G5): Re, Im ~ N(0, S_n / (4 df)) by Box-Muller from the two
// uniforms of Philox counter (bin, channel, stream 3, 0); bins with S_n <= 0 or not finite get 0.  out [3][N][2].
__global__ void k_noise(const double* __restrict__ psd, int64_t N, double df, uint64_t seed, double* __restrict__ out) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (k >= N) return;
    const double s = psd[c * N + k];
    double re = 0.0, im = 0.0;
    if (isfinite(s) && s > 0.0) {
        double u0, u1;
        uniforms2(seed, (uint32_t)c, 3u, (uint32_t)k, u0, u1);
        const double mod = sqrt(s / (4.0 * df)) * sqrt(-2.0 * log(u0));
        double sn, cs;
        sincos(2.0 * kPi * u1, &sn, &cs);
        re = mod * cs;
        im = mod * sn;
    }
    reinterpret_cast<double2*>(out)[c * N + k] = make_double2(re, im);
}

struct PtState {
    double* theta;       // [T][K][11] sampler coordinates
    double* logl;        // [T][K]
    double* betas;       // [T]
    double* prop_theta;  // [T][K/2][11] proposals (sampler coordinates; the hot path converts them itself)
    double* prop_logl;   // [T][K/2]
    double* prop_z;      // [T][K/2]
    unsigned long long* n_accept;   // [T]
    unsigned long long* n_swap;     // [T-1]
    int T, K;
    double a;            // stretch parameter
    uint64_t seed;
};

// Walkers k with k % 2 == half move; moving walker number i of temperature t is k = 2 i + half.
__global__ void k_pt_propose(PtState s, int half, uint32_t step) {
    const int hk = s.K / 2;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= s.T * hk) return;
    const int t = idx / hk, i = idx - t * hk;
    const int k = 2 * i + half;
    double u_z, u_j;
    uniforms2(s.seed, step, 0u, (uint32_t)(t * s.K + k), u_z, u_j);
    const double g = __dadd_rn(__dmul_rn(s.a - 1.0, u_z), 1.0);
    const double z = __ddiv_rn(__dmul_rn(g, g), s.a);                       // eq. 15 by inverting its CDF
    int jj = (int)(u_j * hk);
    jj = min(jj, hk - 1);
    const int j = 2 * jj + (1 - half);                                       // partner from the other half
    const double* xk = s.theta + ((int64_t)t * s.K + k) * MBHL_NPARAM;
    const double* xj = s.theta + ((int64_t)t * s.K + j) * MBHL_NPARAM;
#pragma unroll
    for (int d = 0; d < MBHL_NPARAM; ++d)                                                                   // eq. 14, no contraction
        s.prop_theta[(int64_t)idx * MBHL_NPARAM + d] = __dadd_rn(xj[d], __dmul_rn(z, __dadd_rn(xk[d], -xj[d])));
    s.prop_z[idx] = z;
}

__global__ void k_pt_accept(PtState s, int half, uint32_t step) {
    const int hk = s.K / 2;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= s.T * hk) return;
    const int t = idx / hk, i = idx - t * hk;
    const int k = 2 * i + half;
    const int64_t w = (int64_t)t * s.K + k;
    double u, unused;
    uniforms2(s.seed, step, 1u, (uint32_t)w, u, unused);
    const double ln_new = s.prop_logl[idx], ln_old = s.logl[w], beta = s.betas[t];
    // ln of eq. 16 on the tempered density: (D - 1) ln z + beta (ln L(Y) - ln L(X)); outside the prior box L(Y) = 0
    bool acc = false;
    if (isfinite(ln_new)) {
        const double lnr = (MBHL_NPARAM - 1) * log(s.prop_z[idx]) + (beta * ln_new - beta * ln_old);
        acc = log(u) < lnr;
    }
    if (acc) {
#pragma unroll
        for (int d = 0; d < MBHL_NPARAM; ++d) s.theta[w * MBHL_NPARAM + d] = s.prop_theta[(int64_t)idx * MBHL_NPARAM + d];
        s.logl[w] = ln_new;
        atomicAdd(s.n_accept + t, 1ULL);
    }
}

// one thread per walker slot k: rung pairs (i, i-1) from the hottest down, as eq. 17
__global__ void k_pt_swap(PtState s, uint32_t step) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= s.K) return;
    for (int i = s.T - 1; i >= 1; --i) {
        const int64_t wi = (int64_t)i * s.K + k, wj = (int64_t)(i - 1) * s.K + k;
        double u, unused;
        uniforms2(s.seed, step, 2u, (uint32_t)wi, u, unused);
        const double li = s.logl[wi], lj = s.logl[wj];
        const double lnr = (s.betas[i - 1] - s.betas[i]) * (li - lj);
        if (log(u) < lnr) {
#pragma unroll
            for (int d = 0; d < MBHL_NPARAM; ++d) {
                const double a = s.theta[wi * MBHL_NPARAM + d];
                s.theta[wi * MBHL_NPARAM + d] = s.theta[wj * MBHL_NPARAM + d];
                s.theta[wj * MBHL_NPARAM + d] = a;
            }
            s.logl[wi] = lj;
            s.logl[wj] = li;
            atomicAdd(s.n_swap + (i - 1), 1ULL);
        }
    }
}

}  // namespace mbhl
