// mbhl_model.cuh - device-side waveform model and LISA response (fp64).
//
// Per-walker constants (step a1), PhenomD/PhenomHM amplitude + phase + dphase (a3, PAPER.md:112-126,
// eqs. 5-6) and the fast frequency-domain response with TDI A/E/T (a4, eqs. 7-10).
// Readings: DESIGN.md section 4.  Written from the formulas, shares nothing with oracle/.
#pragma once
#include <math.h>
#include <stdint.h>

#include "mbhl_model_table.inc"

#define MBHL_NMODE 6
#define MBHL_NQ 8

namespace mbhl {

__constant__ double c_table[MBHL_TABLE_N];

// physical constants (SURVEY.md 8(c) "Constants")
constexpr double kPi = 3.141592653589793238462643383279502884;
constexpr double kTwoPi = 6.283185307179586476925286766559005768;
constexpr double kC = 299792458.0;
constexpr double kMtsun = 4.925491025543576e-06;
constexpr double kGpcS = 1.0e9 * 3.0856775814913674e16 / kC;
constexpr double kAuS = 149597870700.0 / kC;
constexpr double kArmS = 2.5e9 / kC;
constexpr double kYearSid = 31558149.7635;
constexpr double kOmega0 = kTwoPi / kYearSid;
constexpr double kEulerGamma = 0.5772156649015328606;
constexpr double kFAmpIns = 0.014;
constexpr double kFPhiIns = 0.018;
constexpr double kLn64 = 4.158883083359671856503;   // ln 64

__constant__ int c_mode_l[MBHL_NMODE] = {2, 3, 4, 2, 3, 4};
__constant__ int c_mode_m[MBHL_NMODE] = {2, 3, 4, 1, 2, 3};

struct cplx {
    double re, im;
};
__host__ __device__ inline cplx cmul(cplx a, cplx b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__host__ __device__ inline cplx cadd(cplx a, cplx b) { return {a.re + b.re, a.im + b.im}; }
__host__ __device__ inline cplx csub(cplx a, cplx b) { return {a.re - b.re, a.im - b.im}; }
__host__ __device__ inline cplx cscale(cplx a, double s) { return {a.re * s, a.im * s}; }

struct ModeConst {
    // piecewise-linear frequency maps f -> f_22 (O3): regions 0 inspiral, 1 intermediate, 2 ringdown
    double fiA, fiP, fr;        // boundaries (Mf): amplitude inspiral end, phase inspiral end, f_RD,lm
    double aA[3], bA[3];        // amplitude map
    double aP[3], bP[3];        // phase map
    double invaP[3], cP[3];     // 1/a_r and continuity constants (mode offset Delta_lm folded in)
    double ampc;                // pi sqrt(2 eta/3) c_lm massfactor
    int vpow;                   // power of V in |H_lm|
    int active;
    double f_lo, f_hi;          // band (Hz)
    double dlog;                // ln(f_hi/f_lo)/(S-1)
    double inv_dlog;            // (S-1)/ln(f_hi/f_lo)
    double ln_flo;
    double P[12];               // mode polarisation tensor: xx,yy,zz,xy,xz,yz as (re,im)
};

struct WalkerConst {
    int valid;
    int pad_;
    double eta, M_s, amp0, t_coal;
    double fRD, fDM, f_peak, f_ref, f_mr;
    double am[7];               // PN amplitude coefficients times pi^(i/3)
    double rho[3];
    double gam1w, gam2ow, w;    // gamma1*w, gamma2/w, w = gamma3 fDM
    double dint[5];             // intermediate amplitude quartic
    double ph[8];               // PN phase coefficients (ph[5] multiplies 1+ln(pi f); ph[6] constant part)
    double pre;                 // 3/(128 eta)
    double inveta;
    double sig[4];
    double bet[3], alp[5];
    double C1i, C2i, C1m, C2m;  // C1 connection constants
    double pshift, tshift;      // alignment: Psi(f_ref) = Psi'(f_ref) = 0
    double k[3];                // propagation vector
    ModeConst mode[MBHL_NMODE];
};

// Compact per-walker record read by the fused dense kernel (step a6/a7): the bin range of every mode's band
// on the init grid (k_lo = min{k: f_k >= f_lo}, k_hi = max{k: f_k <= f_hi}; empty: k_lo > k_hi) and the
// constants of the log-spaced knot grid used to guess a bin's spline interval.
struct DenseMode {
    int k_lo, k_hi;
    double ln_flo, inv_dlog;
};
struct DenseWalker {
    double t_coal;
    int valid;
    int pad_;
    long long pairs;            // sum over modes of in-band bins
    long long bins;             // bins covered by at least one mode
    DenseMode mode[MBHL_NMODE];
};

constexpr double kRoundMagic = 6755399441055744.0;   // 1.5 * 2^52: x + magic - magic = rint(x) for |x| < 2^51

// sin(pi y/2) = y Ps(y^2), cos(pi y/2) = Pc(y^2) on |y| <= 1/2: coefficients from gen_sincos_coeffs.py
// (Chebyshev-node interpolation in 50-digit arithmetic; max error 2.6e-17 / 1.0e-16 before rounding).
// Kept in the constant bank so that DFMA reads them as c[][] operands (as immediates each costs two moves per use).
__constant__ double c_sc[13] = {1.5707963267948966, -0.6459640975062443, 0.07969262624604301, -0.004681754132340976,
                                0.0001604411507421909, -3.59864335298231e-06, 5.633933781537854e-08,
                                -1.2337005501361513, 0.25366950789986475, -0.02086348073494657,
                                0.000919259950041661, -2.520013526428479e-05, 4.6552961874867623e-07};
// The shorter pair used per bin by the fused dense kernel (sincos_qturn_x, mbhl_dense.cuh): sine of degree 4 and cosine of
// degree 5 in y^2 (max error 3.4e-12 / 5.6e-14, gen_sincos_coeffs.py: three multiply-adds fewer per bin, far below the 1e-9
// per-bin bar of the template).  S0..S4, then C0..C5.
__constant__ double c_scd[11] = {1.5707963267881, -0.6459640961467954, 0.07969258272563062, -0.004681266256726245,
                                 0.00015820630355647733,
                                 0.9999999999999444, -1.2337005501201592, 0.25366950715370434, -0.020863468002244645,
                                 0.0009191617369539572, -2.4850963357813638e-05};
#define kS0 c_sc[0]
#define kS1 c_sc[1]
#define kS2 c_sc[2]
#define kS3 c_sc[3]
#define kS4 c_sc[4]
#define kS5 c_sc[5]
#define kS6 c_sc[6]
#define kC1 c_sc[7]
#define kC2 c_sc[8]
#define kC3 c_sc[9]
#define kC4 c_sc[10]
#define kC5 c_sc[11]
#define kC6 c_sc[12]

// sin and cos of p4 quarter turns (angle = p4 pi/2), any |p4| < 2^51.  No conversions, no divides: the
// nearest integer comes from the magic-number add, the quadrant from the low word of that sum.
__device__ __forceinline__ void sincos_qturn(double p4, double& sn, double& cs) {
    const double t = p4 + kRoundMagic;
    const int n = __double2loint(t);
    const double y = p4 - (t - kRoundMagic);
    const double z = y * y;
    double ps = fma(z, kS6, kS5);
    double pc = fma(z, kC6, kC5);
    ps = fma(z, ps, kS4); pc = fma(z, pc, kC4);
    ps = fma(z, ps, kS3); pc = fma(z, pc, kC3);
    ps = fma(z, ps, kS2); pc = fma(z, pc, kC2);
    ps = fma(z, ps, kS1); pc = fma(z, pc, kC1);
    ps = fma(z, ps, kS0); pc = fma(z, pc, 1.0);
    ps *= y;
    const bool odd = (n & 1) != 0;
    const double a = odd ? pc : ps;      // sin(angle) up to sign
    const double b = odd ? ps : pc;      // cos(angle) up to sign
    sn = __hiloint2double(__double2hiint(a) ^ ((n & 2) << 30), __double2loint(a));
    cs = __hiloint2double(__double2hiint(b) ^ (((n + 1) & 2) << 30), __double2loint(b));
}

// ---------------------------------------------------------------------------------------------
// PhenomD pieces (all frequencies are Mf)
// ---------------------------------------------------------------------------------------------
__device__ inline double fit11(int base, double eta, double x) {
    const double* t = c_table + base;
    const double e2 = eta * eta;
    return t[0] + t[1] * eta + x * (t[2] + t[3] * eta + t[4] * e2) + x * x * (t[5] + t[6] * eta + t[7] * e2) +
           x * x * x * (t[8] + t[9] * eta + t[10] * e2);
}

__device__ inline void amp_ins(const WalkerConst& c, double f, double* val, double* der) {
    const double f13 = cbrt(f), f23 = f13 * f13;
    const double invf = 1.0 / f;
    // sum_i am_i f^(i/3), i = 0..6, then the pseudo-PN terms rho_k f^((6+k)/3)
    double p[7];
    p[0] = 1.0; p[1] = f13; p[2] = f23; p[3] = f; p[4] = f * f13; p[5] = f * f23; p[6] = f * f;
    double v = 0.0, d = 0.0;
#pragma unroll
    for (int i = 0; i < 7; ++i) {
        v += c.am[i] * p[i];
        d += c.am[i] * (i / 3.0) * p[i] * invf;
    }
    const double f73 = f * f * f13, f83 = f * f * f23, f3 = f * f * f;
    v += c.rho[0] * f73 + c.rho[1] * f83 + c.rho[2] * f3;
    d += ((7.0 / 3.0) * c.rho[0] * f73 + (8.0 / 3.0) * c.rho[1] * f83 + 3.0 * c.rho[2] * f3) * invf;
    *val = v;
    *der = d;
}

__device__ inline void amp_mr(const WalkerConst& c, double f, double* val, double* der) {
    const double x = f - c.fRD;
    const double lor = 1.0 / (x * x + c.w * c.w);
    const double v = c.gam1w * lor * exp(-c.gam2ow * x);
    *val = v;
    *der = v * (-2.0 * x * lor - c.gam2ow);
}

__device__ inline double amp_hat(const WalkerConst& c, double f) {
    double v, d;
    if (f < kFAmpIns) {
        amp_ins(c, f, &v, &d);
    } else if (f < c.f_peak) {
        v = c.dint[0] + f * (c.dint[1] + f * (c.dint[2] + f * (c.dint[3] + f * c.dint[4])));
    } else {
        amp_mr(c, f, &v, &d);
    }
    return v;
}

// v = cbrt(pi f), from the caller when it already has it (the mode amplitude of an inspiral knot needs the same cube root)
__device__ inline void psi_ins_raw_v(const WalkerConst& c, double f, double v, double* psi, double* dpsi) {
    const double pf = kPi * f;
    const double lnpf = log(pf);
    const double v2 = v * v, v3 = pf, v4 = v2 * v2, v5 = v4 * v, v6 = v3 * v3, v7 = v6 * v;
    const double iv5 = 1.0 / v5;
    const double invf = kPi * (iv5 * v2);               // 1 / f = pi / v^3: one division fewer
    const double c5 = c.ph[5] * (1.0 + lnpf);
    const double c6 = c.ph[6] - (6848.0 / 63.0) * (kLn64 + lnpf);
    // series S = sum_i c_i v^i ; Psi_TF2 = -pi/4 + pre v^-5 S
    const double S = 1.0 + c.ph[2] * v2 + c.ph[3] * v3 + c.ph[4] * v4 + c5 * v5 + c6 * v6 + c.ph[7] * v7;
    // d/df [c_i v^(i-5)] = v^(i-5)/f * ((i-5)/3 c_i + f c_i'), with f c_5' = ph5, f c_6' = -6848/63
    const double dS = (-5.0 / 3.0) + (-1.0) * c.ph[2] * v2 + (-2.0 / 3.0) * c.ph[3] * v3 + (-1.0 / 3.0) * c.ph[4] * v4 +
                      c.ph[5] * v5 + ((1.0 / 3.0) * c6 - 6848.0 / 63.0) * v6 + (2.0 / 3.0) * c.ph[7] * v7;
    const double f13 = v * 0.68278406325529568147, f23 = f13 * f13;     // cbrt(f) = cbrt(pi f) / cbrt(pi): one cube root fewer
    *psi = -0.25 * kPi + c.pre * iv5 * S +
           (c.sig[0] * f + 0.75 * c.sig[1] * f * f13 + 0.6 * c.sig[2] * f * f23 + 0.5 * c.sig[3] * f * f) * c.inveta;
    *dpsi = c.pre * iv5 * dS * invf + (c.sig[0] + c.sig[1] * f13 + c.sig[2] * f23 + c.sig[3] * f) * c.inveta;
}
__device__ inline void psi_ins_raw(const WalkerConst& c, double f, double* psi, double* dpsi) {
    psi_ins_raw_v(c, f, cbrt(kPi * f), psi, dpsi);
}

__device__ inline void psi_int_raw(const WalkerConst& c, double f, double* psi, double* dpsi) {
    const double if1 = 1.0 / f, if2 = if1 * if1;
    *psi = (c.bet[0] * f + c.bet[1] * log(f) - (c.bet[2] / 3.0) * if2 * if1) * c.inveta;
    *dpsi = (c.bet[0] + c.bet[1] * if1 + c.bet[2] * if2 * if2) * c.inveta;
}

__device__ inline void psi_mr_raw(const WalkerConst& c, double f, double* psi, double* dpsi) {
    const double x = f - c.alp[4] * c.fRD;
    const double sq = sqrt(f), f14 = sqrt(sq);
    *psi = (c.alp[0] * f - c.alp[1] / f + (4.0 / 3.0) * c.alp[2] * sq * f14 + c.alp[3] * atan(x / c.fDM)) * c.inveta;
    *dpsi = (c.alp[0] + c.alp[1] / (f * f) + c.alp[2] / f14 + c.alp[3] * c.fDM / (c.fDM * c.fDM + x * x)) * c.inveta;
}

// C1-connected Psi_22 and dPsi_22/df before the alignment of reading G4 (reads neither pshift nor tshift).
__device__ inline void psi22_unaligned(const WalkerConst& c, double f, double* psi, double* dpsi) {
    double p, d;
    if (f < kFPhiIns) {
        psi_ins_raw(c, f, &p, &d);
    } else if (f < c.f_mr) {
        psi_int_raw(c, f, &p, &d);
        p += c.C1i + c.C2i * f;
        d += c.C2i;
    } else {
        psi_mr_raw(c, f, &p, &d);
        p += c.C1m + c.C2m * f;
        d += c.C2m;
    }
    *psi = p;
    *dpsi = d;
}

// Aligned Psi_22 and dPsi_22/df.
__device__ inline void psi22(const WalkerConst& c, double f, double* psi, double* dpsi) {
    double p, d;
    psi22_unaligned(c, f, &p, &d);
    *psi = p - c.pshift - c.tshift * (f - c.f_ref);
    *dpsi = d - c.tshift;
}

// t_lm(f_hz) of eq. 6 for mode index mi.
__device__ inline double t_of_f(const WalkerConst& c, int mi, double f_hz) {
    const ModeConst& mc = c.mode[mi];
    const double f = f_hz * c.M_s;
    const int r = (f < mc.fiP) ? 0 : ((f < mc.fr) ? 1 : 2);
    double p, d;
    psi22(c, mc.aP[r] * f + mc.bP[r], &p, &d);
    return c.t_coal + c.M_s * d * (1.0 / kTwoPi);
}

// ---------------------------------------------------------------------------------------------
// Spin-weight -2 spherical harmonics needed by the six modes (closed forms), theta = iota
// ---------------------------------------------------------------------------------------------
// ct, st = cos, sin of theta; ch, sh = cos, sin of theta / 2 (the caller evaluates them once for both signs of m)
__device__ inline double sYlm_theta(int l, int m, double ct, double st, double ch, double sh) {
    const double ch2 = ch * ch, sh2 = sh * sh;
    if (l == 2) {
        if (m == 2) return sqrt(5.0 / (64.0 * kPi)) * (1.0 + ct) * (1.0 + ct);
        if (m == -2) return sqrt(5.0 / (64.0 * kPi)) * (1.0 - ct) * (1.0 - ct);
        if (m == 1) return sqrt(5.0 / (16.0 * kPi)) * st * (1.0 + ct);
        if (m == -1) return sqrt(5.0 / (16.0 * kPi)) * st * (1.0 - ct);
    } else if (l == 3) {
        if (m == 3) return -sqrt(21.0 / (2.0 * kPi)) * ch2 * ch2 * ch * sh;
        if (m == -3) return sqrt(21.0 / (2.0 * kPi)) * ch * sh2 * sh2 * sh;
        if (m == 2) return 0.5 * sqrt(7.0 / kPi) * ch2 * ch2 * (3.0 * ct - 2.0);
        if (m == -2) return sqrt(7.0 / (4.0 * kPi)) * (2.0 + 3.0 * ct) * sh2 * sh2;
    } else if (l == 4) {
        if (m == 4) return 3.0 * sqrt(7.0 / kPi) * ch2 * ch2 * ch2 * sh2;
        if (m == -4) return 3.0 * sqrt(7.0 / kPi) * ch2 * sh2 * sh2 * sh2;
        if (m == 3) return -3.0 * sqrt(7.0 / (2.0 * kPi)) * ch2 * ch2 * ch * (2.0 * ct - 1.0) * sh;
        if (m == -3) return 3.0 * sqrt(7.0 / (2.0 * kPi)) * ch * (1.0 + 2.0 * ct) * sh2 * sh2 * sh;
    }
    return 0.0;
}

// ---------------------------------------------------------------------------------------------
// Smooth functions of one mode at one frequency: the Q = 8 splined quantities (phase in CYCLES)
// ---------------------------------------------------------------------------------------------
__device__ inline double sinc_pi(double u) {   // sin(pi u)/(pi u); the quarter-turn sine keeps its relative accuracy near 0
    const double x = kPi * u;
    double sn, cs;
    sincos_qturn(2.0 * u, sn, cs);
    return (x == 0.0) ? 1.0 : sn / x;
}

__device__ inline void smooth_quantities(const WalkerConst& c, int mi, double f_hz, double q[MBHL_NQ]) {
    const ModeConst& mc = c.mode[mi];
    const double f = f_hz * c.M_s;
    const int m = c_mode_m[mi];
    // amplitude (O3): A_lm = amp0 * Ahat(f22A) * beta_lm(f)
    const double V = cbrt(kTwoPi * f / m);
    {
        const int r = (f < mc.fiA) ? 0 : ((f < mc.fr) ? 1 : 2);
        const double f22 = mc.aA[r] * f + mc.bA[r];
        double vp = 1.0;
        for (int i = 0; i < mc.vpow; ++i) vp *= V;
        const double beta = mc.ampc * vp / (V * V * V * sqrt(V));
        q[0] = c.amp0 * amp_hat(c, f22) * beta;
    }
    // phase and time (O3, eq. 6)
    double psi, dpsi;
    {
        const int r = (f < mc.fiP) ? 0 : ((f < mc.fr) ? 1 : 2);
        const double f22 = mc.aP[r] * f + mc.bP[r];
        if (r == 0 && f22 < kFPhiIns) {
            // inspiral branch of the map: f22 = (2 / m) f, so cbrt(pi f22) is the V of the amplitude above
            double p_, d_;
            psi_ins_raw_v(c, f22, V, &p_, &d_);
            psi = p_ - c.pshift - c.tshift * (f22 - c.f_ref);
            dpsi = d_ - c.tshift;
        } else {
            psi22(c, f22, &psi, &dpsi);
        }
        psi = psi * mc.invaP[r] + mc.cP[r];
    }
    const double t = c.t_coal + c.M_s * dpsi * (1.0 / kTwoPi);
    // orbit (O4): positions in light-seconds
    double sa, ca;
    sincos_qturn(t * (4.0 / kYearSid), sa, ca);                 // alpha = Omega_0 t, in quarter turns
    const double c2a = ca * ca - sa * sa, s2a = 2.0 * sa * ca;
    const double ecc = kArmS / (2.0 * 1.7320508075688772935 * kAuS);
    const double eR = ecc * kAuS;
    const double cb[3] = {1.0, -0.5, -0.5};
    const double sb[3] = {0.0, 0.86602540378443864676, -0.86602540378443864676};
    double pL[3][3];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        pL[n][0] = eR * 0.5 * ((c2a * cb[n] + s2a * sb[n]) - 3.0 * cb[n]);
        pL[n][1] = eR * 0.5 * ((s2a * cb[n] - c2a * sb[n]) - 3.0 * sb[n]);
        pL[n][2] = -eR * 1.7320508075688772935 * (ca * cb[n] + sa * sb[n]);
    }
    const double kp0 = kAuS * (c.k[0] * ca + c.k[1] * sa);
    const double phiR_cyc = -f_hz * kp0;                       // phi_R / 2 pi
    q[1] = -psi * (1.0 / kTwoPi) + phiR_cyc;
    // the three arms: (s,r) = (3,1),(2,1),(3,2) and their reverses
    const int as_[3] = {2, 1, 2};
    const int ar_[3] = {0, 0, 1};
    cplx gf[3], gb[3];   // forward s->r and backward r->s link kernels without the common prefactor
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int s = as_[a], r = ar_[a];
        const double nx = (pL[r][0] - pL[s][0]) * (1.0 / kArmS);
        const double ny = (pL[r][1] - pL[s][1]) * (1.0 / kArmS);
        const double nz = (pL[r][2] - pL[s][2]) * (1.0 / kArmS);
        const double kn = c.k[0] * nx + c.k[1] * ny + c.k[2] * nz;
        const double kps = c.k[0] * (pL[r][0] + pL[s][0]) + c.k[1] * (pL[r][1] + pL[s][1]) + c.k[2] * (pL[r][2] + pL[s][2]);
        const double w0 = nx * nx, w1 = ny * ny, w2 = nz * nz, w3 = 2.0 * nx * ny, w4 = 2.0 * nx * nz, w5 = 2.0 * ny * nz;
        cplx nPn;
        nPn.re = mc.P[0] * w0 + mc.P[2] * w1 + mc.P[4] * w2 + mc.P[6] * w3 + mc.P[8] * w4 + mc.P[10] * w5;
        nPn.im = mc.P[1] * w0 + mc.P[3] * w1 + mc.P[5] * w2 + mc.P[7] * w3 + mc.P[9] * w4 + mc.P[11] * w5;
        double se, ce;
        sincos_qturn(-2.0 * f_hz * (kArmS + kps), se, ce);     // exp(-i pi f (L + k.(p_r+p_s)))
        const cplx e = cmul({ce, se}, nPn);
        // sinc[pi f L (1 -+ k.n)] = sin / x: the two divisions of an arm share one reciprocal
        const double um = f_hz * kArmS * (1.0 - kn), up = f_hz * kArmS * (1.0 + kn);
        const double xm = kPi * um, xp = kPi * up;
        double snm, snp, unused;
        sincos_qturn(2.0 * um, snm, unused);
        sincos_qturn(2.0 * up, snp, unused);
        const double prod = xm * xp;
        const double inv = 1.0 / prod;
        gf[a] = cscale(e, (prod != 0.0) ? snm * xp * inv : sinc_pi(um));
        gb[a] = cscale(e, (prod != 0.0) ? snp * xm * inv : sinc_pi(up));
    }
    // G_31 = gf[0], G_13 = gb[0], G_21 = gf[1], G_12 = gb[1], G_32 = gf[2], G_23 = gb[2]
    double sz, cz;
    sincos_qturn(-4.0 * f_hz * kArmS, sz, cz);
    const cplx z = {cz, sz};
    const cplx X = csub(cadd(gf[0], cmul(z, gb[0])), cadd(gf[1], cmul(z, gb[1])));
    const cplx Y = csub(cadd(gb[1], cmul(z, gf[1])), cadd(gf[2], cmul(z, gb[2])));
    const cplx Z = csub(cadd(gb[2], cmul(z, gf[2])), cadd(gb[0], cmul(z, gf[0])));
    // common factor (1 - z^2)(-i pi f L)
    const cplx z2 = cmul(z, z);
    const double pfl = kPi * f_hz * kArmS;
    const cplx pref = cmul({1.0 - z2.re, -z2.im}, {0.0, -pfl});
    const cplx A = cmul(pref, cscale(csub(Z, X), 0.70710678118654752440));
    const cplx E = cmul(pref, cscale(cadd(csub(X, cscale(Y, 2.0)), Z), 0.40824829046386301637));
    const cplx T = cmul(pref, cscale(cadd(cadd(X, Y), Z), 0.57735026918962576451));
    q[2] = A.re; q[3] = A.im; q[4] = E.re; q[5] = E.im; q[6] = T.re; q[7] = T.im;
}

// ---------------------------------------------------------------------------------------------
// Step a1 + a2: everything per walker
// ---------------------------------------------------------------------------------------------
__device__ inline void solve5(double A[5][5], double b[5]) {
    for (int col = 0; col < 5; ++col) {
        int piv = col;
        double best = fabs(A[col][col]);
        for (int r = col + 1; r < 5; ++r)
            if (fabs(A[r][col]) > best) { best = fabs(A[r][col]); piv = r; }
        if (piv != col) {
            for (int k = 0; k < 5; ++k) { double t = A[col][k]; A[col][k] = A[piv][k]; A[piv][k] = t; }
            double t = b[col]; b[col] = b[piv]; b[piv] = t;
        }
        const double inv = 1.0 / A[col][col];
        for (int r = col + 1; r < 5; ++r) {
            const double fct = A[r][col] * inv;
            for (int k = col; k < 5; ++k) A[r][k] -= fct * A[col][k];
            b[r] -= fct * b[col];
        }
    }
    for (int r = 4; r >= 0; --r) {
        double s = b[r];
        for (int k = r + 1; k < 5; ++k) s -= A[r][k] * b[k];
        b[r] = s / A[r][r];
    }
}

// Root of a continuous function on a bracket [a, b] with fn(a) = fa and fn(b) = fb of opposite signs
// (Illinois variant of regula falsi, bisection when the secant leaves the bracket).  Stops when the bracket
// is a few ulps wide or |fn| <= ftol; returns the end point whose sign matches fb.
template <typename F>
__device__ inline double bracketed_root(F fn, double a, double fa, double b, double fb, double ftol) {
    if (fb == 0.0) return b;
    const bool up = fb > 0.0;                            // sign of the kept end point
    int side = 0;
    for (int it = 0; it < 200; ++it) {
        if (fabs(b - a) <= 4.5e-16 * fmax(fabs(a), fabs(b))) break;
        double x = (a * fb - b * fa) / (fb - fa);
        if (!((x > a && x < b) || (x < a && x > b))) x = 0.5 * (a + b);
        const double fx = fn(x);
        if ((fx > 0.0) == up || fx == 0.0) {
            b = x; fb = fx;
            if (fabs(fx) <= ftol) break;
            if (side == 1) fa *= 0.5;
            side = 1;
        } else {
            a = x; fa = fx;
            if (side == -1) fb *= 0.5;
            side = -1;
        }
    }
    return b;
}

// Everything per walker.  The per-mode parts run for the modes mode_lo <= mi < mode_hi only: k_walker_consts gives a warp
// to every walker, all lanes run the common part redundantly on one shared-memory record (identical stores)
// and lane L fills mode L % 6.
__device__ inline void build_walker(const double* __restrict__ p, double t0, double f_min, double f_max, int S,
                                    uint32_t mode_mask, WalkerConst& c, int mode_lo, int mode_hi) {
    const double M_T = p[0], q_in = p[1], a1 = p[2], a2 = p[3], D_L = p[4];
    const double phi_ref = p[5], inc = p[6], lam = p[7], beta = p[8], psi_pol = p[9], t_ref = p[10];
    bool ok = true;
    for (int i = 0; i < 11; ++i) ok = ok && isfinite(p[i]);
    ok = ok && (M_T > 0.0) && (D_L > 0.0) && (q_in > 0.0) && (fabs(a1) <= 1.0) && (fabs(a2) <= 1.0);
    c.valid = ok ? 1 : 0;
    c.pad_ = 0;
    for (int mi = 0; mi < MBHL_NMODE; ++mi) c.mode[mi].active = 0;
    __syncwarp();                                       // every lane is past the reset before a lane fills its mode
    if (!ok) return;

    const double q = (q_in >= 1.0) ? q_in : 1.0 / q_in;
    const double m1 = q / (1.0 + q), m2 = 1.0 / (1.0 + q);
    const double eta = m1 * m2, delta = m1 - m2;
    const double e2 = eta * eta, e3 = e2 * eta;
    const double xs = 0.5 * (a1 + a2), xa = 0.5 * (a1 - a2);
    const double chi_pn = (m1 * a1 + m2 * a2) - (38.0 * eta / 113.0) * (a1 + a2);
    const double chi_hat = chi_pn / (1.0 - 76.0 * eta / 113.0);
    const double x = chi_hat - 1.0;
    c.eta = eta;
    c.inveta = 1.0 / eta;
    c.pre = 3.0 / (128.0 * eta);
    c.M_s = M_T * kMtsun;
    c.amp0 = c.M_s * c.M_s / (D_L * kGpcS);
    c.t_coal = t0 + t_ref;

    // final state, quasi-normal modes
    const double Stot = m1 * m1 * a1 + m2 * m2 * a2;
    const double* T = c_table;
    double af;
    {
        const double S2 = Stot * Stot, S3 = S2 * Stot, S4 = S2 * S2;
        af = 2.0 * sqrt(3.0) * eta + T[MT_fs_spin_e2] * e2 + T[MT_fs_spin_e3] * e3 + T[MT_fs_spin_e4] * e2 * e2 +
             eta * (T[MT_fs_spin_s1e1] * Stot + T[MT_fs_spin_s2e1] * S2 + T[MT_fs_spin_s3e1] * S3 + T[MT_fs_spin_s4e1] * S4) +
             e2 * (T[MT_fs_spin_s1e2] * Stot + T[MT_fs_spin_s2e2] * S2 + T[MT_fs_spin_s3e2] * S3 + T[MT_fs_spin_s4e2] * S4) + Stot;
        af = fmin(af, 0.999);
    }
    double Erad;
    {
        const double Sh = Stot / (1.0 - 2.0 * eta);
        const double num = eta * (T[MT_fs_erad_e1] + T[MT_fs_erad_e2] * eta + T[MT_fs_erad_e3] * e2 + T[MT_fs_erad_e4] * e3);
        Erad = num * (1.0 + (T[MT_fs_erad_n0] + T[MT_fs_erad_n1] * eta + T[MT_fs_erad_n2] * e2) * Sh) /
               (1.0 + (T[MT_fs_erad_d0] + T[MT_fs_erad_d1] * eta + T[MT_fs_erad_d2] * e2) * Sh);
    }
    double frd[MBHL_NMODE], fdm[MBHL_NMODE];
    {
        const double oma = 1.0 - af;
        const double ln_oma = log(oma);                       // (1 - a_f)^p = exp(p ln(1 - a_f)): one logarithm serves the 4 powers
        const double inv = 1.0 / (kTwoPi * (1.0 - Erad));
        for (int mi = 0; mi < mode_hi; ++mi) {
            if (mi != 0 && mi < mode_lo) continue;           // mode (2,2) is needed by everyone
            const double* t6 = T + MT_qnm_22_f1 + 6 * mi;
            const double om = t6[0] + t6[1] * exp(t6[2] * ln_oma);
            const double Q = t6[3] + t6[4] * exp(t6[5] * ln_oma);
            frd[mi] = om * inv;
            fdm[mi] = frd[mi] / (2.0 * Q);
        }
    }
    __syncwarp();                                       // the loop above is lane-divergent (mode_lo/mode_hi differ per lane)
    c.fRD = frd[0];
    c.fDM = fdm[0];

    // phenomenological coefficients (O1)
    c.rho[0] = fit11(MT_pd_rho1_l00, eta, x);
    c.rho[1] = fit11(MT_pd_rho2_l00, eta, x);
    c.rho[2] = fit11(MT_pd_rho3_l00, eta, x);
    const double v2 = fit11(MT_pd_v2_l00, eta, x);
    const double g1 = fit11(MT_pd_gamma1_l00, eta, x);
    const double g2 = fit11(MT_pd_gamma2_l00, eta, x);
    const double g3 = fit11(MT_pd_gamma3_l00, eta, x);
    c.sig[0] = fit11(MT_pd_sigma1_l00, eta, x);
    c.sig[1] = fit11(MT_pd_sigma2_l00, eta, x);
    c.sig[2] = fit11(MT_pd_sigma3_l00, eta, x);
    c.sig[3] = fit11(MT_pd_sigma4_l00, eta, x);
    c.bet[0] = fit11(MT_pd_beta1_l00, eta, x);
    c.bet[1] = fit11(MT_pd_beta2_l00, eta, x);
    c.bet[2] = fit11(MT_pd_beta3_l00, eta, x);
    c.alp[0] = fit11(MT_pd_alpha1_l00, eta, x);
    c.alp[1] = fit11(MT_pd_alpha2_l00, eta, x);
    c.alp[2] = fit11(MT_pd_alpha3_l00, eta, x);
    c.alp[3] = fit11(MT_pd_alpha4_l00, eta, x);
    c.alp[4] = fit11(MT_pd_alpha5_l00, eta, x);

    // PN phase coefficients (constant ratios are written (K / D) * x so that they fold at compile time: K * x / D is a
    // run-time division, and this routine is one long dependent chain)
    c.ph[0] = 1.0;
    c.ph[1] = 0.0;
    c.ph[2] = 3715.0 / 756.0 + (55.0 / 9.0) * eta;
    c.ph[3] = -16.0 * kPi + (113.0 / 3.0) * delta * xa + (113.0 / 3.0 - (76.0 / 3.0) * eta) * xs;
    c.ph[4] = 15293365.0 / 508032.0 + (27145.0 / 504.0) * eta + (3085.0 / 72.0) * e2 + (-405.0 / 8.0 + 200.0 * eta) * xa * xa -
              (405.0 / 4.0) * delta * xa * xs + (-405.0 / 8.0 + (5.0 / 2.0) * eta) * xs * xs;
    c.ph[5] = 38645.0 * kPi / 756.0 - (65.0 * kPi / 9.0) * eta + delta * (-732985.0 / 2268.0 - (140.0 / 9.0) * eta) * xa +
              (-732985.0 / 2268.0 + (24260.0 / 81.0) * eta + (340.0 / 9.0) * e2) * xs;
    c.ph[6] = 11583231236531.0 / 4694215680.0 - 6848.0 * kEulerGamma / 21.0 - 640.0 * kPi * kPi / 3.0 +
              (-15737765635.0 / 3048192.0 + 2255.0 * kPi * kPi / 12.0) * eta + (76055.0 / 1728.0) * e2 - (127825.0 / 1296.0) * e3 +
              (2270.0 * kPi / 3.0) * delta * xa + (2270.0 * kPi / 3.0 - 520.0 * kPi * eta) * xs;
    c.ph[7] = 77096675.0 * kPi / 254016.0 + (378515.0 * kPi / 1512.0) * eta - (74045.0 * kPi / 756.0) * e2 +
              delta * (-25150083775.0 / 3048192.0 + (26804935.0 / 6048.0) * eta - (1985.0 / 48.0) * e2) * xa +
              (-25150083775.0 / 3048192.0 + (10566655595.0 / 762048.0) * eta - (1042165.0 / 3024.0) * e2 + (5345.0 / 36.0) * e3) * xs;
    // PN amplitude coefficients, premultiplied by pi^(i/3)
    {
        double a[7];
        a[0] = 1.0;
        a[1] = 0.0;
        a[2] = -323.0 / 224.0 + (451.0 / 168.0) * eta;
        a[3] = (27.0 / 8.0) * delta * xa + (27.0 / 8.0 - (11.0 / 6.0) * eta) * xs;
        a[4] = -27312085.0 / 8128512.0 - (1975055.0 / 338688.0) * eta + (105271.0 / 24192.0) * e2 + (-81.0 / 32.0 + 8.0 * eta) * xa * xa -
               (81.0 / 16.0) * delta * xa * xs + (-81.0 / 32.0 + (17.0 / 8.0) * eta) * xs * xs;
        a[5] = -85.0 * kPi / 64.0 + (85.0 * kPi / 16.0) * eta + delta * (285197.0 / 16128.0 - (1579.0 / 4032.0) * eta) * xa +
               (285197.0 / 16128.0 - (15317.0 / 672.0) * eta - (2227.0 / 1008.0) * e2) * xs;
        a[6] = -177520268561.0 / 8583708672.0 + (545384828789.0 / 5007163392.0 - 205.0 * kPi * kPi / 48.0) * eta -
               (3248849057.0 / 178827264.0) * e2 + (34473079.0 / 6386688.0) * e3 +
               (1614569.0 / 64512.0 - (1873643.0 / 16128.0) * eta + (2167.0 / 42.0) * e2) * xa * xa +
               (31.0 * kPi / 12.0 - (7.0 * kPi / 3.0) * eta) * xs +
               (1614569.0 / 64512.0 - (61391.0 / 1344.0) * eta + (57451.0 / 4032.0) * e2) * xs * xs +
               delta * xa * (31.0 * kPi / 12.0 + (1614569.0 / 32256.0 - (165961.0 / 2688.0) * eta) * xs);
        const double pi13 = cbrt(kPi);
        double pw = 1.0;
        for (int i = 0; i < 7; ++i) { c.am[i] = a[i] * pw; pw *= pi13; }
    }

    // amplitude set-up: f_peak, collocation quartic, f_ref
    c.w = g3 * c.fDM;
    c.gam1w = g1 * c.w;
    c.gam2ow = g2 / c.w;
    if (g2 >= 1.0) c.f_peak = fabs(c.fRD - c.fDM * g3 / g2);
    else c.f_peak = fabs(c.fRD + c.fDM * g3 * (sqrt(1.0 - g2 * g2) - 1.0) / g2);
    {
        const double f1 = kFAmpIns, f3 = c.f_peak, f2 = 0.5 * (f1 + f3);
        double v1, d1, v3, d3;
        amp_ins(c, f1, &v1, &d1);
        amp_mr(c, f3, &v3, &d3);
        double A[5][5] = {{1.0, f1, f1 * f1, f1 * f1 * f1, f1 * f1 * f1 * f1},
                          {1.0, f2, f2 * f2, f2 * f2 * f2, f2 * f2 * f2 * f2},
                          {1.0, f3, f3 * f3, f3 * f3 * f3, f3 * f3 * f3 * f3},
                          {0.0, 1.0, 2.0 * f1, 3.0 * f1 * f1, 4.0 * f1 * f1 * f1},
                          {0.0, 1.0, 2.0 * f3, 3.0 * f3 * f3, 4.0 * f3 * f3 * f3}};
        double b[5] = {v1, v2, v3, d1, d3};
        solve5(A, b);
        for (int i = 0; i < 5; ++i) c.dint[i] = b[i];
    }
    {
        // f_ref: root of g(f) = (5/6)/f - 2x/(x^2+w^2) - gamma2/w above f_peak (reading G4)
        // multiplied through by f (x^2 + w^2) > 0: same sign and root, no division in the iteration
        const double w = c.w, g2w = c.gam2ow, fRD = c.fRD;
        auto g = [&](double f) {
            const double xx = f - fRD;
            const double den = fma(xx, xx, w * w);
            return fma(5.0 / 6.0, den, -f * fma(g2w, den, 2.0 * xx));
        };
        double lo = c.f_peak, hi = c.fRD + 4.0 * w;
        for (int it = 0; it < 64 && g(hi) > 0.0; ++it) hi += w;
        c.f_ref = bracketed_root(g, lo, g(lo), hi, g(hi), 0.0);      // g > 0 at lo, g <= 0 at hi
    }
    // phase connections and alignment
    c.f_mr = 0.5 * c.fRD;
    {
        double pi_, dpi_, pm_, dpm_, pr_, dpr_;
        psi_ins_raw(c, kFPhiIns, &pi_, &dpi_);
        psi_int_raw(c, kFPhiIns, &pm_, &dpm_);
        c.C2i = dpi_ - dpm_;
        c.C1i = pi_ - pm_ - c.C2i * kFPhiIns;
        psi_int_raw(c, c.f_mr, &pm_, &dpm_);
        pm_ += c.C1i + c.C2i * c.f_mr;
        dpm_ += c.C2i;
        psi_mr_raw(c, c.f_mr, &pr_, &dpr_);
        c.C2m = dpm_ - dpr_;
        c.C1m = pm_ - pr_ - c.C2m * c.f_mr;
        // alignment (reading G4) from the unaligned phase, in registers: every field of the shared record is stored
        // exactly once with the same value by every lane, so no lane can observe a half-built record
        double p0, d0;
        psi22_unaligned(c, c.f_ref, &p0, &d0);
        c.pshift = p0;
        c.tshift = d0;
    }

    // extrinsic: propagation vector, polarisation tensors (O4)
    double sl, cl, sbt, cbt, s2p, c2p;
    sincos(lam, &sl, &cl);
    sincos(beta, &sbt, &cbt);
    sincos(2.0 * psi_pol, &s2p, &c2p);
    c.k[0] = -cbt * cl;
    c.k[1] = -cbt * sl;
    c.k[2] = -sbt;
    const double u[3] = {sl, -cl, 0.0};
    const double v[3] = {-sbt * cl, -sbt * sl, cbt};
    // symmetric tensors in order xx,yy,zz,xy,xz,yz
    const int ia[6] = {0, 1, 2, 0, 0, 1}, ib[6] = {0, 1, 2, 1, 2, 2};
    double Pp[6], Pc[6];
    for (int e = 0; e < 6; ++e) {
        const double ep = u[ia[e]] * u[ib[e]] - v[ia[e]] * v[ib[e]];
        const double ec = u[ia[e]] * v[ib[e]] + v[ia[e]] * u[ib[e]];
        Pp[e] = c2p * ep + s2p * ec;
        Pc[e] = -s2p * ep + c2p * ec;
    }

    const double f_i22A = kFAmpIns, f_i22P = kFPhiIns;
    double psi_i, psi_r, dtmp;
    psi22(c, f_i22P, &psi_i, &dtmp);
    psi22(c, c.fRD, &psi_r, &dtmp);
    const double ampbase = kPi * sqrt(2.0 * eta / 3.0);
    for (int mi = mode_lo; mi < mode_hi; ++mi) {
        ModeConst& mc = c.mode[mi];
        const int l = c_mode_l[mi], m = c_mode_m[mi];
        mc.fiA = 0.5 * m * f_i22A;
        mc.fiP = 0.5 * m * f_i22P;
        mc.fr = frd[mi];
        mc.aA[0] = 2.0 / m; mc.bA[0] = 0.0;
        mc.aA[1] = (c.fRD - f_i22A) / (mc.fr - mc.fiA); mc.bA[1] = f_i22A - mc.aA[1] * mc.fiA;
        mc.aA[2] = 1.0; mc.bA[2] = c.fRD - mc.fr;
        mc.aP[0] = 2.0 / m; mc.bP[0] = 0.0;
        mc.aP[1] = (c.fRD - f_i22P) / (mc.fr - mc.fiP); mc.bP[1] = f_i22P - mc.aP[1] * mc.fiP;
        mc.aP[2] = c.fDM / fdm[mi]; mc.bP[2] = c.fRD - mc.aP[2] * mc.fr;
        for (int r = 0; r < 3; ++r) mc.invaP[r] = 1.0 / mc.aP[r];
        const double dphi = T[MT_hm_22_amp + 2 * mi + 1];
        // psi22 at the map images of the boundaries (the maps are continuous: images are f_i22P and fRD)
        double pi_img, pr_img;
        psi22(c, mc.aP[0] * mc.fiP + mc.bP[0], &pi_img, &dtmp);
        psi22(c, mc.aP[1] * mc.fr + mc.bP[1], &pr_img, &dtmp);
        const double c0 = 0.0;
        const double c1 = c0 + pi_img * (mc.invaP[0] - mc.invaP[1]);
        const double c2 = c1 + pr_img * (mc.invaP[1] - mc.invaP[2]);
        mc.cP[0] = c0 - dphi;
        mc.cP[1] = c1 - dphi;
        mc.cP[2] = c2 - dphi;
        const double clm = T[MT_hm_22_amp + 2 * mi];
        double massf = 1.0;
        int vp = 0;
        if (l == 2 && m == 1) { massf = delta; vp = 1; }
        else if (l == 3 && m == 3) { massf = delta; vp = 1; }
        else if (l == 3 && m == 2) { massf = 1.0 - 3.0 * eta; vp = 2; }
        else if (l == 4 && m == 4) { massf = 1.0 - 3.0 * eta; vp = 2; }
        else if (l == 4 && m == 3) { massf = delta * (1.0 - 2.0 * eta); vp = 3; }
        mc.ampc = ampbase * fabs(clm * massf);
        mc.vpow = vp;
        // mode polarisation tensor P_lm = 1/2 Y_{l,-m}(P+ + i Px) + 1/2 (-1)^l conj(Y_lm)(P+ - i Px)
        double ct_i, st_i, ch_i, sh_i;
        sincos(inc, &st_i, &ct_i);
        sincos(0.5 * inc, &sh_i, &ch_i);
        const double ym = sYlm_theta(l, -m, ct_i, st_i, ch_i, sh_i), yp = sYlm_theta(l, m, ct_i, st_i, ch_i, sh_i);
        double sm, cm;
        sincos(m * phi_ref, &sm, &cm);
        const cplx Ym = {ym * cm, -ym * sm};                 // Y_{l,-m} = y e^{-i m phi}
        const double sgn = (l & 1) ? -1.0 : 1.0;
        const cplx Ypc = {sgn * yp * cm, -sgn * yp * sm};    // (-1)^l conj(Y_lm)
        for (int e = 0; e < 6; ++e) {
            const cplx a = cmul(Ym, {Pp[e], Pc[e]});
            const cplx b = cmul(Ypc, {Pp[e], -Pc[e]});
            mc.P[2 * e] = 0.5 * (a.re + b.re);
            mc.P[2 * e + 1] = 0.5 * (a.im + b.im);
        }
        mc.f_lo = mc.f_hi = mc.dlog = mc.inv_dlog = mc.ln_flo = 0.0;       // active was reset before the __syncwarp at the top
    }
    // bands (O5).  On the inspiral branch of the phase map t_lm(f) = t_22(2 f / m), so the
    // six roots of t_lm(f) = 0 are images of ONE root x0 of t_22 in (2,2) geometric frequency, found once.
    auto t22 = [&](double x22) {
        double p_, d_;
        psi22(c, x22, &p_, &d_);
        return c.t_coal + c.M_s * d_ * (1.0 / kTwoPi);
    };
    const double t_top = t22(kFPhiIns);                 // t_lm at the end of every mode's inspiral branch
    double x0 = -1.0;
    for (int mi = mode_lo; mi < mode_hi; ++mi) {
        if (!((mode_mask >> mi) & 1u)) continue;
        ModeConst& mc = c.mode[mi];
        const int m = c_mode_m[mi];
        const double f_top = 0.5 * m * kFPhiIns / c.M_s;
        const double f_hi = fmin(f_max, 0.2 * fmax(1.0, 0.5 * m) / c.M_s);
        double f_lo;
        const double t_min = t_of_f(c, mi, f_min);
        if (t_min >= 0.0) {
            f_lo = f_min;
        } else if (f_top <= f_min || t_top < 0.0) {
            f_lo = fmax(f_top, f_min);
        } else {
            if (x0 < 0.0) {
                // the time to coalescence tau = t_coal - t_22 falls off like x^(-8/3) (P6), so tau^(-3/8) is nearly
                // linear in x: the secant steps run on g(x) = tau(x)^(-3/8) - t_coal^(-3/8), which has the sign of t_22
                const double xa = mc.aP[0] * (f_min * c.M_s);        // t22(xa) = t_min < 0 <= t_top
                auto p38 = [](double tau) { return exp(-0.375 * log(tau)); };     // tau^(-3/8); only the sign and zero of g matter
                const double g0 = p38(c.t_coal);
                auto g = [&](double x22) {
                    const double tau = c.t_coal - t22(x22);
                    return (tau > 0.0) ? p38(tau) - g0 : 1e300;
                };
                const double ga = p38(c.t_coal - t_min) - g0;
                const double gb = (c.t_coal - t_top > 0.0) ? p38(c.t_coal - t_top) - g0 : 1e300;
                x0 = bracketed_root(g, xa, ga, kFPhiIns, gb, 4e-16 * g0);
            }
            f_lo = fmax(f_min, x0 * (0.5 * m) / c.M_s);
        }
        if (f_hi > f_lo) {
            mc.active = 1;
            mc.f_lo = f_lo;
            mc.f_hi = f_hi;
            const double lg = log(f_hi / f_lo);
            mc.dlog = lg / (S - 1);
            mc.inv_dlog = (S - 1) / lg;
            mc.ln_flo = log(f_lo);
        }
    }
}

}  // namespace mbhl
