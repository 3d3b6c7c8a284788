"""Seeded synthetic inputs shaped like the paper's workloads.

Holds NONE of the method's arithmetic: grids, prior draws, the analytic SciRD
A/E/T noise PSD, Gaussian noise and a flat-LCDM luminosity distance.  Injections
are produced by a caller-supplied template function (tests pass the oracle's,
bench.py passes the library's own mbhl_template), so this module imports neither.

The paper measures on its own fabricated injections with the LDC "tdi" PSD
package (not available offline); these inputs stand in for them.
"""
import math

import numpy as np

C_SI = 299792458.0
ARM_S = 2.5e9 / C_SI
YEAR_JULIAN_S = 31557600.0
SEED0 = 200501827
PARAM_NAMES = ("M_T", "q", "a1", "a2", "D_L", "phi_ref", "inc", "lam", "beta", "psi", "t_ref")


def lum_dist_gpc(z, H0=67.7, Om=0.31, n=4096):
    """Flat-LCDM luminosity distance in Gpc (composite Simpson); pinned to PAPER.md Tables I-II (P17)."""
    zz = np.linspace(0.0, z, 2 * n + 1)
    y = 1.0 / np.sqrt(Om * (1.0 + zz) ** 3 + 1.0 - Om)
    h = zz[1] - zz[0]
    integral = h / 3.0 * (y[0] + y[-1] + 4.0 * y[1:-1:2].sum() + 2.0 * y[2:-1:2].sum())
    return (1.0 + z) * (C_SI / 1000.0 / H0) * integral / 1000.0      # Mpc -> Gpc


def scird_psd_aet(f):
    """Analytic SciRD noise PSD of TDI A, E, T (first generation, fractional-frequency units); no Galactic term."""
    f = np.asarray(f, dtype=np.float64)
    x = 2.0 * math.pi * f * ARM_S
    s_oms = (15.0e-12) ** 2 * (1.0 + (2.0e-3 / f) ** 4) * (2.0 * math.pi * f / C_SI) ** 2
    s_acc = (3.0e-15) ** 2 * (1.0 + (0.4e-3 / f) ** 2) * (1.0 + (f / 8.0e-3) ** 4) / (2.0 * math.pi * f * C_SI) ** 2
    sx2 = np.sin(x) ** 2
    s_ae = 8.0 * sx2 * (2.0 * s_acc * (3.0 + 2.0 * np.cos(x) + np.cos(2.0 * x)) + s_oms * (2.0 + np.cos(x)))
    s_t = 16.0 * s_oms * (1.0 - np.cos(x)) * sx2 + 128.0 * s_acc * sx2 * np.sin(0.5 * x) ** 4
    return np.stack([s_ae, s_ae, s_t])


def grid(T_obs_yr, n_bins, f_start):
    """Uniform Fourier grid f_k = (k0 + k)/T_obs, k0 = ceil(f_start T_obs) (at least 1)."""
    df = 1.0 / (T_obs_yr * YEAR_JULIAN_S)
    k0 = max(1, int(math.ceil(f_start / df)))
    return (k0 + np.arange(n_bins, dtype=np.float64)) * df


def draw_prior(rng, M_T, T_obs_s, q_range=(1.0, 5.0), z_range=(1.0, 4.0), M_log_range=None):
    """One parameter set in the order of PAPER.md:65 with the prior shapes of Table I / BASELINE config 0."""
    if M_log_range is not None:
        M_T = 10.0 ** rng.uniform(math.log10(M_log_range[0]), math.log10(M_log_range[1]))
    q = rng.uniform(*q_range)
    a1 = rng.uniform(-0.99, 0.99)
    a2 = rng.uniform(-0.99, 0.99)
    z = rng.uniform(*z_range)
    D_L = lum_dist_gpc(z, n=256)
    phi_ref = rng.uniform(0.0, 2.0 * math.pi)
    inc = math.acos(rng.uniform(-1.0, 1.0))
    lam = rng.uniform(0.0, 2.0 * math.pi)
    beta = math.asin(rng.uniform(-1.0, 1.0))
    psi = rng.uniform(0.0, math.pi)
    t_ref = rng.uniform(0.05, 0.95) * T_obs_s
    return np.array([M_T, q, a1, a2, D_L, phi_ref, inc, lam, beta, psi, t_ref])


def perturb(rng, p, n, width=1e-3):
    """n walkers around p: relative Gaussian for M_T, q, D_L, t_ref; absolute for spins and angles."""
    out = np.tile(p, (n, 1))
    g = rng.standard_normal((n, 11)) * width
    rel = [0, 1, 4, 10]
    ab = [2, 3, 5, 6, 7, 8, 9]
    out[:, rel] *= 1.0 + g[:, rel]
    out[:, ab] += g[:, ab]
    out[:, 2:4] = np.clip(out[:, 2:4], -0.99, 0.99)
    return out


def noise(rng, psd, df):
    """Complex Gaussian noise, Re and Im ~ N(0, S_n/(4 df)) per bin (reading G5 of eq. 12)."""
    sig = np.sqrt(psd / (4.0 * df))
    return sig * (rng.standard_normal(psd.shape) + 1j * rng.standard_normal(psd.shape))


def build(config, template_fn, n_bins=None, batch=None, with_noise=True):
    """Builds BASELINE.json config 0, 1 or 2 (optionally shrunk with n_bins/batch for tests).

    template_fn(params[11], freqs[N], S) -> complex128 [3, N] produces the injections.
    Returns dict(freqs, data, psd, params, S, t0, injections).
    """
    rng = np.random.default_rng(SEED0 + config)
    if config == 0:
        T, N, f0, S, B = 0.1, 1 << 16, 1e-4, 256, 4
    elif config == 1:
        T, N, f0, S, B = 1.0, 1 << 20, 1e-5, 512, 64
    elif config == 2:
        T, f0, S, B = 1.33, 0.0, 1024, 1024
        N = int(math.floor(0.1 * T * YEAR_JULIAN_S))
    else:
        raise ValueError("config must be 0, 1 or 2")
    if n_bins is not None:
        N = n_bins
    if batch is not None:
        B = batch
    T_s = T * YEAR_JULIAN_S
    freqs = grid(T, N, f0)
    df = 1.0 / T_s
    psd = scird_psd_aet(freqs)
    if config == 0:
        params = np.stack([draw_prior(rng, 1e6, T_s) for _ in range(B)])
        injections = params[:1].copy()
    elif config == 1:
        inj = draw_prior(rng, 1e6, T_s)
        inj[:5] = [1e6, 3.0, 0.6, -0.3, lum_dist_gpc(2.0)]
        inj[10] = 0.95 * T_s
        injections = inj[None, :]
        params = perturb(rng, inj, B)
    else:
        injections = []
        for (M, q, z) in ((1e5, 1.5, 1.0), (1e6, 5.0, 3.0), (1e8, 10.0, 8.0)):
            inj = draw_prior(rng, M, T_s)
            inj[0], inj[1], inj[4], inj[10] = M, q, lum_dist_gpc(z), 0.95 * T_s
            injections.append(inj)
        injections = np.stack(injections)
        counts = [B - 2 * (B // 3), B // 3, B // 3]
        params = np.concatenate([perturb(rng, injections[i], counts[i]) for i in range(3)])
    data = np.zeros((3, N), dtype=np.complex128)
    for inj in injections:
        data += np.asarray(template_fn(inj, freqs, S))
    if with_noise:
        data += noise(rng, psd, df)
    return dict(freqs=freqs, data=data, psd=psd, params=params, S=S, t0=0.0, injections=injections,
                T_obs_yr=T, config=config)


def sparse_batch(batch=16384, seed_offset=3):
    """BASELINE.json config 3: parameter sets from the config-0 priors with M_T log-uniform [1e5, 1e8]."""
    rng = np.random.default_rng(SEED0 + seed_offset)
    T_s = 1.33 * YEAR_JULIAN_S
    return np.stack([draw_prior(rng, None, T_s, M_log_range=(1e5, 1e8)) for _ in range(batch)])


def het_edges(freqs, n_coarse, f_lo=None, f_hi=None):
    """Coarse-bin edges (bin indices, first 0, last N, strictly increasing) for the heterodyned likelihood variant
    (row (f).4).  An INPUT of that variant, shared by the oracle and the library: half of the
    n_coarse bins are log-spaced in frequency between f_lo and f_hi (the band the caller expects the signal in, e.g. the
    first and last knot of the reference's (2,2) mode; default: the whole grid) - the envelope evolves on the scale of
    f itself at the low end of a band -, the other half uniform in frequency (the time-shift term of the phase)."""
    f = np.asarray(freqs, dtype=np.float64)
    N = f.size
    f_lo = f[0] if f_lo is None else max(f[0], float(f_lo))
    f_hi = f[-1] if f_hi is None else min(f[-1], float(f_hi))
    n1 = max(1, n_coarse // 2)
    n2 = max(1, n_coarse - n1)
    e_log = np.searchsorted(f, f_lo * (f_hi / f_lo) ** (np.arange(n1 + 1) / float(n1)), side="left")
    e_lin = np.searchsorted(f, f[0] + (f[-1] - f[0]) * np.arange(1, n2) / float(n2), side="left")
    e = np.unique(np.concatenate([[0], e_log, e_lin, [N]]))
    return e[(e >= 0) & (e <= N)].astype(np.int64)
