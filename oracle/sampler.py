"""Oracle for the sampler-side steps next to the likelihood (section II.B).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Plain numpy restatement, step by step, of

  - the sampler's coordinates and prior box (PAPER.md:67-81 Table I, :559): walkers live in
    theta = (ln M_T, q, a1, a2, ln D_L, phi_ref, cos iota, lambda, sin beta, psi, ln t_ref),
    every component uniform between the bounds of Table I;
  - the affine-invariant stretch move (eqs. 14-16, a = 1.15 :222);
  - the temperature swap of parallel tempering (eq. 17).

Random numbers are the method's inputs: both this oracle and the CUDA library draw them from the
counter-based generator Philox4x32-10 (Salmon et al. 2011), each with its own implementation, keyed by
(seed, step, stream) and counted by walker, so the two sides see the same uniforms.

Pins (tests/test_oracle_sampler.py): Table I bounds against the values PAPER.md prints; unpack is the inverse
of the transforms the workload generator applies; Philox against the known-answer vectors of its paper
(counter = key = 0 and counter = key = 0xffffffff); the stretch proposal's z distribution against the closed
form CDF of g(z) ~ 1/sqrt(z) on [1/a, a]; detailed balance of the stretch move and of the swap on a
Gaussian target (sample mean / variance of a long chain).
"""
import math

import numpy as np

# Table I: lower and upper bound of every sampled coordinate
PRIOR_LO = np.array([math.log(1e3), 0.05, -0.99, -0.99, math.log(0.044), 0.0, -1.0, 0.0, -1.0, 0.0, math.log(1.0)])
PRIOR_HI = np.array([math.log(1e9), 1.0, 0.99, 0.99, math.log(1298.00), 2.0 * math.pi, 1.0, 2.0 * math.pi, 1.0, math.pi,
                     math.log(3.15576e8)])
NDIM = 11
STRETCH_A = 1.15


def in_prior(theta):
    """True where every coordinate lies inside the box of Table I (uniform prior: the log prior is a constant there)."""
    theta = np.asarray(theta, dtype=np.float64)
    return np.all(np.isfinite(theta) & (theta >= PRIOR_LO) & (theta <= PRIOR_HI), axis=-1)


def unpack_sampled(theta):
    """theta [.., 11] (sampler coordinates) -> physical parameters in the order of PAPER.md:65."""
    theta = np.asarray(theta, dtype=np.float64)
    p = np.array(theta, dtype=np.float64, copy=True)
    p[..., 0] = np.exp(theta[..., 0])
    p[..., 4] = np.exp(theta[..., 4])
    p[..., 6] = np.arccos(theta[..., 6])
    p[..., 8] = np.arcsin(theta[..., 8])
    p[..., 10] = np.exp(theta[..., 10])
    return p


# ---------------------------------------------------------------------------------------------
# Philox4x32-10: counter (4 x uint32), key (2 x uint32) -> 4 x uint32
# ---------------------------------------------------------------------------------------------
_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = 0x9E3779B9, 0xBB67AE85


def philox4x32(counter, key):
    """counter [.., 4] uint32, key [.., 2] uint32 (broadcastable) -> [.., 4] uint32, ten rounds."""
    c = np.array(np.broadcast_to(np.asarray(counter, dtype=np.uint32), np.broadcast_shapes(np.shape(counter), np.shape(key)[:-1] + (4,))),
                 dtype=np.uint32)
    k = np.asarray(key, dtype=np.uint32)
    k0 = np.broadcast_to(k[..., 0], c.shape[:-1]).astype(np.uint64)
    k1 = np.broadcast_to(k[..., 1], c.shape[:-1]).astype(np.uint64)
    c0, c1, c2, c3 = (c[..., i].astype(np.uint64) for i in range(4))
    mask = np.uint64(0xFFFFFFFF)
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & mask
        hi1, lo1 = p1 >> np.uint64(32), p1 & mask
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0) & mask, lo1, (hi0 ^ c3 ^ k1) & mask, lo0
        k0 = (k0 + np.uint64(_W0)) & mask
        k1 = (k1 + np.uint64(_W1)) & mask
    return np.stack([c0, c1, c2, c3], axis=-1).astype(np.uint32)


def uniforms(seed, step, stream, index):
    """Two uniforms in (0, 1) per index: counter = (index, step, stream, 0), key = (seed lo, seed hi); each from 52 random bits."""
    index = np.asarray(index, dtype=np.uint32)
    ctr = np.stack([index, np.full_like(index, step), np.full_like(index, stream), np.zeros_like(index)], axis=-1)
    key = np.array([seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF], dtype=np.uint32)
    r = philox4x32(ctr, key).astype(np.uint64)
    u0 = ((r[..., 0] << np.uint64(20)) | (r[..., 1] >> np.uint64(12))).astype(np.float64)
    u1 = ((r[..., 2] << np.uint64(20)) | (r[..., 3] >> np.uint64(12))).astype(np.float64)
    return (u0 + 0.5) * 2.0 ** -52, (u1 + 0.5) * 2.0 ** -52


# ---------------------------------------------------------------------------------------------
# stretch move and temperature swap
# ---------------------------------------------------------------------------------------------
def stretch_z(u, a=STRETCH_A):
    """z with density g(z) ~ 1/sqrt(z) on [1/a, a] (eq. 15) from a uniform u by inverting the CDF."""
    return ((a - 1.0) * u + 1.0) ** 2 / a


def stretch_propose(x_active, x_partner, z):
    """eq. 14: Y = X_j + z (X_k - X_j), X_k the walker being moved, X_j its partner from the other half."""
    return x_partner + z[..., None] * (x_active - x_partner)


def stretch_log_accept(z, logp_new, logp_old, ndim=NDIM):
    """ln of eq. 16: z^(D-1) p(Y)/p(X); the move is accepted when ln u < this."""
    return (ndim - 1) * np.log(z) + logp_new - logp_old


def swap_log_accept(beta_i, beta_j, logl_i, logl_j):
    """ln of eq. 17: [L(x_i)/L(x_j)]^(beta_j - beta_i) for adjacent rungs i, j."""
    return (beta_j - beta_i) * (logl_i - logl_j)


def stretch_half_step(theta, logl, betas, half, seed, step, loglike_fn):
    """One half of an ensemble update at every temperature.

    theta [T, K, 11] walker coordinates, logl [T, K] their log-likelihoods, betas [T] inverse temperatures
    (the last may be 0: T_max = infinity).  Walkers k with k % 2 == half move, each with a partner
    drawn from the other half of the same temperature.  loglike_fn(theta[M, 11]) -> logL[M].  The tempered
    density is prior x L^beta; the prior is uniform on the box of Table I, so a proposal outside
    the box is rejected.  Returns the updated (theta, logl, accepted[T, K]).
    """
    T, K, D = theta.shape
    act = np.arange(half, K, 2)
    oth = np.arange(1 - half, K, 2)
    idx = (np.arange(T)[:, None] * K + act[None, :]).astype(np.uint32)          # global walker index
    u_z, u_j = uniforms(seed, step, 0, idx)
    u_acc, _ = uniforms(seed, step, 1, idx)
    z = stretch_z(u_z)
    j = oth[np.minimum((u_j * oth.size).astype(np.int64), oth.size - 1)]
    x_act = theta[:, act, :]
    x_par = np.take_along_axis(theta, j[:, :, None].repeat(D, axis=2), axis=1)
    y = stretch_propose(x_act, x_par, z)
    ok = in_prior(y)
    logl_new = np.full((T, act.size), -np.inf)
    if ok.any():
        logl_new[ok] = loglike_fn(y[ok])
    lnr = stretch_log_accept(z, betas[:, None] * logl_new, betas[:, None] * logl[:, act])
    lnr = np.where(ok & np.isfinite(logl_new), lnr, -np.inf)
    acc = np.log(u_acc) < lnr
    theta = theta.copy()
    logl = logl.copy()
    theta[:, act, :] = np.where(acc[:, :, None], y, x_act)
    logl[:, act] = np.where(acc, logl_new, logl[:, act])
    accepted = np.zeros((T, K), dtype=bool)
    accepted[:, act] = acc
    return theta, logl, accepted


def swap_step(theta, logl, betas, seed, step):
    """Temperature swaps (eq. 17): from the hottest pair down, walker k of rung i and walker k of rung i-1 exchange
    positions with probability min(1, exp((beta_{i-1} - beta_i)(logL_i - logL_{i-1}))).  Returns (theta, logl, swapped[T-1, K])."""
    T, K, _ = theta.shape
    theta = theta.copy()
    logl = logl.copy()
    swapped = np.zeros((T - 1, K), dtype=bool)
    for i in range(T - 1, 0, -1):
        idx = (np.uint32(i) * np.uint32(K) + np.arange(K, dtype=np.uint32))
        u, _ = uniforms(seed, step, 2, idx)
        lnr = swap_log_accept(betas[i], betas[i - 1], logl[i], logl[i - 1])
        do = np.log(u) < lnr
        ti, tl = theta[i].copy(), logl[i].copy()
        theta[i] = np.where(do[:, None], theta[i - 1], theta[i])
        logl[i] = np.where(do, logl[i - 1], logl[i])
        theta[i - 1] = np.where(do[:, None], ti, theta[i - 1])
        logl[i - 1] = np.where(do, tl, logl[i - 1])
        swapped[i - 1] = do
    return theta, logl, swapped


def ladder(n_temps=10, base=2.04807, t_max_inf=True):
    """Geometric temperature ladder of ptemcee: T_i = base^i, last rung at infinite temperature."""
    betas = base ** -np.arange(n_temps, dtype=np.float64)
    if t_max_inf:
        betas[-1] = 0.0
    return betas


def noise_aet(psd, df, seed):
    """Frequency-domain noise realisation for the three TDI channels (eq. 12; reading G5 of DESIGN.md).

    psd [3, N] one-sided PSD.  The paper draws a modulus N(0, 1/(2 sqrt(df))) sqrt(S_n) and a uniform phase; a normal
    draw used as a modulus is ambiguous (G5), so this is the standard circular complex Gaussian it approximates:
    Re and Im independent N(0, S_n / (4 df)), i.e. a Rayleigh modulus sqrt(S_n/(4 df)) sqrt(-2 ln u0) with the
    uniform phase 2 pi u1 (Box-Muller).  The uniforms come from Philox with counter (bin, channel, stream 3, 0)
    and key = seed.  Bins with S_n <= 0 or not finite get 0.  Returns complex128 [3, N].
    """
    psd = np.asarray(psd, dtype=np.float64)
    C, N = psd.shape
    out = np.zeros((C, N), dtype=np.complex128)
    key = np.array([seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF], dtype=np.uint32)
    k = np.arange(N, dtype=np.uint32)
    for c in range(C):
        ctr = np.stack([k, np.full_like(k, c), np.full_like(k, 3), np.zeros_like(k)], axis=-1)
        r = philox4x32(ctr, key).astype(np.uint64)
        u0 = (((r[:, 0] << np.uint64(20)) | (r[:, 1] >> np.uint64(12))).astype(np.float64) + 0.5) * 2.0 ** -52
        u1 = (((r[:, 2] << np.uint64(20)) | (r[:, 3] >> np.uint64(12))).astype(np.float64) + 0.5) * 2.0 ** -52
        ok = np.isfinite(psd[c]) & (psd[c] > 0.0)
        sig = np.sqrt(np.where(ok, psd[c], 0.0) / (4.0 * df))
        mod = sig * np.sqrt(-2.0 * np.log(u0))
        ang = 2.0 * math.pi * u1
        out[c] = mod * np.cos(ang) + 1j * mod * np.sin(ang)
    return out


# ---------------------------------------------------------------------------------------------
# LISA-frame sampling coordinates ("sampled in the LISA frame and then converted to the SSB frame
# before waveform generation"; :222 "8 sky location posterior modes in the LISA reference frame").  The paper
# cites Marsat et al. [40] for the formulas and prints none: DESIGN.md section 4 reading G20 fixes them from
# the orbit of O4 (oracle/response.py orbit()).
# ---------------------------------------------------------------------------------------------
def lisa_frame(alpha):
    """The 3x3 matrix R whose columns are the LISA-frame basis vectors x_L, y_L, z_L in SSB components (v_SSB = R v_L):
    R = R_z(alpha) R_y(-pi/3) R_z(-alpha), alpha = Omega_0 t the orbital phase of the constellation
    centre.  z_L is the normal of the constellation plane (60 degrees from the ecliptic pole, precessing once per
    year) and the frame also carries the cartwheel rotation: in it the three spacecraft of the O4 orbit sit at the
    fixed positions (L/sqrt 3)(cos phi_n, sin phi_n, 0), phi_n = pi, -pi/3, +pi/3 (pinned in tests)."""
    ca, sa = math.cos(alpha), math.sin(alpha)
    rz = np.array([[ca, -sa, 0.0], [sa, ca, 0.0], [0.0, 0.0, 1.0]])
    ct, st = 0.5, -math.sqrt(3.0) / 2.0                  # cos, sin of -pi/3
    ry = np.array([[ct, 0.0, st], [0.0, 1.0, 0.0], [-st, 0.0, ct]])
    return rz @ ry @ rz.T


def _sky_basis(lam, beta):
    """n (towards the source), u, v of oracle/response.source_frame for sky angles (lam, beta) in any frame."""
    cl, sl, cb, sb = math.cos(lam), math.sin(lam), math.cos(beta), math.sin(beta)
    return np.array([cb * cl, cb * sl, sb]), np.array([sl, -cl, 0.0]), np.array([-sb * cl, -sb * sl, cb])


def lisa_to_ssb(t_L, lam_L, beta_L, psi_L, t0=0.0):
    """(t_L, lambda_L, beta_L, psi_L) -> (t_ref, lambda, beta, psi) in the SSB frame (reading G20).

    The frame is taken at the orbital phase alpha = Omega_0 (t0 + t_L) of the LISA-frame time itself, which makes the
    map explicit.  Sky direction and polarisation basis are rotated as vectors (the wave is the same physical
    tensor in both frames); t_L is the arrival time of the wavefront at the constellation centre,
    t_L = t_ref + k.p_0/c with k = -n the propagation vector (a delay tau multiplies by exp(-2 pi i f tau), O0)."""
    from .constants import AU_S, YEAR_SIDEREAL_S
    alpha = 2.0 * math.pi / YEAR_SIDEREAL_S * (t0 + t_L)
    R = lisa_frame(alpha)
    n_L, u_L, v_L = _sky_basis(lam_L, beta_L)
    n = R @ n_L
    beta = math.asin(max(-1.0, min(1.0, n[2])))
    lam = math.atan2(n[1], n[0]) % (2.0 * math.pi)
    _, u, v = _sky_basis(lam, beta)
    u_rot = R @ u_L
    delta = math.atan2(float(u_rot @ v), float(u_rot @ u))
    psi = (psi_L + delta) % math.pi
    p0 = AU_S * np.array([math.cos(alpha), math.sin(alpha), 0.0])
    t_ref = t_L + float(n @ p0)                          # t_L - k.p_0/c
    return t_ref, lam, beta, psi


def ssb_to_lisa(t_ref, lam, beta, psi, t0=0.0):
    """Inverse of lisa_to_ssb: the orbital phase depends on t_L itself, so t_L is found by fixed-point iteration
    (contraction factor Omega_0 R/c = 1e-4)."""
    from .constants import AU_S, YEAR_SIDEREAL_S
    n, u, v = _sky_basis(lam, beta)
    t_L = t_ref
    for _ in range(60):
        alpha = 2.0 * math.pi / YEAR_SIDEREAL_S * (t0 + t_L)
        p0 = AU_S * np.array([math.cos(alpha), math.sin(alpha), 0.0])
        t_new = t_ref - float(n @ p0)
        if t_new == t_L:
            break
        t_L = t_new
    alpha = 2.0 * math.pi / YEAR_SIDEREAL_S * (t0 + t_L)
    R = lisa_frame(alpha)
    n_L = R.T @ n
    beta_L = math.asin(max(-1.0, min(1.0, n_L[2])))
    lam_L = math.atan2(n_L[1], n_L[0]) % (2.0 * math.pi)
    _, u_L, v_L = _sky_basis(lam_L, beta_L)
    u_rot = R.T @ u
    delta = math.atan2(float(u_rot @ v_L), float(u_rot @ u_L))
    return t_L, lam_L, beta_L, (psi + delta) % math.pi


def unpack_sampled_lisa(theta, t0=0.0):
    """theta [.., 11] = (ln M_T, q, a1, a2, ln D_L, phi_ref, cos iota, lambda_L, sin beta_L, psi_L, ln t_L) with the
    sky, polarisation and time coordinates in the LISA frame -> physical SSB parameters."""
    theta = np.asarray(theta, dtype=np.float64)
    p = unpack_sampled(theta)
    flat = p.reshape(-1, NDIM)
    for row in flat:
        if np.all(np.isfinite(row)):
            row[10], row[7], row[8], row[9] = lisa_to_ssb(row[10], row[7], row[8], row[9], t0)
    return flat.reshape(p.shape)
