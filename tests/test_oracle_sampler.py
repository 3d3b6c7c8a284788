"""Pins of oracle/sampler.py and of the per-mode products: Table I, Philox known answers, the
stretch proposal's distribution, detailed balance on a Gaussian target, linearity of <d|h> over the modes."""
import math
import os

import numpy as np

from oracle import likelihood as L
from oracle import sampler as S
from paper_2005_01827_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_tables.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def test_prior_box_is_table_one():
    g = golden()
    lo, hi = S.PRIOR_LO, S.PRIOR_HI
    assert abs(math.exp(lo[0]) / g["prior_MT_lo"] - 1) < 1e-14
    assert abs(math.exp(hi[0]) / g["prior_MT_hi"] - 1) < 1e-14
    assert (lo[1], hi[1]) == (g["prior_q_lo"], g["prior_q_hi"])
    assert (lo[2], hi[2], lo[3], hi[3]) == (g["prior_a_lo"], g["prior_a_hi"], g["prior_a_lo"], g["prior_a_hi"])
    assert abs(math.exp(lo[4]) / g["DL_z0.01"] - 1) < 1e-14 and abs(math.exp(hi[4]) / g["DL_z100"] - 1) < 1e-14
    assert (lo[5], lo[7], lo[9]) == (0.0, 0.0, 0.0) and hi[5] == hi[7] == 2 * math.pi and hi[9] == math.pi
    assert (lo[6], hi[6], lo[8], hi[8]) == (-1.0, 1.0, -1.0, 1.0)
    assert abs(math.exp(lo[10]) / g["prior_tref_lo"] - 1) < 1e-14 and abs(math.exp(hi[10]) / g["prior_tref_hi"] - 1) < 1e-14
    assert S.STRETCH_A == g["stretch_a"]


def test_unpack_sampled_inverts_the_generator_transforms():
    rng = np.random.default_rng(3)
    p = np.stack([W.draw_prior(rng, 1e6, 3e7, q_range=(0.05, 1.0)) for _ in range(50)])
    theta = p.copy()
    theta[:, 0], theta[:, 4], theta[:, 10] = np.log(p[:, 0]), np.log(p[:, 4]), np.log(p[:, 10])
    theta[:, 6], theta[:, 8] = np.cos(p[:, 6]), np.sin(p[:, 8])
    assert np.all(S.in_prior(theta))
    back = S.unpack_sampled(theta)
    assert np.max(np.abs(back / p - 1.0)) < 1e-13
    bad = theta[:3].copy()
    bad[0, 1] = 1.2
    bad[1, 6] = -1.0000001
    bad[2, 10] = np.nan
    assert not S.in_prior(bad).any()


def test_philox_known_answers():
    # Random123 known-answer vectors of philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11)
    kat = [((0, 0, 0, 0), (0, 0), (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
           ((0xffffffff,) * 4, (0xffffffff,) * 2, (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
           ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0), (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1))]
    for ctr, key, want in kat:
        got = S.philox4x32(np.array(ctr, dtype=np.uint32), np.array(key, dtype=np.uint32))
        assert tuple(int(x) for x in got) == want
    u0, u1 = S.uniforms(12345, 7, 1, np.arange(100000))
    assert 0.0 < u0.min() and u0.max() < 1.0 and abs(u0.mean() - 0.5) < 5e-3 and abs(np.corrcoef(u0, u1)[0, 1]) < 1e-2


def test_stretch_z_has_the_density_of_eq_15():
    a = S.STRETCH_A
    u = np.linspace(0.0, 1.0, 1001)
    z = S.stretch_z(u)
    assert z[0] == 1.0 / a and abs(z[-1] - a) < 1e-15
    cdf = (np.sqrt(z) - 1.0 / math.sqrt(a)) / (math.sqrt(a) - 1.0 / math.sqrt(a))      # integral of z^(-1/2) normalised on [1/a, a]
    assert np.max(np.abs(cdf - u)) < 1e-14


def test_stretch_move_and_swaps_sample_a_tempered_gaussian():
    # detailed balance (eqs. 16, 17): a Gaussian likelihood inside the box must come out with variance sigma^2 / beta
    mu = 0.5 * (S.PRIOR_LO + S.PRIOR_HI)
    sig = 0.01 * (S.PRIOR_HI - S.PRIOR_LO)
    fn = lambda th: -0.5 * np.sum(((th - mu) / sig) ** 2, axis=-1)
    betas = np.array([1.0, 0.5, 0.25])
    T, K = 3, 48
    rng = np.random.default_rng(11)
    theta = mu + sig * rng.standard_normal((T, K, 11)) / np.sqrt(betas)[:, None, None]
    logl = fn(theta)
    acc, samples = [], []
    for step in range(1500):
        for half in (0, 1):
            theta, logl, a = S.stretch_half_step(theta, logl, betas, half, seed=99, step=2 * step + half, loglike_fn=fn)
            acc.append(a.mean() * 2)
        theta, logl, _ = S.swap_step(theta, logl, betas, seed=99, step=step)
        if step >= 300:
            samples.append(theta.copy())
    assert np.allclose(logl, fn(theta), rtol=0, atol=1e-9)                      # bookkeeping of logl through moves and swaps
    s = np.stack(samples)                                                        # [steps, T, K, 11]
    for t in range(T):
        x = (s[:, t] - mu) / sig
        assert np.max(np.abs(x.mean(axis=(0, 1)))) < 0.15 / math.sqrt(betas[t])
        ratio = x.var(axis=(0, 1)) * betas[t]
        assert np.all(np.abs(ratio - 1.0) < 0.15), (t, ratio)
    assert 0.2 < np.mean(acc) < 0.95


def test_mode_products_are_linear_in_the_modes(table):
    tf = lambda p, f, Sp: L.template(table, p, f, Sp)
    wl = W.build(0, tf, n_bins=4096, batch=2)
    p = wl["params"][1]
    dh, hh = L.mode_products(table, p, wl["freqs"], wl["data"], wl["psd"], wl["S"])
    tdh, thh, _ = L.loglike_parts(table, p, wl["freqs"], wl["data"], wl["psd"], wl["S"])
    assert abs(dh.sum() - tdh) <= 1e-12 * (np.abs(dh).sum() + abs(tdh))        # <d|h> is linear in h
    assert np.all(hh >= 0.0) and hh[0] == hh.max()                               # (2,2) dominates
    assert thh <= np.sum(np.sqrt(hh)) ** 2 * (1 + 1e-12)                         # triangle inequality
    assert abs(thh - hh.sum()) > 1e-6 * thh                                      # modes mix


def test_noise_realisation_has_the_psd_it_was_drawn_from():
    # eq. 12 / reading G5: E[4 df |n|^2 / S_n] = 2 per bin, Re and Im independent N(0, S_n/(4 df)), channels independent
    N, df = 200000, 3.0e-8
    f = (1.0 + np.arange(N)) * df * 50.0
    psd = W.scird_psd_aet(f)
    psd[1, 10] = 0.0
    psd[2, 11] = np.nan
    n = S.noise_aet(psd, df, seed=77)
    assert n[1, 10] == 0.0 and n[2, 11] == 0.0 and np.all(np.isfinite(n.view(np.float64)))
    good = np.isfinite(psd) & (psd > 0.0)
    z = np.where(good, n / np.sqrt(np.where(good, psd, 1.0) / (4.0 * df)), 0.0)      # unit-variance Re and Im
    for c in range(3):
        zc = z[c][good[c]]
        assert abs(zc.real.mean()) < 0.01 and abs(zc.imag.mean()) < 0.01
        assert abs(zc.real.var() - 1.0) < 0.015 and abs(zc.imag.var() - 1.0) < 0.015
        assert abs(np.mean(zc.real * zc.imag)) < 0.01
        assert abs(np.mean(np.abs(zc) ** 2) - 2.0) < 0.02                              # 4 df |n|^2 / S_n averages 2
        assert abs(np.mean(np.abs(zc) ** 4) - 8.0) < 0.3                               # Rayleigh modulus: E r^4 = 8
    assert abs(np.mean(z[0] * np.conj(z[1]))) < 0.01 and abs(np.mean(z[0] * np.conj(z[2]))) < 0.01
    # reproducible, and a different seed gives a different stream
    assert np.array_equal(n, S.noise_aet(psd, df, seed=77)) and not np.array_equal(n, S.noise_aet(psd, df, seed=78))


# ---------------------------------------------------------------------------------------------
# LISA-frame coordinates (reading G20)
# ---------------------------------------------------------------------------------------------
def test_lisa_frame_is_the_constellation_frame_of_the_orbit():
    # in the frame R(alpha) the spacecraft of the O4 orbit are at rest in the plane z_L = 0, at radius L/sqrt(3) and
    # angles pi, -pi/3, +pi/3; a wrong tilt sign, a missing cartwheel rotation or a wrong phase fails this
    from oracle import response
    from oracle.constants import ARM_S
    for t in (0.0, 1.1e6, 9.7e6, 2.9e7, 5.5e7):
        _, pL = response.orbit(np.float64(t))
        R = S.lisa_frame(response.OMEGA0 * t)
        assert np.max(np.abs(R @ R.T - np.eye(3))) < 1e-15 and abs(np.linalg.det(R) - 1.0) < 1e-15
        assert abs(R[2, 2] - 0.5) < 1e-15                                   # plane inclined by 60 degrees
        for n, phi in ((1, math.pi), (2, -math.pi / 3.0), (3, math.pi / 3.0)):
            q = R.T @ pL[n]
            want = ARM_S / math.sqrt(3.0) * np.array([math.cos(phi), math.sin(phi), 0.0])
            assert np.max(np.abs(q - want)) < 1e-13 * ARM_S, (t, n, q / ARM_S)


def test_lisa_to_ssb_rotates_the_wave_tensor_and_round_trips():
    from oracle import response
    from oracle.constants import AU_S
    rng = np.random.default_rng(31)
    for _ in range(20):
        t_L = rng.uniform(1e5, 6e7)
        lam_L, beta_L, psi_L = rng.uniform(0, 2 * math.pi), math.asin(rng.uniform(-1, 1)), rng.uniform(0, math.pi)
        t_ref, lam, beta, psi = S.lisa_to_ssb(t_L, lam_L, beta_L, psi_L)
        assert 0.0 <= lam < 2 * math.pi and 0.0 <= psi < math.pi and abs(beta) <= math.pi / 2
        # the same physical wave: k, P+ and Px built from the LISA-frame angles and rotated to the SSB are those of the SSB angles
        R = S.lisa_frame(response.OMEGA0 * t_L)
        kL, PpL, PcL = response.source_frame(lam_L, beta_L, psi_L)
        k, Pp, Pc = response.source_frame(lam, beta, psi)
        assert np.max(np.abs(R @ kL - k)) < 1e-14
        assert np.max(np.abs(R @ PpL @ R.T - Pp)) < 1e-13 and np.max(np.abs(R @ PcL @ R.T - Pc)) < 1e-13
        # so k.n for every link is the same number in both frames (links are fixed vectors in the LISA frame)
        _, pL = response.orbit(np.float64(t_L))
        for (s_, r_) in response.LINKS:
            n_ssb = pL[r_] - pL[s_]
            assert abs(k @ n_ssb - kL @ (R.T @ n_ssb)) < 1e-13 * np.linalg.norm(n_ssb)
        # time: t_L is the arrival of the wavefront at the constellation centre
        p0, _ = response.orbit(np.float64(t_L))
        assert abs((t_L - t_ref) - float(k @ p0)) < 4e-16 * t_L + 1e-10 and abs(t_L - t_ref) <= AU_S * (1 + 1e-12)
        # round trip
        back = S.ssb_to_lisa(t_ref, lam, beta, psi)
        assert abs(back[0] - t_L) < 1e-13 * t_L
        assert abs(math.remainder(back[1] - lam_L, 2 * math.pi)) < 1e-12 and abs(back[2] - beta_L) < 1e-12
        assert abs(math.remainder(back[3] - psi_L, math.pi)) < 1e-12
    # a source in the direction of the constellation centre as seen from the Sun is reached R/c EARLIER than the SSB
    t_L = 4.0e6
    t_ref, lam, beta, psi = S.lisa_to_ssb(t_L, 0.3, 0.2, 0.1)
    back = S.ssb_to_lisa(1.0e7, response.OMEGA0 * 1.0e7 % (2 * math.pi), 0.0, 0.4)
    assert abs((back[0] - 1.0e7) + AU_S) < 1e-3               # alpha moves by Omega_0 R/c = 1e-4 rad in between


def test_eight_sky_modes_in_the_lisa_frame():
    # in the LISA frame the sky posterior has 8 modes, longitudes separated by pi/2, latitudes +-beta_L.
    # With a frozen constellation at low frequency (x = 2 pi f L/c << 1) the A, E responses of the 8 points
    # (lambda_L + k pi/2, +-beta_L; the reflected ones with iota -> pi - iota, psi_L -> pi - psi_L) have equal moduli up
    # to O(x); the same operations applied to SSB angles change them by O(1).
    from oracle import response
    from oracle.constants import ARM_S
    t, f = 1.3e7, 1e-4
    x = 2 * math.pi * f * ARM_S
    lam_L, beta_L, psi_L, inc, phi = 1.0, 0.5, 0.7, 1.1, 2.0

    def moduli(lam_L, beta_L, psi_L, inc, frame):
        if frame == "lisa":
            _, lam, beta, psi = S.lisa_to_ssb(t, lam_L, beta_L, psi_L)
        else:
            lam, beta, psi = lam_L, beta_L, psi_L
        _, (A, E, T) = response.transfer(np.float64(f), np.float64(t), lam, beta, psi, inc, phi, 2, 2)
        return abs(A), abs(E)

    for frame, near in (("lisa", True), ("ssb", False)):
        a0, e0 = moduli(lam_L, beta_L, psi_L, inc, frame)
        worst = 0.0
        for k in range(4):
            a1, e1 = moduli(lam_L + k * math.pi / 2, beta_L, psi_L + k * math.pi / 2, inc, frame)
            a2, e2 = moduli(lam_L + k * math.pi / 2, -beta_L, math.pi - psi_L + k * math.pi / 2, math.pi - inc, frame)
            worst = max(worst, abs(a1 / a0 - 1), abs(e1 / e0 - 1), abs(a2 / a0 - 1), abs(e2 / e0 - 1))
        if near:
            assert worst < 0.5 * x, (worst, x)
        else:
            assert worst > 0.05, worst


def test_unpack_sampled_lisa_is_unpack_then_frame_conversion():
    rng = np.random.default_rng(33)
    th = rng.uniform(S.PRIOR_LO, S.PRIOR_HI, size=(5, 11))
    th[:, 10] = np.log(rng.uniform(1e5, 3e7, 5))
    p = S.unpack_sampled_lisa(th, t0=123.0)
    q = S.unpack_sampled(th)
    for b in range(5):
        t_ref, lam, beta, psi = S.lisa_to_ssb(q[b, 10], q[b, 7], q[b, 8], q[b, 9], 123.0)
        assert np.array_equal(p[b, [10, 7, 8, 9]], [t_ref, lam, beta, psi])
        assert np.array_equal(p[b, :7], q[b, :7])
