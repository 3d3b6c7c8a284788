"""Pins P6-P8, P13 of the oracle's PhenomD / PhenomHM restatement."""
import math

import numpy as np
import pytest

from oracle.constants import GPC_S, MODES, MTSUN_S
from oracle.phenom import F_AMP_INS, F_PHI_INS, Intrinsic
from oracle.response import sYlm

CASES = [(1e6, 3.0, 0.6, -0.3), (2e6, 1.0, 0.0, 0.0), (1e5, 1.5, -0.9, 0.8), (1e8, 10.0, 0.95, -0.95),
         (3e5, 20.0, -0.99, -0.99)]


@pytest.mark.parametrize("M,q,a1,a2", CASES)
def test_p6_newtonian_time_to_coalescence(table, M, q, a1, a2):
    # eq. 6 with phi = -Psi must give t_22(f) -> t_coal - (5/256) Mc^(-5/3) (pi f)^(-8/3), sign included
    I = Intrinsic(table, M, q, a1, a2, 10.0)
    Mc = I.M_s * I.eta ** 0.6
    t_coal = 1234.5
    rel = []
    for Mf in (1e-5, 1e-6, 1e-7):
        f = Mf / I.M_s
        t = float(I.t_of_f(2, 2, np.float64(f), t_coal))
        newt = -(5.0 / 256.0) * Mc ** (-5.0 / 3.0) * (math.pi * f) ** (-8.0 / 3.0)
        assert t < 0.0
        rel.append(abs((t - t_coal) / newt - 1.0))
    assert rel[2] < rel[1] < rel[0]
    assert rel[2] < 2e-3                                   # O(v^2) with v = (pi Mf)^(1/3) ~ 7e-3
    assert 3.0 < rel[0] / rel[1] < 6.0                     # v^2 scaling: 10^(2/3) = 4.64


@pytest.mark.parametrize("M,q,a1,a2", CASES)
def test_p7_newtonian_amplitude(table, M, q, a1, a2):
    D = 7.0
    I = Intrinsic(table, M, q, a1, a2, D)
    Mc = I.M_s * I.eta ** 0.6
    fac = 0.5 * abs(sYlm(2, 2, 0.0, 0.0) + np.conj(sYlm(2, -2, 0.0, 0.0)))
    rel = []
    for Mf in (1e-5, 1e-7):
        f = Mf / I.M_s
        got = fac * float(I.amp_lm(2, 2, np.float64(Mf)))
        ref = math.sqrt(5.0 / 24.0) * math.pi ** (-2.0 / 3.0) * Mc ** (5.0 / 6.0) * f ** (-7.0 / 6.0) / (D * GPC_S)
        rel.append(abs(got / ref - 1.0))
    assert rel[1] < rel[0] < 2e-3 and rel[1] < 1e-4


@pytest.mark.parametrize("M,q,a1,a2", CASES)
def test_p8_c1_continuity_and_phase_derivative(table, M, q, a1, a2):
    I = Intrinsic(table, M, q, a1, a2, 10.0)
    eps = 1e-9
    for fb in (F_PHI_INS, I.f_mr):                          # phase region boundaries
        lo, hi = np.float64(fb * (1 - eps)), np.float64(fb * (1 + eps))
        (p1, d1), (p2, d2) = I.psi22(lo), I.psi22(hi)
        assert abs(p2 - p1) <= abs(d1) * 2.1 * eps * fb + 1e-10 * max(1.0, abs(p1))
        assert abs(d2 - d1) <= 1e-6 * abs(d1) + 1e-6        # slope jump bounded by Psi'' * 2 eps f
    for fb in (F_AMP_INS, I.f_peak):                        # amplitude region boundaries
        a1_, a2_ = I.amp_hat(np.float64(fb * (1 - eps))), I.amp_hat(np.float64(fb * (1 + eps)))
        assert abs(a2_ - a1_) <= 1e-7 * abs(a1_)
        def slope_jump(h):
            sl = (I.amp_hat(np.float64(fb - h)) - I.amp_hat(np.float64(fb - 2 * h))) / h
            sr = (I.amp_hat(np.float64(fb + 2 * h)) - I.amp_hat(np.float64(fb + h))) / h
            return abs(sr - sl)
        # C1: the one-sided slopes differ only by curvature * O(h), so the jump shrinks with h
        assert slope_jump(1e-7 * fb) <= 0.02 * slope_jump(1e-5 * fb) + 1e-6 * abs(a1_) / fb
    # analytic derivative vs central finite difference in every region
    for f0 in (1e-3, 0.01, 0.017, 0.019, 0.03, 0.45 * I.fRD, 0.6 * I.fRD, I.fRD, 1.2 * I.fRD):
        h = 1e-5 * f0
        fd = (I.psi22(np.float64(f0 + h))[0] - I.psi22(np.float64(f0 - h))[0]) / (2 * h)
        an = I.psi22(np.float64(f0))[1]
        assert abs(fd - an) <= 1e-7 * max(abs(an), 1.0) + 1e-6 * abs(I.psi22(np.float64(f0))[0]) / f0 * 1e-3
    # alignment (G4): f_ref maximises f^2 A_22 and Psi(f_ref) = Psi'(f_ref) = 0
    ff = np.linspace(0.8 * I.f_ref, 1.2 * I.f_ref, 20001)
    g = ff ** 2 * I.amp22(ff)
    assert abs(ff[np.argmax(g)] - I.f_ref) <= 2 * (ff[1] - ff[0])
    p, d = I.psi22(np.float64(I.f_ref))
    assert abs(p) < 1e-9 and abs(d) < 1e-7


@pytest.mark.parametrize("M,q,a1,a2", CASES[:4])
def test_p13_higher_mode_maps(table, M, q, a1, a2):
    I = Intrinsic(table, M, q, a1, a2, 10.0)
    eps = 1e-10
    for (l, m) in MODES:
        # continuity of A_lm and Psi_lm at the map boundaries
        for fb in (0.5 * m * F_AMP_INS, 0.5 * m * F_PHI_INS, I.f_rd[(l, m)]):
            lo, hi = np.float64(fb * (1 - eps)), np.float64(fb * (1 + eps))
            if I.amp_lm(l, m, lo) > 0:
                assert abs(I.amp_lm(l, m, hi) / I.amp_lm(l, m, lo) - 1.0) < 1e-6
            p1, d1 = I.psi_lm(l, m, lo)
            p2, d2 = I.psi_lm(l, m, hi)
            assert abs(p2 - p1) < 1e-6 * max(1.0, abs(p1))
            assert abs(d2 - d1) < 1e-5 * max(1.0, abs(d1))
        # inspiral: Psi_lm(f) = (m/2) Psi_22(2f/m) - Delta_lm and t_lm(f) = t_22(2f/m)
        f = np.array([1e-4, 1e-3, 4e-3]) * m / 2.0
        p, d = I.psi_lm(l, m, f)
        p22, d22 = I.psi22(2.0 * f / m)
        assert np.allclose(p, 0.5 * m * p22 - table[f"hm.{l}{m}.dphi"], rtol=1e-13, atol=1e-9)
        assert np.allclose(d, d22, rtol=1e-13)
    # (2,2) is PhenomD itself
    f = np.geomspace(1e-4, 0.3, 50)
    assert np.allclose(I.amp_lm(2, 2, f), I.amp22(f), rtol=1e-13)
    assert np.allclose(I.psi_lm(2, 2, f)[0], I.psi22(f)[0], rtol=1e-13, atol=1e-10)
    # equal masses: odd-m modes vanish (delta = 0)
    Ieq = Intrinsic(table, M, 1.0, a1, a2, 10.0)
    for (l, m) in ((3, 3), (2, 1), (4, 3)):
        assert np.all(Ieq.amp_lm(l, m, f) == 0.0)


def test_mass_ratio_reading_g15(table):
    # q and 1/q describe the same binary; a1 always belongs to the heavier body
    A = Intrinsic(table, 1e6, 4.0, 0.3, -0.2, 10.0)
    B = Intrinsic(table, 1e6, 0.25, 0.3, -0.2, 10.0)
    assert A.eta == B.eta and A.chi_hat == B.chi_hat and A.f_ref == B.f_ref


def test_amplitudes_positive_and_inspiral_monotone(table):
    for q in (1.0, 2.0, 5.0, 20.0):
        for a in (-0.99, 0.0, 0.99):
            I = Intrinsic(table, 1e6, q, a, -a, 10.0)
            f = np.geomspace(1e-5, I.f_ref, 3000)
            assert np.all(np.diff(I.psi22(f)[1]) > 0.0)        # t(f) strictly increasing up to merger
            assert np.all(I.amp_hat(np.geomspace(1e-5, 0.5, 3000)) > 0.0)
            assert I.gamma2 < 1.0 and 0.5 * I.fRD > F_PHI_INS and I.f_peak > F_AMP_INS


def test_higher_mode_table_rows_follow_from_the_leading_pn_multipoles(table):
    # hm.<lm>.amp / hm.<lm>.dphi (model_data/phenomhm_table.csv, tag "derived") against the textbook leading-PN
    # time-domain multipoles h_lm = 2 eta M x / R sqrt(16 pi/5) H_lm exp(-i m phi) (Kidder 2008 / Blanchet's review):
    # the stationary-phase factor of mode m is sqrt(2/m) and the mode content at f > 0 is the transform of
    # h_{l,-m} = (-1)^l conj(h_lm) (reading G3), so
    #   c_lm = sqrt(2/m) |H_lm| (mass factors and powers of x stripped),  Delta_lm = (1 - m/2) pi/4 + arg[(-1)^l conj(H_lm)].
    s = math.sqrt
    H = {(2, 2): 1.0 + 0.0j, (2, 1): -1j / 3.0, (3, 3): -0.75j * s(15.0 / 14.0), (3, 2): s(5.0 / 7.0) / 3.0 + 0.0j,
         (4, 4): -8.0 / 9.0 * s(5.0 / 7.0) + 0.0j, (4, 3): -9j / (4.0 * s(70.0))}
    for (l, m) in MODES:
        c = s(2.0 / m) * abs(H[(l, m)])
        z = (-1.0) ** l * np.conj(H[(l, m)])
        dphi = (1.0 - 0.5 * m) * math.pi / 4.0 + math.atan2(z.imag, z.real)
        assert abs(table[f"hm.{l}{m}.amp"] - c) < 1e-15, (l, m)
        d = table[f"hm.{l}{m}.dphi"] - dphi
        assert abs(d - 2 * math.pi * round(d / (2 * math.pi))) < 1e-14, (l, m)


def _newtonian_chirp_spectrum(eta, delta, l, m, dt=1.0, n=1 << 20):
    """|FFT| of the leading-PN time-domain multipole h_{l,-m}(t) = (-1)^l conj(h_lm) of a Newtonian quasi-circular inspiral
    (geometric units, M = 1, R = 1):  h_lm = 2 eta x sqrt(16 pi/5) H_lm(x) exp(-i m phi),  x = (omega_orb)^(2/3),
    Theta = eta (t_c - t)/5,  x = Theta^(-1/4)/4,  phi = -Theta^(5/8)/eta  (textbook, Blanchet's review / Kidder 2008).
    H_lm with their mass factors and powers of x are typed here from that literature, independently of oracle/phenom.py.
    The record runs from orbital M omega = 0.004 to 0.055 with a smooth taper over 0.004-0.006 and 0.040-0.055, zero-padded
    to n samples.  Returns (f [cycles per M], |h~(f)|) on the FFT grid."""
    s = math.sqrt
    tau = lambda om: 5.0 / (256.0 * eta) * om ** (-8.0 / 3.0)          # time to coalescence at orbital frequency om
    t = np.arange(-tau(0.004), -tau(0.055), dt)                        # t_c = 0
    assert t.size < n
    theta = eta * (-t) / 5.0
    x = 0.25 * theta ** -0.25
    om = x ** 1.5
    phi = -theta ** 0.625 / eta
    H = {(2, 2): 1.0 + 0.0 * x,
         (2, 1): -1j / 3.0 * delta * x ** 0.5,
         (3, 3): -0.75j * s(15.0 / 14.0) * delta * x ** 0.5,
         (3, 2): s(5.0 / 7.0) / 3.0 * (1.0 - 3.0 * eta) * x,
         (4, 4): -8.0 / 9.0 * s(5.0 / 7.0) * (1.0 - 3.0 * eta) * x,
         (4, 3): -9j / (4.0 * s(70.0)) * delta * (1.0 - 2.0 * eta) * x ** 1.5}[(l, m)]
    h = 2.0 * eta * x * s(16.0 * math.pi / 5.0) * H * np.exp(-1j * m * phi)
    h = (-1.0) ** l * np.conj(h)                           # h_{l,-m}: the positive-frequency content (reading G3)

    def ramp(u):                                           # C-infinity step from 0 (u <= 0) to 1 (u >= 1)
        u = np.clip(u, 2e-3, 1.0 - 2e-3)
        return 1.0 / (1.0 + np.exp(1.0 / u - 1.0 / (1.0 - u)))
    w = ramp((t + tau(0.004)) / (tau(0.004) - tau(0.006))) * ramp((-tau(0.055) - t) / (tau(0.040) - tau(0.055)))
    spec = np.fft.fft(h * w, n) * dt
    return np.fft.fftfreq(n, dt), np.abs(spec)


@pytest.mark.parametrize("q", [3.0, 5.0, 1.5])
def test_beta_lm_structure_against_the_fft_of_a_newtonian_chirp(table, q):
    # Pins WHICH mass factor (delta, 1 - 3 eta, delta (1 - 2 eta)) and WHICH power of V every mode amplitude carries in
    # Intrinsic.beta_lm, and its V^(-7/2) sqrt(2/m) stationary-phase prefactor: the FFT of the time-domain leading-PN
    # multipole of a Newtonian chirp, divided by the (2,2) spectrum at the same orbital frequency, must equal
    # beta_lm(f) / beta_22(2 f / m).  Three mass ratios so that delta, (1 - 3 eta) and (1 - 2 eta) all move; several orbital
    # frequencies so that a wrong power of V shows as a slope.  Measured agreement is ~1e-3 (stationary phase: omega_dot /
    # omega^2 ~ 1e-3 here, plus taper ripple); the bar is 1 %.
    I = Intrinsic(table, 1e6, q, 0.0, 0.0, 10.0)
    eta, delta = I.eta, I.delta
    f22, s22 = _newtonian_chirp_spectrum(eta, delta, 2, 2)
    pos = f22 > 0
    for (l, m) in MODES:
        # orbital M omega: V = omega^(1/3) = 0.20 ... 0.27, a factor 1.36 in V, so one power of V off is a 36 % slope.  The m = 1
        # mode has half the cycles of (2,2) at a given orbital frequency and its taper ripple passes 1 % above 0.015
        omegas = np.array([0.008, 0.011, 0.015, 0.020]) if m > 1 else np.array([0.008, 0.011, 0.015])
        flm, slm = _newtonian_chirp_spectrum(eta, delta, l, m)
        f_m = m * omegas / (2.0 * math.pi)
        f_2 = 2.0 * omegas / (2.0 * math.pi)
        got_lm = np.interp(f_m, flm[pos], slm[pos])
        got_22 = np.interp(f_2, f22[pos], s22[pos])
        # absolute level of every mode against the oracle's formula (1 %: stationary phase + taper ripple)
        want = I.beta_lm(l, m, f_m)
        assert np.max(np.abs(got_lm / want - 1.0)) < 1e-2, ((l, m), got_lm / want)
        # ratio to (2,2) at the same orbital frequency: what amp_lm multiplies A_22 by in the inspiral
        ratio_fft = got_lm / got_22
        ratio_oracle = I.beta_lm(l, m, f_m) / I.beta_lm(2, 2, f_2)
        assert np.max(np.abs(ratio_fft / ratio_oracle - 1.0)) < 1e-2, ((l, m), ratio_fft / ratio_oracle)


@pytest.mark.parametrize("M,q,a1,a2", CASES[:4])
def test_ringdown_amplitude_of_every_mode_is_the_22_lorentzian_shifted_to_its_own_f_rd(table, M, q, a1, a2):
    # in the ringdown region the amplitude map is the SHIFT f_22 = f - (f_RD,lm - f_RD,22), slope one (the phase
    # map has slope f_damp,22 / f_damp,lm instead).  Stated without the map: with R_lm(f) = A_lm(f) / beta_lm(f), the leading-PN
    # factor stripped, R_lm(f_RD,lm + x) = R_22(f_RD,22 + x) for x >= 0, so the Lorentzian of every mode peaks at the same offset
    # from its own ringdown frequency and has the (2,2) width.  A slope other than one changes the measured half-width below.
    I = Intrinsic(table, M, q, a1, a2, 10.0)
    R = lambda l, m, f: I.amp_lm(l, m, np.float64(f)) / I.beta_lm(l, m, np.float64(f))
    w22 = I.gamma3 * I.fDM

    def half_width(l, m):
        # x > 0 with R(f_RD + x) = R(f_RD) / 2, by bisection on the measured curve
        f0 = I.f_rd[(l, m)]
        r0 = R(l, m, f0)
        lo, hi = 0.0, 20.0 * w22
        assert R(l, m, f0 + hi) < 0.5 * r0
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if R(l, m, f0 + mid) > 0.5 * r0 else (lo, mid)
        return 0.5 * (lo + hi)

    hw22 = half_width(2, 2)
    assert 0.2 * w22 < hw22 < 3.0 * w22                    # of the order of the Lorentzian's width gamma3 f_damp,22
    for (l, m) in MODES[1:]:
        if I.beta_lm(l, m, np.float64(0.1)) == 0.0:
            continue                                       # odd-m modes of an equal-mass binary vanish
        for x in (0.0, 0.3 * w22, w22, 4.0 * w22):
            assert R(l, m, I.f_rd[(l, m)] + x) == pytest.approx(R(2, 2, I.fRD + x), rel=1e-11), ((l, m), x)
        assert half_width(l, m) == pytest.approx(hw22, rel=1e-9), (l, m)
