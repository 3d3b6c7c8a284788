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
