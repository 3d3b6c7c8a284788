"""Pins P9-P12 of the oracle's LISA response (eqs. 7-10)."""
import math

import numpy as np

from oracle import response
from oracle.constants import ARM_S, AU_S, MODES, YEAR_SIDEREAL_S

PI = math.pi


def test_p10_harmonics_closed_forms_and_orthonormality():
    for th in (0.0, 0.3, 1.2, 2.9):
        for ph in (0.0, 0.7, 4.0):
            y22 = math.sqrt(5.0 / (64.0 * PI)) * (1.0 + math.cos(th)) ** 2 * complex(math.cos(2 * ph), math.sin(2 * ph))
            y2m2 = math.sqrt(5.0 / (64.0 * PI)) * (1.0 - math.cos(th)) ** 2 * complex(math.cos(2 * ph), -math.sin(2 * ph))
            y21 = math.sqrt(5.0 / (16.0 * PI)) * math.sin(th) * (1.0 + math.cos(th)) * complex(math.cos(ph), math.sin(ph))
            assert abs(response.sYlm(2, 2, th, ph) - y22) < 1e-13
            assert abs(response.sYlm(2, -2, th, ph) - y2m2) < 1e-13
            assert abs(response.sYlm(2, 1, th, ph) - y21) < 1e-13
    # orthonormality over the sphere by Gauss-Legendre x uniform-phi quadrature (exact for these degrees)
    x, wx = np.polynomial.legendre.leggauss(24)
    nphi = 16
    phis = 2.0 * PI * np.arange(nphi) / nphi
    lms = [(l, s * m) for (l, m) in MODES for s in (1, -1)]
    vals = {lm: np.array([[response.sYlm(lm[0], lm[1], math.acos(xi), p) for p in phis] for xi in x]) for lm in lms}
    for a in lms:
        for b in lms:
            integral = np.sum(wx[:, None] * vals[a] * np.conj(vals[b])) * (2.0 * PI / nphi)
            assert abs(integral - (1.0 if a == b else 0.0)) < 1e-12, (a, b, integral)


def test_p11_orbit_is_a_rigid_rotating_triangle():
    t = np.linspace(0.0, 2.0 * YEAR_SIDEREAL_S, 2001)
    p0, pL = response.orbit(t)
    for (s, r) in response.LINKS:
        arm = np.sqrt(np.sum((pL[r] - pL[s]) ** 2, axis=0))
        assert np.max(np.abs(arm / ARM_S - 1.0)) < 1e-13
    cen = (pL[1] + pL[2] + pL[3]) / 3.0
    assert np.max(np.abs(cen)) < 1e-13 * AU_S
    assert np.allclose(np.sqrt(np.sum(p0 ** 2, axis=0)), AU_S, rtol=1e-15)
    # one-sidereal-year periodicity and cyclic symmetry n -> n+1 after a third of a year... of constellation rotation
    p0b, pLb = response.orbit(t + YEAR_SIDEREAL_S)
    for n in (1, 2, 3):
        assert np.max(np.abs(pLb[n] - pL[n])) < 1e-9 * ARM_S
    # eccentricity of the stated construction
    assert abs(response.ECC - 0.0048242) < 1e-6


def _time_domain_X(f, k, P, pos, tau):
    """First-generation Michelson X(tau) from literal delays for H(t) = P exp(2 pi i f t), frozen positions."""
    def H(t):
        return P * np.exp(2j * PI * f * t)

    def y(s, r, t):
        n = (pos[r] - pos[s]) / ARM_S
        num = n @ (H(t - ARM_S - k @ pos[s]) - H(t - k @ pos[r])) @ n
        return 0.5 * num / (1.0 - k @ n)

    L = ARM_S
    X = (y(3, 1, tau) + y(1, 3, tau - L) + y(2, 1, tau - 2 * L) + y(1, 2, tau - 3 * L)
         - (y(2, 1, tau) + y(1, 2, tau - L) + y(3, 1, tau - 2 * L) + y(1, 3, tau - 3 * L)))
    Y = (y(1, 2, tau) + y(2, 1, tau - L) + y(3, 2, tau - 2 * L) + y(2, 3, tau - 3 * L)
         - (y(3, 2, tau) + y(2, 3, tau - L) + y(1, 2, tau - 2 * L) + y(2, 1, tau - 3 * L)))
    Z = (y(2, 3, tau) + y(3, 2, tau - L) + y(1, 3, tau - 2 * L) + y(3, 1, tau - 3 * L)
         - (y(1, 3, tau) + y(3, 1, tau - L) + y(2, 3, tau - 2 * L) + y(3, 2, tau - 3 * L)))
    return X, Y, Z


def test_p9_frozen_constellation_time_domain_brute_force():
    rng = np.random.default_rng(9)
    for trial in range(6):
        lam, beta, psi = rng.uniform(0, 2 * PI), math.asin(rng.uniform(-1, 1)), rng.uniform(0, PI)
        inc, phi_ref = math.acos(rng.uniform(-1, 1)), rng.uniform(0, 2 * PI)
        l, m = MODES[trial]
        f = 10.0 ** rng.uniform(-4, -1)
        t_star = rng.uniform(0, YEAR_SIDEREAL_S)
        k, Pp, Pc = response.source_frame(lam, beta, psi)
        P = response.mode_polarisation(l, m, inc, phi_ref, Pp, Pc)
        p0, pL = response.orbit(np.float64(t_star))
        pos = {n: p0 + pL[n] for n in (1, 2, 3)}
        tau = 0.37 * ARM_S                                  # any instant: the common factor exp(2 pi i f tau) divides out
        X, Y, Z = _time_domain_X(f, k, P, pos, tau)
        ph = np.exp(2j * PI * f * tau)
        G, _ = response.link_kernels(np.float64(f), np.float64(t_star), k, P, with_doppler=True)
        A, E, T = response.tdi_aet(np.float64(f), G)
        A_td = (Z - X) / math.sqrt(2.0) / ph
        E_td = (X - 2 * Y + Z) / math.sqrt(6.0) / ph
        T_td = (X + Y + Z) / math.sqrt(3.0) / ph
        scale = max(abs(A_td), abs(E_td))
        assert abs(A - A_td) < 1e-11 * scale and abs(E - E_td) < 1e-11 * scale and abs(T - T_td) < 1e-11 * scale
        # the Doppler factorisation (G8): T = exp(i phi_R) T-hat
        phi_R, (Ah, Eh, Th) = response.transfer(np.float64(f), np.float64(t_star), lam, beta, psi, inc, phi_ref, l, m)
        rot = np.exp(1j * phi_R)
        assert abs(rot * Ah - A) < 1e-12 * scale and abs(rot * Eh - E) < 1e-12 * scale and abs(rot * Th - T) < 1e-12 * scale
        assert abs(phi_R + 2 * PI * f * (k @ p0)) < 1e-9


def test_p12_t_channel_suppressed_at_low_frequency():
    lam, beta, psi, inc, phi_ref = 1.1, 0.4, 0.7, 1.0, 2.0
    ratios = []
    for f in (1e-3, 1e-4, 1e-5):
        _, (A, E, T) = response.transfer(np.float64(f), np.float64(3.0e6), lam, beta, psi, inc, phi_ref, 2, 2)
        ratios.append(abs(T) / math.hypot(abs(A), abs(E)))
    # For this exactly rigid equilateral constellation the GW response of T vanishes through O(x^2),
    # x = 2 pi f L/c: |T|/|A,E| = c x^3 with the same c at every f (SURVEY.md P12 guessed O(x))
    x = [2 * PI * f * ARM_S for f in (1e-3, 1e-4, 1e-5)]
    c = [r / xi ** 3 for r, xi in zip(ratios, x)]
    assert ratios[0] < 1e-4
    assert abs(c[0] / c[1] - 1.0) < 0.02 and abs(c[1] / c[2] - 1.0) < 0.02 and c[0] < 0.1


def test_spacecraft_relabelling_symmetry():
    # rotating the source by the constellation's internal 120-degree symmetry is not a symmetry of the
    # sky, but A^2+E^2 (a rotation-invariant pair) must be unchanged under cyclic relabelling 1->2->3->1
    lam, beta, psi, inc, phi_ref = 2.1, -0.3, 0.2, 0.8, 1.0
    f, t = np.float64(3e-3), np.float64(1.0e7)
    k, Pp, Pc = response.source_frame(lam, beta, psi)
    P = response.mode_polarisation(2, 2, inc, phi_ref, Pp, Pc)
    G, _ = response.link_kernels(f, t, k, P, with_doppler=True)
    A, E, T = response.tdi_aet(f, G)
    perm = {1: 2, 2: 3, 3: 1}
    Gp = {(perm[s], perm[r]): g for (s, r), g in G.items()}
    A2, E2, T2 = response.tdi_aet(f, Gp)
    assert abs(abs(A) ** 2 + abs(E) ** 2 - abs(A2) ** 2 - abs(E2) ** 2) < 1e-12 * (abs(A) ** 2 + abs(E) ** 2)
    assert abs(T - T2) < 1e-12 * max(abs(T), abs(A) * 1e-6)
