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


def test_p12_t_channel_vanishes_through_relative_order_x2(table=None):
    # DESIGN.md section 4 (reading P12) derives it: in X + Y + Z every term that is even in mu = k.n is a function of
    # the ARM, not of the link direction, and cancels pairwise; the first direction-dependent term of the round-trip
    # factor sinc[x/2 (1 - mu)] + exp(-ix) sinc[x/2 (1 + mu)] is + i x^3 mu / 12 (x = 2 pi f L/c).  Hence
    #   T -> (1/sqrt 3) (1 - z^2) (-i x/2) (i x^3/12) 2 [a_31 mu_31 + a_12 mu_12 + a_23 mu_23],  a_sr = n_sr.P.n_sr,
    # so |T|/|A,E| = c x^3 (SURVEY.md P12 guessed O(x)); the closed form pins the leading coefficient, sign included.
    lam, beta, psi, inc, phi_ref = 1.1, 0.4, 0.7, 1.0, 2.0
    t = np.float64(3.0e6)
    k, Pp, Pc = response.source_frame(lam, beta, psi)
    P = response.mode_polarisation(2, 2, inc, phi_ref, Pp, Pc)
    _, pL = response.orbit(t)
    lead = 0.0
    for (s, r) in ((3, 1), (1, 2), (2, 3)):
        n = (pL[r] - pL[s]) / ARM_S
        lead = lead + (n @ P @ n) * (k @ n)
    ratios, xs = [], []
    for f, tol in ((1e-3, 0.2), (3e-4, 0.05), (1e-4, 0.02)):
        x = 2 * PI * f * ARM_S
        _, (A, E, T) = response.transfer(np.float64(f), t, lam, beta, psi, inc, phi_ref, 2, 2)
        z = np.exp(-1j * x)
        T_lead = (1.0 - z * z) * (-0.5j * x) * (1j * x ** 3 / 12.0) * 2.0 * lead / math.sqrt(3.0)
        assert abs(T / T_lead - 1.0) < tol, (f, T, T_lead)
        ratios.append(abs(T) / math.hypot(abs(A), abs(E)))
        xs.append(x)
    c = [r / xi ** 3 for r, xi in zip(ratios, xs)]
    assert ratios[0] < 1e-4
    assert abs(c[0] / c[1] - 1.0) < 0.05 and abs(c[1] / c[2] - 1.0) < 0.02 and c[0] < 0.1


def test_source_frame_is_a_right_handed_transverse_traceless_basis():
    # pins response.source_frame (O4): k = -n(lambda, beta); P+, Px symmetric, traceless, transverse, normalised and
    # mutually orthogonal; psi rotates them like a spin-2 pair; (u, v, k) is right handed so that psi is measured from u
    # towards v as seen along the propagation direction
    rng = np.random.default_rng(11)
    for _ in range(8):
        lam, beta, psi = rng.uniform(0, 2 * PI), math.asin(rng.uniform(-1, 1)), rng.uniform(0, PI)
        k, Pp, Pc = response.source_frame(lam, beta, psi)
        nhat = np.array([math.cos(beta) * math.cos(lam), math.cos(beta) * math.sin(lam), math.sin(beta)])
        assert np.max(np.abs(k + nhat)) < 1e-15 and abs(k @ k - 1.0) < 1e-15
        for Q in (Pp, Pc):
            assert np.max(np.abs(Q - Q.T)) < 1e-15 and abs(np.trace(Q)) < 1e-15 and np.max(np.abs(Q @ k)) < 1e-15
        assert abs(np.sum(Pp * Pp) - 2.0) < 1e-14 and abs(np.sum(Pc * Pc) - 2.0) < 1e-14 and abs(np.sum(Pp * Pc)) < 1e-14
        _, Pp4, Pc4 = response.source_frame(lam, beta, psi + PI / 4)
        assert np.max(np.abs(Pp4 - Pc)) < 1e-14 and np.max(np.abs(Pc4 + Pp)) < 1e-14
        _, Pp2, Pc2 = response.source_frame(lam, beta, psi + PI / 2)
        assert np.max(np.abs(Pp2 + Pp)) < 1e-14 and np.max(np.abs(Pc2 + Pc)) < 1e-14
        # at psi = 0: P+ = u u - v v with u along increasing... u = dn/dlambda direction reversed, v = dn/dbeta;
        # handedness u x v = k
        _, e_p, e_c = response.source_frame(lam, beta, 0.0)
        v = np.array([-math.sin(beta) * math.cos(lam), -math.sin(beta) * math.sin(lam), math.cos(beta)])   # d n / d beta
        u = np.cross(v, k)                                                                                 # so that u x v = k
        assert np.max(np.abs(e_p - (np.outer(u, u) - np.outer(v, v)))) < 1e-14
        assert np.max(np.abs(e_c - (np.outer(u, v) + np.outer(v, u)))) < 1e-14


def test_mode_polarisation_is_the_positive_frequency_part_of_the_mode_sum():
    # pins response.mode_polarisation against the DEFINITION (reading G3):
    #   h+ - i hx = sum_{l, +-m} Y_lm(iota, phi_ref) h_lm(t),  h_{l,-m} = (-1)^l conj(h_lm)   (non-precessing),
    #   H(t) = h+ P+ + hx Px,
    # and eq. 5's mode content at f > 0 is, with the Fourier kernel exp(-2 pi i f t) of reading G2, the transform of
    # h_{l,-m}(t), the member of the pair that carries exp(+i m Omega t).  With a toy h_lm(t) = a exp(-i m Omega t)
    # the exp(+i m Omega t) coefficient of H(t) (a discrete Fourier projection) must equal P_lm x (-1)^l conj(a).
    rng = np.random.default_rng(12)
    nt = 64
    tt = np.arange(nt) / nt                                  # one period of Omega = 2 pi
    for (l, m) in MODES:
        lam, beta, psi = rng.uniform(0, 2 * PI), math.asin(rng.uniform(-1, 1)), rng.uniform(0, PI)
        inc, phi_ref = math.acos(rng.uniform(-1, 1)), rng.uniform(0, 2 * PI)
        a = complex(rng.standard_normal(), rng.standard_normal())
        _, Pp, Pc = response.source_frame(lam, beta, psi)
        h_pos = a * np.exp(-1j * m * 2 * PI * tt)            # h_{l,m}(t)
        h_neg = (-1.0) ** l * np.conj(h_pos)                 # h_{l,-m}(t)
        hc = response.sYlm(l, m, inc, phi_ref) * h_pos + response.sYlm(l, -m, inc, phi_ref) * h_neg
        hp, hx = hc.real, -hc.imag
        H = hp[:, None, None] * Pp[None] + hx[:, None, None] * Pc[None]          # [nt, 3, 3], real
        coeff = np.tensordot(np.exp(-1j * m * 2 * PI * tt), H, axes=(0, 0)) / nt  # projection on exp(+i m Omega t)
        P = response.mode_polarisation(l, m, inc, phi_ref, Pp, Pc)
        content = (-1.0) ** l * np.conj(a)                   # amplitude of h_{l,-m}: the f > 0 mode content
        assert np.max(np.abs(coeff - P * content)) < 1e-12 * abs(a), (l, m)
        assert np.max(np.abs(P)) > 1e-3                      # not trivially zero


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
