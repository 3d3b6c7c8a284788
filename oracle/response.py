"""Oracle: fast frequency-domain LISA response, TDI A/E/T (eqs. 7-10).

Follows SURVEY.md 8(c) O4.  The single-link kernel is derived from the
time-domain two-point definition
    y_sr(t) = 1/2 n.[H(t - L/c - k.p_s/c) - H(t - k.p_r/c)].n / (1 - k.n)
for a Fourier component H(t) = P exp(+2 pi i f t) (convention O0), with all
positions frozen at t = t_lm(f).  TEST INFRASTRUCTURE - see oracle/__init__.py.
"""
import math

import numpy as np

from .constants import ARM_S, AU_S, YEAR_SIDEREAL_S

PI = math.pi
OMEGA0 = 2.0 * PI / YEAR_SIDEREAL_S
ECC = ARM_S / (2.0 * math.sqrt(3.0) * AU_S)      # e = L / (2 sqrt(3) R)
LINKS = ((3, 1), (1, 3), (2, 1), (1, 2), (3, 2), (2, 3))   # (sender, receiver)


def _fact(n):
    return float(math.factorial(n))


def wigner_d(l, mp, m, theta):
    """Wigner small-d matrix element d^l_{mp,m}(theta) (textbook sum formula)."""
    c, s = math.cos(0.5 * theta), math.sin(0.5 * theta)
    pre = math.sqrt(_fact(l + mp) * _fact(l - mp) * _fact(l + m) * _fact(l - m))
    tot = 0.0
    for k in range(0, 2 * l + 1):
        d1, d2, d3, d4 = l + m - k, k, l - k - mp, k - m + mp
        if d1 < 0 or d3 < 0 or d4 < 0:
            continue
        tot += ((-1.0) ** (k - m + mp)) / (_fact(d1) * _fact(d2) * _fact(d3) * _fact(d4)) \
            * c ** (2 * l - 2 * k + m - mp) * s ** (2 * k - m + mp)
    return pre * tot


def sYlm(l, m, theta, phi, s=-2):
    """Spin-weighted spherical harmonic sY_lm = (-1)^s sqrt((2l+1)/4pi) d^l_{m,-s}(theta) e^{i m phi}."""
    return ((-1.0) ** s) * math.sqrt((2 * l + 1) / (4.0 * PI)) * wigner_d(l, m, -s, theta) \
        * complex(math.cos(m * phi), math.sin(m * phi))


def orbit(t):
    """Equal-arm first-order-in-e orbit (O4).  Returns p0[3,...] and pL[n][3,...] = p_n - p0, in light-seconds."""
    t = np.asarray(t, dtype=np.float64)
    alpha = OMEGA0 * t
    ca, sa = np.cos(alpha), np.sin(alpha)
    p0 = AU_S * np.array([ca, sa, np.zeros_like(ca)])
    pL = {}
    for n in (1, 2, 3):
        bn = 2.0 * PI * (n - 1) / 3.0
        pL[n] = ECC * AU_S * np.array([
            0.5 * (np.cos(2.0 * alpha - bn) - 3.0 * math.cos(bn)),
            0.5 * (np.sin(2.0 * alpha - bn) - 3.0 * math.sin(bn)),
            -math.sqrt(3.0) * np.cos(alpha - bn)])
    return p0, pL


def source_frame(lam, beta, psi):
    """Propagation vector k and polarisation tensors P_+, P_x in the SSB frame (O4)."""
    cl, sl, cb, sb = math.cos(lam), math.sin(lam), math.cos(beta), math.sin(beta)
    k = -np.array([cb * cl, cb * sl, sb])
    u = np.array([sl, -cl, 0.0])
    v = np.array([-sb * cl, -sb * sl, cb])
    e_plus = np.outer(u, u) - np.outer(v, v)
    e_cross = np.outer(u, v) + np.outer(v, u)
    c2, s2 = math.cos(2.0 * psi), math.sin(2.0 * psi)
    return k, c2 * e_plus + s2 * e_cross, -s2 * e_plus + c2 * e_cross


def mode_polarisation(l, m, inc, phi_ref, P_plus, P_cross):
    """P_lm = 1/2 Y_{l,-m} (P+ + i Px) + 1/2 (-1)^l conj(Y_{lm}) (P+ - i Px)   (O4, convention O0)."""
    y_minus = sYlm(l, -m, inc, phi_ref)
    y_plus = sYlm(l, m, inc, phi_ref)
    return 0.5 * y_minus * (P_plus + 1j * P_cross) + 0.5 * ((-1.0) ** l) * np.conj(y_plus) * (P_plus - 1j * P_cross)


def link_kernels(f, t, k, P, with_doppler):
    """G_sr(f, t) for the six links; if not with_doppler the common factor exp(i phi_R) is removed.

    Returns ({(s,r): G}, phi_R) with phi_R = -2 pi f k.p0(t)/c.
    """
    f = np.asarray(f, dtype=np.float64)
    p0, pL = orbit(t)
    kp0 = k[0] * p0[0] + k[1] * p0[1] + k[2] * p0[2]
    phi_R = -2.0 * PI * f * kp0
    G = {}
    for (s, r) in LINKS:
        n = (pL[r] - pL[s]) / ARM_S
        kn = k[0] * n[0] + k[1] * n[1] + k[2] * n[2]
        nPn = np.zeros(f.shape, dtype=np.complex128)
        for a in range(3):
            for b in range(3):
                nPn = nPn + n[a] * P[a, b] * n[b]
        kps = sum(k[a] * (pL[r][a] + pL[s][a]) for a in range(3))
        x = PI * f * ARM_S * (1.0 - kn)
        sinc = np.sinc(x / PI)
        phase = -PI * f * (ARM_S + kps)
        if with_doppler:
            phase = phase + phi_R
        G[(s, r)] = (-1j * PI * f * ARM_S) * sinc * np.exp(1j * phase) * nPn
    return G, phi_R


def tdi_aet(f, G):
    """First-generation Michelson X,Y,Z from link kernels, then eqs. 8-10."""
    z = np.exp(-2j * PI * np.asarray(f) * ARM_S)
    pref = 1.0 - z * z
    X = pref * ((G[(3, 1)] + z * G[(1, 3)]) - (G[(2, 1)] + z * G[(1, 2)]))
    Y = pref * ((G[(1, 2)] + z * G[(2, 1)]) - (G[(3, 2)] + z * G[(2, 3)]))
    Z = pref * ((G[(2, 3)] + z * G[(3, 2)]) - (G[(1, 3)] + z * G[(3, 1)]))
    A = (Z - X) / math.sqrt(2.0)
    E = (X - 2.0 * Y + Z) / math.sqrt(6.0)
    T = (X + Y + Z) / math.sqrt(3.0)
    return A, E, T


def transfer(f, t, lam, beta, psi, inc, phi_ref, l, m):
    """Doppler-factored transfer functions: returns phi_R and T-hat^{A,E,T} with T = exp(i phi_R) T-hat (G8)."""
    k, Pp, Pc = source_frame(lam, beta, psi)
    P = mode_polarisation(l, m, inc, phi_ref, Pp, Pc)
    G, phi_R = link_kernels(f, t, k, P, with_doppler=False)
    return phi_R, tdi_aet(f, G)
