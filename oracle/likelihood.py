"""Oracle: sparse stage, spline/direct templates, inner products and logL.

Follows SURVEY.md 8(c) O5-O9 (PAPER.md:124-129 band, :171 sparse grid + spline +
interpolation, :177 modes summed before the product, eqs. 2, 3, 11 inner
product).  TEST INFRASTRUCTURE - see oracle/__init__.py.
"""
import math

import numpy as np

from . import response, spline
from .constants import MODES
from .phenom import F_PHI_INS, Intrinsic

PI = math.pi
TWO_PI_LD = 2.0 * np.longdouble("3.14159265358979323846264338327950288")
PARAM_NAMES = ("M_T", "q", "a1", "a2", "D_L", "phi_ref", "inc", "lam", "beta", "psi", "t_ref")
NQ = 8     # splined quantities per (walker, mode): A, Phi, Re/Im T-hat^{A,E,T}   (G8)


def mode_band(intr, l, m, t_coal, f_min, f_max):
    """O5: [f_lo, f_hi] of one mode on a grid spanning [f_min, f_max]; None if empty.

    f_lo: root of t_lm(f) = 0 on the inspiral branch of the phase
    map (f <= (m/2) 0.018 / M), where t_lm is monotone; clamped to the branch
    ends when there is no sign change.  f_hi = 0.2 max(1, m/2) / M  [reading G10].
    """
    f_top = 0.5 * m * F_PHI_INS / intr.M_s
    f_hi = min(f_max, 0.2 * max(1.0, 0.5 * m) / intr.M_s)
    tl = float(intr.t_of_f(l, m, np.float64(f_min), t_coal))
    if tl >= 0.0:
        f_lo = f_min
    elif f_top <= f_min or float(intr.t_of_f(l, m, np.float64(f_top), t_coal)) < 0.0:
        f_lo = max(f_top, f_min)
    else:
        lo, hi = f_min, f_top
        while True:
            mid = 0.5 * (lo + hi)
            if mid <= lo or mid >= hi:
                break
            if float(intr.t_of_f(l, m, np.float64(mid), t_coal)) < 0.0:
                lo = mid
            else:
                hi = mid
        f_lo = hi
    if not (f_hi > f_lo):
        return None
    return f_lo, f_hi


def knots_for_band(f_lo, f_hi, S):
    """O5: S log-spaced knots with exact end points."""
    s = np.arange(S, dtype=np.float64)
    k = f_lo * np.exp(s * (math.log(f_hi / f_lo) / (S - 1)))
    k[0] = f_lo
    k[-1] = f_hi
    return k


def smooth_quantities(intr, ext, l, m, f_hz, t_coal):
    """The Q=8 smooth functions of one mode at frequencies f_hz (O2-O4, eqs. 5-10).

    Rows: A_lm; Phi_lm = phi_lm + phi_R (rad, the linear term -2 pi f t_coal left out, G9);
    Re, Im of T-hat^A, T-hat^E, T-hat^T.
    """
    f_hz = np.asarray(f_hz, dtype=np.float64)
    fM = f_hz * intr.M_s
    amp = intr.amp_lm(l, m, fM)
    psi, dpsi = intr.psi_lm(l, m, fM)
    t = t_coal + intr.M_s * dpsi / (2.0 * PI)                      # eq. 6
    phi_R, (TA, TE, TT) = response.transfer(f_hz, t, ext["lam"], ext["beta"], ext["psi"],
                                            ext["inc"], ext["phi_ref"], l, m)
    return np.stack([amp, -psi + phi_R, TA.real, TA.imag, TE.real, TE.imag, TT.real, TT.imag])


def unpack(params):
    p = dict(zip(PARAM_NAMES, [float(v) for v in params]))
    return p


def walker_valid(p):
    """8(b): out-of-domain walkers get logL = -inf."""
    vals = list(p.values())
    if not all(math.isfinite(v) for v in vals):
        return False
    return p["M_T"] > 0.0 and p["D_L"] > 0.0 and p["q"] > 0.0 and abs(p["a1"]) <= 1.0 and abs(p["a2"]) <= 1.0


def sparse_stage(table, params, f_min, f_max, S, t0=0.0, knots_override=None):
    """Steps a1-a5 for one walker: per mode None or dict(knots, y[8,S], coef[S-1,8,4])."""
    p = unpack(params)
    intr = Intrinsic(table, p["M_T"], p["q"], p["a1"], p["a2"], p["D_L"])
    t_coal = t0 + p["t_ref"]
    out = []
    for i, (l, m) in enumerate(MODES):
        band = mode_band(intr, l, m, t_coal, f_min, f_max)
        if band is None:
            out.append(None)
            continue
        knots = knots_for_band(band[0], band[1], S) if knots_override is None else knots_override[i]
        y = smooth_quantities(intr, p, l, m, knots, t_coal)
        coef = np.stack([spline.coefficients(knots, y[qi]) for qi in range(NQ)], axis=1)   # [S-1, 8, 4]
        out.append(dict(knots=knots, y=y, coef=coef))
    return out, t_coal


def _combine(amp, Phi, That, f, t_coal):
    """O7: A exp(i theta) T-hat with theta = Phi - 2 pi f t_coal, the linear term taken exactly (G9)."""
    lin = np.asarray(f, dtype=np.longdouble) * np.longdouble(t_coal)        # cycles
    lin = lin - np.rint(lin)
    cyc = Phi / (2.0 * PI)
    cyc = (cyc - np.rint(cyc)) - lin.astype(np.float64)
    theta = 2.0 * PI * cyc
    e = amp * (np.cos(theta) + 1j * np.sin(theta))
    return [e * T for T in That]


def template(table, params, freqs, S, t0=0.0, mode="spline", mode_mask=0x3F):
    """h^{A,E,T} on freqs [3, N] complex128 for one walker; bins outside a mode's band get 0 from it."""
    freqs = np.asarray(freqs, dtype=np.float64)
    h = np.zeros((3, freqs.size), dtype=np.complex128)
    p = unpack(params)
    if not walker_valid(p):
        return h
    intr = Intrinsic(table, p["M_T"], p["q"], p["a1"], p["a2"], p["D_L"])
    t_coal = t0 + p["t_ref"]
    f_min, f_max = freqs[0], freqs[-1]
    for i, (l, m) in enumerate(MODES):
        if not (mode_mask >> i) & 1:
            continue
        band = mode_band(intr, l, m, t_coal, f_min, f_max)
        if band is None:
            continue
        sel = np.nonzero((freqs >= band[0]) & (freqs <= band[1]))[0]
        if sel.size == 0:
            continue
        f = freqs[sel]
        if mode == "direct":                                         # O9
            q = smooth_quantities(intr, p, l, m, f, t_coal)
        else:                                                        # O5-O7
            knots = knots_for_band(band[0], band[1], S)
            y = smooth_quantities(intr, p, l, m, knots, t_coal)
            q = np.stack([spline.evaluate(knots, spline.coefficients(knots, y[qi]), f) for qi in range(NQ)])
        That = [q[2] + 1j * q[3], q[4] + 1j * q[5], q[6] + 1j * q[7]]
        for c, hc in enumerate(_combine(q[0], q[1], That, f, t_coal)):
            h[c, sel] += hc
    return h


def weights(freqs, psd):
    """w = 4 df / S_n; 0 where S_n <= 0 or not finite (G6).  df = (f_{N-1} - f_0)/(N-1)  (G13)."""
    freqs = np.asarray(freqs, dtype=np.float64)
    df = (freqs[-1] - freqs[0]) / (freqs.size - 1)
    psd = np.asarray(psd, dtype=np.float64)
    ok = np.isfinite(psd) & (psd > 0.0)
    w = np.zeros_like(psd)
    w[ok] = 4.0 * df / psd[ok]
    return w


def inner(a, b, w):
    """<a|b> = sum_c sum_k w_ck Re(a conj(b))   (eqs. 3, 11; rectangle rule G13), long-double accumulation."""
    prod = (a.real * b.real + a.imag * b.imag) * w
    return float(np.sum(prod.astype(np.longdouble)))


def loglike_parts(table, params, freqs, data, psd, S, t0=0.0, mode="spline"):
    """Returns (<d|h>, <h|h>, logL) with logL = <d|h> - 1/2<h|h> - 1/2<d|d> (eq. 2)."""
    p = unpack(params)
    if not walker_valid(p):
        return 0.0, 0.0, -math.inf
    w = weights(freqs, psd)
    h = template(table, params, freqs, S, t0, mode)
    dh = inner(data, h, w)
    hh = inner(h, h, w)
    dd = inner(data, data, w)
    return dh, hh, dh - 0.5 * hh - 0.5 * dd


def loglike_direct_residual(table, params, freqs, data, psd, S, t0=0.0, mode="spline"):
    """-1/2 <d-h|d-h> accumulated directly (left side of eq. 2)."""
    w = weights(freqs, psd)
    h = template(table, params, freqs, S, t0, mode)
    r = data - h
    return -0.5 * inner(r, r, w)


def mode_products(table, params, freqs, data, psd, S, t0=0.0):
    """Per-mode inner products (Table III :292-300): for each mode evaluated in isolation,
    (<d|h_lm>, <h_lm|h_lm>); the optimal SNR of the mode alone is <h_lm|h_lm>^(1/2).
    Returns two arrays of length 6 in the mode order of PAPER.md:122."""
    w = weights(freqs, psd)
    dh = np.zeros(len(MODES))
    hh = np.zeros(len(MODES))
    for i in range(len(MODES)):
        h = template(table, params, freqs, S, t0, mode_mask=1 << i)
        dh[i] = inner(data, h, w)
        hh[i] = inner(h, h, w)
    return dh, hh
