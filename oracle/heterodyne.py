"""Oracle: heterodyned ("relative binning") likelihood, an accuracy-controlled variant of the hot path.

PAPER.md:177 leaves this open ("In the future, we may test different approximations in our GPU implementation to gain
even more performance"); SURVEY.md 8(f).4 names heterodyned / relative-binning sums.  The definition used here
(reading H1) follows the algorithm step by step.  TEST INFRASTRUCTURE - see oracle/__init__.py.

Reference parameters Theta0 give, per mode m, a reference phasor on the fine grid
    E0_m(k) = exp(i theta0_m(f_k))   inside the reference band of mode m, 0 outside,
theta0_m the total phase of the SPLINE template of Theta0 (Phi - 2 pi f t_coal, O7).  A walker's template is written as
    h^c(f_k) = sum_m r_{c,m}(f_k) E0_m(k),   r_{c,m}(f) = A_m(f) That^c_m(f) exp(i [theta_m(f) - theta0_m(f)]),
and r, which is smooth for a walker near Theta0, is replaced on every coarse bin b = [e_b, e_{b+1}) by the parabola
through its values at the bin's first frequency f_L, its centre fbar = (f_L + f_R)/2 and its last frequency f_R:
r ~ r0 + r1 x + r2 x^2, x = f - fbar, s = (f_R - f_L)/2, r0 = r(fbar), r1 = (r(f_R) - r(f_L))/(2 s),
r2 = (r(f_R) - 2 r(fbar) + r(f_L))/(2 s^2) (r1 = r2 = 0 for a one-bin coarse bin).  Then (eqs. 2, 3, 11), with the
moments A_n = sum_{k in b} w_c conj(d_c) E0_m x_k^n and B_n = sum_{k in b} w_c E0_m conj(E0_m') x_k^n, n = 0, 1, 2,
    <d|h> ~ Re sum_{c,m,b} [A0 r0 + A1 r1 + A2 r2],
    <h|h> ~ Re sum_{c,b} sum_{m,m'} [B0 r0 conj(r0') + B1 (r1 conj(r0') + r0 conj(r1')) + B2 (r2 conj(r0') + r1 conj(r1') + r0 conj(r2'))]
(terms in x^3, x^4 dropped).  The summary data A, B are computed once per reference; a walker
costs its sparse stage plus 3 n_b spline evaluations per mode.  The band of a mode is taken to be the reference's
(the summary data hold it); where f_L or f_R lies outside the band common to walker and reference, r is taken at the
nearest frequency inside it (no spline is ever extrapolated) - but only on coarse bins that the walker's own band
reaches: a coarse bin lying wholly outside the walker's band [f_lo, f_hi] of a mode gets r = 0 for that mode, as in the
brute-force sums, where the mode contributes nothing there (reading H1, amended: moving all three points of such a bin to
the band edge would give it a constant non-zero envelope, an error that does not shrink with the bin width).  The coarse bins actually used are the caller's edges
REFINED by the reference's band edges (first in-band bin and one past the last of every mode), so that on every coarse
bin a mode is either in band throughout or absent: without this the bins that hold a band edge dominate the error.
With one fine bin per coarse bin the variant IS the
brute-force spline likelihood (for a walker whose bands hold the same bins as the reference's).
"""
import math

import numpy as np

from . import likelihood as L
from . import spline as ospline
from .constants import MODES

TWO_PI = 2.0 * math.pi


def _cycles(Phi, f, t_coal):
    """Total phase Phi - 2 pi f t_coal in cycles mod 1, the linear term taken exactly (G9), as L._combine does."""
    lin = np.asarray(f, dtype=np.longdouble) * np.longdouble(t_coal)
    lin = lin - np.rint(lin)
    cyc = Phi / TWO_PI
    return (cyc - np.rint(cyc)) - lin.astype(np.float64)


def setup(table, params_ref, freqs, data, psd, S, edges, t0=0.0):
    """Summary data of the reference Theta0 on the coarse bins given by `edges` (bin indices, 0 ... N)."""
    freqs = np.asarray(freqs, dtype=np.float64)
    w = L.weights(freqs, psd)
    modes, t_coal = L.sparse_stage(table, params_ref, freqs[0], freqs[-1], S, t0)
    band = []
    for mo in modes:
        if mo is not None:
            k_lo = int(np.searchsorted(freqs, mo["knots"][0], side="left"))
            k_hi = int(np.searchsorted(freqs, mo["knots"][-1], side="right")) - 1
            if k_hi >= k_lo:
                band += [k_lo, k_hi + 1]
    edges = np.unique(np.concatenate([np.asarray(edges, dtype=np.int64), np.asarray(band, dtype=np.int64)]))
    nb = edges.size - 1
    E0 = np.zeros((len(MODES), freqs.size), dtype=np.complex128)
    for m, mo in enumerate(modes):
        if mo is None:
            continue
        x = mo["knots"]
        sel = np.nonzero((freqs >= x[0]) & (freqs <= x[-1]))[0]
        Phi = ospline.evaluate(x, mo["coef"][:, 1, :], freqs[sel])
        th = TWO_PI * _cycles(Phi, freqs[sel], t_coal)
        E0[m, sel] = np.cos(th) + 1j * np.sin(th)
    fL = freqs[edges[:-1]]
    fR = freqs[edges[1:] - 1]
    fbar = 0.5 * (fL + fR)
    A0 = np.zeros((3, len(MODES), nb), dtype=np.complex128)
    A1 = np.zeros_like(A0)
    A2 = np.zeros_like(A0)
    B0 = np.zeros((3, len(MODES), len(MODES), nb), dtype=np.complex128)
    B1 = np.zeros_like(B0)
    B2 = np.zeros_like(B0)
    for b in range(nb):
        k = slice(edges[b], edges[b + 1])
        d = freqs[k] - fbar[b]
        for c in range(3):
            wd = w[c, k] * np.conj(data[c, k])
            for m in range(len(MODES)):
                A0[c, m, b] = np.sum(wd * E0[m, k])
                A1[c, m, b] = np.sum(wd * E0[m, k] * d)
                A2[c, m, b] = np.sum(wd * E0[m, k] * d * d)
                for mp in range(len(MODES)):
                    pr = w[c, k] * E0[m, k] * np.conj(E0[mp, k])
                    B0[c, m, mp, b] = np.sum(pr)
                    B1[c, m, mp, b] = np.sum(pr * d)
                    B2[c, m, mp, b] = np.sum(pr * d * d)
    return dict(edges=edges, fL=fL, fR=fR, A0=A0, A1=A1, A2=A2, B0=B0, B1=B1, B2=B2, ref_modes=modes, ref_t_coal=t_coal,
                dd=L.inner(data, data, w), freqs=freqs, S=S, t0=t0)


def _envelope(walker_modes, t_coal, summary, f):
    """r[c, m, :] at frequencies f, each moved to the nearest frequency inside the band common to walker and reference."""
    r = np.zeros((3, len(MODES), f.size), dtype=np.complex128)
    f_in = f
    for m in range(len(MODES)):
        mo, ref = walker_modes[m], summary["ref_modes"][m]
        if mo is None or ref is None:
            continue
        lo, hi = max(mo["knots"][0], ref["knots"][0]), min(mo["knots"][-1], ref["knots"][-1])
        if not lo <= hi:
            continue
        f = np.clip(f_in, lo, hi)
        q = np.stack([ospline.evaluate(mo["knots"], mo["coef"][:, qi, :], f) for qi in range(L.NQ)])
        Phi0 = ospline.evaluate(ref["knots"], ref["coef"][:, 1, :], f)
        dth = TWO_PI * (_cycles(q[1], f, t_coal) - _cycles(Phi0, f, summary["ref_t_coal"]))
        e = q[0] * (np.cos(dth) + 1j * np.sin(dth))
        # coarse bins (f has one entry per bin) that the walker's own band does not reach: the mode is absent there
        reached = (summary["fR"] >= mo["knots"][0]) & (summary["fL"] <= mo["knots"][-1])
        for c in range(3):
            r[c, m] = np.where(reached, e * (q[2 + 2 * c] + 1j * q[3 + 2 * c]), 0.0)
    return r


def loglike_parts(table, summary, params):
    """(<d|h>, <h|h>, logL) of one walker from the summary data (the heterodyned sums above)."""
    p = L.unpack(params)
    if not L.walker_valid(p):
        return 0.0, 0.0, -math.inf
    modes, t_coal = L.sparse_stage(table, params, summary["freqs"][0], summary["freqs"][-1], summary["S"], summary["t0"])
    fL, fR = summary["fL"], summary["fR"]
    rL = _envelope(modes, t_coal, summary, fL)
    rM = _envelope(modes, t_coal, summary, 0.5 * (fL + fR))
    rR = _envelope(modes, t_coal, summary, fR)
    s = 0.5 * (fR - fL)
    ok = s > 0.0
    s1 = np.where(ok, s, 1.0)
    r0 = rM
    r1 = np.where(ok, (rR - rL) / (2.0 * s1), 0.0)
    r2 = np.where(ok, (rR - 2.0 * rM + rL) / (2.0 * s1 * s1), 0.0)
    dh = float(np.sum((summary["A0"] * r0 + summary["A1"] * r1 + summary["A2"] * r2).real.astype(np.longdouble)))
    a = lambda r: r[:, :, None, :]                 # mode m
    bc = lambda r: np.conj(r[:, None, :, :])       # conj, mode m'
    t = (summary["B0"] * a(r0) * bc(r0)
         + summary["B1"] * (a(r1) * bc(r0) + a(r0) * bc(r1))
         + summary["B2"] * (a(r2) * bc(r0) + a(r1) * bc(r1) + a(r0) * bc(r2)))
    hh = float(np.sum(t.real.astype(np.longdouble)))
    return dh, hh, dh - 0.5 * hh - 0.5 * summary["dd"]
