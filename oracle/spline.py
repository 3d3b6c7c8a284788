"""Oracle: not-a-knot cubic spline ("cubic spline ... Scipy").

Unknowns are the knot slopes s_j; the tridiagonal system is solved with the
Thomas algorithm.  TEST INFRASTRUCTURE - see oracle/__init__.py.
"""
import numpy as np


def notaknot_slopes(x, y):
    """Slopes s_j of the not-a-knot cubic spline through (x_j, y_j); needs len(x) >= 4."""
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    S = x.size
    h = np.diff(x)
    dl = np.diff(y) / h                      # delta_j
    lower = np.zeros(S)
    diag = np.zeros(S)
    upper = np.zeros(S)
    rhs = np.zeros(S)
    for j in range(1, S - 1):
        lower[j] = h[j]
        diag[j] = 2.0 * (h[j - 1] + h[j])
        upper[j] = h[j - 1]
        rhs[j] = 3.0 * (h[j] * dl[j - 1] + h[j - 1] * dl[j])
    diag[0] = h[1]
    upper[0] = h[0] + h[1]
    rhs[0] = ((3.0 * h[0] + 2.0 * h[1]) * h[1] * dl[0] + h[0] ** 2 * dl[1]) / (h[0] + h[1])
    lower[S - 1] = h[S - 2] + h[S - 3]
    diag[S - 1] = h[S - 3]
    rhs[S - 1] = (h[S - 2] ** 2 * dl[S - 3] + (2.0 * h[S - 3] + 3.0 * h[S - 2]) * h[S - 3] * dl[S - 2]) \
        / (h[S - 3] + h[S - 2])
    # Thomas algorithm
    cp = np.zeros(S)
    dp = np.zeros(S)
    cp[0] = upper[0] / diag[0]
    dp[0] = rhs[0] / diag[0]
    for j in range(1, S):
        den = diag[j] - lower[j] * cp[j - 1]
        cp[j] = upper[j] / den
        dp[j] = (rhs[j] - lower[j] * dp[j - 1]) / den
    s = np.zeros(S)
    s[S - 1] = dp[S - 1]
    for j in range(S - 2, -1, -1):
        s[j] = dp[j] - cp[j] * s[j + 1]
    return s


def coefficients(x, y):
    """Per-interval (y_j, s_j, c_j, d_j): p(tau) = y_j + s_j tau + c_j tau^2 + d_j tau^3, tau = f - x_j."""
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    s = notaknot_slopes(x, y)
    h = np.diff(x)
    dl = np.diff(y) / h
    c = (3.0 * dl - 2.0 * s[:-1] - s[1:]) / h
    d = (s[:-1] + s[1:] - 2.0 * dl) / (h * h)
    return np.stack([y[:-1], s[:-1], c, d], axis=1)       # [S-1, 4]


def evaluate(x, coef, f):
    """Evaluates the spline at f (right-continuous interval choice, G12; f must lie in [x_0, x_{S-1}])."""
    x = np.asarray(x, dtype=np.float64)
    f = np.asarray(f, dtype=np.float64)
    j = np.clip(np.searchsorted(x, f, side="right") - 1, 0, x.size - 2)
    tau = f - x[j]
    c = coef[j]
    return c[:, 0] + tau * (c[:, 1] + tau * (c[:, 2] + tau * c[:, 3]))
