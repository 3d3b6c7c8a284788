#!/usr/bin/env python3
"""Prints the polynomial coefficients of sincos_qturn() in mbhl_kernels.cuh.

sin(pi y / 2) = y * Ps(y^2) and cos(pi y / 2) = Pc(y^2) for |y| <= 1/2 (y in quarter turns).
Ps, Pc: degree-6 polynomials in z = y^2 on [0, 1/4], obtained by interpolation at Chebyshev nodes in
50-digit arithmetic (near-minimax), converted to the monomial basis and rounded to double.  The script
also reports the maximum error of the rounded polynomials evaluated in 50-digit arithmetic.
Run: python paper_2005_01827_b200/csrc/gen_sincos_coeffs.py      (documentation of provenance; not imported)
"""
import mpmath as mp

mp.mp.dps = 50
DEG = 6
A, B = mp.mpf(0), mp.mpf(1) / 4


def gs(z):
    if z == 0:
        return mp.pi / 2
    r = mp.sqrt(z)
    return mp.sin(mp.pi * r / 2) / r


def gc(z):
    return mp.cos(mp.pi * mp.sqrt(z) / 2)


def cheb_fit(g, deg):
    n = deg + 1
    nodes = [(A + B) / 2 + (B - A) / 2 * mp.cos(mp.pi * (2 * k + 1) / (2 * n)) for k in range(n)]
    V = mp.matrix(n, n)
    rhs = mp.matrix(n, 1)
    for i, x in enumerate(nodes):
        for j in range(n):
            V[i, j] = x ** j
        rhs[i] = g(x)
    return [mp.lu_solve(V, rhs)[j] for j in range(n)]


def max_err(coefs, fn, odd):
    worst = mp.mpf(0)
    for i in range(0, 4001):
        y = mp.mpf(i) / 8000
        z = y * y
        p = mp.mpf(0)
        for c in reversed(coefs):
            p = p * z + mp.mpf(c)
        val = p * y if odd else p
        worst = max(worst, abs(val - fn(mp.pi * y / 2)))
    return worst


for name, g, fn, odd in (("S", gs, mp.sin, True), ("C", gc, mp.cos, False)):
    c = [float(v) for v in cheb_fit(g, DEG)]
    print(f"// {name}: max abs error of the rounded polynomial = {mp.nstr(max_err(c, fn, odd), 3)}")
    for k, v in enumerate(c):
        print(f"constexpr double k{name}{k} = {v!r};")

# the shorter pair of the fused dense kernel (sincos_qturn_x in mbhl_dense.cuh, array c_scd): sine of degree 4 and
# cosine of degree 5 in z; their errors (3.4e-12, 5.6e-14) sit far below the 1e-9 per-bin bar of the template
for name, g, fn, odd, deg in (("DS", gs, mp.sin, True, 4), ("DC", gc, mp.cos, False, 5)):
    c = [float(v) for v in cheb_fit(g, deg)]
    print(f"// {name} (degree {deg}): max abs error of the rounded polynomial = {mp.nstr(max_err(c, fn, odd), 3)}")
    for k, v in enumerate(c):
        print(f"constexpr double k{name}{k} = {v!r};")
