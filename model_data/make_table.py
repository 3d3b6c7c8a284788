#!/usr/bin/env python3
"""Writes model_data/phenomhm_table.csv -- the numeric table of the waveform model.

PAPER.md:110-116 uses PhenomHM [70,71,76]; PAPER.md prints none of that model's
numbers and the cited papers are not available offline.
The *structure* of the model (which fits exist, their functional forms) follows
SURVEY.md 8(c) O1-O3; the *numbers* are kept in one data file with a provenance
tag per entry:

  derived    closed form re-derived for this build (DESIGN.md says from what)
  published  short rounded values printed in the cited literature, recalled
             offline and NOT re-verified (treat as surrogate if in doubt)
  surrogate  smooth stand-in designed here so that the model is well behaved
             (positive amplitudes, monotone inspiral t(f), gamma2 < 1, ...);
             NOT the published PhenomD/PhenomHM calibration.

This file is data for both the oracle and the CUDA library (each parses or
bakes it with its own code).  It contains no arithmetic of the method.
Run:  python model_data/make_table.py   (rewrites the CSV deterministically)
"""
import math
import os

import numpy as np

ORDER11 = ["l00", "l10", "l01", "l11", "l21", "l02", "l12", "l22", "l03", "l13", "l23"]

# name: (n0, n1, s1, s2, s3, n2, (u1,u2,u3))
#   Lambda(eta, chi) = (n0 + n1 eta) (1 + s1 chi + s2 chi^2 + s3 chi^3)
#                      + n2 eta^2 (chi - 1)(u1 + u2 chi + u3 chi^2)
# re-expanded in x = chi - 1 into the 11 slots of the bilinear-cubic fit form
# of SURVEY.md 8(c) O1.
DESIGN = {
    # inspiral amplitude pseudo-PN terms
    "rho1":   (3900.0, -17400.0, 0.10, 0.02, 0.00, 900.0, (1.0, 0.3, 0.1)),
    "rho2":   (-40100.0, 112000.0, 0.12, -0.03, 0.01, -5000.0, (1.0, -0.2, 0.1)),
    "rho3":   (83200.0, -191000.0, 0.08, 0.02, -0.01, 9000.0, (1.0, 0.2, -0.1)),
    # intermediate amplitude collocation value at f2
    "v2":     (0.92, 1.90, 0.10, 0.03, 0.01, 0.4, (1.0, 0.2, 0.1)),
    # merger-ringdown amplitude
    "gamma1": (0.0105, 0.0460, 0.15, 0.05, 0.02, 0.004, (1.0, 0.2, 0.1)),
    "gamma2": (0.78, 0.28, -0.08, 0.02, 0.01, 0.10, (1.0, -0.3, 0.1)),
    "gamma3": (1.31, -0.02, -0.03, 0.01, 0.00, 0.05, (1.0, 0.2, 0.0)),
    # inspiral phase pseudo-PN terms
    "sigma1": (2100.0, 1460.0, 0.05, 0.01, 0.00, 300.0, (1.0, 0.1, 0.1)),
    "sigma2": (-300.0, -1000.0, 0.10, 0.02, 0.01, -400.0, (1.0, 0.2, 0.1)),
    "sigma3": (500.0, 2000.0, 0.10, 0.02, 0.01, 900.0, (1.0, 0.2, 0.1)),
    # sigma4 carries the curvature that keeps t(f) monotone for anti-aligned spins
    "sigma4": (-8000.0, 0.0, 6.25, -1.25, 0.0, 2000.0, (1.0, 0.2, 0.1)),
    # intermediate phase
    "beta1":  (97.9, -42.7, 0.05, 0.01, 0.00, 10.0, (1.0, 0.1, 0.1)),
    "beta2":  (-3.28, -9.05, 0.10, 0.03, 0.01, -1.0, (1.0, 0.2, 0.1)),
    "beta3":  (-2.5e-5, 1.98e-5, 0.15, 0.04, 0.01, -3.0e-6, (1.0, 0.2, 0.1)),
    # merger-ringdown phase
    "alpha1": (43.3, 639.0, 0.05, 0.01, 0.00, 30.0, (1.0, 0.1, 0.1)),
    "alpha2": (-0.070, -0.162, 0.10, 0.03, 0.01, -0.02, (1.0, 0.2, 0.1)),
    "alpha3": (9.6, -397.0, 0.08, 0.02, 0.01, -20.0, (1.0, 0.2, 0.1)),
    "alpha4": (0.030, 1.02, 0.06, 0.02, 0.01, 0.10, (1.0, 0.2, 0.1)),
    "alpha5": (0.9974, -0.0079, 0.004, -0.002, 0.001, 0.004, (1.0, 0.2, 0.1)),
}


def eleven(n0, n1, s1, s2, s3, n2, u):
    # P(chi) = 1 + s1 chi + s2 chi^2 + s3 chi^3 with chi = x + 1
    P = np.polynomial.polynomial.Polynomial([1.0, s1, s2, s3])
    Px = P(np.polynomial.polynomial.Polynomial([1.0, 1.0])).coef  # in powers of x
    Px = np.pad(Px, (0, 4 - len(Px)))
    # Q(chi) = (chi-1)(u1 + u2 chi + u3 chi^2) = x (u1 + u2 (x+1) + u3 (x+1)^2)
    u1, u2, u3 = u
    q1 = u1 + u2 + u3
    q2 = u2 + 2.0 * u3
    q3 = u3
    vals = {
        "l00": n0 * Px[0], "l10": n1 * Px[0],
        "l01": n0 * Px[1], "l11": n1 * Px[1], "l21": n2 * q1,
        "l02": n0 * Px[2], "l12": n1 * Px[2], "l22": n2 * q2,
        "l03": n0 * Px[3], "l13": n1 * Px[3], "l23": n2 * q3,
    }
    return [vals[k] for k in ORDER11]


def rows():
    out = []
    for name, d in DESIGN.items():
        for k, v in zip(ORDER11, eleven(*d)):
            out.append((f"pd.{name}.{k}", v, "surrogate"))
    # Final spin, polynomial in eta and total spin S = m1^2 a1 + m2^2 a2 (form of ref [70]).
    tag = "published"
    for k, v in [("e2", -4.399), ("e3", 9.397), ("e4", -13.181),
                 ("s1e1", -0.085), ("s2e1", 0.102), ("s3e1", -1.355), ("s4e1", -0.868),
                 ("s1e2", -5.837), ("s2e2", -2.097), ("s3e2", 4.109), ("s4e2", 2.064)]:
        out.append((f"fs.spin.{k}", v, tag))
    # Radiated energy, rational in effective spin S/(1-2 eta) (form of ref [70]).
    for k, v in [("e1", 0.0559745), ("e2", 0.580951), ("e3", -0.960673), ("e4", 3.35241),
                 ("n0", -0.00303023), ("n1", -2.00661), ("n2", 7.70506),
                 ("d0", -0.671440), ("d1", -1.47569), ("d2", 7.30468)]:
        out.append((f"fs.erad.{k}", v, tag))
    # Quasi-normal modes (l,m,0): M omega = f1 + f2 (1-a)^f3, Q = q1 + q2 (1-a)^q3
    qnm = {
        "22": (1.5251, -1.1568, 0.1292, 0.7000, 1.4187, -0.4990),
        "33": (1.8956, -1.3043, 0.1818, 0.9000, 2.3430, -0.4810),
        "44": (2.3000, -1.5056, 0.2244, 1.1929, 3.1191, -0.4825),
        "21": (0.6000, -0.2339, 0.4175, -0.3000, 2.3561, -0.2277),
        "32": (1.1481, -0.5552, 0.3002, 0.8313, 2.3773, -0.3655),
        "43": (1.6869, -0.8862, 0.2822, 1.4812, 2.8096, -0.4271),
    }
    for lm, v in qnm.items():
        for k, x in zip(("f1", "f2", "f3", "q1", "q2", "q3"), v):
            out.append((f"qnm.{lm}.{k}", x, tag))
    # Leading-PN frequency-domain mode amplitudes |H_lm| = c_lm * massfactor * V^p
    # (derived from the time-domain multipoles by the stationary-phase factor
    # sqrt(2/m); DESIGN.md section "Higher modes"), and the constant phase offsets
    # Delta_lm = (1 - m/2) pi/4 + arg[(-1)^l conj(H^TD_lm)].
    s = math.sqrt
    pi = math.pi
    hm = {
        "22": (1.0, 0.0),
        "33": (0.75 * s(5.0 / 7.0), -pi / 8.0 - pi / 2.0),
        "44": (4.0 / 9.0 * s(10.0 / 7.0), -pi / 4.0 + pi),
        "21": (s(2.0) / 3.0, pi / 8.0 + pi / 2.0),
        "32": (1.0 / 3.0 * s(5.0 / 7.0), pi),
        "43": (0.75 * s(3.0 / 35.0), -pi / 8.0 + pi / 2.0),
    }
    for lm, (c, dphi) in hm.items():
        out.append((f"hm.{lm}.amp", c, "derived"))
        out.append((f"hm.{lm}.dphi", dphi, "derived"))
    return out


def main():
    here = os.path.dirname(os.path.abspath(__file__))
    path = os.path.join(here, "phenomhm_table.csv")
    with open(path, "w") as fh:
        fh.write("# name,value,provenance  -- written by model_data/make_table.py; see its docstring\n")
        for name, v, tag in rows():
            fh.write(f"{name},{float(v)!r},{tag}\n")
    print("wrote", path, len(rows()), "entries")


if __name__ == "__main__":
    main()
