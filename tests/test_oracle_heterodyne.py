"""Pins of the heterodyned likelihood variant's oracle (oracle/heterodyne.py)."""
import numpy as np

from oracle import heterodyne as H
from oracle import likelihood as L
from paper_2005_01827_b200 import workloads as W


def small_problem(table, n_bins=4096, S=64):
    wl = W.build(0, lambda p, f, Sp: L.template(table, p, f, Sp), n_bins=n_bins, batch=4)
    wl["S"] = S
    return wl


def test_one_fine_bin_per_coarse_bin_is_the_brute_force_likelihood(table):
    # with edges = 0, 1, ..., N every envelope value is used where it was evaluated: the variant reduces to eqs. 2, 3, 11
    wl = small_problem(table, n_bins=1500)
    edges = np.arange(wl["freqs"].size + 1)
    inj = wl["injections"][0]
    summ = H.setup(table, inj, wl["freqs"], wl["data"], wl["psd"], wl["S"], edges)
    rng = np.random.default_rng(51)
    for p in [inj] + list(W.perturb(rng, inj, 2, 1e-5)):
        dh, hh, ll = H.loglike_parts(table, summ, p)
        rdh, rhh, rll = L.loglike_parts(table, p, wl["freqs"], wl["data"], wl["psd"], wl["S"])
        # (the two differ only where the walker's band and the reference's differ by a bin, reading H1: not here)
        assert abs(hh - rhh) <= 1e-9 * rhh and abs(dh - rdh) <= 1e-9 * max(abs(rdh), rhh), (dh, rdh, hh, rhh)
        assert abs(ll - rll) <= 1e-8 * (1.0 + abs(rll))


def test_error_is_small_and_falls_with_the_coarse_bin_width(table):
    # parabolic interpolation of a smooth envelope: already 64 coarse bins over 4096 fine bins give <h|h> to 1e-5; the
    # error falls with the bin width (not monotonically at every step: what remains comes from the few coarse bins that
    # hold a band edge or a C1 kink of the model) and logL agrees with brute force to a small fraction of a unit
    wl = small_problem(table)
    inj = wl["injections"][0]
    rng = np.random.default_rng(52)
    walker = W.perturb(rng, inj, 1, 3e-6)[0]
    ref = L.loglike_parts(table, walker, wl["freqs"], wl["data"], wl["psd"], wl["S"])
    ref0 = L.loglike_parts(table, inj, wl["freqs"], wl["data"], wl["psd"], wl["S"])
    errs, errs0, dll = [], [], []
    for nb in (32, 64, 256, 1024):
        edges = W.het_edges(wl["freqs"], nb)
        summ = H.setup(table, inj, wl["freqs"], wl["data"], wl["psd"], wl["S"], edges)
        dh, hh, ll = H.loglike_parts(table, summ, walker)
        errs.append(max(abs(hh - ref[1]), abs(dh - ref[0])) / ref[1])
        dll.append(abs(ll - ref[2]))
        errs0.append(abs(H.loglike_parts(table, summ, inj)[1] - ref0[1]) / ref0[1])
    assert max(errs) < 1e-5 and max(errs0) < 1e-5, (errs, errs0)
    assert errs[3] < 1e-7 and errs[3] < max(errs[:2]) / 20.0 and errs[2] < max(errs[:2]) / 3.0, errs
    assert dll[3] < 1e-3 and dll[1] < 0.05, dll


def test_edges_generator_and_degenerate_inputs(table):
    wl = small_problem(table, n_bins=700)
    e = W.het_edges(wl["freqs"], 50)
    assert e[0] == 0 and e[-1] == wl["freqs"].size and np.all(np.diff(e) > 0) and e.size <= 51
    summ = H.setup(table, wl["injections"][0], wl["freqs"], wl["data"], wl["psd"], wl["S"], e)
    bad = wl["injections"][0].copy()
    bad[4] = -1.0
    assert H.loglike_parts(table, summ, bad)[2] == -np.inf
    heavy = wl["injections"][0].copy()
    heavy[0] = 1e10                                   # every band below the grid: no signal
    dh, hh, ll = H.loglike_parts(table, summ, heavy)
    assert dh == 0.0 and hh == 0.0 and ll == -0.5 * summ["dd"]
