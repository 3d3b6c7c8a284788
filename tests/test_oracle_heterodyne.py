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


def test_order_of_convergence_on_a_window_without_band_edges_or_model_kinks(table):
    # What mbhl.h promises for mbhl_het_*: the error falls at least with the CUBE of the coarse bin width.  A parabola through
    # three points of a smooth envelope leaves an error r''' x (x^2 - s^2) / 6, odd about the bin centre, whose sum against
    # slowly varying weights cancels to leading order - so on clean bins the sums converge with the FOURTH power (a factor 16
    # per halving).  The window is chosen so that nothing else contributes: 0.3-1.2 mHz for a 1e6 Msun binary 2e7 s before
    # merger lies inside the band of all six modes (every f_lo is below the window, every f_hi above) and inside the inspiral
    # region of every mode's amplitude and phase maps ((2,1): M f < 0.007), the data are the noise-free injection, and the
    # walker sits 1e-4 (relative) away from the reference so that the errors stay far above rounding.  Dropping the
    # second-order moments (A2, B2) or mis-centring the parabola turns this into second-order convergence (a factor 4).
    n = 4096
    freqs = np.linspace(3e-4, 1.2e-3, n)
    psd = W.scird_psd_aet(freqs)
    S = 128
    inj = np.array([1e6, 3.0, 0.6, -0.3, 10.0, 1.3, 0.9, 2.1, 0.4, 0.7, 2.0e7])
    for mo in L.sparse_stage(table, inj, freqs[0], freqs[-1], S, 0.0)[0]:
        assert mo is not None and mo["knots"][0] == freqs[0] and mo["knots"][-1] == freqs[-1]     # in band throughout
    data = L.template(table, inj, freqs, S)
    walker = W.perturb(np.random.default_rng(5), inj, 1, 1e-4)[0]
    rdh, rhh, _ = L.loglike_parts(table, walker, freqs, data, psd, S)
    e_hh, e_dh = [], []
    for nb in (8, 16, 32, 64):
        edges = np.unique(np.round(np.linspace(0, n, nb + 1)).astype(np.int64))
        summ = H.setup(table, inj, freqs, data, psd, S, edges)
        assert summ["edges"].size == nb + 1                                                       # no band edge refined the bins
        dh, hh, _ = H.loglike_parts(table, summ, walker)
        e_hh.append(abs(hh - rhh) / rhh)
        e_dh.append(abs(dh - rdh) / rhh)
    for a, b in ((0, 1), (1, 2)):
        assert 10.0 < e_hh[a] / e_hh[b] < 24.0, e_hh          # fourth order: 16 per halving
        assert e_dh[a] / e_dh[b] > 8.0, e_dh                   # at least third
    assert e_hh[0] / e_hh[3] > 512.0 and e_dh[0] / e_dh[3] > 512.0, (e_hh, e_dh)      # at least the cube over three halvings
    assert e_hh[0] < 1e-3 and e_hh[3] < 1e-6


def test_coarse_bins_outside_the_walkers_own_band_contribute_nothing(table):
    # Reading H1 (amended): a walker whose band starts LATER than the reference's (a smaller t_ref: every f_lo moves up) has no
    # signal in the coarse bins between the two band edges; the brute-force sums skip those bins, so must the heterodyned ones.
    # With one fine bin per coarse bin the parabola plays no role and the two must agree to rounding - before the amendment the
    # bins in between carried the envelope of the band edge (a few bins per mode here, a relative error of ~1e-3).
    wl = small_problem(table, n_bins=1500)
    freqs = wl["freqs"]
    inj = wl["injections"][0]
    summ = H.setup(table, inj, freqs, wl["data"], wl["psd"], wl["S"], np.arange(freqs.size + 1))
    walker = inj.copy()
    walker[10] *= 0.97
    ref_modes = L.sparse_stage(table, inj, freqs[0], freqs[-1], wl["S"])[0]
    w_modes = L.sparse_stage(table, walker, freqs[0], freqs[-1], wl["S"])[0]
    df = freqs[1] - freqs[0]
    gaps = [(w["knots"][0] - r["knots"][0]) / df for w, r in zip(w_modes, ref_modes) if w is not None and r is not None]
    assert min(gaps) > 1.5, gaps                       # every mode's band starts at least two fine bins later than the reference's
    dh, hh, ll = H.loglike_parts(table, summ, walker)
    rdh, rhh, rll = L.loglike_parts(table, walker, freqs, wl["data"], wl["psd"], wl["S"])
    assert abs(hh - rhh) <= 1e-9 * rhh and abs(dh - rdh) <= 1e-9 * max(abs(rdh), rhh), (dh, rdh, hh, rhh)
    assert abs(ll - rll) <= 1e-8 * (1.0 + abs(rll))
