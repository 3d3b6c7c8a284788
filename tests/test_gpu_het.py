"""GPU parity of the heterodyned likelihood variant (mbhl_het_*) against oracle/heterodyne.py, and its
accuracy against the brute-force path (mbhl_loglike_parts) on the same device."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import heterodyne as H
from oracle import likelihood as L
from paper_2005_01827_b200 import binding as M
from paper_2005_01827_b200 import workloads as W

DEV = "cuda:0"


def dev(x):
    return torch.as_tensor(np.ascontiguousarray(x), device=DEV)


def test_het_parity_small(table):
    wl = W.build(0, lambda p, f, Sp: L.template(table, p, f, Sp), n_bins=4096, batch=4)
    S = 64
    ctx = M.mbhl_init(dev(wl["freqs"]), dev(wl["data"]), dev(wl["psd"]), sparse_points=S, t0=wl["t0"])
    inj = wl["injections"][0]
    rng = np.random.default_rng(61)
    walkers = np.concatenate([inj[None, :], W.perturb(rng, inj, 3, 3e-6), W.perturb(rng, inj, 2, 1e-4)])
    bad = inj.copy()
    bad[4] = -1.0
    heavy = inj.copy()
    heavy[0] = 1e10
    walkers = np.concatenate([walkers, bad[None, :], heavy[None, :]])
    brute = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(walkers))]
    for nb in (37, 256, wl["freqs"].size):
        edges = W.het_edges(wl["freqs"], nb) if nb < wl["freqs"].size else np.arange(wl["freqs"].size + 1)
        summ = H.setup(table, inj, wl["freqs"], wl["data"], wl["psd"], S, edges, wl["t0"])
        het = M.mbhl_het_init(ctx, dev(inj), edges)
        dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_het_loglike(het, dev(walkers))]
        for b in range(6):
            rdh, rhh, rll = H.loglike_parts(table, summ, walkers[b])
            assert abs(hh[b] - rhh) <= 1e-8 * rhh, (nb, b, hh[b], rhh)
            assert abs(dh[b] - rdh) <= 1e-8 * max(abs(rdh), rhh), (nb, b, dh[b], rdh)
            assert abs(ll[b] - rll) <= 1e-6 * (1.0 + abs(rll)), (nb, b, ll[b], rll)
        assert np.isneginf(ll[6]) and dh[6] == 0.0 and hh[6] == 0.0
        assert ll[7] == -0.5 * M.mbhl_data_norm(ctx) and hh[7] == 0.0
        if nb == wl["freqs"].size:      # one fine bin per coarse bin: the variant is the brute-force likelihood
            for b in range(4):
                assert abs(hh[b] - brute[1][b]) <= 1e-9 * brute[1][b] and abs(ll[b] - brute[2][b]) <= 1e-8 * (1.0 + abs(brute[2][b]))
        M.mbhl_het_free(het)
    # argument checks
    with pytest.raises(M.MbhlError):
        M.mbhl_het_init(ctx, dev(inj), np.array([0, 5, 5, wl["freqs"].size]))
    with pytest.raises(M.MbhlError):
        M.mbhl_het_init(ctx, dev(inj), np.array([1, 5, wl["freqs"].size]))
    with pytest.raises(M.MbhlError):
        M.mbhl_het_init(ctx, dev(bad), W.het_edges(wl["freqs"], 16))
    M.mbhl_free(ctx)


def test_het_walker_with_a_band_that_starts_later_than_the_references(table):
    # Reading H1 as amended in round 3: coarse bins that the walker's own band does not reach contribute nothing.  A walker with
    # a smaller t_ref has every f_lo above the reference's.  GPU against the oracle on ragged coarse bins, and - with one fine
    # bin per coarse bin, where the parabola plays no role - GPU heterodyne against the GPU brute-force path.
    wl = W.build(0, lambda p, f, Sp: L.template(table, p, f, Sp), n_bins=1500, batch=4)
    S = 64
    freqs = wl["freqs"]
    ctx = M.mbhl_init(dev(freqs), dev(wl["data"]), dev(wl["psd"]), sparse_points=S, t0=wl["t0"])
    inj = wl["injections"][0]
    shifted = inj.copy()
    shifted[10] *= 0.97                                  # bands start a few fine bins later in every mode
    later = inj.copy()
    later[10] *= 0.999
    walkers = np.stack([shifted, later, inj])
    brute = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(walkers))]
    for nb in (64, freqs.size):
        edges = W.het_edges(freqs, nb) if nb < freqs.size else np.arange(freqs.size + 1)
        summ = H.setup(table, inj, freqs, wl["data"], wl["psd"], S, edges, wl["t0"])
        het = M.mbhl_het_init(ctx, dev(inj), edges)
        dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_het_loglike(het, dev(walkers))]
        for b in range(3):
            rdh, rhh, rll = H.loglike_parts(table, summ, walkers[b])
            assert abs(hh[b] - rhh) <= 1e-8 * rhh and abs(dh[b] - rdh) <= 1e-8 * max(abs(rdh), rhh), (nb, b, dh[b], rdh, hh[b], rhh)
            assert abs(ll[b] - rll) <= 1e-6 * (1.0 + abs(rll)), (nb, b, ll[b], rll)
            if nb == freqs.size:
                assert abs(hh[b] - brute[1][b]) <= 1e-9 * brute[1][b] and abs(dh[b] - brute[0][b]) <= 1e-9 * max(abs(brute[0][b]), brute[1][b]), b
        M.mbhl_het_free(het)
    M.mbhl_free(ctx)


def test_het_config2_scale_parity_and_accuracy(table):
    # config-2 grid (N = 4 197 160, S = 1024), reference = the 1e6 Msun injection, walkers at posterior-like distances
    wl = W.build(2, lambda p, f, S: L.template(table, p, f, S) if p[0] == 1e6 else np.zeros((3, f.size), dtype=np.complex128))
    freqs, S = wl["freqs"], wl["S"]
    ctx = M.mbhl_init(dev(freqs), dev(wl["data"]), dev(wl["psd"]), sparse_points=S, t0=wl["t0"])
    inj = wl["injections"][1]
    rng = np.random.default_rng(62)
    walkers = np.concatenate([inj[None, :], W.perturb(rng, inj, 3, 1e-7), W.perturb(rng, inj, 2, 1e-6)])
    # coarse bins: half of them log-spaced over the band of the reference's modes (read from the library's own knots)
    kn = M.mbhl_sparse(ctx, dev(inj[None, :]), want_coef=False)[0].cpu().numpy()[0]
    f_lo, f_hi = kn[kn[:, 0] > 0, 0].min(), kn[:, -1].max()
    edges = W.het_edges(freqs, 512, f_lo, f_hi)
    het = M.mbhl_het_init(ctx, dev(inj), edges)
    dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_het_loglike(het, dev(walkers))]
    bdh, bhh, bll = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(walkers))]
    summ = H.setup(table, inj, freqs, wl["data"], wl["psd"], S, edges, wl["t0"])
    for b in (0, 2, 5):
        rdh, rhh, rll = H.loglike_parts(table, summ, walkers[b])
        # phases reach ~2.5e7 rad here: one ulp is 3.7e-9 rad and both implementations carry ~10 roundings of that size in
        # their (independent) spline evaluations, i.e. ~4e-8 relative noise on an envelope value; the walker that IS
        # the reference (b = 0) cancels exactly on both sides
        tol = 1e-8 if b == 0 else 3e-7
        assert abs(hh[b] - rhh) <= tol * rhh and abs(dh[b] - rdh) <= tol * max(abs(rdh), rhh), (b, dh[b], rdh, hh[b], rhh)
        assert abs(ll[b] - rll) <= 1e-6 * (1.0 + abs(rll)), (b, ll[b], rll)          # the north_star bar on logL itself
    # accuracy against the brute-force path: a small fraction of <h|h>, shrinking with more coarse bins
    err512 = np.max(np.abs(hh - bhh) / bhh)
    het2 = M.mbhl_het_init(ctx, dev(inj), W.het_edges(freqs, 2048, f_lo, f_hi))
    dh2, hh2, ll2 = [t.cpu().numpy() for t in M.mbhl_het_loglike(het2, dev(walkers))]
    err2048 = np.max(np.abs(hh2 - bhh) / bhh)
    print('het accuracy at config-2 scale: rel <h|h> error', err512, err2048, 'max |dlogL|', np.max(np.abs(ll - bll)), np.max(np.abs(ll2 - bll)))
    assert err512 < 1e-5 and err2048 < 1e-7 and err2048 < err512 / 10.0, (err512, err2048)
    assert np.max(np.abs(ll2 - bll)) < 0.05, (ll2, bll)
    M.mbhl_het_free(het)
    M.mbhl_het_free(het2)
    M.mbhl_free(ctx)
