"""Per-bin parity of the fused dense kernel itself (k_dense) against the oracle, through the C ABI.

mbhl_loglike_parts never returns the template, only its inner products.  With PROBE DATA - a flat PSD chosen so that
every weight w = 4 df / S_n is exactly 1 and a data stream that is zero except for one unit entry (1 or i) in one
channel at one bin k - eq. 3 collapses to <d|h> = Re h^c(k) (resp. Im h^c(k)): six probes per bin read the template
value the dense kernel formed at that bin, with its own bookkeeping (staged-interval cache, knot straddles, band-edge
gating, scratch and per-bin lookups), at the north_star bar of 1e-9 of max|h^c|.  Bins are chosen around the features
that switch the kernel between its paths; a host-side mirror of the kernel's classification rules (csrc/mbhl_dense.cuh)
asserts that every path is hit.  Config 0 grid and the config-2 grid (t_coal ~ 4e7 s, phases of 1e6 cycles).
"""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import likelihood as L
from oracle import spline as ospline
from paper_2005_01827_b200 import binding as M
from paper_2005_01827_b200 import workloads as W

DEV = "cuda:0"
CHUNK, WARP_TILE, GEN_SLOTS = 512, 128, 6          # csrc/mbhl_kernels.cuh: kChunk, kWarpTile; mbhl_dense.cuh: kGenSlots


def dev(x):
    return torch.as_tensor(np.ascontiguousarray(x), device=DEV)


class Probe:
    """One-hot data streams on a fixed grid with unit weights; reads h^c(k) of every walker through <d|h>."""

    def __init__(self, freqs, S, t0):
        self.freqs, self.S, self.t0 = freqs, S, t0
        self.N = freqs.size
        df = (freqs[-1] - freqs[0]) / (self.N - 1)
        self.f_d = dev(freqs)
        self.psd_d = torch.full((3, self.N), 4.0 * df, dtype=torch.float64, device=DEV)      # w = 1
        self.data_d = torch.zeros((3, self.N, 2), dtype=torch.float64, device=DEV)

    def read(self, params, bins):
        """h [B, 3, len(bins)] complex128 as the dense kernel evaluated it."""
        p = dev(params)
        out = np.zeros((params.shape[0], 3, len(bins)), dtype=np.complex128)
        for i, k in enumerate(bins):
            for c in range(3):
                for comp in range(2):
                    self.data_d[c, k, comp] = 1.0
                    ctx = M.mbhl_init(self.f_d, self.data_d, self.psd_d, sparse_points=self.S, t0=self.t0)
                    dh, hh, ll = M.mbhl_loglike_parts(ctx, p)
                    v = dh.cpu().numpy()
                    assert abs(M.mbhl_data_norm(ctx) - 1.0) < 1e-12
                    M.mbhl_free(ctx)
                    self.data_d[c, k, comp] = 0.0
                    out[:, c, i] += v if comp == 0 else 1j * v
        return out


def oracle_at_bins(table, p, freqs, S, t0, bins):
    """Oracle spline template at the given bins: per-mode contributions [6, 3, n] (also filled at edge bins), edge flags
    (bin within one of a band edge, reading G10), in-band flags, per-mode (knots, k_lo, k_hi)."""
    modes, t_coal = L.sparse_stage(table, p, freqs[0], freqs[-1], S, t0)
    f = freqs[bins]
    contrib = np.zeros((6, 3, len(bins)), dtype=np.complex128)
    edge = np.zeros((6, len(bins)), dtype=bool)
    inband = np.zeros((6, len(bins)), dtype=bool)
    info = []
    for mi, mo in enumerate(modes):
        if mo is None:
            info.append(None)
            continue
        x = mo["knots"]
        k_lo = int(np.searchsorted(freqs, x[0], side="left"))
        k_hi = int(np.searchsorted(freqs, x[-1], side="right")) - 1
        info.append((x, k_lo, k_hi))
        edge[mi] = (np.abs(bins - k_lo) <= 1) | (np.abs(bins - k_hi) <= 1)        # reading G10
        inband[mi] = (f >= x[0]) & (f <= x[-1])
        sel = np.nonzero(inband[mi] | edge[mi])[0]              # edge bins: the end interval's cubic, whichever side
        if sel.size == 0:
            continue
        q = np.stack([ospline.evaluate(x, mo["coef"][:, qi, :], f[sel]) for qi in range(8)])
        That = [q[2] + 1j * q[3], q[4] + 1j * q[5], q[6] + 1j * q[7]]
        for c, hc in enumerate(L._combine(q[0], q[1], That, f[sel], t_coal)):
            contrib[mi, c, sel] = hc
    return contrib, edge, inband, info


def interval_of(x, f):
    return int(np.clip(np.searchsorted(x, f, side="right") - 1, 0, x.size - 2))


def kernel_path(freqs, x, k_lo, k_hi, k):
    """Mirror of k_dense's classification for bin k of one (walker, mode) with knots x and band [k_lo, k_hi]."""
    if k < k_lo or k > k_hi:
        return "out"
    c0 = (k // CHUNK) * CHUNK
    a, b = max(c0, k_lo), min(c0 + CHUNK - 1, k_hi, freqs.size - 1)
    ja, jb = interval_of(x, freqs[a]), interval_of(x, freqs[b])
    t0 = c0 + ((k - c0) // WARP_TILE) * WARP_TILE
    t1 = t0 + WARP_TILE - 1
    ta, tb = max(t0, k_lo), min(t1, k_hi, freqs.size - 1)
    full = ta == t0 and tb == t1
    jta, jtb = interval_of(x, freqs[ta]), interval_of(x, freqs[tb])
    if jb - ja <= 1:                       # one or two staged records for the chunk
        if full and jta == jtb:
            return "fast"
        return "straddle" if jta != jtb else "edge-gated"
    if full and jta == jtb:
        return "general-uniform"
    return "general-scratch" if jtb - jta < GEN_SLOTS else "general-perbin"


def feature_bins(freqs, info, rng, n_random=4):
    """Bins around the features that switch the dense kernel between its paths, for one walker."""
    N = freqs.size
    ks = set()
    for item in info:
        if item is None:
            continue
        x, k_lo, k_hi = item
        for e in (k_lo, k_hi):
            ks.update(range(e - 3, e + 4))
        S = x.size
        for j in (1, 2, 3, S // 8, S // 4, S // 2, 3 * S // 4, S - 3, S - 2):
            kk = int(np.searchsorted(freqs, x[j]))
            ks.update(range(kk - 2, kk + 2))
        kk = int(np.searchsorted(freqs, x[S // 2]))
        c0 = (kk // CHUNK) * CHUNK
        ks.update([c0 - 1, c0, c0 + 1, c0 + WARP_TILE - 1, c0 + WARP_TILE, c0 + CHUNK - 1, c0 + CHUNK])
        if k_hi > k_lo:
            ks.update(int(v) for v in rng.integers(k_lo, k_hi + 1, n_random))
    ks.update([0, 1, N - 2, N - 1])
    return np.array(sorted(k for k in ks if 0 <= k < N), dtype=np.int64)


def check_window(table, probe, params, bins, global_max, local_tol):
    """Compares the probed template with the oracle at `bins` for every walker; returns the set of kernel paths seen."""
    h_gpu = probe.read(params, bins)
    seen = set()
    for b in range(params.shape[0]):
        contrib, edge, inband, info = oracle_at_bins(table, params[b], probe.freqs, probe.S, probe.t0, bins)
        for i, k in enumerate(bins):
            for mi, item in enumerate(info):
                if item is not None and not edge[mi, i]:
                    seen.add(kernel_path(probe.freqs, item[0], item[1], item[2], int(k)))
            # a mode whose band edge is within one bin may be in or out (G10): either value is valid
            cands = [sum(contrib[mi, :, i] for mi in range(6) if inband[mi, i] and not edge[mi, i]) + np.zeros(3, dtype=np.complex128)]
            for mi in range(6):
                if edge[mi, i]:
                    cands = cands + [v + contrib[mi, :, i] for v in cands]
            err = min(np.max(np.abs(h_gpu[b, :, i] - v) / global_max[b]) for v in cands)
            assert err <= 1e-9, (b, int(k), err, h_gpu[b, :, i], cands[0])          # north_star: 1e-9 of max|h^c|
            loc = max(np.max(np.abs(v)) for v in cands)
            if loc > 0.0:
                errl = min(np.max(np.abs(h_gpu[b, :, i] - v)) for v in cands) / loc
                assert errl <= local_tol, (b, int(k), errl)                            # no mis-gated or misplaced bin
            else:
                assert np.all(h_gpu[b, :, i] == 0.0), (b, int(k))
    return seen


def test_dense_kernel_per_bin_config0(table):
    tf = lambda p, f, S: L.template(table, p, f, S)
    wl = W.build(0, tf)
    params = wl["params"].copy()
    params[3, 0] = 3e7                       # a heavy binary: band ends inside the grid (upper band edges)
    probe = Probe(wl["freqs"], wl["S"], wl["t0"])
    rng = np.random.default_rng(21)
    gmax = np.stack([np.max(np.abs(L.template(table, p, wl["freqs"], wl["S"], wl["t0"])), axis=1) for p in params])
    bins = set()
    for b in (0, 3):
        _, _, _, info = oracle_at_bins(table, params[b], wl["freqs"], wl["S"], wl["t0"], np.array([0]))
        bins.update(feature_bins(wl["freqs"], info[:2] + info[3:4], rng).tolist())
    bins = np.array(sorted(bins), dtype=np.int64)
    seen = check_window(table, probe, params, bins, gmax, 2e-9)
    # (band edges of this grid fall where a chunk holds three or more intervals; the gated staged path is hit at config-2 scale)
    assert {"fast", "straddle", "general-uniform", "general-scratch", "general-perbin", "out"} <= seen, seen


def test_dense_kernel_per_bin_config2_scale(table):
    # the config-2 grid (N = 4 197 160 bins up to 0.1 Hz, S = 1024, t_coal ~ 4e7 s): one walker per injection group
    wl = W.build(2, lambda p, f, S: np.zeros((3, f.size), dtype=np.complex128), with_noise=False)
    sel = [0, 500, 1023]
    params = wl["params"][sel]
    freqs, S = wl["freqs"], wl["S"]
    probe = Probe(freqs, S, wl["t0"])
    rng = np.random.default_rng(22)
    # max|h^c| over the grid from every 64th bin (the envelope A |T-hat| is smooth on that scale; a slightly smaller
    # scale only tightens the bar)
    f_dec = np.append(freqs[::64], freqs[-1])
    gmax = np.stack([np.max(np.abs(L.template(table, p, f_dec, S, wl["t0"])), axis=1) for p in params])
    bins = set()
    for b in range(3):
        _, _, _, info = oracle_at_bins(table, params[b], freqs, S, wl["t0"], np.array([0]))
        bins.update(feature_bins(freqs, [info[0], info[3]], rng, n_random=3).tolist())     # modes (2,2) and (2,1)
    for f_w in (1e-4, 2e-3, 5e-2):                                                          # fixed windows as well
        k = int(f_w / (freqs[1] - freqs[0]))
        bins.update(range(k, k + 3))
    bins = np.array(sorted(bins), dtype=np.int64)
    # phases reach ~4e6 cycles at the lowest knots: ulp = 9e-10 cycles = 6e-9 rad in BOTH implementations' knot values,
    # so relative to the LOCAL amplitude a few 1e-8 is rounding; a mis-gated or misplaced bin would be O(1)
    seen = check_window(table, probe, params, bins, gmax, 1e-7)
    assert {"fast", "straddle", "edge-gated", "general-scratch", "general-perbin", "out"} <= seen, seen
    assert (freqs.size - 1) in bins and (freqs.size % CHUNK) != 0                          # the ragged last chunk


def test_template_parity_config2_scale_on_seeded_bins(table):
    # mbhl_template (spline path) on 2e4 seeded frequencies of the config-2 band, t_coal ~ 4e7 s, against the oracle
    wl = W.build(2, lambda p, f, S: np.zeros((3, f.size), dtype=np.complex128), with_noise=False)
    freqs, S = wl["freqs"], wl["S"]
    rng = np.random.default_rng(23)
    f_out = np.sort(np.concatenate([10.0 ** rng.uniform(math.log10(freqs[0]), -1.0, 15000),
                                    rng.uniform(freqs[0], freqs[-1], 5000)]))
    f_out = f_out[(f_out >= freqs[0]) & (f_out <= freqs[-1])]
    ctx = M.mbhl_init(dev(freqs), torch.zeros((3, freqs.size, 2), dtype=torch.float64, device=DEV),
                      torch.ones((3, freqs.size), dtype=torch.float64, device=DEV), sparse_points=S, t0=wl["t0"])
    sel = [1, 400, 900]
    h_gpu = M.mbhl_template(ctx, dev(wl["params"][sel]), freqs_out=dev(f_out)).cpu().numpy()
    for i, b in enumerate(sel):
        modes, t_coal = L.sparse_stage(table, wl["params"][b], freqs[0], freqs[-1], S, wl["t0"])
        h_ref = np.zeros((3, f_out.size), dtype=np.complex128)
        near_edge = np.zeros(f_out.size, dtype=bool)
        for mo in modes:
            if mo is None:
                continue
            x = mo["knots"]
            for e in (x[0], x[-1]):
                near_edge |= np.abs(f_out - e) <= 4e-16 * e                       # a sample ON an edge may be in or out
            s_ = np.nonzero((f_out >= x[0]) & (f_out <= x[-1]))[0]
            q = np.stack([ospline.evaluate(x, mo["coef"][:, qi, :], f_out[s_]) for qi in range(8)])
            That = [q[2] + 1j * q[3], q[4] + 1j * q[5], q[6] + 1j * q[7]]
            for c, hc in enumerate(L._combine(q[0], q[1], That, f_out[s_], t_coal)):
                h_ref[c, s_] += hc
        keep = ~near_edge
        for c in range(3):
            scale = np.max(np.abs(h_ref[c]))
            assert scale > 0
            assert np.max(np.abs(h_gpu[i, c][keep] - h_ref[c][keep])) <= 1e-9 * scale, (b, c)
    M.mbhl_free(ctx)
