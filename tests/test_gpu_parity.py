"""GPU parity tests: the CUDA path through the C ABI against the CPU oracle, element by element.

Tolerances (BASELINE.json north_star): |dlogL| <= 1e-6 (1 + |logL|); per-bin template error <= 1e-9
relative to max|h^c| per channel (G6), band-edge bins excluded (G10).
"""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import likelihood as L
from oracle import spline as ospline
from oracle.constants import MODES
from oracle.phenom import Intrinsic
from paper_2005_01827_b200 import binding as M
from paper_2005_01827_b200 import workloads as W

DEV = "cuda:0"


def dev(x):
    return torch.as_tensor(np.ascontiguousarray(x), device=DEV)


def make_ctx(wl, **kw):
    return M.mbhl_init(dev(wl["freqs"]), dev(wl["data"]), dev(wl["psd"]), sparse_points=wl["S"], t0=wl["t0"], **kw)


@pytest.fixture(scope="module")
def cfg0(table):
    tf = lambda p, f, S: L.template(table, p, f, S)
    wl = W.build(0, tf)
    # extra walkers: equal masses (odd modes vanish), q < 1 (reading G15), extreme spins, a heavy binary
    extra = wl["params"][:4].copy()
    extra[0, 1] = 1.0
    extra[1, 1] = 1.0 / extra[1, 1]
    extra[2, 2:4] = [-0.99, 0.99]
    extra[3, 0] = 3e7
    wl["params"] = np.concatenate([wl["params"], extra])
    return wl


def edge_mask(table, params, freqs, t0):
    """True for bins within +-1 of any mode's band edge (membership may legitimately differ, G10)."""
    p = L.unpack(params)
    intr = Intrinsic(table, p["M_T"], p["q"], p["a1"], p["a2"], p["D_L"])
    mask = np.zeros(freqs.size, dtype=bool)
    for (l, m) in MODES:
        band = L.mode_band(intr, l, m, t0 + p["t_ref"], freqs[0], freqs[-1])
        if band is None:
            continue
        for edge in band:
            k = int(np.searchsorted(freqs, edge))
            mask[max(0, k - 2):k + 2] = True
    return mask


def check_sparse_stage(table, params, knots, y, coef, f_lo, f_hi, S, t0):
    """Element-by-element comparison of mbhl_sparse's three outputs with the oracle's sparse stage; returns the number of active modes."""
    n_active = 0
    for b in range(params.shape[0]):
        modes, _ = L.sparse_stage(table, params[b], f_lo, f_hi, S, t0)
        for mi, mo in enumerate(modes):
            if mo is None:
                assert np.all(knots[b, mi] == 0.0) and np.all(coef[b, mi] == 0.0)
                continue
            n_active += 1
            assert np.max(np.abs(knots[b, mi] / mo["knots"] - 1.0)) < 1e-13
            yo = mo["y"]
            amp_scale = np.max(np.abs(yo[0]))
            if amp_scale > 0:
                assert np.max(np.abs(y[b, mi, 0] - yo[0])) <= 1e-10 * amp_scale
            assert np.max(np.abs(y[b, mi, 1] - yo[1])) <= 2e-8                       # radians
            tscale = np.max(np.abs(yo[2:]))
            assert np.max(np.abs(y[b, mi, 2:] - yo[2:])) <= 1e-10 * tscale
            # spline coefficients (phase row in cycles, y_j reduced mod 1)
            co = mo["coef"].copy()                    # [S-1, 8, 4]
            co[:, 1, :] /= 2.0 * math.pi
            cg = coef[b, mi]
            hj = np.diff(mo["knots"])
            for q in range(8):
                # compare each coefficient through its contribution at the far end of the interval
                # (c_j h^2 and d_j h^3 are differences of O(y) terms: that is their natural error scale)
                yscale = 1.0 if q == 1 else (np.max(np.abs(co[:, 0, 0])) if q == 0 else np.max(np.abs(co[:, 2:, 0])))
                tol = 1e-10 * yscale if q != 1 else 2e-9          # phase: cycles
                for col in range(4):
                    d = (cg[:, q, col] - co[:, q, col]) * hj ** col
                    if q == 1 and col == 0:
                        d = d - np.rint(d)
                        assert np.max(np.abs(cg[:, q, col])) <= 0.5 + 1e-12
                    assert np.max(np.abs(d)) <= tol, (b, mi, q, col, np.max(np.abs(d)), tol)
    return n_active


def test_sparse_stage_parity(table, cfg0):
    ctx = make_ctx(cfg0)
    params = cfg0["params"]
    knots, y, coef = [t.cpu().numpy() for t in M.mbhl_sparse(ctx, dev(params))]
    check_sparse_stage(table, params, knots, y, coef, cfg0["freqs"][0], cfg0["freqs"][-1], cfg0["S"], cfg0["t0"])
    M.mbhl_free(ctx)


@pytest.mark.parametrize("S", [512, 1024])
def test_sparse_stage_parity_at_benchmark_knot_counts(table, S):
    # The knot counts of BASELINE configs 1-4 (S a multiple of 32 up to 1024: the fast 32-row sweeps of k_sparse_spline), on
    # config 3's own grid (T_obs = 1.33 yr, f up to 0.1 Hz) with 16 walkers from config 3's prior (M_T log-uniform 1e5-1e8 Msun,
    # workloads.sparse_batch): bands that start at the grid's first bin, bands that end inside it, heavy binaries whose modes
    # span barely a decade.  Same element-by-element bars as the S = 256 case above.
    freqs = W.grid(1.33, int(0.1 * 1.33 * W.YEAR_JULIAN_S), 0.0)
    n = freqs.size
    ctx = M.mbhl_init(dev(freqs), torch.zeros((3, n, 2), dtype=torch.float64, device=DEV),
                      torch.ones((3, n), dtype=torch.float64, device=DEV), sparse_points=S)
    params = W.sparse_batch(16)
    assert params[:, 0].min() < 1e6 < 1e7 < params[:, 0].max()              # light and heavy binaries both drawn
    knots, y, coef = [t.cpu().numpy() for t in M.mbhl_sparse(ctx, dev(params))]
    n_active = check_sparse_stage(table, params, knots, y, coef, freqs[0], freqs[-1], S, 0.0)
    assert n_active >= 80                                                  # nearly all of the 96 (walker, mode) pairs are in band
    f_hi = knots[:, :, -1]
    assert np.any((f_hi > 0) & (f_hi < 0.99 * freqs[-1])) and np.any(f_hi > 0.99 * freqs[-1])   # bands ending inside / at the grid edge
    M.mbhl_free(ctx)


@pytest.mark.parametrize("direct", [False, True])
def test_template_parity_config0(table, cfg0, direct):
    ctx = make_ctx(cfg0)
    params = cfg0["params"]
    h_gpu = M.mbhl_template(ctx, dev(params), direct=direct).cpu().numpy()
    for b in range(params.shape[0]):
        h_ref = L.template(table, params[b], cfg0["freqs"], cfg0["S"], cfg0["t0"], mode="direct" if direct else "spline")
        keep = ~edge_mask(table, params[b], cfg0["freqs"], cfg0["t0"])
        for c in range(3):
            scale = np.max(np.abs(h_ref[c]))
            assert scale > 0
            err = np.max(np.abs(h_gpu[b, c][keep] - h_ref[c][keep])) / scale
            assert err <= 1e-9, (b, c, err)
        # edge bins: either side's value is a valid one (in or out of band): |diff| bounded by the local amplitude
        assert np.all(np.abs(h_gpu[b] - h_ref)[:, ~keep] <= 1.0001 * np.maximum(np.abs(h_gpu[b]), np.abs(h_ref))[:, ~keep] + 1e-300)
    M.mbhl_free(ctx)


def test_template_on_another_grid(table, cfg0):
    ctx = make_ctx(cfg0)
    f_out = np.sort(np.random.default_rng(5).uniform(cfg0["freqs"][0], cfg0["freqs"][-1], 3001))
    p = cfg0["params"][:2]
    h_gpu = M.mbhl_template(ctx, dev(p), freqs_out=dev(f_out)).cpu().numpy()
    for b in range(2):
        # the bands come from the init grid; evaluate the oracle's splines at f_out
        modes, t_coal = L.sparse_stage(table, p[b], cfg0["freqs"][0], cfg0["freqs"][-1], cfg0["S"], cfg0["t0"])
        h_ref = np.zeros((3, f_out.size), dtype=np.complex128)
        for mo in modes:
            if mo is None:
                continue
            sel = np.nonzero((f_out >= mo["knots"][0]) & (f_out <= mo["knots"][-1]))[0]
            q = np.stack([ospline.evaluate(mo["knots"], mo["coef"][:, qi, :], f_out[sel]) for qi in range(8)])
            That = [q[2] + 1j * q[3], q[4] + 1j * q[5], q[6] + 1j * q[7]]
            for c, hc in enumerate(L._combine(q[0], q[1], That, f_out[sel], t_coal)):
                h_ref[c, sel] += hc
        for c in range(3):
            assert np.max(np.abs(h_gpu[b, c] - h_ref[c])) <= 1e-9 * np.max(np.abs(h_ref[c]))
    M.mbhl_free(ctx)


def test_loglike_parity_config0(table, cfg0):
    ctx = make_ctx(cfg0)
    params = cfg0["params"]
    dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(params))]
    ll2 = M.mbhl_loglike(ctx, dev(params)).cpu().numpy()
    assert np.array_equal(ll, ll2)                                  # deterministic reductions
    pairs, bins = M.mbhl_last_work(ctx)
    assert 0 < bins <= params.shape[0] * cfg0["freqs"].size and bins <= pairs <= 6 * bins
    w = L.weights(cfg0["freqs"], cfg0["psd"])
    dd = L.inner(cfg0["data"], cfg0["data"], w)
    assert abs(M.mbhl_data_norm(ctx) / dd - 1.0) < 1e-13
    for b in range(params.shape[0]):
        rdh, rhh, rll = L.loglike_parts(table, params[b], cfg0["freqs"], cfg0["data"], cfg0["psd"], cfg0["S"], cfg0["t0"])
        assert abs(ll[b] - rll) <= 1e-6 * (1.0 + abs(rll)), (b, ll[b], rll)
        assert abs(hh[b] - rhh) <= 1e-8 * rhh and abs(dh[b] - rdh) <= 1e-8 * max(abs(rdh), rhh)
        assert abs(ll[b] - (dh[b] - 0.5 * hh[b] - 0.5 * M.mbhl_data_norm(ctx))) <= 1e-9 * (dd + hh[b])
    # host-buffer entry point gives the same numbers
    ph = torch.from_numpy(params.copy()).pin_memory()
    lh = torch.empty(params.shape[0], dtype=torch.float64).pin_memory()
    M.mbhl_loglike_host(ctx, ph, lh)
    assert np.array_equal(lh.numpy(), ll)
    M.mbhl_free(ctx)


def test_noise_free_injection_gives_logl_zero_and_distance_scaling(table):
    tf = lambda p, f, S: L.template(table, p, f, S)
    wl = W.build(0, tf, with_noise=False)
    ctx = make_ctx(wl)
    inj = wl["injections"][0]
    p = np.stack([inj, inj, inj])
    p[1, 4] *= 2.0
    # a mass offset large enough to leave the peak: this short grid (T_obs = 0.1 yr, SNR ~ 130) has a posterior width of a
    # few 1e-5 in ln M_T, so the 1e-5 offset first written here moved logL by less than one unit; 1e-3 is ~30 sigma
    p[2, 0] *= 1.0 + 1e-3
    dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(p))]
    assert abs(ll[0]) < 1e-6 and hh[0] > 1e3
    assert abs(hh[1] * 4.0 / hh[0] - 1.0) < 1e-12
    assert ll[2] < -1.0
    M.mbhl_free(ctx)


def test_edge_cases(table, cfg0):
    # ragged grid (N not a multiple of the chunk or of 32), PSD zeros / non-finite, mode mask, domain errors
    n = 5 * 512 + 37
    sl = slice(20000, 20000 + n)
    freqs = cfg0["freqs"][sl].copy()
    data = cfg0["data"][:, sl].copy()
    psd = cfg0["psd"][:, sl].copy()
    psd[0, 11] = 0.0
    psd[1, 12] = np.inf
    psd[2, 13] = np.nan
    psd[1, 14] = -1.0
    params = cfg0["params"][:4].copy()
    bad = params[:3].copy()
    bad[0, 4] = -5.0           # D_L <= 0
    bad[1, 2] = 1.5            # |a1| > 1
    bad[2, 10] = np.nan
    heavy = params[:1].copy()
    heavy[0, 0] = 1e10         # every band below the grid
    allp = np.concatenate([params, bad, heavy])
    for mask in (0, 0b000001, 0b101010):
        ctx = M.mbhl_init(dev(freqs), dev(data), dev(psd), sparse_points=64, mode_mask=mask)
        ll = M.mbhl_loglike(ctx, dev(allp)).cpu().numpy()
        dd = M.mbhl_data_norm(ctx)
        w = L.weights(freqs, psd)
        assert abs(dd / L.inner(data, data, w) - 1.0) < 1e-13
        assert np.all(np.isneginf(ll[4:7])) and ll[7] == -0.5 * dd and not np.any(np.isnan(ll))
        for b in range(4):
            h = L.template(table, allp[b], freqs, 64, 0.0, mode_mask=mask if mask else 0x3F)
            ref = L.inner(data, h, w) - 0.5 * L.inner(h, h, w) - 0.5 * L.inner(data, data, w)
            assert abs(ll[b] - ref) <= 1e-6 * (1.0 + abs(ref))
        # B = 0 is a no-op
        M.mbhl_loglike(ctx, torch.empty((0, 11), dtype=torch.float64, device=DEV))
        M.mbhl_free(ctx)


def test_host_pointers_at_init_and_workspace_api(table, cfg0):
    ctx_d = make_ctx(cfg0)
    ctx_h = M.mbhl_init(cfg0["freqs"], np.ascontiguousarray(cfg0["data"]), np.ascontiguousarray(cfg0["psd"]),
                        sparse_points=cfg0["S"], t0=cfg0["t0"])
    p = dev(cfg0["params"])
    a = M.mbhl_loglike(ctx_d, p).cpu().numpy()
    b = M.mbhl_loglike(ctx_h, p).cpu().numpy()
    assert np.array_equal(a, b)
    need = M.mbhl_workspace_bytes(ctx_h, p.shape[0])
    assert need > 0
    ws = torch.empty(need, dtype=torch.uint8, device=DEV)
    M.mbhl_set_workspace(ctx_h, ws)
    assert np.array_equal(M.mbhl_loglike(ctx_h, p).cpu().numpy(), a)
    small = torch.empty(1024, dtype=torch.uint8, device=DEV)
    M.mbhl_set_workspace(ctx_h, small)
    with pytest.raises(M.MbhlError, match="workspace"):
        M.mbhl_loglike(ctx_h, p)
    M.mbhl_set_workspace(ctx_h, None)
    assert np.array_equal(M.mbhl_loglike(ctx_h, p).cpu().numpy(), a)
    assert M.mbhl_launch_count(ctx_h) > 0
    M.mbhl_free(ctx_d)
    M.mbhl_free(ctx_h)


def test_two_live_contexts_with_different_sparse_sizes(table, cfg0):
    # k_spline's dynamic shared memory limit is per function, not per context (ADVICE): a second context with a smaller S
    # must not break the first one
    big = make_ctx(cfg0)                                             # S = 256
    p = dev(cfg0["params"])
    a = M.mbhl_loglike(big, p).cpu().numpy()
    n = 4 * 512
    small = M.mbhl_init(dev(cfg0["freqs"][:n]), dev(cfg0["data"][:, :n]), dev(cfg0["psd"][:, :n]), sparse_points=16)
    M.mbhl_loglike(small, p)
    huge = M.mbhl_init(dev(cfg0["freqs"][:n]), dev(cfg0["data"][:, :n]), dev(cfg0["psd"][:, :n]), sparse_points=2048)
    assert torch.isfinite(M.mbhl_loglike(huge, p)).all()
    assert np.array_equal(M.mbhl_loglike(big, p).cpu().numpy(), a)
    assert torch.isfinite(M.mbhl_loglike(small, p)).all()
    for c in (big, small, huge):
        M.mbhl_free(c)
    with pytest.raises(M.MbhlError, match="invalid argument"):
        M.mbhl_init(dev(cfg0["freqs"][:n]), dev(cfg0["data"][:, :n]), dev(cfg0["psd"][:, :n]), sparse_points=2049)
    # workspace sizing is monotone in B and covers one slice for any larger batch (ADVICE)
    c = make_ctx(cfg0)
    sizes = [M.mbhl_workspace_bytes(c, b) for b in (1, 2, 7, 8, 9, 64, 1000, 32768, 40000, 10 ** 6)]
    assert all(x <= y for x, y in zip(sizes, sizes[1:])) and sizes[-1] == sizes[-3]
    M.mbhl_free(c)


def test_hot_path_is_capturable_in_a_cuda_graph(table, cfg0):
    # with max_batch set the call only enqueues kernels and a memset on the context's stream: one graph launch replays it
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        ctx = M.mbhl_init(dev(cfg0["freqs"]), dev(cfg0["data"]), dev(cfg0["psd"]), sparse_points=cfg0["S"], t0=cfg0["t0"],
                          max_batch=8, stream=s)
        p = dev(cfg0["params"])
        out = torch.empty(p.shape[0], dtype=torch.float64, device=DEV)
        ref = M.mbhl_loglike(ctx, p).clone()
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            M.mbhl_loglike(ctx, p, out)
        out.zero_()
        g.replay()
        s.synchronize()
        assert torch.equal(out, ref)
        p[0, 0] *= 1.0001                       # new walker positions in the same buffer: replay evaluates them
        g.replay()
        s.synchronize()
        assert torch.equal(out, M.mbhl_loglike(ctx, p)) and not torch.equal(out, ref)
        s.synchronize()
        M.mbhl_free(ctx)


def test_init_rejects_bad_grids(cfg0):
    f = cfg0["freqs"][:1000].copy()
    d = np.ascontiguousarray(cfg0["data"][:, :1000])
    s = np.ascontiguousarray(cfg0["psd"][:, :1000])
    bad = f.copy()
    bad[500] *= 1.001                                  # non-uniform
    with pytest.raises(M.MbhlError, match="invalid argument"):
        M.mbhl_init(bad, d, s)
    with pytest.raises(M.MbhlError, match="invalid argument"):
        M.mbhl_init(f[::-1].copy(), d, s)              # decreasing
    with pytest.raises(M.MbhlError, match="invalid argument"):
        M.mbhl_init(f[:3].copy(), d[:, :3].copy(), s[:, :3].copy())
    with pytest.raises(M.MbhlError, match="invalid argument"):
        M.mbhl_init(f, d, s, sparse_points=4)


def test_loglike_parity_config1_sampled_walkers(table):
    # BASELINE config 1 at full size (N = 2^20, S = 512, B = 64): the oracle checks sampled walkers one by one
    tf = lambda p, f, S: L.template(table, p, f, S)
    wl = W.build(1, tf)
    ctx = make_ctx(wl)
    ll = M.mbhl_loglike(ctx, dev(wl["params"])).cpu().numpy()
    assert ll.shape == (64,) and np.all(np.isfinite(ll))
    for b in (0, 17, 63):
        ref = L.loglike_parts(table, wl["params"][b], wl["freqs"], wl["data"], wl["psd"], wl["S"], wl["t0"])[2]
        assert abs(ll[b] - ref) <= 1e-6 * (1.0 + abs(ref)), (b, ll[b], ref)
    # the injection itself is close to the maximum: logL(injection) ~ -(number of noise dof)/1 + ... >> typical walker
    inj = M.mbhl_loglike(ctx, dev(wl["injections"])).cpu().numpy()[0]
    ref = L.loglike_parts(table, wl["injections"][0], wl["freqs"], wl["data"], wl["psd"], wl["S"], wl["t0"])[2]
    assert abs(inj - ref) <= 1e-6 * (1.0 + abs(ref))
    M.mbhl_free(ctx)


def test_loglike_parity_config2_full_size_in_the_bench_launch_configuration(table):
    # BASELINE config 2 at full size (B = 1024, S = 1024, N = 4 197 160), the batch and launch shape bench.py times:
    # one walker per injection group plus the group boundaries are checked by the oracle one by one, the rest
    # through properties that hold at any size.
    tf = lambda p, f, S: L.template(table, p, f, S)
    wl = W.build(2, tf)
    B = wl["params"].shape[0]
    assert B == 1024 and wl["freqs"].size == 4197160 and wl["S"] == 1024
    ctx = make_ctx(wl, max_batch=B)
    p = dev(wl["params"])
    dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, p)]
    dd = M.mbhl_data_norm(ctx)
    assert np.all(np.isfinite(ll)) and np.all(hh > 0.0)
    assert np.max(np.abs(ll - (dh - 0.5 * hh - 0.5 * dd)) / (dd + hh)) <= 1e-12       # eq. 2
    assert np.array_equal(M.mbhl_loglike(ctx, p).cpu().numpy(), ll)                     # bitwise reproducible
    # a walker's result does not depend on its position in the batch or on its tile mates (tiles of 8 walkers)
    perm = np.random.default_rng(7).permutation(B)
    assert np.array_equal(M.mbhl_loglike(ctx, dev(wl["params"][perm])).cpu().numpy(), ll[perm])
    sub = [3, 341, 342, 700, 1023]
    # a small batch takes another launch shape (chunks per CTA), i.e. another summation order
    ll_sub = M.mbhl_loglike(ctx, dev(wl["params"][sub])).cpu().numpy()
    assert np.max(np.abs(ll_sub - ll[sub]) / (dd + hh[sub])) <= 1e-13
    pairs, bins = M.mbhl_last_work(ctx)
    assert 0 < bins <= len(sub) * wl["freqs"].size and bins <= pairs <= 6 * bins
    for b in (0, 341, 342, 683, 1023):
        rdh, rhh, rll = L.loglike_parts(table, wl["params"][b], wl["freqs"], wl["data"], wl["psd"], wl["S"], wl["t0"])
        assert abs(ll[b] - rll) <= 1e-6 * (1.0 + abs(rll)), (b, ll[b], rll)
        assert abs(hh[b] - rhh) <= 1e-8 * rhh, (b, hh[b], rhh)
    M.mbhl_free(ctx)


def test_batches_beyond_the_grid_limit_are_sliced(table, cfg0):
    # B > 65535 walkers: the library processes slices of 32768; every copy of a walker must give the same number
    n = 3 * 512 + 5
    sl = slice(30000, 30000 + n)
    ctx = M.mbhl_init(dev(cfg0["freqs"][sl]), dev(cfg0["data"][:, sl]), dev(cfg0["psd"][:, sl]), sparse_points=32)
    base = cfg0["params"][:4]
    ref = M.mbhl_loglike(ctx, dev(base)).cpu().numpy()
    B = 70003
    big = np.tile(base, (B // 4 + 1, 1))[:B]
    dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(big))]
    assert ll.shape == (B,)
    # slices of 32768 walkers and the last partial slice take other launch shapes: same sums up to rounding order
    dd = M.mbhl_data_norm(ctx)
    for k in range(4):
        assert np.max(np.abs(ll[k::4] - ref[k])) <= 1e-12 * (dd + np.max(hh[k::4]))
    # the host-buffer entry point stages parameters in the workspace: sliced the same way
    lh = torch.empty(B, dtype=torch.float64).pin_memory()
    M.mbhl_loglike_host(ctx, torch.from_numpy(big.copy()).pin_memory(), lh)
    assert np.array_equal(lh.numpy(), ll)
    M.mbhl_free(ctx)


def test_tiny_grids_and_few_knots(table, cfg0):
    # the smallest inputs the boundary accepts (N >= 4 bins, S >= 8 knots) and a handful of sizes around the tile edges
    for n, S, k0 in ((4, 8, 20000), (7, 8, 100), (127, 9, 40000), (129, 17, 60000), (513, 33, 5)):
        sl = slice(k0, k0 + n)
        f, d, s_ = cfg0["freqs"][sl].copy(), np.ascontiguousarray(cfg0["data"][:, sl]), np.ascontiguousarray(cfg0["psd"][:, sl])
        ctx = M.mbhl_init(dev(f), dev(d), dev(s_), sparse_points=S)
        p = cfg0["params"][:3]
        ll = M.mbhl_loglike(ctx, dev(p)).cpu().numpy()
        for b in range(3):
            ref = L.loglike_parts(table, p[b], f, d, s_, S, 0.0)[2]
            assert abs(ll[b] - ref) <= 1e-6 * (1.0 + abs(ref)), (n, S, b, ll[b], ref)
        M.mbhl_free(ctx)


def test_many_knots_up_to_the_documented_ceiling(table, cfg0):
    # S above 1024 (up to the ceiling mbhl.h documents, 2048): the sweeps of the fused sparse kernel leave their 32-row fast
    # path, a CTA's shared memory holds twice the rows; S = 1056 is the first multiple of 32 beyond the fast path
    sl = slice(1000, 9000)
    f, d, s_ = cfg0["freqs"][sl].copy(), np.ascontiguousarray(cfg0["data"][:, sl]), np.ascontiguousarray(cfg0["psd"][:, sl])
    p = cfg0["params"][:2]
    for S in (1056, 1536, 2048):
        ctx = M.mbhl_init(dev(f), dev(d), dev(s_), sparse_points=S)
        dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(p))]
        for b in range(2):
            rdh, rhh, rll = L.loglike_parts(table, p[b], f, d, s_, S, 0.0)
            assert abs(ll[b] - rll) <= 1e-6 * (1.0 + abs(rll)), (S, b, ll[b], rll)
            assert abs(hh[b] - rhh) <= 1e-8 * max(rhh, 1e-300), (S, b, hh[b], rhh)
        M.mbhl_free(ctx)


def test_narrow_interval_regime_random_masses(table):
    # BASELINE config 4 corner: few bins per spline interval (N = 2^14 bins up to 0.1 Hz with S = 1024 knots) and walkers
    # from 1e5 to 1e8 solar masses in one batch: every path of the dense kernel (staged, knot straddles, scratch, per bin)
    N = 1 << 14
    df = 0.1 / N
    freqs = (1.0 + np.arange(N, dtype=np.float64)) * df
    psd = W.scird_psd_aet(freqs)
    params = W.sparse_batch(12, seed_offset=9)
    params[:, 10] *= (1.0 / df) / (1.33 * W.YEAR_JULIAN_S)          # t_ref as the same fraction of T_obs = 1/df
    rng = np.random.default_rng(9)
    data = L.template(table, params[0], freqs, 1024) + W.noise(rng, psd, df)
    ctx = M.mbhl_init(dev(freqs), dev(data), dev(psd), sparse_points=1024)
    dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(params))]
    pairs, bins = M.mbhl_last_work(ctx)
    assert pairs > 0
    for b in range(params.shape[0]):
        rdh, rhh, rll = L.loglike_parts(table, params[b], freqs, data, psd, 1024)
        assert abs(ll[b] - rll) <= 1e-6 * (1.0 + abs(rll)), (b, ll[b], rll)
        assert abs(hh[b] - rhh) <= 1e-8 * max(rhh, 1e-300), (b, hh[b], rhh)
    h_gpu = M.mbhl_template(ctx, dev(params[:3])).cpu().numpy()
    for b in range(3):
        h_ref = L.template(table, params[b], freqs, 1024)
        keep = ~edge_mask(table, params[b], freqs, 0.0)
        for c in range(3):
            scale = np.max(np.abs(h_ref[c]))
            if scale > 0:
                assert np.max(np.abs(h_gpu[b, c][keep] - h_ref[c][keep])) <= 1e-9 * scale
    M.mbhl_free(ctx)


def test_random_grids_knot_counts_and_masses(table):
    # seeded sweep over what the boundary accepts: grid length, start and spacing, knots per mode, walkers from 1e4 to 3e8
    # solar masses with mass ratios up to 20 and merger times inside, at the edge of and beyond the observation
    rng = np.random.default_rng(200501827)
    worst = 0.0
    for trial in range(10):
        N = int(rng.integers(600, 40000))
        S = int(rng.choice([8, 16, 33, 64, 128, 257, 512]))
        T_yr = 10.0 ** rng.uniform(-1.5, 0.3)
        freqs = W.grid(T_yr, N, 10.0 ** rng.uniform(-5.0, -3.3))
        df = freqs[1] - freqs[0]
        psd = W.scird_psd_aet(freqs)
        P = np.stack([W.draw_prior(rng, None, T_yr * W.YEAR_JULIAN_S, q_range=(1.0, 20.0), z_range=(0.5, 10.0), M_log_range=(1e4, 3e8))
                      for _ in range(5)])
        P[:, 10] = rng.uniform(0.02, 1.5, 5) * T_yr * W.YEAR_JULIAN_S
        data = L.template(table, P[0], freqs, S) + W.noise(rng, psd, df)
        ctx = M.mbhl_init(dev(freqs), dev(data), dev(psd), sparse_points=S)
        dh, hh, ll = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(P))]
        for b in range(P.shape[0]):
            rdh, rhh, rll = L.loglike_parts(table, P[b], freqs, data, psd, S)
            assert abs(ll[b] - rll) <= 1e-6 * (1.0 + abs(rll)), (trial, N, S, b, ll[b], rll)
            assert abs(hh[b] - rhh) <= 1e-8 * rhh + 1e-300, (trial, N, S, b, hh[b], rhh)
            worst = max(worst, abs(ll[b] - rll) / (1.0 + abs(rll)))
        M.mbhl_free(ctx)
    assert worst < 1e-9
