"""GPU parity tests of the sampler-side calls: per-mode products, sampler coordinates,
parallel-tempered stretch-move ensemble, each against oracle/ on the same seeded inputs."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import likelihood as L
from oracle import sampler as S
from paper_2005_01827_b200 import binding as M
from paper_2005_01827_b200 import workloads as W

DEV = "cuda:0"


def dev(x):
    return torch.as_tensor(np.ascontiguousarray(x), device=DEV)


def to_sampled(p):
    """Physical parameters -> the sampler's coordinates; q is mapped into (0, 1] (q and 1/q are the same binary, G15)."""
    th = np.array(p, dtype=np.float64, copy=True)
    th[..., 0], th[..., 4], th[..., 10] = np.log(p[..., 0]), np.log(p[..., 4]), np.log(p[..., 10])
    th[..., 1] = np.where(p[..., 1] > 1.0, 1.0 / p[..., 1], p[..., 1])
    th[..., 6], th[..., 8] = np.cos(p[..., 6]), np.sin(p[..., 8])
    return th


@pytest.fixture(scope="module")
def small(table):
    wl = W.build(0, lambda p, f, Sp: L.template(table, p, f, Sp), n_bins=4096, batch=4)
    wl["S"] = 64
    return wl


def make_ctx(wl):
    return M.mbhl_init(dev(wl["freqs"]), dev(wl["data"]), dev(wl["psd"]), sparse_points=wl["S"], t0=wl["t0"])


def test_mode_products_parity(table, small):
    ctx = make_ctx(small)
    p = small["params"]
    dh, hh = [t.cpu().numpy() for t in M.mbhl_mode_products(ctx, dev(p))]
    tdh, thh, _ = [t.cpu().numpy() for t in M.mbhl_loglike_parts(ctx, dev(p))]
    for b in range(p.shape[0]):
        rdh, rhh = L.mode_products(table, p[b], small["freqs"], small["data"], small["psd"], small["S"], small["t0"])
        assert np.all(np.abs(hh[b] - rhh) <= 1e-8 * rhh.max())
        assert np.all(np.abs(dh[b] - rdh) <= 1e-8 * max(np.abs(rdh).max(), rhh.max()))
        assert abs(dh[b].sum() - tdh[b]) <= 1e-10 * (np.abs(dh[b]).sum() + abs(tdh[b]))       # <d|h> is linear over the modes
    # a mode disabled at init gives zero
    ctx2 = M.mbhl_init(dev(small["freqs"]), dev(small["data"]), dev(small["psd"]), sparse_points=small["S"], mode_mask=0b000101)
    dh2, hh2 = [t.cpu().numpy() for t in M.mbhl_mode_products(ctx2, dev(p))]
    assert np.all(hh2[:, [1, 3, 4, 5]] == 0.0) and np.all(dh2[:, [1, 3, 4, 5]] == 0.0)
    assert np.allclose(hh2[:, [0, 2]], hh[:, [0, 2]], rtol=1e-13, atol=0.0)
    M.mbhl_free(ctx)
    M.mbhl_free(ctx2)


def test_loglike_sampled_parity(table, small):
    ctx = make_ctx(small)
    p = small["params"]
    th = to_sampled(p)
    assert np.all(S.in_prior(th))
    ll = M.mbhl_loglike_sampled(ctx, dev(th)).cpu().numpy()
    for b in range(p.shape[0]):
        ref = L.loglike_parts(table, S.unpack_sampled(th[b]), small["freqs"], small["data"], small["psd"], small["S"], small["t0"])[2]
        assert abs(ll[b] - ref) <= 1e-6 * (1.0 + abs(ref)), (b, ll[b], ref)
    bad = th.copy()
    bad[0, 1] = 1.5                 # q outside Table I
    bad[1, 6] = 1.0 + 1e-12         # cos(iota) > 1
    bad[2, 0] = math.log(1e10)      # M_T above the box
    bad[3, 10] = np.nan
    out = M.mbhl_loglike_sampled(ctx, dev(bad)).cpu().numpy()
    assert np.all(np.isneginf(out))
    # a batch larger than one slice of the hot path (32768 walkers)
    n = 40001
    big = np.tile(th, (n // th.shape[0] + 1, 1))[:n]
    out = M.mbhl_loglike_sampled(ctx, dev(big)).cpu().numpy()
    for b in range(th.shape[0]):
        assert np.max(np.abs(out[b::th.shape[0]] - ll[b])) <= 1e-9 * (1.0 + abs(ll[b]))
    M.mbhl_free(ctx)


def test_lisa_frame_coordinates_parity(table, small):
    # walkers handed over in the LISA frame; the conversion runs inside the per-walker constants kernel
    ctx = make_ctx(small)
    rng = np.random.default_rng(41)
    n = 64
    th = rng.uniform(S.PRIOR_LO, S.PRIOR_HI, size=(n, 11))
    th[:, 10] = np.log(rng.uniform(1e4, 6e7, n))
    th[:4, 8] = [1.0, -1.0, 0.0, 1.0 - 1e-16]                        # poles and the LISA-plane equator
    th[4, 7], th[5, 7], th[6, 9] = 0.0, 2.0 * math.pi, 0.0
    for coords, unpack in ((M.COORDS_SAMPLED, S.unpack_sampled), (M.COORDS_SAMPLED_LISA, lambda t: S.unpack_sampled_lisa(t, small["t0"]))):
        got = M.mbhl_unpack_coords(ctx, dev(th), coords).cpu().numpy()
        ref = unpack(th)
        assert np.max(np.abs(got[:, :7] - ref[:, :7]) / np.abs(ref[:, :7]).clip(1e-300)) <= 4e-16 + 1e-15
        # angles: compare as directions (lambda is undefined at a pole, psi is defined mod pi there only jointly with lambda)
        nonpole = np.abs(np.abs(ref[:, 8]) - math.pi / 2) > 1e-6
        dl = np.abs(np.remainder(got[:, 7] - ref[:, 7] + math.pi, 2 * math.pi) - math.pi)
        dp = np.abs(np.remainder(got[:, 9] - ref[:, 9] + math.pi / 2, math.pi) - math.pi / 2)
        assert np.max(dl[nonpole]) <= 1e-12 and np.max(dp[nonpole]) <= 1e-12
        assert np.max(np.abs(got[:, 8] - ref[:, 8])) <= 2e-8                      # asin near +-1 amplifies rounding like 1/cos(beta)
        assert np.max(np.abs(got[nonpole, 8] - ref[nonpole, 8]) * np.cos(ref[nonpole, 8])) <= 1e-14
        assert np.max(np.abs(got[:, 10] - ref[:, 10]) / ref[:, 10]) <= 1e-15
        assert np.all((got[:, 7] >= 0) & (got[:, 7] < 2 * math.pi + 1e-15) & (got[:, 9] >= 0) & (got[:, 9] <= math.pi))
    # likelihood through the LISA-frame entry point against the oracle on converted parameters; walkers around the injection
    inj = small["params"]
    thL = to_sampled(inj)
    for b in range(inj.shape[0]):
        t_L, lam_L, beta_L, psi_L = S.ssb_to_lisa(inj[b, 10], inj[b, 7], inj[b, 8], inj[b, 9], small["t0"])
        thL[b, 7], thL[b, 8], thL[b, 9], thL[b, 10] = lam_L, math.sin(beta_L), psi_L, math.log(t_L)
    ll = M.mbhl_loglike_coords(ctx, dev(thL), M.COORDS_SAMPLED_LISA).cpu().numpy()
    ll_ssb = M.mbhl_loglike(ctx, dev(inj)).cpu().numpy()
    for b in range(inj.shape[0]):
        ref = L.loglike_parts(table, S.unpack_sampled_lisa(thL[b], small["t0"]), small["freqs"], small["data"], small["psd"], small["S"], small["t0"])[2]
        assert abs(ll[b] - ref) <= 1e-6 * (1.0 + abs(ref)), (b, ll[b], ref)
        assert abs(ll[b] - ll_ssb[b]) <= 1e-5 * (1.0 + abs(ref))                  # the same binaries (round trip through the frames)
    bad = thL.copy()
    bad[0, 8] = 1.5
    assert np.isneginf(M.mbhl_loglike_coords(ctx, dev(bad), M.COORDS_SAMPLED_LISA).cpu().numpy()[0])
    with pytest.raises(M.MbhlError):
        M.mbhl_loglike_coords(ctx, dev(thL), 7)
    M.mbhl_free(ctx)


@pytest.mark.parametrize("coords", [1, 2])
def test_pt_ensemble_parity(table, small, coords):
    # T = 3 rungs (the last at infinite temperature), K = 8 walkers, a few steps: GPU ensemble against the oracle's,
    # with the walkers living in the SSB frame (coords 1) or in the LISA frame (coords 2)
    ctx = make_ctx(small)
    T, K = 3, 8
    betas = np.array([1.0, 0.4, 0.0])
    rng = np.random.default_rng(5)
    th0 = to_sampled(small["injections"][0])
    unpack = S.unpack_sampled
    if coords == 2:
        inj = small["injections"][0]
        t_L, lam_L, beta_L, psi_L = S.ssb_to_lisa(inj[10], inj[7], inj[8], inj[9], small["t0"])
        th0[7], th0[8], th0[9], th0[10] = lam_L, math.sin(beta_L), psi_L, math.log(t_L)
        unpack = lambda t: S.unpack_sampled_lisa(t, small["t0"])
    width = np.array([1e-4, 1e-3, 1e-3, 1e-3, 1e-2, 1e-2, 1e-2, 1e-2, 1e-2, 1e-2, 1e-5])
    theta = th0 + width * rng.standard_normal((T, K, 11))
    theta[..., 1] = np.clip(theta[..., 1], 0.06, 0.999)
    theta[..., 6] = np.clip(theta[..., 6], -0.999, 0.999)
    theta[..., 8] = np.clip(theta[..., 8], -0.999, 0.999)
    theta[..., 9] = np.clip(theta[..., 9], 1e-3, math.pi - 1e-3)
    assert np.all(S.in_prior(theta))

    def fn(th):
        return np.array([L.loglike_parts(table, unpack(t), small["freqs"], small["data"], small["psd"], small["S"], small["t0"])[2]
                         for t in th])

    logl = fn(theta.reshape(-1, 11)).reshape(T, K)
    pt = M.mbhl_pt_init(ctx, dev(theta), betas, seed=2005018270001, stretch_a=S.STRETCH_A, coords=coords)
    g_theta, g_logl, _, _ = M.mbhl_pt_state(pt, T, K, DEV)
    assert np.array_equal(g_theta.cpu().numpy(), theta)
    assert np.max(np.abs(g_logl.cpu().numpy() - logl) / (1.0 + np.abs(logl))) <= 1e-6
    n_acc = np.zeros(T, dtype=np.int64)
    n_swp = np.zeros(T - 1, dtype=np.int64)
    for step in range(5):
        for half in (0, 1):
            theta, logl, a = S.stretch_half_step(theta, logl, betas, half, 2005018270001, 2 * step + half, fn)
            n_acc += a.sum(axis=1)
        theta, logl, sw = S.swap_step(theta, logl, betas, 2005018270001, step)
        n_swp += sw.sum(axis=1)
        M.mbhl_pt_step(pt, 1)
        g_theta, g_logl, g_acc, g_swp = M.mbhl_pt_state(pt, T, K, DEV)
        assert np.max(np.abs(g_theta.cpu().numpy() - theta)) <= 1e-12, step
        assert np.max(np.abs(g_logl.cpu().numpy() - logl) / (1.0 + np.abs(logl))) <= 1e-6, step
        assert np.array_equal(g_acc, n_acc) and np.array_equal(g_swp, n_swp), step
    assert n_acc.sum() > 0 and n_acc[-1] > 0          # the infinite-temperature rung accepts in-prior moves with z^(D-1)
    M.mbhl_pt_free(pt)
    # argument checks
    with pytest.raises(M.MbhlError):
        M.mbhl_pt_init(ctx, dev(theta[:, :7]), betas)          # odd number of walkers
    with pytest.raises(M.MbhlError):
        M.mbhl_pt_init(ctx, dev(theta), np.array([1.0, -0.5, 0.0]))
    outside = theta.copy()
    outside[2, 3, 1] = 1.5                                      # a starting walker outside the Table I box (ADVICE: it could never move at beta = 0)
    with pytest.raises(M.MbhlError, match="prior box"):
        M.mbhl_pt_init(ctx, dev(outside), betas)
    M.mbhl_free(ctx)


def test_noise_realisation_parity():
    N, df = 100003, 3.0e-8
    f = (1.0 + np.arange(N)) * df * 100.0
    psd = W.scird_psd_aet(f)
    psd[0, 5] = 0.0
    psd[2, 7] = np.inf
    ref = S.noise_aet(psd, df, seed=2005018270002)
    got = M.mbhl_noise(dev(psd), df, seed=2005018270002).cpu().numpy()
    scale = np.sqrt(np.where(np.isfinite(psd) & (psd > 0), psd, 0.0) / (4.0 * df))
    assert got[0, 5] == 0.0 and got[2, 7] == 0.0
    # same uniforms on both sides: only the rounding of log / sqrt / sincos differs
    assert np.max(np.abs(got - ref) / np.maximum(scale, 1e-300)) <= 1e-13
