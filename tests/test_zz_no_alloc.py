"""GPU test of mbhl_unpack_coords_static, the entry point for callers that must not allocate device memory.

Who needs it: a sampler that shares the GPU with a framework whose memory pool already holds all free HBM (a cudaMalloc
inside the library would fail), a job under a fixed memory quota, or a loop that cannot take the stall cudaMalloc /
cudaFree put on the device's other streams.  mbhl_unpack_coords may allocate its workspace on the first call; the
_static form runs the same kernel with its scratch records in a fixed 2.6 MB array inside libmbhl.so and allocates
nothing, at the price of a limit of 1024 walkers per call and of one array shared by all callers on a device.

What is checked: on two calls in a row (the second with fewer rows and other coordinates, so that it runs over the
first call's left-over records) the output equals that of the existing mbhl_unpack_coords bit for bit, NaN rows
included - the repository's tolerance for this conversion is a few ulps against the oracle (test_gpu_sampler.py); the
two GPU paths run identical arithmetic, so equality is the right bar between them.  Also: a batch above the limit and
overlapping buffers are refused with a clear message, and the call itself leaves the device's allocated memory
unchanged.

This file is named test_zz_* so that pytest collects it last: with `-x` a failure here cannot hide any other test.
It builds its own small context and inputs, so it passes alone in a fresh process as well as after the other files.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2005_01827_b200 import binding as M

DEV = "cuda:0"
# Table I box of the sampler's coordinates: ln M_T, q, a1, a2, ln D_L, phi_ref, cos iota, lambda, sin beta, psi, ln t
LO = np.array([np.log(1e3), 0.05, -0.99, -0.99, np.log(0.044), 0.0, -1.0, 0.0, -1.0, 0.0, np.log(1.0)])
HI = np.array([np.log(1e9), 1.0, 0.99, 0.99, np.log(1298.0), 2 * np.pi, 1.0, 2 * np.pi, 1.0, np.pi, np.log(3.15576e8)])


def dev(x):
    return torch.as_tensor(np.ascontiguousarray(x), device=DEV)


def make_ctx():
    """A small context of its own: 4096 uniform bins, flat PSD, zero data (the conversion does not look at the data)."""
    n = 4096
    freqs = 1e-4 + np.arange(n) * 2.4e-5
    data = np.zeros((3, n), dtype=np.complex128)
    psd = np.full((3, n), 1e-40)
    return M.mbhl_init(dev(freqs), dev(data), dev(psd), sparse_points=64, t0=1.0e6)


def rows_for(seed, n):
    rng = np.random.default_rng(seed)
    th = rng.uniform(LO, HI, size=(n, 11))
    th[:, 10] = np.log(rng.uniform(1e4, 6e7, n))
    th[0, 1] = 1.5                   # outside the box: the row comes back as NaN on both paths
    th[1, 8] = 1.0                   # a pole of the LISA frame
    return th


def test_static_scratch_entry_point_matches_the_allocating_path_on_two_calls_in_a_row():
    ctx = make_ctx()
    first = rows_for(7, M.STATIC_MAX_WALKERS)           # fills the whole fixed array
    second = rows_for(8, 37)                            # then a short, ragged batch over its left-overs
    for th, coords in ((first, M.COORDS_SAMPLED_LISA), (second, M.COORDS_SAMPLED)):
        rows = dev(th)
        want = M.mbhl_unpack_coords(ctx, rows, coords)                  # existing path (context workspace)
        out = torch.full((th.shape[0], M.NPARAM), -7.0, dtype=torch.float64, device=DEV)
        torch.cuda.synchronize()
        before = torch.cuda.mem_get_info()[0]
        got = M.mbhl_unpack_coords_static(ctx, rows, coords, out)       # fixed-array path
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] >= before                   # the call took no device memory
        np.testing.assert_array_equal(got.cpu().numpy(), want.cpu().numpy())   # bit for bit; NaN == NaN here
        assert np.all(np.isnan(got[0].cpu().numpy())) and np.all(np.isfinite(got[1:].cpu().numpy()))
    # and once more with the first batch: a repeat after the short call still agrees
    again = M.mbhl_unpack_coords_static(ctx, dev(first), M.COORDS_SAMPLED_LISA,
                                        torch.empty((first.shape[0], M.NPARAM), dtype=torch.float64, device=DEV))
    np.testing.assert_array_equal(again.cpu().numpy(), M.mbhl_unpack_coords(ctx, dev(first), M.COORDS_SAMPLED_LISA).cpu().numpy())
    M.mbhl_free(ctx)


def test_static_scratch_entry_point_refuses_what_it_cannot_hold():
    ctx = make_ctx()
    too_many = dev(rows_for(9, M.STATIC_MAX_WALKERS + 1))
    out = torch.empty_like(too_many)
    with pytest.raises(M.MbhlError, match="MBHL_STATIC_MAX_WALKERS"):
        M.mbhl_unpack_coords_static(ctx, too_many, M.COORDS_SAMPLED, out)
    rows = dev(rows_for(10, 16))
    with pytest.raises(M.MbhlError, match="overlap"):
        M.mbhl_unpack_coords_static(ctx, rows, M.COORDS_SAMPLED, rows)   # in place is not allowed
    with pytest.raises(M.MbhlError):
        M.mbhl_unpack_coords_static(ctx, rows, 7, torch.empty_like(rows))
    empty = torch.empty((0, M.NPARAM), dtype=torch.float64, device=DEV)
    assert M.mbhl_unpack_coords_static(ctx, empty, M.COORDS_SAMPLED, torch.empty_like(empty)).shape[0] == 0
    M.mbhl_free(ctx)
