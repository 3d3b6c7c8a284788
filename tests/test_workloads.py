"""Host logic of the synthetic-input generators (no method arithmetic there)."""
import numpy as np

from paper_2005_01827_b200 import workloads as W


def zero_template(p, f, S):
    return np.zeros((3, f.size), dtype=np.complex128)


def test_grids_and_shapes_follow_baseline_configs():
    wl = W.build(0, zero_template)
    assert wl["freqs"].size == 1 << 16 and wl["S"] == 256 and wl["params"].shape == (4, 11)
    df = 1.0 / (0.1 * W.YEAR_JULIAN_S)
    assert abs(wl["freqs"][1] - wl["freqs"][0] - df) < 1e-20 and wl["freqs"][0] >= 1e-4 > wl["freqs"][0] - df
    assert np.all(wl["params"][:, 0] == 1e6) and np.all((wl["params"][:, 1] >= 1) & (wl["params"][:, 1] <= 5))
    wl1 = W.build(1, zero_template, n_bins=4096)
    assert wl1["S"] == 512 and wl1["params"].shape == (64, 11)
    assert np.max(np.abs(wl1["params"][:, 0] / 1e6 - 1.0)) < 1e-2
    wl2 = W.build(2, zero_template, n_bins=4096, batch=30)
    assert wl2["S"] == 1024 and wl2["params"].shape == (30, 11) and wl2["injections"].shape == (3, 11)
    assert int(np.floor(0.1 * 1.33 * W.YEAR_JULIAN_S)) == 4197160


def test_seeding_is_deterministic_and_noise_has_the_stated_variance():
    a = W.build(0, zero_template, n_bins=4096)
    b = W.build(0, zero_template, n_bins=4096)
    assert np.array_equal(a["data"], b["data"]) and np.array_equal(a["params"], b["params"])
    rng = np.random.default_rng(0)
    psd = np.full((3, 200000), 2.0)
    n = W.noise(rng, psd, 0.5)
    # Re, Im ~ N(0, S/(4 df)): E[4 df |n|^2 / S] = 2 per bin (reading G5)
    assert abs(np.mean(4 * 0.5 * np.abs(n) ** 2 / psd) - 2.0) < 0.02


def test_psd_shape():
    f = np.array([1e-4, 1e-3, 1e-2])
    s = W.scird_psd_aet(f)
    assert s.shape == (3, 3) and np.all(s > 0) and np.array_equal(s[0], s[1])
    assert np.all(s[2] < s[0])            # T is the quiet channel at low frequency
