"""The seeded input generators: shapes, determinism, window bounds, recipe facts."""
import numpy as np
import pytest

from paper_1808_10375_b200 import synth


def test_config_table_matches_baseline_json():
    want = [(64, 100, 1, 1, 160, 160), (128, 2500, 2, 1, 640, 640), (128, 10000, 4, 1, 760, 760),
            (256, 4096, 4, 2, 1300, 1300), (512, 2000, 3, 1, 1800, 2100)]
    got = [(c.N, c.n_views, c.K, c.L, c.obj_h, c.obj_w) for c in synth.CONFIGS]
    assert got == want
    assert [c.mode_views for c in synth.CONFIGS] == [100, 5000, 40000, 32768, 6000]
    assert [c.n_iter for c in synth.CONFIGS] == [50, 100, 100, 100, 50]
    assert all(c.obj_w % 2 == 0 for c in synth.CONFIGS)


@pytest.mark.parametrize("i", range(5))
def test_positions_inside_object_for_full_configs(i):
    c = synth.CONFIGS[i]
    pos = synth.make_positions(c, np.random.default_rng(0))
    assert pos.shape == (c.n_views, 2) and pos.dtype == np.int32
    assert pos.min() >= 0
    assert (pos[:, 0] + c.N).max() <= c.obj_h and (pos[:, 1] + c.N).max() <= c.obj_w
    # raster order, x fastest
    assert np.all(np.abs(np.diff(pos[:c.nx, 1]) - c.step) <= 2 * c.jit)


def test_problem_is_deterministic_and_typed():
    a = synth.make_problem(0)
    b = synth.make_problem(0)
    for f in ("positions", "intensities", "probe0", "object0"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    assert a.intensities.dtype == np.float32 and a.probe0.dtype == np.complex64
    assert a.object0.dtype == np.complex64 and a.positions.dtype == np.int32
    c = a.cfg
    assert a.intensities.shape == (100, 64, 64) and a.object0.shape == (1, 160, 160)
    assert np.all(a.object0 == 1) and np.allclose(a.probe0, 0.9 * a.probe_true)
    assert 0.8 <= np.abs(a.object_true).min() and np.abs(a.object_true).max() <= 1.0
    ph = np.angle(a.object_true[0])
    assert abs(ph.min() + np.pi / 2) < 1e-6 and abs(ph.max() - np.pi / 2) < 1e-6
    # config 0 is noise-free: I = |FFT2(P O)|^2 exactly (float32-rounded)
    y, x = a.positions[7]
    want = np.abs(np.fft.fft2(a.probe_true[0].astype(complex) * a.object_true[0, y:y + 64, x:x + 64])) ** 2
    assert np.allclose(a.intensities[7], want, rtol=1e-4, atol=1e-4 * want.max())


def test_poisson_scaling_keeps_units_and_photon_budget():
    pr = synth.make_problem(synth.CONFIGS[1].scaled(4, 4))
    c = pr.cfg
    assert pr.probe0.shape == (2, 128, 128) and pr.intensities.min() >= 0
    # mean counts per frame ~ photons once rescaled; intensities stay in |FFT|^2 units
    clean = np.zeros_like(pr.intensities, dtype=np.float64)
    for j, (y, x) in enumerate(pr.positions):
        for k in range(c.K):
            clean[j] += np.abs(np.fft.fft2(pr.probe_true[k].astype(complex) * pr.object_true[0, y:y + 128, x:x + 128])) ** 2
    assert abs(pr.intensities.sum() / clean.sum() - 1) < 1e-2
    s = c.photons / clean.sum(axis=(1, 2)).mean()
    counts = pr.intensities.astype(np.float64) * s
    assert np.abs(counts - np.round(counts)).max() < 1e-2        # integer photon counts


def test_modes_are_distinct_and_weighted():
    P = synth.make_probe(synth.CONFIGS[2])
    pw = (np.abs(P) ** 2).sum((1, 2))
    assert np.allclose(pw / pw.sum(), [0.4, 0.3, 0.2, 0.1])
    assert not np.allclose(P[0] / np.sqrt(0.4), P[1] / np.sqrt(0.3))
