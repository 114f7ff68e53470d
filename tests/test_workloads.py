"""Seeded input generators: shapes, determinism, the stated recipe.  CPU only."""
import numpy as np

from harness import workloads as wl


def test_config_table_sizes():
    sizes = [(768, 64, 1, 1, 49152), (49152, 256, 3, 1, 12582912), (12288, 256, 1, 256, 805306368),
             (49152, 512, 1, 1, 25165824), (786432, 1024, 8, 1, 805306368)]
    for i, (npix, n_los, nf, batch, samples) in enumerate(sizes):
        w = wl.config(i)
        assert (w.npix, w.n_los, w.n_freq, w.batch, w.los_samples) == (npix, n_los, nf, batch, samples)
        assert w.params.dtype == np.float32


def test_draws_are_deterministic_and_in_range():
    a, b = wl.config(1), wl.config(1)
    assert np.array_equal(a.params, b.params)
    p = a.params[0]
    assert 3 <= p[0] <= 9 and 15 <= p[1] / wl.DEG <= 35 and 0 <= p[2] / wl.DEG <= 2 and 10 <= p[3] / wl.DEG <= 40
    w2 = wl.config(2)
    r = w2.params.astype(np.float64) / wl.FULL16_NOMINAL
    assert r.min() >= 0.8 - 1e-6 and r.max() <= 1.2 + 1e-6 and r.std() > 0.1
    c1 = a.cotangents(); c2 = b.cotangents()
    assert all(np.array_equal(x, y) for x, y in zip(c1, c2))
    assert c1[0].shape == (1, 3, 49152) and abs(c1[1].std() - 1) < 0.02
    ones = wl.config(0).cotangents(ones=True)
    assert np.all(ones[2] == 1)
    f = wl.config(4).freqs
    assert f[0] == 0.408e9 and abs(f[-1] - 30e9) < 1 and np.allclose(np.diff(np.log(f)), np.log(f[1] / f[0]))


def test_grid_recipe():
    w = wl.config(3)
    assert w.params.shape == (128, 128, 32, 3) and w.box == (40.0, 40.0, 8.0)
    X, Y, Z = wl.grid_nodes((128, 128, 32), w.box)
    spiral = wl.spiral_pattern(X, Y, Z, *wl.DISC4_NOMINAL)
    d = w.params.astype(np.float64) - spiral
    assert abs(np.sqrt(np.mean(np.sum(d * d, -1))) - 3.0) < 1e-3      # GRF rms 3 uG
    assert abs(d.mean()) < 1e-6                                       # k = 0 mode removed
    rho = np.hypot(X, Y)
    assert np.all(spiral[(rho <= 3) | (rho >= 20)] == 0)
    # red spectrum: neighbouring nodes are strongly correlated
    c = np.mean(d[1:, :, :, 0] * d[:-1, :, :, 0]) / np.mean(d[..., 0] ** 2)
    assert c > 0.5


def test_scaled_keeps_model():
    w = wl.config(2).scaled(nside=4, n_los=32, batch=3)
    assert w.params.shape == (3, 16) and w.npix == 192 and w.los_samples == 192 * 32 * 3
