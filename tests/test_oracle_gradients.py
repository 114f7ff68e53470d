"""Pins for the oracle's hand-derived reverse sweep: central finite
differences of the (separately pinned) oracle forward for EVERY parameter of every model kind,
linearity in the cotangent, and Euler homogeneity in b0.  CPU only."""
import numpy as np
import pytest

import oracle
from harness import workloads as wl


def loss(model_factory, p, geom, cots, pix):
    I, Q, U = oracle.forward(model_factory(p), *geom, pix=pix)
    return float((cots[0] * I).sum() + (cots[1] * Q).sum() + (cots[2] * U).sum())


def fd_check(model_factory, p, geom, pix, seed, rel=1e-5, h_rel=1e-6, idx=None, abs_floor=0.0):
    nfreq = len(geom[3])
    rng = np.random.default_rng(seed)
    shape = (1, nfreq, len(pix))
    cots = [rng.standard_normal(shape) for _ in range(3)]
    g = oracle.vjp(model_factory(p), *geom, *cots, pix=pix).ravel()
    flat = np.asarray(p, dtype=np.float64).ravel()
    for j in (range(flat.size) if idx is None else idx):
        h = h_rel * max(abs(flat[j]), 1e-3)
        pp, pm = flat.copy(), flat.copy()
        pp[j] += h; pm[j] -= h
        fd = (loss(model_factory, pp.reshape(np.shape(p)), geom, cots, pix) -
              loss(model_factory, pm.reshape(np.shape(p)), geom, cots, pix)) / (2 * h)
        assert g[j] == pytest.approx(fd, rel=rel, abs=abs_floor), (j, g[j], fd)
    return g


def test_fd_disc4_cfg0_all_pixels():
    w = wl.config(0)
    aux = w.aux.astype(np.float64)
    geom = (w.nside, w.n_los, w.s_max, w.freqs)
    fd_check(lambda p: oracle.Model("disc4", p, aux=aux), w.params.astype(np.float64)[0], geom,
             np.arange(w.npix), seed=1)


def test_fd_disc4_low_frequency_strong_faraday():
    w = wl.config(0)
    aux = w.aux.astype(np.float64)
    geom = (16, 128, 20.0, np.array([0.408e9, 2.4e9]))
    pix = np.array([1400, 1500, 1530, 1600, 1700])   # near the plane: large Faraday depth
    fd_check(lambda p: oracle.Model("disc4", p, aux=aux), w.params.astype(np.float64)[0], geom, pix, seed=2,
             rel=2e-5)


@pytest.mark.parametrize("cfg", [2, 4])
def test_fd_full16_three_sightlines(cfg):
    w = wl.config(cfg)
    rng = np.random.default_rng(100 + cfg)
    pix = np.sort(rng.choice(w.npix, 3, replace=False))
    # add one in-plane pixel so the Faraday terms are exercised hard
    pix = np.append(pix, w.npix // 2 + 3)
    geom = (w.nside, min(w.n_los, 256), w.s_max, w.freqs)
    p = w.params.astype(np.float64)[min(7, w.batch - 1)]
    fd_check(lambda q: oracle.Model("full16", q), p, geom, pix, seed=3, rel=1e-5)


def test_fd_full16_alpha_not_three():
    p = wl.FULL16_NOMINAL.copy(); p[12] = 2.7
    geom = (4, 64, 25.0, np.array([0.408e9, 1.4e9, 23e9]))
    fd_check(lambda q: oracle.Model("full16", q), p, geom, np.array([3, 77, 90, 101, 188]), seed=4)


def test_fd_uniform_all_six():
    p = np.array([2.0, -3.0, 1.5, 4e-5, 0.02, 2.8])
    geom = (2, 32, 3.0, np.array([0.408e9, 2.4e9]))
    fd_check(lambda q: oracle.Model("uniform", q), p, geom, np.arange(48), seed=5)


def test_fd_grid_64_random_node_components():
    rng = np.random.default_rng(6)
    shape, box = (9, 8, 5), (40.0, 40.0, 8.0)
    X, Y, Z = wl.grid_nodes(shape, box)
    G = wl.spiral_pattern(X, Y, Z, *wl.DISC4_NOMINAL) + rng.normal(size=shape + (3,))
    aux = wl.AUX_NOMINAL
    geom = (4, 64, 20.0, np.array([0.408e9]))
    pix = np.arange(192)
    # pick 64 node-components that the sightlines actually touch
    cots0 = [np.ones((1, 1, 192))] * 3
    touched = np.flatnonzero(oracle.vjp(oracle.Model("grid_b", G, aux=aux, box=box), *geom, *cots0, pix=pix).ravel() != 0)
    idx = rng.choice(touched, 64, replace=False)
    g = fd_check(lambda q: oracle.Model("grid_b", q, aux=aux, box=box), G, geom, pix, seed=7, idx=idx, rel=2e-5, h_rel=1e-5,
                 abs_floor=3e-8)  # floor = FD round-off: eps*|loss|/(2h)
    # nodes no sightline sample touches get exactly zero
    untouched = np.setdiff1d(np.arange(G.size), touched)
    assert np.all(g[untouched] == 0.0)


def test_vjp_linear_in_cotangent_and_none_is_zero():
    w = wl.config(4).scaled(nside=2, n_los=64)
    m = oracle.Model("full16", w.params.astype(np.float64))
    geom = (w.nside, w.n_los, w.s_max, w.freqs)
    rng = np.random.default_rng(8)
    c1 = [rng.standard_normal((1, 8, 48)) for _ in range(3)]
    c2 = [rng.standard_normal((1, 8, 48)) for _ in range(3)]
    g1 = oracle.vjp(m, *geom, *c1)
    g2 = oracle.vjp(m, *geom, *c2)
    g12 = oracle.vjp(m, *geom, *[2.0 * a - 0.5 * b for a, b in zip(c1, c2)])
    np.testing.assert_allclose(g12, 2.0 * g1 - 0.5 * g2, rtol=1e-9, atol=1e-12 * np.abs(g1).max())
    gI = oracle.vjp(m, *geom, c1[0], None, None)
    gQ = oracle.vjp(m, *geom, None, c1[1], None)
    gU = oracle.vjp(m, *geom, None, None, c1[2])
    np.testing.assert_allclose(gI + gQ + gU, g1, rtol=1e-9, atol=1e-12 * np.abs(g1).max())


def test_b0_homogeneity_without_faraday():
    # n_e = 0: I,Q,U are homogeneous of degree (alpha+1)/2 in b0 -> b0 dL/db0 = (alpha+1)/2 * L
    w = wl.config(0)
    aux = w.aux.astype(np.float64); aux[4] = 0.0; aux[3] = 3.0
    p = w.params.astype(np.float64)[0]
    m = oracle.Model("disc4", p, aux=aux)
    geom = (w.nside, w.n_los, w.s_max, w.freqs)
    rng = np.random.default_rng(9)
    cots = [rng.standard_normal((1, 1, w.npix)) for _ in range(3)]
    I, Q, U = oracle.forward(m, *geom)
    L = (cots[0] * I).sum() + (cots[1] * Q).sum() + (cots[2] * U).sum()
    g = oracle.vjp(m, *geom, *cots)
    assert g[0, 0] == pytest.approx(2.0 / p[0] * L, rel=1e-10)
    # with n_e != 0 the Faraday term adds to it
    aux2 = aux.copy(); aux2[4] = 0.03
    m2 = oracle.Model("disc4", p, aux=aux2)
    I, Q, U = oracle.forward(m2, 8, 64, 20.0, [0.408e9])
    L2 = (cots[0] * I).sum() + (cots[1] * Q).sum() + (cots[2] * U).sum()
    g2 = oracle.vjp(m2, 8, 64, 20.0, [0.408e9], *cots)
    assert abs(g2[0, 0] - 2.0 / p[0] * L2) > 1e-3 * abs(g2[0, 0])


@pytest.mark.parametrize("zero", [(0,), (5,), (9,), (13,), (0, 13)])
def test_fd_full16_zero_amplitudes(zero):
    """Amplitude parameters exactly at zero (b0 at the edge of the paper's U[0,10] prior, n_e0 = 0 to switch Faraday
    rotation off, ...): the derivative with respect to an amplitude is the unit-amplitude field (App. D.3:
    dB/db0 = B_disc / b0), finite there; checked by central differences straddling zero."""
    p = wl.FULL16_NOMINAL.copy()
    scale = {0: 6.0, 5: 2.0, 9: 2.1e-4, 13: 0.03}
    for j in zero:
        p[j] = 0.0
    geom = (4, 64, 25.0, np.array([0.408e9, 1.4e9]))
    pix = np.array([3, 77, 90, 101, 188])
    rng = np.random.default_rng(40)
    cots = [rng.standard_normal((1, 2, len(pix))) for _ in range(3)]
    model = lambda q: oracle.Model("full16", q)   # noqa: E731
    g = oracle.vjp(model(p), *geom, *cots, pix=pix).ravel()
    assert np.all(np.isfinite(g))
    for j in zero:
        h = (1e-7 if j == 13 else 1e-5) * scale[j]   # n_e0 enters through cos / sin of up to ~1500 rad x n_e0 / 0.03
        pp, pm = p.copy(), p.copy()
        pp[j] += h; pm[j] -= h
        fd = (loss(model, pp, geom, cots, pix) - loss(model, pm, geom, cots, pix)) / (2 * h)
        assert g[j] == pytest.approx(fd, rel=2e-6, abs=1e-9 * np.abs(g).max()), (j, g[j], fd)
    if 9 in zero:      # N_0 = 0: no emission, every other derivative vanishes exactly
        assert np.all(g[np.arange(16) != 9] == 0.0) and g[9] != 0.0
