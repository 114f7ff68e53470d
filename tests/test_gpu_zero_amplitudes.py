"""Amplitude parameters exactly at zero: the adjoint accumulates amplitude derivatives with the unit-amplitude field
(App. D.3: dB/db0 = B_disc / b0 etc.), so they stay finite -- no 0/0 -- and match the oracle."""
import numpy as np
import pytest

from harness import parity
from harness import workloads as wl

pytestmark = pytest.mark.gpu


def _check(w, what):
    maps, _ = parity.gpu_forward(w)
    ref = parity.oracle_forward(w)
    for m, r in zip(maps, ref):
        rms = np.sqrt(np.mean(r * r, axis=-1, keepdims=True))
        assert np.all(np.abs(m - r) <= parity.MAP_TOL * rms + 0.0), what   # zero maps must be exactly zero
    cots = w.cotangents()
    g, gr = parity.gpu_vjp(w, cots), parity.oracle_vjp(w, cots)
    assert np.all(np.isfinite(g)), (what, g)
    nz = gr != 0
    assert np.all(np.abs(g - gr)[nz] <= parity.GRAD_TOL * np.abs(gr)[nz]), (what, np.abs(g - gr)[nz] / np.abs(gr)[nz])
    assert np.all(g[~nz] == 0.0), (what, g[~nz])


@pytest.mark.parametrize("zero", [(0,), (5,), (9,), (13,), (0, 13), (0, 5)])
@pytest.mark.parametrize("lanes", [1, 8])
def test_full16_zero_amplitudes(zero, lanes):
    w = wl.config(4).scaled(nside=8, n_los=256)
    p = w.params.copy()
    for j in zero:
        p[0, j] = 0.0
    w.params = p
    maps, _ = parity.gpu_forward(w, lanes=lanes)
    ref = parity.oracle_forward(w)
    for m, r in zip(maps, ref):
        rms = np.sqrt(np.mean(r * r, axis=-1, keepdims=True))
        assert np.all(np.abs(m - r) <= parity.MAP_TOL * rms), zero
    cots = w.cotangents()
    g, gr = parity.gpu_vjp(w, cots, lanes=lanes), parity.oracle_vjp(w, cots)
    assert np.all(np.isfinite(g)), (zero, g)
    nz = gr != 0
    assert np.all(np.abs(g - gr)[nz] <= parity.GRAD_TOL * np.abs(gr)[nz]), (zero, np.abs(g - gr)[nz] / np.abs(gr)[nz])
    assert np.all(g[~nz] == 0.0), (zero, g[~nz])


def test_disc4_zero_b0():
    w = wl.config(1).scaled(nside=8, n_los=128)
    p = w.params.copy(); p[0, 0] = 0.0
    w.params = p
    _check(w, "disc4 b0 = 0")


def test_stack16_zero_b0_of_one_spiral():
    w = wl.stack16(nside=8, n_los=128, freqs=(1.4e9, 23e9))
    p = w.params.copy(); p[0, 4] = 0.0
    w.params = p
    _check(w, "stack16 b0_2 = 0")


@pytest.mark.parametrize("which", [3, 4])
def test_uniform_zero_density(which):
    w = wl.uniform_toy(bvec=(2.0, -3.0, 1.5), nside=4, n_los=48, freqs=(0.408e9, 2.4e9))
    p = w.params.copy(); p[0, which] = 0.0
    w.params = p
    _check(w, f"uniform p[{which}] = 0")
