"""The paper's own 16-parameter model (Eq. 16; Table 3): oracle pins, GPU parity."""
import numpy as np
import pytest

import oracle
from harness import parity
from harness import workloads as wl

W = (0.6, 0.3, 0.1, 0.3)                                  # weights printed in Eq. (16)
SRC = ((0, 1, 2), (0, 2, 1), (2, 1, 0), (1, 0, 2))        # B_x = .6 B1x + .3 B2x + .1 B3z + .3 B4y, etc.


def test_stack_is_the_printed_combination_of_four_wmap_spirals():
    rng = np.random.Generator(np.random.PCG64(16))
    r = rng.uniform(-1, 1, (300, 3)) * np.array([22.0, 22.0, 3.0])
    B, N0, ne, al = oracle.eval_fields(oracle.Model("stack16", wl.STACK16_TABLE3, aux=wl.AUX_NOMINAL), r)
    tot = np.zeros_like(B)
    for k in range(4):
        Bk, N0k, nek, _ = oracle.eval_fields(oracle.Model("disc4", wl.STACK16_TABLE3[4 * k:4 * k + 4], aux=wl.AUX_NOMINAL), r)
        for c in range(3):
            tot[:, c] += W[k] * Bk[:, SRC[k][c]]
    assert np.abs(B - tot).max() < 1e-15 and np.array_equal(N0, N0k) and np.array_equal(ne, nek) and np.all(al == 3.0)
    rho = np.hypot(r[:, 0], r[:, 1])
    assert np.all(B[(rho <= 3) | (rho >= 20)] == 0.0) and np.any(B[(rho > 3) & (rho < 20)] != 0.0)


def test_single_component_reduces_to_disc4():
    """b0 of spirals 2-4 set to zero: the maps are those of DISC4 with b0 -> 0.6 b0_1 (identity permutation)."""
    p = wl.STACK16_TABLE3.copy()
    p[[4, 8, 12]] = 0.0
    w = wl.stack16(nside=4, n_los=64)
    w.params = p[None, :].astype(np.float32)
    m = parity.oracle_forward(w)
    q = w.params[0, :4].astype(np.float64) * np.array([0.6, 1, 1, 1])
    d = oracle.forward(oracle.Model("disc4", q, aux=w.aux.astype(np.float64)), w.nside, w.n_los, w.s_max, w.freqs)
    for a, b in zip(m, d):
        assert np.allclose(a, b, rtol=1e-12, atol=1e-300)


def test_stack16_gradient_matches_finite_differences():
    w = wl.stack16(nside=2, n_los=48, freqs=(1.4e9, 23e9))
    cots = w.cotangents()
    g = parity.oracle_vjp(w, cots)[0]
    base = w.params.astype(np.float64)
    for j in range(16):
        h = 1e-6 * abs(base[0, j])
        vals = []
        for sgn in (1, -1):
            q = base.copy(); q[0, j] += sgn * h
            I, Q, U = oracle.forward(oracle.Model("stack16", q, aux=w.aux.astype(np.float64)), w.nside, w.n_los, w.s_max, w.freqs)
            vals.append((I * cots[0]).sum() + (Q * cots[1]).sum() + (U * cots[2]).sum())
        fd = (vals[0] - vals[1]) / (2 * h)
        assert abs(fd - g[j]) <= 3e-5 * abs(g[j]), (j, fd, g[j])


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["2.4GHz", "408MHz_f64", "batch", "clip_ne_grid"])
def test_gpu_stack16_parity(case):
    if case == "2.4GHz":
        w = wl.stack16(nside=16, n_los=256, freqs=(2.4e9, 23e9))
    elif case == "408MHz_f64":
        w = wl.stack16(nside=16, n_los=1024, freqs=(0.408e9, 1.4e9))
    elif case == "batch":
        w = wl.stack16(nside=8, n_los=100, freqs=(23e9,), batch=5)
    else:
        w = wl.stack16(nside=8, n_los=256, freqs=(1.4e9,))
        w.clip_box = (40.0, 40.0, 10.0)
        w.ne_grid, w.ne_box = wl.clumpy_disc_grid((32, 32, 16), w.clip_box, 0.03, 20.0, 1.0, seed=83), w.clip_box
    maps, _ = parity.gpu_forward(w)
    parity.assert_maps_close(maps, parity.oracle_forward(w), what=f"stack16 forward {case}")
    cots = w.cotangents()
    g, ref = parity.gpu_vjp(w, cots), parity.oracle_vjp(w, cots)
    rel = np.abs(g - ref) / np.abs(ref)
    assert rel.max() <= parity.GRAD_TOL, (case, rel.max(), np.unravel_index(rel.argmax(), rel.shape))
