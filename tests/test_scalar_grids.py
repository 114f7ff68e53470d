"""Gridded n_e / N_0: oracle pins on CPU, GPU parity for DISC4 and GRID_B models."""
import numpy as np
import pytest

import oracle
from harness import parity
from harness import workloads as wl

BOX = (40.0, 40.0, 10.0)


def _disc4():
    return oracle.Model("disc4", wl.DISC4_NOMINAL, aux=wl.AUX_NOMINAL)


def test_trilinear_scalar_reproduces_linear_functions_and_is_zero_outside():
    ax = [np.linspace(-l / 2, l / 2, n) for n, l in zip((9, 7, 5), BOX)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    lin = lambda x, y, z: 0.01 + 0.001 * x - 0.002 * y + 0.003 * z   # noqa: E731
    rng = np.random.Generator(np.random.PCG64(4))
    r = rng.uniform(-1, 1, (200, 3)) * np.array(BOX) * 0.5
    r[:3] = [[20.0, 20.0, 5.0], [-20.0, -20.0, -5.0], [20.0, 0.0, 0.0]]          # corners / faces are inside
    with oracle.scalar_grids(ne=lin(X, Y, Z), ne_box=BOX, n0=2.0 * lin(X, Y, Z), n0_box=BOX):
        B, N0, ne, _ = oracle.eval_fields(_disc4(), r)
        assert np.abs(ne - lin(*r.T)).max() < 1e-15 and np.abs(N0 - 2 * lin(*r.T)).max() < 1e-15
        _, N0o, neo, _ = oracle.eval_fields(_disc4(), [[20.0001, 0, 0], [0, -20.1, 0], [0, 0, 5.01]])
        assert np.all(neo == 0.0) and np.all(N0o == 0.0)
    _, N0a, nea, _ = oracle.eval_fields(_disc4(), r[:5])                          # grids removed: analytic discs again
    assert np.all(nea > 0) and not np.allclose(nea, lin(*r[:5].T))


def test_grid_sampled_from_the_analytic_disc_converges_to_the_analytic_maps():
    """Fig. 6 lower for the scalar fields: error falls as the grid is refined (second order)."""
    wr = wl.config(1).scaled(nside=4, n_los=128)
    wr.clip_box = BOX                                                             # stay inside the grids
    ref = parity.oracle_forward(wr)
    a = wl.AUX_NOMINAL
    err_I, err_P = [], []
    for n in (17, 33, 65):
        X, Y, Z = wl.grid_nodes((n, n, n), BOX)
        disc = lambda amp, hr, hz: amp * np.exp(-np.hypot(X, Y) / hr) / np.cosh(Z / hz) ** 2   # noqa: E731
        w = wl.config(1).scaled(nside=4, n_los=128)
        w.clip_box = BOX
        w.ne_grid, w.ne_box = disc(a[4], a[5], a[6]).astype(np.float32), BOX
        w.n0_grid, w.n0_box = disc(a[0], a[1], a[2]).astype(np.float32), BOX
        m = parity.oracle_forward(w)
        e = [np.abs(m[k] - ref[k]).max() / np.abs(ref[k]).max() for k in range(3)]
        err_I.append(e[0]); err_P.append(max(e[1], e[2]))
    assert err_I[0] / err_I[1] > 3.0 and err_I[1] / err_I[2] > 3.0 and err_I[2] < 1e-3     # second order in the spacing
    assert err_P[0] > err_P[1] > err_P[2] and err_P[2] < 0.03


def test_gridded_ne_gradient_matches_finite_differences():
    w = wl.config(1).scaled(nside=2, n_los=48)
    w.ne_grid, w.ne_box = wl.clumpy_disc_grid((17, 17, 9), BOX, 0.03, 20.0, 1.0, seed=77), BOX
    w.clip_box = BOX
    cots = w.cotangents()
    g = parity.oracle_vjp(w, cots)[0]
    base = w.params.astype(np.float64)
    for j in range(4):
        h = 1e-6 * abs(base[0, j])
        vals = []
        for sgn in (1, -1):
            q = base.copy(); q[0, j] += sgn * h
            ww = wl.config(1).scaled(nside=2, n_los=48)
            ww.ne_grid, ww.ne_box, ww.clip_box = w.ne_grid, BOX, BOX
            with oracle.scalar_grids(ne=w.ne_grid, ne_box=BOX):
                I, Q, U = oracle.forward(oracle.Model("disc4", q, aux=w.aux.astype(np.float64)), w.nside, w.n_los, w.s_max,
                                         w.freqs, clip_box=BOX)
            vals.append((I * cots[0]).sum() + (Q * cots[1]).sum() + (U * cots[2]).sum())
        fd = (vals[0] - vals[1]) / (2 * h)
        assert abs(fd - g[j]) <= 2e-5 * abs(g[j]), (j, fd, g[j])


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["disc4_ne", "disc4_ne_n0_lowfreq", "gridb_ne_n0"])
def test_gpu_gridded_scalars_parity(case):
    """The paper's section 3.1 set-up in miniature: WMAP B (4 parameters) analytic, n_e on a grid."""
    if case == "disc4_ne":
        w = wl.config(1).scaled(nside=16, n_los=256)
        w.ne_grid, w.ne_box = wl.clumpy_disc_grid((64, 64, 16), BOX, 0.03, 20.0, 1.0, seed=78), BOX
    elif case == "disc4_ne_n0_lowfreq":
        w = wl.config(1).scaled(nside=16, n_los=512)
        w.freqs = np.array([0.408e9, 1.4e9])                                      # strong rotation: float64 chain
        w.ne_grid, w.ne_box = wl.clumpy_disc_grid((64, 64, 16), BOX, 0.03, 20.0, 1.0, seed=79), BOX
        w.n0_grid, w.n0_box = wl.clumpy_disc_grid((32, 32, 16), BOX, 2.1038e-4, 5.0, 1.0, seed=80, contrast=0.1), BOX
    else:
        w = wl.config(3).scaled(nside=8, n_los=256)
        w.ne_grid, w.ne_box = wl.clumpy_disc_grid((32, 32, 8), (40.0, 40.0, 8.0), 0.03, 20.0, 1.0, seed=81), (40.0, 40.0, 8.0)
        w.n0_grid, w.n0_box = wl.clumpy_disc_grid((32, 32, 8), (40.0, 40.0, 8.0), 2.1038e-4, 5.0, 1.0, seed=82, contrast=0.1), (40.0, 40.0, 8.0)
    maps, _ = parity.gpu_forward(w)
    parity.assert_maps_close(maps, parity.oracle_forward(w), what=f"gridded scalars forward {case}")
    cots = w.cotangents()
    g, ref = parity.gpu_vjp(w, cots), parity.oracle_vjp(w, cots)
    if w.kind == "grid_b":
        rms = np.sqrt(np.mean(ref[ref != 0] ** 2))
        assert np.all(np.abs(g - ref) <= 1e-3 * np.abs(ref) + 1e-4 * rms) and np.array_equal(ref == 0.0, g == 0.0)
    else:
        assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref))


@pytest.mark.gpu
def test_gpu_paper_section31_workload_full_size():
    """PAPER.md section 3.1 at the paper's sizes (L180): NSIDE 64, N_int 512, n_e on a (256, 256, 64) grid (16.8 MB: another
    cache regime than the small grids above), WMAP B with the paper's true values, box-clipped integration; forward and
    gradient against the oracle on every pixel."""
    w = wl.paper_section31()
    assert w.ne_grid.shape == (256, 256, 64) and w.npix * w.n_los == 25165824
    maps, _ = parity.gpu_forward(w)
    parity.assert_maps_close(maps, parity.oracle_forward(w), what="section 3.1 forward")
    cots = w.cotangents()
    g, ref = parity.gpu_vjp(w, cots), parity.oracle_vjp(w, cots)
    assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref)), np.abs(g - ref) / np.abs(ref)


@pytest.mark.gpu
@pytest.mark.parametrize("ne_amp", [0.12, 0.5])
def test_gpu_strong_ne_grid_with_zero_aux_ne(ne_amp):
    """The aux n_e entries are ignored when a gridded n_e is given (synax.h), so the caller may leave them at zero: the
    float64 chain's tile length (fp32 in-tile Faraday angle) must then be sized from the grid itself.  n_e grid 4-17 x
    the nominal disc at 408 MHz, few samples (several rad per step)."""
    w = wl.config(1).scaled(nside=16, n_los=128)
    w.freqs = np.array([0.408e9])
    w.aux = w.aux.copy(); w.aux[4] = 0.0
    w.ne_grid, w.ne_box = wl.clumpy_disc_grid((64, 64, 16), BOX, ne_amp, 20.0, 1.0, seed=83), BOX
    ref = parity.oracle_forward(w)
    for precision in (0, 2):
        maps, _ = parity.gpu_forward(w, precision=precision)
        parity.assert_maps_close(maps, ref, what=f"strong n_e grid, aux ne0 = 0, precision {precision}")
    cots = w.cotangents()
    gr = parity.oracle_vjp(w, cots)
    for precision in (0, 2):
        g = parity.gpu_vjp(w, cots, precision=precision)
        assert np.all(np.abs(g - gr) <= parity.GRAD_TOL * np.abs(gr)), (precision, np.abs(g - gr) / np.abs(gr))


@pytest.mark.gpu
def test_gpu_gridded_scalars_rejected_for_full16():
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(2).scaled(nside=4, n_los=32, batch=1)
    plan = sx.Plan(w.nside, w.n_los, w.s_max, w.freqs)
    g = torch.zeros((4, 4, 4), device="cuda")
    with pytest.raises(sx.SynaxError):
        sx.forward(plan, sx.Model("full16", ne_grid=g, ne_box=BOX), torch.from_numpy(w.params).cuda())
    plan.close()
