"""synax_forward_f64 / synax_vjp_f64: the paper's own arithmetic -- every step in float64 ("the default
precision is double ... for all examples") -- against the float64 oracle on float64 inputs (not fp32-rounded ones).
Bound: 1e-10 x map RMS per map, 1e-9 relative per gradient component (the two sides differ in summation order and in
their float64 math libraries only)."""
import numpy as np
import pytest

import oracle
from harness import parity
from harness import workloads as wl

pytestmark = pytest.mark.gpu

MAP_TOL_F64 = 1.0e-10
GRAD_TOL_F64 = 1.0e-9


def _run(w, params64, lanes=0):
    import torch
    import paper_2410_01136_b200 as sx
    plan = sx.Plan(w.nside, w.n_los, w.s_max, w.freqs, observer=w.observer)
    if w.clip_box is not None:
        plan.set_box(w.clip_box)
    if lanes:
        plan.set_option("lanes", lanes)
    sg = {}
    if w.ne_grid is not None:
        sg.update(ne_grid=torch.from_numpy(w.ne_grid).cuda().contiguous(), ne_box=w.ne_box)
    model = sx.Model(w.kind, aux=w.aux, **sg)
    p = torch.from_numpy(np.ascontiguousarray(params64)).cuda()
    maps = tuple(t.cpu().numpy() for t in sx.forward_f64(plan, model, p))
    rng = np.random.Generator(np.random.PCG64(w.cot_seed + 17))
    cots = [rng.standard_normal(maps[0].shape) for _ in range(3)]
    g = sx.vjp_f64(plan, model, p, *[torch.from_numpy(c).cuda() for c in cots]).cpu().numpy()
    plan.close()
    aux = None if w.aux is None else w.aux.astype(np.float64)
    m = oracle.Model(w.kind, params64, aux=aux)
    with oracle.scalar_grids(ne=w.ne_grid, ne_box=w.ne_box, n0=None, n0_box=None):
        ref = oracle.forward(m, w.nside, w.n_los, w.s_max, w.freqs, observer=w.observer, clip_box=w.clip_box)
        gr = oracle.vjp(m, w.nside, w.n_los, w.s_max, w.freqs, *cots, observer=w.observer, clip_box=w.clip_box)
    return maps, ref, g, gr


def _check(w, params64, what, lanes=0):
    maps, ref, g, gr = _run(w, params64, lanes)
    e = parity.map_errors(maps, ref)
    assert np.all(np.isfinite(e)) and e.max() <= MAP_TOL_F64, (what, e.reshape(3, -1).max(1))
    nz = gr != 0
    rel = np.abs(g - gr)[nz] / np.abs(gr)[nz]
    assert rel.max() <= GRAD_TOL_F64, (what, rel)
    assert np.all(g[~nz] == 0.0)
    return e.max(), rel.max()


@pytest.mark.parametrize("cfg,lanes", [(0, 0), (0, 1), (1, 0)])
def test_f64_mode_cfg0_cfg1(cfg, lanes):
    w = wl.config(cfg)
    if cfg == 1:
        w = w.scaled(nside=32)
    rng = np.random.Generator(np.random.PCG64(50 + cfg))
    p = w.params.astype(np.float64) * (1.0 + 1e-3 * rng.uniform(-1, 1, w.params.shape))   # not representable in fp32
    em, eg = _check(w, p, f"cfg{cfg}", lanes)
    print(f"float64 mode cfg{cfg}: maps {em:.1e} x RMS, gradient {eg:.1e}")


@pytest.mark.parametrize("lanes", [8, 32])
def test_f64_mode_cfg4_nside16_strong_rotation(lanes):
    w = wl.config(4).scaled(nside=16, n_los=1024)
    p = wl.FULL16_NOMINAL[None, :] * (1.0 + 1e-3 * np.linspace(-1, 1, 16))
    em, eg = _check(w, p, "cfg4 @ nside 16", lanes)
    print(f"float64 mode cfg4@nside16: maps {em:.1e} x RMS, gradient {eg:.1e}")


def test_f64_mode_alpha_not_three_and_batch():
    w = wl.config(2).scaled(nside=4, n_los=100, batch=5)
    p = w.params.astype(np.float64)
    p[:, 12] = [2.5, 2.8, 3.0, 3.2, 3.4]
    w.freqs = np.array([0.408e9, 1.4e9, 23e9])
    _check(w, p, "full16 alpha != 3, batch 5, 3 frequencies")


def test_f64_mode_stack16_uniform_boxclip_and_grid_ne():
    w = wl.stack16(nside=8, n_los=128, freqs=(1.4e9, 23e9))
    _check(w, w.params.astype(np.float64), "stack16")
    w = wl.uniform_toy(bvec=(2.0, -3.0, 1.5), nside=4, n_los=48, freqs=(0.408e9, 2.4e9))
    w.clip_box = (40.0, 40.0, 10.0)
    _check(w, w.params.astype(np.float64), "uniform, box-clipped")
    w = wl.config(1).scaled(nside=8, n_los=128)
    w.ne_grid, w.ne_box = wl.clumpy_disc_grid((32, 32, 8), (40.0, 40.0, 10.0), 0.03, 20.0, 1.0, seed=91), (40.0, 40.0, 10.0)
    _check(w, w.params.astype(np.float64), "disc4 with gridded n_e")


def test_f64_mode_rejects_grid_b():
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(3).scaled(nside=2, n_los=16)
    plan = sx.Plan(w.nside, w.n_los, w.s_max, w.freqs)
    model = sx.Model("grid_b", aux=w.aux, grid_shape=w.params.shape[:3], box=w.box)
    with pytest.raises(sx.SynaxError) as ei:
        sx.forward_f64(plan, model, torch.from_numpy(w.params.astype(np.float64)).cuda())
    assert ei.value.status == 2
    plan.close()
