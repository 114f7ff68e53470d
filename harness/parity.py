"""Shared helpers for the GPU parity tests: run the CUDA library and the oracle on the same seeded
inputs (harness.workloads) and compare per map.  Imported only by tests/, bench.py and __graft_entry__.smoke()."""
from __future__ import annotations

import numpy as np

import oracle
from harness import workloads as wl

MAP_TOL = 1.0e-4    # max |delta| <= MAP_TOL * RMS(oracle map), per (batch, frequency, Stokes) -- BASELINE.json north_star
GRAD_TOL = 1.0e-3   # relative error per gradient component -- BASELINE.json north_star


def oracle_model(w: wl.Workload) -> oracle.Model:
    p = w.params.astype(np.float64)
    aux = None if w.aux is None else w.aux.astype(np.float64)
    return oracle.Model(w.kind, p, aux=aux, box=w.box)


def _grids(w):
    return oracle.scalar_grids(ne=w.ne_grid, ne_box=w.ne_box, n0=w.n0_grid, n0_box=w.n0_box)


def oracle_forward(w: wl.Workload, pix=None):
    with _grids(w):
        return _oracle_forward(w, pix)


def oracle_vjp(w: wl.Workload, cots, pix=None):
    with _grids(w):
        return _oracle_vjp(w, cots, pix)


def _oracle_forward(w: wl.Workload, pix=None):
    return oracle.forward(oracle_model(w), w.nside, w.n_los, w.s_max, w.freqs, observer=w.observer, pix=pix,
                          clip_box=w.clip_box)


def _oracle_vjp(w: wl.Workload, cots, pix=None):
    return oracle.vjp(oracle_model(w), w.nside, w.n_los, w.s_max, w.freqs, *cots, observer=w.observer, pix=pix,
                      clip_box=w.clip_box)


def gpu_objects(w: wl.Workload, pix_range=None, pix_stride=1, **options):
    import torch
    import paper_2410_01136_b200 as sx
    plan = sx.Plan(w.nside, w.n_los, w.s_max, w.freqs, observer=w.observer, pix_range=pix_range, pix_stride=pix_stride)
    if w.clip_box is not None:
        plan.set_box(w.clip_box)
    for k, v in options.items():
        plan.set_option(k, v)
    sg = {}
    if w.ne_grid is not None:
        sg.update(ne_grid=torch.from_numpy(w.ne_grid).cuda().contiguous(), ne_box=w.ne_box)
    if w.n0_grid is not None:
        sg.update(n0_grid=torch.from_numpy(w.n0_grid).cuda().contiguous(), n0_box=w.n0_box)
    if w.kind == "grid_b":
        model = sx.Model("grid_b", aux=w.aux, grid_shape=w.params.shape[:3], box=w.box, **sg)
    else:
        model = sx.Model(w.kind, aux=w.aux, **sg)
    params = torch.from_numpy(w.params).cuda().contiguous()
    return plan, model, params


def gpu_forward(w: wl.Workload, **options):
    import torch
    import paper_2410_01136_b200 as sx
    plan, model, params = gpu_objects(w, **options)
    I, Q, U = sx.forward(plan, model, params)
    torch.cuda.synchronize()
    out = tuple(t.cpu().numpy().astype(np.float64) for t in (I, Q, U))
    stats = plan.stats()
    plan.close()
    return out, stats


def gpu_vjp(w: wl.Workload, cots, **options):
    import torch
    import paper_2410_01136_b200 as sx
    plan, model, params = gpu_objects(w, **options)
    d = [None if c is None else torch.from_numpy(np.ascontiguousarray(c, dtype=np.float32)).cuda() for c in cots]
    g = sx.vjp(plan, model, params, *d)
    torch.cuda.synchronize()
    out = g.cpu().numpy().astype(np.float64)
    plan.close()
    return out


def map_errors(gpu_maps, ref_maps):
    """max |delta| / RMS(ref) per (Stokes, batch, freq) -> array [3][batch][n_freq]."""
    errs = []
    for g, r in zip(gpu_maps, ref_maps):
        rms = np.sqrt(np.mean(r * r, axis=-1))
        errs.append(np.abs(g - r).max(axis=-1) / rms)
    return np.array(errs)


def assert_maps_close(gpu_maps, ref_maps, tol=MAP_TOL, what=""):
    e = map_errors(gpu_maps, ref_maps)
    assert np.all(np.isfinite(e)), f"{what}: non-finite map"
    assert e.max() <= tol, f"{what}: max|d|/RMS = {e.max():.3e} > {tol:g} (I,Q,U worst: {e.reshape(3, -1).max(1)})"
    return e


def assert_sampled_maps_close(gpu_sub, ref_sub, rms_mask, tol=MAP_TOL, what=""):
    """Full-size runs checked on sampled pixels: the map RMS (C-2#16) is taken over the UNIFORMLY sampled pixels only
    (rms_mask), every sampled pixel -- the extra ill-conditioned in-plane ones included -- is held to tol x that RMS."""
    worst = 0.0
    for g, r in zip(gpu_sub, ref_sub):
        rms = np.sqrt(np.mean(r[..., rms_mask] ** 2, axis=-1, keepdims=True))
        e = np.abs(g - r) / rms
        assert np.all(np.isfinite(e)), f"{what}: non-finite map"
        assert e.max() <= tol, f"{what}: max|d|/RMS = {e.max():.3e} > {tol:g} (per map: {e.max(axis=-1)})"
        worst = max(worst, float(e.max()))
    return worst


def assert_log_gradient_close(g, ref, theta, what="", rel=GRAD_TOL, floor=1.0e-5):
    """Gradient check away from the configs' own parameters (random draws, reading C-2#14b): in log-parameter
    space, |d(g_j theta_j)| <= rel |g_j theta_j| + floor max_k |g_k theta_k|.  The floor is the fp32 round-off of the
    accumulations (~1e-6 .. 1e-5 of the largest terms): a component more than 100x below the largest one is a cancelling
    sum whose RELATIVE error the arithmetic does not bound."""
    lg, lref = np.asarray(g) * theta, np.asarray(ref) * theta
    bound = rel * np.abs(lref) + floor * np.abs(lref).max(axis=-1, keepdims=True)
    assert np.all(np.abs(lg - lref) <= bound), f"{what}: {np.abs(lg - lref) / np.abs(lref)}"
