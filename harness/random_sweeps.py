"""Seeded random sweeps of the CUDA path against the oracle, beyond the BASELINE configs.

    python -m harness.random_sweeps mid     7000 7840   # 12 k ... 390 k sightlines, cotangents on ~400 pixels
    python -m harness.random_sweeps grid    8000 8150   # GRID_B: non-cubic grids, arbitrary boxes
    python -m harness.random_sweeps options 9000 9700   # small maps, every option, 1 ... 600 samples, 1-32 frequencies

One line per draw ("ok" / "FAIL" with the worst map error in units of the map RMS and the gradient verdicts), the count of
failures at the end.  Bounds as in tests/: maps 1e-4 x RMS, gradients 1e-3 in log-parameter space (reading C-2#14b), grid
gradients 1e-3 |g| + 1e-4 RMS(g) (C-2#14).  Every draw checks the forward, the adjoint with nothing stored by the plan and
the adjoint after the forward.  A few of the draws are kept as tests/test_gpu_fuzz.py; the outcomes of the full ranges are
recorded in profiles/r02_random_sweeps.md.  Test infrastructure (it runs the oracle), not product code.
"""
from __future__ import annotations

import sys

import numpy as np

from harness import parity
from harness import workloads as wl


def _sparse(w, seed, n_pix=400):
    step = max(7, w.npix // n_pix) | 1
    pix = np.arange(seed % step, w.npix, step)
    full = w.cotangents()
    cots = tuple(np.zeros_like(c) for c in full)
    for c, f in zip(cots, full):
        c[..., pix] = f[..., pix]
    return pix, cots


def _run_analytic(w, opts, pix, cots_h):
    """(map error / RMS on `pix`, verdicts of the two adjoint routes, escalated sightlines)."""
    import torch
    import paper_2410_01136_b200 as sx
    plan, model, params = parity.gpu_objects(w, **opts)
    d = [torch.from_numpy(c).cuda() for c in cots_h]
    sub = tuple(np.ascontiguousarray(c[..., pix]) for c in cots_h)
    ref = parity.oracle_vjp(w, sub, pix=pix)
    refm = parity.oracle_forward(w, pix=pix)
    th = w.params.astype(np.float64)
    g_alone = sx.vjp(plan, model, params, *d).cpu().numpy().astype(np.float64)
    maps = tuple(t.cpu().numpy().astype(np.float64)[..., pix] for t in sx.forward(plan, model, params))
    g_after = sx.vjp(plan, model, params, *d).cpu().numpy().astype(np.float64)
    torch.cuda.synchronize()
    esc = plan.stats()["escalated"]
    plan.close()
    e = parity.map_errors(maps, refm)
    verdicts = []
    for g in (g_alone, g_after):
        try:
            parity.assert_log_gradient_close(g, ref, th)
            verdicts.append(bool(np.isfinite(g).all()))
        except AssertionError:
            verdicts.append(False)
    return float(e.max()) if np.isfinite(e).all() else float("inf"), verdicts, esc


def sweep_mid(seed):
    w = wl.random_mid(seed)
    pix, cots = _sparse(w, seed)
    e, v, esc = _run_analytic(w, {}, pix, cots)
    ok = e <= parity.MAP_TOL and all(v)
    return ok, (f"{w.name} nside {w.nside} batch {w.batch} n_los {w.n_los} n_freq {w.n_freq} f_min {w.freqs[0] / 1e9:.2f} GHz "
                f"box {w.clip_box is not None} escalated {esc}/{w.npix * w.batch}: map {e:.2e}, adjoint alone / after {v}")


def sweep_options(seed):
    w, opts = wl.random_options(seed)
    e, v, esc = _run_analytic(w, opts, np.arange(w.npix), w.cotangents())
    ok = e <= parity.MAP_TOL and all(v)
    return ok, (f"{w.name} nside {w.nside} batch {w.batch} n_los {w.n_los} n_freq {w.n_freq} f_min {w.freqs[0] / 1e9:.2f} GHz "
                f"box {w.clip_box is not None} n_e grid {w.ne_grid is not None} N_0 grid {w.n0_grid is not None} {opts}: "
                f"map {e:.2e}, adjoint alone / after {v}")


def sweep_grid(seed):
    w = wl.random_grid(seed)
    maps, _ = parity.gpu_forward(w)
    e = parity.map_errors(maps, parity.oracle_forward(w))
    cots = w.cotangents()
    g, ref = parity.gpu_vjp(w, cots), parity.oracle_vjp(w, cots)
    rms = np.sqrt(np.mean(ref * ref))
    bad = int((np.abs(g - ref) > parity.GRAD_TOL * np.abs(ref) + 1.0e-4 * rms).sum())
    zeros = bool(np.array_equal(ref == 0.0, g == 0.0))
    ok = bool(np.isfinite(e).all()) and e.max() <= parity.MAP_TOL and bad == 0 and zeros
    return ok, (f"{w.name} grid {w.params.shape[:3]} box {tuple(round(v, 3) for v in w.box)} nside {w.nside} n_los {w.n_los} "
                f"n_freq {w.n_freq} f_min {w.freqs[0] / 1e9:.2f} GHz clip {w.clip_box is not None}: map {e.max():.2e}, "
                f"grid-gradient components out of tolerance {bad}, worst {np.abs(g - ref).max() / rms:.2e} RMS, untouched cells equal {zeros}")


SWEEPS = {"mid": sweep_mid, "grid": sweep_grid, "options": sweep_options}


def main(argv):
    if len(argv) != 3 or argv[0] not in SWEEPS:
        raise SystemExit(__doc__)
    fn, bad = SWEEPS[argv[0]], 0
    for seed in range(int(argv[1]), int(argv[2])):
        ok, line = fn(seed)
        bad += not ok
        print("ok  " if ok else "FAIL", line, flush=True)
    print(f"{int(argv[2]) - int(argv[1])} draws, {bad} outside the bounds")
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:]))
