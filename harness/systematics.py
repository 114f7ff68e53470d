"""Fig. 6 of the paper through the CUDA path (section 4.1), on the section 3.1 model:

  upper panel  std(Map_N - Map_2048) for N_int in {256, 512, 1024}, NSIDE 64;
  lower panel  std(Map_Nx - Map_analytic) for B on (N_x, N_x, N_x / 4) grids filled from the analytic spiral, N_int 512;

plus the timing of the section 3.1 forward + gradient evaluation (the paper: ~100 ms on an A100 in float64, L226).
The paper's n_e is the YMW16 model (not available here): a seeded clumpy disc on the same (256, 256, 64) grid stands in,
so the numbers are this stand-in's, to be read next to the paper's (< 4e-5 K for N_int >= 256; sub-mK at N_x = 64,
~1e-5 K at N_x = 512).

    python -m harness.systematics [--out profiles/r02_systematics.md] [--nx-max 512]
"""
from __future__ import annotations

import argparse
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))


def gpu_maps(w, **options):
    from harness import parity
    maps, _ = parity.gpu_forward(w, **options)
    return [m[0] for m in maps]          # [Stokes][n_freq][npix]


def timed_step(w, reps=10):
    import torch
    import paper_2410_01136_b200 as sx
    from harness import parity
    plan, model, params = parity.gpu_objects(w)
    cots = [torch.from_numpy(c).cuda() for c in w.cotangents()]
    out = sx.forward(plan, model, params)
    grad = sx.vjp(plan, model, params, *cots)
    torch.cuda.synchronize()
    e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    tf = tv = 0.0
    for _ in range(reps):
        e[0].record(); sx.forward(plan, model, params, out=out); e[1].record()
        sx.vjp(plan, model, params, *cots, out=grad); e[2].record()
        torch.cuda.synchronize()
        tf += e[0].elapsed_time(e[1]); tv += e[1].elapsed_time(e[2])
    plan.close()
    return tf / reps, tv / reps


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=str(ROOT / "profiles" / "r02_systematics.md"))
    ap.add_argument("--nx-max", type=int, default=512)
    args = ap.parse_args()
    from harness import workloads as wl
    lines = ["# Round 2 -- Fig. 6 systematics and the section 3.1 workload on the CUDA path", "",
             "Command: `python -m harness.systematics` (one B200).  Model: PAPER.md section 3.1 (WMAP B with the paper's true",
             "values, WMAP N_0, n_e on a (256, 256, 64) grid -- a seeded clumpy disc standing in for YMW16 --, NSIDE 64, 2.4 GHz,",
             "integration to the faces of the (40, 40, 10) kpc box).  std over the 49,152 pixels, Kelvin.", ""]
    base = wl.paper_section31()
    tf, tv = timed_step(base)
    lines += [f"Section 3.1 evaluation (NSIDE 64, N_int 512, 2.52e7 samples): forward {tf:.3f} ms + gradient (VJP) {tv:.3f} ms = "
              f"{tf + tv:.3f} ms per likelihood-gradient evaluation, fp32 device arithmetic with the float64 Faraday chain where needed "
              "(the paper: ~100 ms per evaluation on an A100 in float64, PAPER.md L226).", ""]
    # upper panel
    ref = gpu_maps(wl.paper_section31(n_los=2048))
    lines += ["## N_int (Fig. 6 upper; paper: < 4e-5 K for N_int >= 256)", "", "| N_int | std(I - I_2048) | std(Q - Q_2048) | std(U - U_2048) |", "|---|---|---|---|"]
    for n in (256, 512, 1024):
        m = gpu_maps(wl.paper_section31(n_los=n))
        lines.append(f"| {n} | " + " | ".join(f"{np.std(a[0] - b[0]):.2e}" for a, b in zip(m, ref)) + " |")
    # lower panel
    ana = gpu_maps(base)
    lines += ["", "## Grid size (Fig. 6 lower; paper: sub-mK at N_x = 64, ~1e-5 K at N_x = 512)", "",
              "| N_x | grid | std(I - I_ana) | std(Q - Q_ana) | std(U - U_ana) | forward ms |", "|---|---|---|---|---|---|"]
    for nx in (64, 128, 256, 512):
        if nx > args.nx_max:
            continue
        wg = wl.section31_gridded_b(nx, base)
        t0 = time.perf_counter()
        m = gpu_maps(wg)
        tfg, _ = timed_step(wg, reps=3)
        lines.append(f"| {nx} | {nx} x {nx} x {nx // 4} | " + " | ".join(f"{np.std(a[0] - b[0]):.2e}" for a, b in zip(m, ana)) + f" | {tfg:.3f} |")
        print(f"N_x = {nx}: done in {time.perf_counter() - t0:.1f} s", flush=True)
    lines += ["", f"Map scale for reference: std(I) = {np.std(ana[0][0]):.3e} K, std(Q) = {np.std(ana[1][0]):.3e} K, std(U) = {np.std(ana[2][0]):.3e} K.", ""]
    Path(args.out).write_text("\n".join(lines))
    print("\n".join(lines))


if __name__ == "__main__":
    main()
