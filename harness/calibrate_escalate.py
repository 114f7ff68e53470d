"""Calibration of the forward's escalation threshold `escalate_rad`: map error against the oracle
and share of sightlines on the float64 Faraday chain as a function of the threshold, on 786,432-sightline calls (nside
256: the regime where the fp32 chain and the float64 chain each take their own list of sightlines), for the cfg-4 model
at two sample counts, three rescalings of n_e and B, and the cfg-1 disc at 408 MHz.  The oracle is evaluated on every
16th pixel (49,152 sightlines per workload).

    python -m harness.calibrate_escalate [--out profiles/r02_escalate_calibration.md]
"""
from __future__ import annotations

import argparse
import dataclasses
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

THRESHOLDS = (100.0, 200.0, 300.0, 500.0, 1000.0, 3000.0)


def workloads():
    from harness import workloads as wl
    c4 = wl.config(4)
    out = [("cfg 4 (1024 samples)", c4), ("cfg 4, 256 samples", dataclasses.replace(c4, n_los=256))]
    for name, fne, fb in (("cfg 4, n_e x 2", 2.0, 1.0), ("cfg 4, n_e x 0.5, B x 1.5", 0.5, 1.5), ("cfg 4, n_e x 4, B x 0.7", 4.0, 0.7)):
        p = c4.params.copy(); p[0, 13] *= fne; p[0, 0] *= fb; p[0, 5] *= fb
        out.append((name, dataclasses.replace(c4, params=p)))
    c1 = wl.config(1)
    out.append(("cfg-1 disc, 408 MHz + 1.4 GHz, 512 samples", dataclasses.replace(c1, nside=256, n_los=512, freqs=np.array([0.408e9, 1.4e9]))))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=str(ROOT / "profiles" / "r02_escalate_calibration.md"))
    args = ap.parse_args()
    from harness import parity
    lines = ["# Round 2 -- calibration of `escalate_rad` (forward, precision 0)", "",
             "Command: `python -m harness.calibrate_escalate` (one B200).  nside 256 (786,432 sightlines per call); the oracle on",
             "every 16th pixel.  Entry = max over the Q and U maps of all frequencies of max|GPU - oracle| / RMS(oracle map) over",
             "the sampled pixels (bound: 1e-4), and the share of sightlines on the float64 Faraday chain.", "",
             "| workload | fp32 only | " + " | ".join(f"{t:g} rad" for t in THRESHOLDS) + " | float64 chain everywhere |", "|---|---|" + "---|" * (len(THRESHOLDS) + 1)]
    worst = {t: 0.0 for t in THRESHOLDS}
    for name, w in workloads():
        pix = np.arange(0, w.npix, 16)
        ref = parity.oracle_forward(w, pix=pix)

        def err(**opt):
            maps, stats = parity.gpu_forward(w, **opt)
            e = parity.map_errors(tuple(m[..., pix] for m in maps), ref)
            return float(e[1:].max()), stats["escalated"] / (w.npix * w.batch)

        row = [f"{err(precision=1)[0]:.1e}"]
        for t in THRESHOLDS:
            e, share = err(escalate_rad=t)
            worst[t] = max(worst[t], e)
            row.append(f"{e:.1e} ({100 * share:.0f} %)")
        row.append(f"{err(precision=2)[0]:.1e}")
        lines.append(f"| {name} | " + " | ".join(row) + " |")
        print(lines[-1], flush=True)
    lines += ["", "Worst case per threshold: " + ", ".join(f"{t:g} rad: {worst[t]:.1e}" for t in THRESHOLDS) + ".", ""]
    Path(args.out).write_text("\n".join(lines))


if __name__ == "__main__":
    main()
