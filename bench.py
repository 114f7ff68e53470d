#!/usr/bin/env python
"""bench.py -- throughput of the synax hot path (forward + VJP) on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: synax_forward followed by
synax_vjp on the same stream (BASELINE.json metric "LoS samples/s (fwd,
fwd+VJP) at nside=256 x 1024 pts").  Default workload = BASELINE.json configs[4] (nside=256, 1024 samples,
8 frequencies, 16-parameter model).  LoS samples = npix * n_los * batch per call (frequencies not
multiplied in).  `value` = samples / (forward + VJP time), inputs resident in HBM.  `e2e` = the same
through synax_forward_host / synax_vjp_host with pinned HOST buffers (copies inside the timed region).

N > 1 (torchrun, one rank per GPU): the partition of SURVEY.md 8(e) -- RING pixel shards of ONE map (interleaved: rank r takes
pixels r, r + N, ..., so that every rank sees every latitude and the ranks take equally long), no exchange in the forward, one sum all-reduce of the gradient per VJP ("scaling": "strong": the map is fixed).
--scaling weak runs independent parameter vectors (HMC chains) per rank instead, with no data-path collective
(DESIGN.md section 9).

--impl reference: the float64 CPU oracle (oracle/), as it stands, on the host cores, on a bounded pixel
subset of the same workload; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "LoS samples/s (fwd+VJP)"
UNIT = "samples/s"

# Algorithmic FP32 lane-instructions per LoS sample (DESIGN.md section 7 / SURVEY.md 8(d) table), fixed
# before tuning: shared part + per-frequency part, forward and VJP (VJP = recompute + adjoint).
ALG_FP = {
    "disc4":  dict(fwd=(70, 12), vjp=(70 + 90, 12 + 14)),
    "full16": dict(fwd=(85, 12), vjp=(85 + 125, 12 + 14)),
    "grid_b": dict(fwd=(120, 12), vjp=(120 + 60, 12 + 14)),
    "uniform": dict(fwd=(30, 12), vjp=(60, 26)),
}
ALG_MUFU = {"disc4": (14, 2), "full16": (19, 2), "grid_b": (10, 2), "uniform": (0, 2), "stack16": (24, 2)}
ALG_FP["stack16"] = dict(fwd=(110, 12), vjp=(110 + 150, 12 + 14))
SM_COUNT, FP32_LANES, MUFU_LANES = 148, 128, 16


def alg_mufu(kind, n_freq, which):
    s, f = ALG_MUFU[kind]
    return s + f * n_freq + (2 if which == "vjp" else 0)     # the adjoint re-evaluates the forward's MUFU work + 2


def bound_seconds(kind, n_freq, samples, sm_mhz, legs=("fwd", "vjp")):
    """cycles per sample = max(FP32 / 128, MUFU / 16) per SM, summed over the legs as ONE instruction mix."""
    fp = sum(alg_fp(kind, n_freq, leg) for leg in legs)
    mu = sum(alg_mufu(kind, n_freq, leg) for leg in legs)
    return max(fp / FP32_LANES, mu / MUFU_LANES) * samples / (SM_COUNT * sm_mhz * 1e6)


def alg_fp(kind, n_freq, which):
    s, f = ALG_FP[kind][which]
    return s + f * n_freq


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d.get("sm_max_mhz", 1965.0)), "MEASURED_PEAKS.json sm_max_mhz"
    return 1965.0, "fallback 1965 MHz (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi -lms sampling of SM clock and throttle reasons during the timed region."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, reasons, mx, pw = [], set(), None, []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        try:
            for line in Path(self.path).read_text().splitlines():
                c = [x.strip() for x in line.split(",")]
                if len(c) < 7:
                    continue
                try:
                    sm.append(float(c[0])); mx = float(c[1]); pw.append(float(c[2]))
                except ValueError:
                    continue
                for n, v in zip(names, c[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=mx, reasons=sorted(reasons), samples=len(sm),
                       sm_mhz_min=float(min(sm)), power_w_max=float(max(pw)) if pw else None)
        return out


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def rank_workload(cfg, rank):
    """Weak scaling: rank r > 0 takes the config's model with its own parameter vector(s) (an independent
    chain): each analytic parameter scaled by (1 + 0.05 u), u ~ U[-1,1] from seed 7000 + r.  Rank 0 is the
    config as BASELINE.json states it."""
    from harness import workloads as wl
    w = wl.config(cfg)
    if rank > 0 and w.kind != "grid_b":
        rng = np.random.Generator(np.random.PCG64(7000 + rank))
        w.params = np.ascontiguousarray((w.params.astype(np.float64) * (1.0 + 0.05 * rng.uniform(-1, 1, w.params.shape))).astype(np.float32))
    elif rank > 0:
        rng = np.random.Generator(np.random.PCG64(7000 + rank))
        w.params = np.ascontiguousarray((w.params.astype(np.float64) * (1.0 + 0.05 * rng.uniform(-1, 1))).astype(np.float32))
    return w


def apply_overrides(w, args):
    """--nside / --n-los / --freq-hz: the config's model at another map size, sample count or at one frequency
    (the Fig. 7-style runtime sweep of PAPER.md L260, L277); the workload name says so."""
    if args.nside or args.n_los:
        w = w.scaled(nside=args.nside or None, n_los=args.n_los or None)
    if args.freq_hz:
        w.freqs = np.array([float(args.freq_hz)])
        w.name += f"@{args.freq_hz:g}Hz"
    return w


# ------------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline of the default run, and --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_sample_pixels(w, target_samples):
    """Bounded sample of the workload: pixels p = 0 (mod stride), stride chosen so that the sample holds about
    `target_samples` LoS samples (all batch elements, all frequencies, all n_los points of those pixels)."""
    per_pix = w.n_los * w.batch
    want = max(1, int(target_samples // per_pix))
    stride = max(1, w.npix // want)
    return np.arange(0, w.npix, stride, dtype=np.int64), stride


def oracle_step(w, pix, cots_sub):
    """One forward + VJP of the oracle over the pixel subset; returns seconds."""
    from harness import parity
    t = time.perf_counter()
    parity.oracle_forward(w, pix=pix)
    t1 = time.perf_counter()
    parity.oracle_vjp(w, cots_sub, pix=pix)
    t2 = time.perf_counter()
    return t1 - t, t2 - t1


def oracle_baseline(w, seconds_budget=15.0, steps=1, warmup=0, threads=None):
    import oracle
    oracle.build()
    all_cores = oracle.num_threads()
    if threads is not None:
        oracle.set_num_threads(threads)
    try:
        return _oracle_baseline(w, seconds_budget, steps, warmup, oracle.num_threads())
    finally:
        oracle.set_num_threads(all_cores)


def _oracle_baseline(w, seconds_budget, steps, warmup, cores):
    # ~7 us per sample per core for FULL16 at 8 frequencies forward+VJP (measured on the build box): size the
    # sample so one step is about `seconds_budget` of wall time on this host
    per_sample_core = 1.2e-6 * (1.0 + 0.6 * w.n_freq)
    target = seconds_budget * cores / per_sample_core
    pix, stride = oracle_sample_pixels(w, min(target, w.los_samples))
    cots = w.cotangents()
    cots_sub = tuple(np.ascontiguousarray(c[..., pix]) for c in cots)
    n_samples = pix.size * w.n_los * w.batch
    for _ in range(warmup):
        oracle_step(w, pix, cots_sub)
    tf = tv = 0.0
    for _ in range(steps):
        a, b = oracle_step(w, pix, cots_sub)
        tf += a; tv += b
    tf /= steps; tv /= steps
    return dict(value=n_samples / (tf + tv), unit=UNIT, cores=int(cores), kind="oracle",
                sample=f"pixels p = 0 (mod {stride}) of {w.name}: {pix.size} sightlines x {w.n_los} samples x batch {w.batch} "
                       f"= {n_samples} LoS samples per step, forward + VJP, float64, OpenMP over sightlines",
                forward_samples_per_s=n_samples / tf, ms_per_step=1e3 * (tf + tv), samples_per_step=int(n_samples))


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    from harness import workloads as wl
    w = apply_overrides(wl.config(args.config), args)
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    # keep the whole run within a few minutes: total oracle time ~ 120 s split over steps + warm-ups
    budget = min(15.0, 120.0 / (steps + warmup))
    # torchrun exports OMP_NUM_THREADS=1 to its workers when the variable is unset; rank 0 is the only one that works here,
    # so it takes the cores the process may run on, as a stand-alone `python bench.py --impl reference` does
    threads = len(os.sched_getaffinity(0)) if world > 1 else None
    cb = oracle_baseline(w, seconds_budget=budget, steps=steps, warmup=warmup, threads=threads)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": world, "steps": steps,
            "warmup": warmup, "ms_per_step": cb["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded, workloads.py)",
            "config": {"workload": w.name, "nside": w.nside, "n_los": w.n_los, "n_freq": w.n_freq, "batch": w.batch,
                       "model": w.kind, "sample": cb["sample"]},
            "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "forward_samples_per_s": cb["forward_samples_per_s"]}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def time_config(sx, torch, w, steps, warmup, flush_buf, want_e2e=True, pix_range=None, pix_stride=1, reduce_grad=False, graph=False, lanes=0, f64=False):
    """Device-resident timing of forward and VJP with CUDA events on the launching stream, L2 flushed between
    timed calls; then (optionally) the host-buffer entry points.  pix_range: this rank's pixel shard (strong
    scaling), with the one gradient all-reduce of the method inside the timed VJP when reduce_grad is set."""
    from paper_2410_01136_b200 import sharding
    plan = sx.Plan(w.nside, w.n_los, w.s_max, w.freqs, observer=w.observer, pix_range=pix_range, pix_stride=pix_stride)
    if want_e2e:   # the *_host calls stage hundreds of MB per call in the stream-ordered pool: keep it mapped (opt-in)
        plan.set_option("pool_release_threshold_mb", 4096)
    if lanes:
        plan.set_option("lanes", lanes)
    npix = plan.npix
    p0 = 0 if pix_range is None else pix_range[0]
    if w.kind == "grid_b":
        model = sx.Model("grid_b", aux=w.aux, grid_shape=w.params.shape[:3], box=w.box)
    else:
        model = sx.Model(w.kind, aux=w.aux)
    params = torch.from_numpy(w.params).cuda().contiguous()
    cots_h = tuple(np.ascontiguousarray(c[..., p0:p0 + npix * pix_stride:pix_stride]) for c in w.cotangents())
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    out = tuple(torch.empty((w.batch, w.n_freq, npix), dtype=torch.float32, device="cuda") for _ in range(3))
    grad = torch.empty_like(params)
    stream = torch.cuda.current_stream()

    def step(ev=None):
        if ev: ev[0].record(stream)
        sx.forward(plan, model, params, out=out)
        if ev: ev[1].record(stream)
        sx.vjp(plan, model, params, *cots, out=grad)
        if reduce_grad: sharding.reduce_gradient(grad)
        if ev: ev[2].record(stream)

    for _ in range(warmup):
        step()
        flush_buf.add_(1.0)
    torch.cuda.synchronize()
    l0 = plan.stats()["launches"]
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    for k in range(steps):
        step(evs[k])
        flush_buf.add_(1.0)          # > L2 (126 MB): every timed step starts with a cold L2
    torch.cuda.synchronize()
    l1 = plan.stats()["launches"]
    tf = np.array([e[0].elapsed_time(e[1]) for e in evs]) * 1e-3
    tv = np.array([e[1].elapsed_time(e[2]) for e in evs]) * 1e-3
    stat = lambda a: {"mean": float(1e3 * a.mean()), "median": float(1e3 * np.median(a)), "best": float(1e3 * a.min())}  # noqa: E731
    res = dict(t_fwd=float(tf.mean()), t_vjp=float(tv.mean()), t_fwd_min=float(tf.min()), t_vjp_min=float(tv.min()),
               launches=int(l1 - l0), escalated=plan.stats()["escalated"],
               timing={"forward_ms": stat(tf), "vjp_ms": stat(tv), "step_ms": stat(tf + tv)})
    if not reduce_grad:
        # The adjoint of a step reuses what the step's own forward stored (Faraday totals, tile bases).  For the record, the same
        # adjoint on its own: the stored values are dropped before every call (setting the option does that), so each call
        # runs its Faraday-only pass first (long multi-frequency calls), the forward-order kernel (one frequency), or its
        # in-kernel pre-pass (small calls).  A few calls, no synchronisation between them.
        ea = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(1 + min(steps, 5))]
        for e in ea:
            plan.set_option("use_forward_totals", 1)
            e[0].record(stream); sx.vjp(plan, model, params, *cots, out=grad); e[1].record(stream)
            flush_buf.add_(1.0)
        torch.cuda.synchronize()
        ts = [e[0].elapsed_time(e[1]) for e in ea[1:]]
        res["timing"]["vjp_standalone_ms"] = {"mean": float(np.mean(ts)), "median": float(np.median(ts)), "best": float(np.min(ts))}
    if f64 and w.kind != "grid_b" and not reduce_grad:
        # the paper's own arithmetic (float64 throughout): synax_forward_f64 / synax_vjp_f64 on float64 buffers
        p64 = params.double()
        c64 = [c.double() for c in cots]
        o64 = tuple(torch.empty((w.batch, w.n_freq, npix), dtype=torch.float64, device="cuda") for _ in range(3))
        g64 = torch.empty_like(p64)
        n64 = 1 + min(steps, 5)
        e64 = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(n64)]
        for e in e64:
            e[0].record(stream); sx.forward_f64(plan, model, p64, out=o64)
            e[1].record(stream); sx.vjp_f64(plan, model, p64, *c64, out=g64)
            e[2].record(stream)
            flush_buf.add_(1.0)
        torch.cuda.synchronize()
        tf64 = np.array([e[0].elapsed_time(e[1]) for e in e64[1:]]); tv64 = np.array([e[1].elapsed_time(e[2]) for e in e64[1:]])
        res["float64_mode"] = {"forward_ms": float(np.median(tf64)), "vjp_ms": float(np.median(tv64)),
                               "note": "synax_forward_f64 / synax_vjp_f64: every step in float64 (the paper's default precision), "
                                       "float64 buffers; medians of %d calls, L2 flushed between" % (n64 - 1)}
        del p64, c64, o64, g64
    if graph and not reduce_grad:
        # the whole step captured once in a CUDA graph and replayed (pays off when a step is launch-bound: cfg 0, 1)
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            step()
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            step()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            g.replay()
        e1.record(stream)
        torch.cuda.synchronize()
        res["t_graph"] = e0.elapsed_time(e1) * 1e-3 / steps
    if want_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()  # noqa: E731
        hp = pin(w.params); hc = [pin(c) for c in cots_h]
        ho = tuple(torch.empty((w.batch, w.n_freq, npix), dtype=torch.float32).pin_memory() for _ in range(3))
        hg = torch.empty(w.params.shape, dtype=torch.float32).pin_memory()
        npv = lambda t: t.numpy()  # noqa: E731

        def host_step():
            sx.forward_host(plan, model, npv(hp), out=tuple(npv(t) for t in ho))
            sx.vjp_host(plan, model, npv(hp), *[npv(c) for c in hc], out=npv(hg))
            if reduce_grad:
                gd = hg.cuda(non_blocking=True)
                sharding.reduce_gradient(gd)
                hg.copy_(gd)

        n_e2e = max(3, min(steps, 10))
        for _ in range(2):
            host_step()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            host_step()            # each *_host call synchronises its stream before returning
        torch.cuda.synchronize()
        res["t_e2e"] = (time.perf_counter() - t0) / n_e2e
        res["h2d"] = int(2 * hp.numel() * 4 + sum(c.numel() for c in hc) * 4)
        res["d2h"] = int(sum(t.numel() for t in ho) * 4 + hg.numel() * 4)
        if not reduce_grad:
            # The paper's inner loop (HMC / ADAM step) through the fused call: the observed Q/U maps
            # stay resident, per step only the parameters go up and (logL, gradient) come back.
            obs_q = (out[1][0] + 1.0e-3 * torch.randn_like(out[1][0])).contiguous()
            obs_u = (out[2][0] + 1.0e-3 * torch.randn_like(out[2][0])).contiguous()
            ll = torch.empty((w.batch,), dtype=torch.float64, device="cuda")
            hll = torch.empty((w.batch,), dtype=torch.float64).pin_memory()

            def fused_step():
                params.copy_(hp, non_blocking=True)
                sx.loglike_vjp(plan, model, params, None, obs_q, obs_u, (0.0, 1.0e6, 1.0e6), out=(ll, grad))
                hll.copy_(ll, non_blocking=True)
                hg.copy_(grad, non_blocking=True)
                torch.cuda.current_stream().synchronize()

            for _ in range(2):
                fused_step()
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                fused_step()
            res["t_fused"] = (time.perf_counter() - t0) / n_e2e
            res["fused_h2d"] = int(hp.numel() * 4)
            res["fused_d2h"] = int(hll.numel() * 8 + hg.numel() * 4)
    plan.close()
    return res


def wl_config(i):
    from harness import workloads as wl
    return wl.config(i)


def committed_csv(name):
    """profiles/<name>: rows of a committed ncu summary as dicts (first line = header), or []."""
    f = ROOT / "profiles" / name
    if not f.exists():
        return []
    import csv
    rows = list(csv.reader(ln for ln in f.read_text().splitlines() if ln.strip() and not ln.startswith("#")))
    return [dict(zip(rows[0], r)) for r in rows[1:]]


def alu_roofline(w, r, local_samples, peak, sm_max, peak_src, strong, clocks):
    """Analytic path: bound by plain ALU issue.  Dominant kernel = the adjoint."""
    fp_vjp, fp_fwd = alg_fp(w.kind, w.n_freq, "vjp"), alg_fp(w.kind, w.n_freq, "fwd")
    achieved = fp_vjp * local_samples / r["t_vjp"] / 1e12
    t_bound = bound_seconds(w.kind, w.n_freq, local_samples, sm_max)
    traffic, ncu = None, None
    if w.name.startswith("cfg4") and not strong:
        for row in committed_csv("r02_cfg4_dram_traffic.csv"):
            if row.get("kernel") == "vjp_kernel":
                traffic = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
        rows = committed_csv("r02_cfg4_pipes.csv")
        if rows:   # ncu --set full capture of the committed build (profiles/r02_cfg4_ncu_full.md): % of peak, sustained active
            ncu = {"source": "profiles/r02_cfg4_ncu_full.md (ncu --set full of the committed build; % of peak, sustained active)",
                   "kernels": {row["kernel"]: {k: float(v) for k, v in row.items() if k != "kernel"} for row in rows}}
    out = {"bound": "alu",
           "kernel": ("vjp_kernel (analytic adjoint; long calls: vjp_classify_kernel + the fp32-angle / float64-angle pair of vjp_kernel "
                      "launches on two streams, timed as one call)"),
           "achieved": achieved, "peak": peak, "unit": "T fp32 lane-instr/s", "frac": achieved / peak, "traffic": traffic,
           "peak_source": f"148 SM x 128 FP32 lanes x {sm_max:.0f} MHz ({peak_src})",
           "alg_fp32_per_sample": fp_vjp, "alg_mufu_per_sample": alg_mufu(w.kind, w.n_freq, "vjp"),
           "forward": {"alg_fp32_per_sample": fp_fwd, "alg_mufu_per_sample": alg_mufu(w.kind, w.n_freq, "fwd"),
                       "achieved": fp_fwd * local_samples / r["t_fwd"] / 1e12,
                       "frac": fp_fwd * local_samples / r["t_fwd"] / 1e12 / peak,
                       "xu_bound_frac": bound_seconds(w.kind, w.n_freq, local_samples, sm_max, legs=("fwd",)) / r["t_fwd"]},
           # the whole step against SURVEY.md 8(d)'s FP32/SFU bound for forward + VJP (north_star's >= 0.50 bar)
           "step_bound_ms": 1e3 * t_bound, "step_frac": t_bound / (r["t_fwd"] + r["t_vjp"]),
           "ncu": ncu}
    if clocks and clocks.get("sm_mhz"):
        out["frac_at_sustained_clock"] = achieved / (peak * clocks["sm_mhz"] / sm_max)
    return out


def grid_roofline(w, r, local_samples):
    """Gridded path: bound by L1/L2 gathers (forward) and L2 vector reductions (adjoint); the ceilings are measured live
    by the two microbenchmarks of SURVEY.md 8(d) on cfg 3's actual index stream (paper_2410_01136_b200/ubench)."""
    try:
        from paper_2410_01136_b200.ubench.__main__ import run as ubench_run
        txt = ubench_run("grid_streams")
        m = json.loads([ln for ln in txt.splitlines() if ln.startswith("JSON ")][-1][5:])
    except Exception as ex:   # no nvcc on the box: say so rather than guess
        return {"bound": "red", "kernel": "grid_vjp_kernel", "achieved": None, "peak": None, "frac": None, "traffic": None,
                "note": f"microbenchmarks unavailable: {ex}"}
    scale = local_samples / m["samples"]      # the microbenchmarks run cfg 3's geometry (49,152 x 512 samples)
    reds = m["red_v4_count"] * scale
    # the adjoint takes the sightlines in a permuted group order (grid_vjp_kernel); the ceiling is the faster of the two orders
    r_ms = min(m["red_v4_ms"], m.get("red_v4_group_order_ms", m["red_v4_ms"]))
    return {"bound": "red", "kernel": "grid_vjp_kernel (two sweeps; per-cell register aggregation with the crossed face's 4 corners "
                                      "carried into the next cell, red.global.v4.f32.add)",
            "achieved": reds / r["t_vjp"], "peak": m["red_v4_count"] / (r_ms * 1e-3), "unit": "red.v4/s",
            "frac": (r_ms * 1e-3 * scale) / r["t_vjp"], "traffic": None,
            "frac_vs_pixel_order_stream": (m["red_v4_ms"] * 1e-3 * scale) / r["t_vjp"],
            "peak_source": "ubench grid_streams (R): red.global.v4.f32.add on the kernel's index stream, per-cell aggregated, measured in this "
                           "run with the sightlines in the adjoint's own (permuted group) order and in pixel order; the faster of the two",
            "alg_red_v4_per_call": reds,
            "note": "achieved / peak count the reference stream of SURVEY.md 8(d): 8 vector reds per cell a lane leaves. The kernel "
                    "itself issues fewer (4 per face crossing + 8 per chunk end; 1.70e7 against 2.35e7 at cfg 3, ncu "
                    "lts__t_requests_srcunit_tex_op_red in profiles/r02_cfg3_grid.md); frac = time of the reference stream / time of the call",
            "forward": {"bound": "l2-gather", "kernel": "grid_forward_kernel",
                        "achieved": m["gather_bytes"] * scale / r["t_fwd"] / 1e9, "peak": m["gather_bytes"] / (m["gather_ms"] * 1e-3) / 1e9,
                        "unit": "GB/s requested (96 B per in-box sample)", "frac": (m["gather_ms"] * 1e-3 * scale) / r["t_fwd"],
                        "peak_source": "ubench grid_streams (G): 8-corner x 3 gather on the kernel's index stream, measured in this run",
                        "frac_vs_padded_gather": (m["gather_v4_ms"] * 1e-3 * scale) / r["t_fwd"]},
            "ceilings_ms": {k: m[k] for k in ("gather_ms", "gather_v4_ms", "red_v4_ms", "red_v4_group_order_ms") if k in m}}


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the synax hot path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank % torch.cuda.device_count())
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", torch.cuda.current_device()))
    import paper_2410_01136_b200 as sx
    sx.load_library()                       # fails loudly when libsynax.so is missing
    strong = args.scaling == "strong" and world > 1
    pix_range, pix_stride = None, 1
    if strong:      # one map, pixel shards, one gradient all-reduce per step
        from paper_2410_01136_b200 import sharding
        from harness import workloads as wl
        w = apply_overrides(wl.config(args.config), args)
        # interleaved shards (rank r: pixels r, r + N, ...): every rank sees every latitude, so the ranks take equally long
        begin, pix_stride, count = sharding.strided_shard_of(w.npix, rank, world)
        pix_range = (begin, count)
    else:           # independent chains: every rank integrates the whole sky for its own parameter vector
        w = apply_overrides(rank_workload(args.config, rank), args)
    kw = dict(pix_range=pix_range, pix_stride=pix_stride, reduce_grad=strong, lanes=args.lanes)
    flush_buf = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device="cuda")   # 256 MB > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # untimed first touch (context, module load)
    time_config(sx, torch, w, 1, 1, flush_buf, want_e2e=False, **kw)
    barrier()
    sampler = ClockSampler(torch.cuda.current_device())
    if rank == 0:
        sampler.start()
    barrier()
    r = time_config(sx, torch, w, args.steps, args.warmup, flush_buf, want_e2e=False, graph=args.graph, f64=args.f64, **kw)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    e = time_config(sx, torch, w, min(args.steps, 5), 1, flush_buf, want_e2e=True, **kw)
    t_step = r["t_fwd"] + r["t_vjp"]
    vals = torch.tensor([t_step, r["t_fwd"], r["t_vjp"], e["t_e2e"]], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(vals, op=dist.ReduceOp.MAX)
    t_step, t_fwd, t_vjp, t_e2e = (float(v) for v in vals.cpu())
    samples = w.los_samples                 # per rank (weak) or of the whole map (strong)
    local_samples = samples if not strong else pix_range[1] * w.n_los * w.batch
    total = samples if strong else world * samples
    line = None
    if rank == 0:
        sm_max, peak_src = peaks()
        peak = SM_COUNT * FP32_LANES * sm_max * 1e6 / 1e12       # T lane-instr/s
        line = {
            "metric": METRIC, "value": total / t_step, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_step, "higher_is_better": True, "scaling": "strong" if strong else "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic (seeded, harness/workloads.py)",
            "config": {"workload": w.name, "nside": w.nside, "n_los": w.n_los, "n_freq": w.n_freq, "batch": w.batch,
                       "model": w.kind, "samples_per_step": samples, "l2": "flushed between timed steps (256 MB write)",
                       "parallelism": ("single GPU" if world == 1 else f"interleaved pixel shards x{world} + gradient all-reduce" if strong
                                       else f"independent parameter vectors x{world}")},
            "forward_samples_per_s": total / t_fwd, "vjp_samples_per_s": total / t_vjp,
            "ms_forward": 1e3 * t_fwd, "ms_vjp": 1e3 * t_vjp,
            "timing": r["timing"],          # per timed step on this rank: mean / median / best, ms; vjp_standalone_ms = the
                                            # adjoint on its own (nothing stored by a forward: Faraday-only pass or pre-pass first)
            "sample_freq_per_s": total * w.n_freq / t_step,
            "e2e": {"value": total / t_e2e, "unit": UNIT, "h2d_bytes_per_step": e["h2d"], "d2h_bytes_per_step": e["d2h"],
                    "ms_per_step": 1e3 * t_e2e,
                    "note": "synax_forward_host + synax_vjp_host on page-locked host buffers: parameters and cotangents "
                            "copied host -> device inside the call, gradient copied back, the I/Q/U maps stored by the "
                            "forward kernel straight into the host buffers (d2h bytes = the bytes that land there)"},
            "e2e_loglike": None if "t_fused" not in e else {
                "value": total / e["t_fused"], "unit": UNIT, "ms_per_step": 1e3 * e["t_fused"],
                "h2d_bytes_per_step": e["fused_h2d"], "d2h_bytes_per_step": e["fused_d2h"],
                "note": "synax_loglike_vjp (Eq. 15 likelihood + gradient fused: forward, residuals, VJP) with pinned host "
                        "parameters in and (logL, grad) out per step; observed Q/U maps resident on the device"},
            "gpu_launches": r["launches"], "escalated_sightlines": r["escalated"],
            "clocks": clocks,
        }
        line["roofline"] = (grid_roofline(w, r, local_samples) if w.kind == "grid_b"
                            else alu_roofline(w, r, local_samples, peak, sm_max, peak_src, strong, clocks))
        if "float64_mode" in r:
            line["float64_mode"] = dict(r["float64_mode"], value=samples / (1e-3 * (r["float64_mode"]["forward_ms"] + r["float64_mode"]["vjp_ms"])), unit=UNIT)
        if "t_graph" in r:
            line["cuda_graph"] = {"ms_per_step": 1e3 * r["t_graph"], "value": samples / r["t_graph"], "unit": UNIT,
                                  "note": "forward + VJP captured once, replayed back to back (no L2 flush between replays)"}
        if world == 1 and not args.no_cpu_baseline:
            wo = apply_overrides(wl_config(args.config), args)
            cb = oracle_baseline(wo, seconds_budget=args.cpu_seconds)
            line["cpu_baseline"] = {k: v for k, v in cb.items() if k in ("value", "unit", "cores", "kind", "sample", "forward_samples_per_s")}
            if cb["cores"] > 1:   # the oracle on one core as well, on a 1/cores share of the same sample
                c1 = oracle_baseline(wo, seconds_budget=args.cpu_seconds / 3.0, threads=1)
                line["cpu_baseline"]["one_core"] = {k: c1[k] for k in ("value", "unit", "cores", "sample", "forward_samples_per_s")}
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs index (default 4: the metric's workload)")
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--scaling", choices=("weak", "strong"), default="strong",
                    help="N > 1: strong (default) = pixel shards of one map + one gradient all-reduce per step (SURVEY.md 8(e)); "
                         "weak = one parameter vector (chain) per rank, no collective")
    ap.add_argument("--nside", type=int, default=0, help="override the config's nside (runtime sweeps)")
    ap.add_argument("--n-los", type=int, default=0, help="override the config's samples per sightline")
    ap.add_argument("--freq-hz", type=float, default=0.0, help="run at this single frequency instead of the config's")
    ap.add_argument("--lanes", type=int, default=0, help="plan option 'lanes' (threads per sightline: 1, 8 or 32; 0 = the library's choice)")
    ap.add_argument("--f64", action="store_true", help="also time the all-float64 entry points (synax_forward_f64 / synax_vjp_f64)")
    ap.add_argument("--graph", action="store_true", help="also time the step captured in a CUDA graph (launch-bound configs)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="wall-time budget of the cpu_baseline oracle sample")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
