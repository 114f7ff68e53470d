"""The adjoint sweeps each sightline backwards and needs its Faraday total first: it takes it from what the plan's last
forward stored (one float64 per sightline) when that forward ran with exactly the same parameters and settings, else
from a pre-pass of its own.  Both routes must give the oracle's gradient; a stale store must never be used."""
import numpy as np
import pytest

from harness import parity
from harness import workloads as wl

pytestmark = pytest.mark.gpu


def _grad(plan, model, params, cots):
    import torch
    import paper_2410_01136_b200 as sx
    g = sx.vjp(plan, model, params, *cots)
    torch.cuda.synchronize()
    return g.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("case", ["cfg1", "cfg4_408MHz", "cfg2_batch", "stack16", "uniform"])
def test_adjoint_after_forward_and_alone(case):
    import torch
    import paper_2410_01136_b200 as sx
    if case == "cfg1":
        w = wl.config(1).scaled(nside=16, n_los=200)
    elif case == "cfg4_408MHz":
        w = wl.config(4).scaled(nside=16, n_los=512)          # strong rotation: float64-angle variants
    elif case == "cfg2_batch":
        w = wl.config(2).scaled(nside=8, n_los=128, batch=3)
    elif case == "stack16":
        w = wl.stack16(nside=8, n_los=128, freqs=(1.4e9, 23e9))
    else:
        w = wl.uniform_toy(bvec=(2.0, -3.0, 1.5), nside=4, n_los=100, freqs=(0.408e9, 2.4e9))
    cots_h = w.cotangents()
    ref = parity.oracle_vjp(w, cots_h)
    nz = ref != 0
    plan, model, params = parity.gpu_objects(w, lanes=1, batch_share=1)   # one thread per sightline: the route with the store
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    g_alone = _grad(plan, model, params, cots)                # nothing stored yet: pre-pass
    sx.forward(plan, model, params)
    g_after = _grad(plan, model, params, cots)                # totals from the forward
    for g, what in ((g_alone, "pre-pass"), (g_after, "stored totals")):
        assert np.all(np.abs(g - ref)[nz] <= parity.GRAD_TOL * np.abs(ref)[nz]), (case, what, np.abs(g - ref)[nz] / np.abs(ref)[nz])
    # other parameters: the store is stale and must not be used
    p2 = (params * 1.07).contiguous()
    w2 = wl.Workload(w.name, w.kind, w.nside, w.n_los, w.s_max, w.freqs, p2.cpu().numpy(), w.aux, cot_seed=w.cot_seed)
    ref2 = parity.oracle_vjp(w2, cots_h)
    g2 = _grad(plan, model, p2, cots)
    assert np.all(np.abs(g2 - ref2)[nz] <= parity.GRAD_TOL * np.abs(ref2)[nz]), (case, "stale store", np.abs(g2 - ref2)[nz] / np.abs(ref2)[nz])
    # ... and the original parameters again are recognised again
    g3 = _grad(plan, model, params, cots)
    assert np.array_equal(g3, g_after)
    plan.close()


def test_store_is_dropped_when_the_geometry_or_the_settings_change():
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(4).scaled(nside=8, n_los=256)
    cots_h = w.cotangents()
    plan, model, params = parity.gpu_objects(w, lanes=1)
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    sx.forward(plan, model, params)
    box = (40.0, 40.0, 10.0)
    plan.set_box(box)                                         # other sample positions: the stored totals are void
    w.clip_box = box
    ref = parity.oracle_vjp(w, cots_h)
    g = _grad(plan, model, params, cots)
    assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref)), np.abs(g - ref) / np.abs(ref)
    sx.forward(plan, model, params)
    plan.set_option("precision", 2)                           # float64 angles everywhere: totals of an fp32 forward are not enough
    g = _grad(plan, model, params, cots)
    assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref))
    plan.close()


@pytest.mark.parametrize("n_los,precision", [(500, 0), (97, 0), (512, 2), (33, 2)])
def test_tile_bases_from_the_forward(n_los, precision):
    """Strong rotation (408 MHz), one thread per sightline: the float64-chain forward stores the Faraday depth before every
    32nd sample and the adjoint runs fp32 tile-local angles on those bases instead of a float64 chain of its own --
    sample counts that are not multiples of 32, the flagged-list route (8 lanes per sightline add their lane offsets) and
    float64 everywhere (precision 2)."""
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(4).scaled(nside=16, n_los=n_los)
    w.params = w.params.copy()
    w.params[0, 13] *= 2.0                                     # n_e doubled: fp32 angles alone miss the bound (2.4e-3)
    cots_h = w.cotangents()
    ref = parity.oracle_vjp(w, cots_h)
    plan, model, params = parity.gpu_objects(w, lanes=1, precision=precision)
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    sx.forward(plan, model, params)
    g = _grad(plan, model, params, cots)
    assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref)), np.abs(g - ref) / np.abs(ref)
    plan.set_option("use_forward_totals", 0)                  # the same without them: pre-pass + float64-angle variants
    g0 = _grad(plan, model, params, cots)
    assert np.all(np.abs(g0 - ref) <= parity.GRAD_TOL * np.abs(ref)), np.abs(g0 - ref) / np.abs(ref)
    plan.close()


def test_long_call_forward_then_adjoint_sparse_cotangent():
    """786,432 sightlines (forward in split mode: the two chains side by side, the missed list afterwards), then the adjoint
    on the stored totals and tile bases; cotangent on every 96th pixel, oracle over those."""
    import torch
    import paper_2410_01136_b200 as sx
    w4 = wl.config(4)
    w = wl.Workload("cfg4_long", w4.kind, 256, 100, w4.s_max, np.array([0.408e9, 1.4e9, 23e9]), w4.params, w4.aux, cot_seed=2204)
    pix = np.arange(7, w.npix, 96)
    full = w.cotangents()
    cots_h = tuple(np.zeros_like(c) for c in full)
    for c, f in zip(cots_h, full):
        c[..., pix] = f[..., pix]
    ref = parity.oracle_vjp(w, tuple(np.ascontiguousarray(c[..., pix]) for c in cots_h), pix=pix)
    plan, model, params = parity.gpu_objects(w)
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    sx.forward(plan, model, params)
    torch.cuda.synchronize()
    stats = plan.stats()
    assert 0.02 * w.npix < stats["escalated"] < 0.9 * w.npix, stats     # split mode
    g = _grad(plan, model, params, cots)
    assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref)), np.abs(g - ref) / np.abs(ref)
    assert np.array_equal(g, _grad(plan, model, params, cots))          # bit-reproducible
    plan.close()


@pytest.mark.parametrize("warm", [True, False])
def test_stored_totals_inside_a_cuda_graph(warm):
    """forward + adjoint captured in one CUDA graph with one thread per sightline: the store, the device-side comparison of
    the parameters and the consumer all replay; new parameter values in the same buffers are picked up.  warm = False: the
    capture is the plan's first call, the store's buffers cannot be allocated inside it, and the adjoint must fall back."""
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(4).scaled(nside=8, n_los=256)
    cots_h = w.cotangents()
    plan, model, params = parity.gpu_objects(w, lanes=1)
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    out = tuple(torch.empty((1, w.n_freq, plan.npix), device="cuda") for _ in range(3))
    g = torch.empty_like(params)
    s = torch.cuda.Stream()
    if warm:
        with torch.cuda.stream(s):
            sx.forward(plan, model, params, out=out)
            sx.vjp(plan, model, params, *cots, out=g)
        s.synchronize()
    else:
        torch.zeros(1, device="cuda").add_(1)
        torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        sx.forward(plan, model, params, out=out)
        sx.vjp(plan, model, params, *cots, out=g)
    for scale in (1.0, 1.05):
        params.mul_(scale)
        graph.replay()
        torch.cuda.synchronize()
        w2 = wl.Workload(w.name, w.kind, w.nside, w.n_los, w.s_max, w.freqs, params.cpu().numpy(), w.aux, cot_seed=w.cot_seed)
        ref = parity.oracle_vjp(w2, cots_h)
        got = g.cpu().numpy().astype(np.float64)
        assert np.all(np.abs(got - ref) <= parity.GRAD_TOL * np.abs(ref)), (warm, scale, np.abs(got - ref) / np.abs(ref))
    plan.close()


def test_tile_bases_with_batch_and_frequency_blocks():
    """Three parameter vectors (different rotation strengths) x 13 frequencies (passes of 8 + 4 + 1) at one thread per
    sightline: the stored totals / tile bases are indexed by (vector, pixel) and shared by all frequency passes."""
    import torch
    import paper_2410_01136_b200 as sx
    w4 = wl.config(4)
    params = np.repeat(w4.params, 3, axis=0).copy()
    params[1, 13] *= 2.0; params[2, 13] *= 0.1; params[2, 0] *= 1.3
    w = wl.Workload("cfg4_b3_f13", w4.kind, 8, 320, w4.s_max, np.geomspace(0.408e9, 30e9, 13), params, w4.aux, cot_seed=2304)
    cots_h = w.cotangents()
    ref = parity.oracle_vjp(w, cots_h)
    plan, model, dparams = parity.gpu_objects(w, lanes=1)
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    maps = tuple(t.cpu().numpy().astype(np.float64) for t in sx.forward(plan, model, dparams))
    parity.assert_maps_close(maps, parity.oracle_forward(w), what="batch 3 x 13 frequencies forward")
    g = _grad(plan, model, dparams, cots)
    assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref)), np.abs(g - ref) / np.abs(ref)
    plan.close()


@pytest.mark.parametrize("nside,freqs,n_los", [(48, (0.408e9, 1.4e9), 500), (48, (23e9,), 500), (48, (0.408e9, 2.4e9, 23e9), 1024),
                                               (64, (0.408e9, 2.4e9, 23e9), 1024)])
def test_mid_size_forward_with_lanes_then_one_thread_adjoint(nside, freqs, n_los):
    """27,648 sightlines (49,152 in the last case, which is long enough for the forward's split mode: one list per chain,
    8 lanes each), the library's own lane choice: the forward runs with 8 lanes per sightline and still stores the
    Faraday totals (and, from its float64 chain, the tile bases -- written per lane and shifted by the lane offsets); the
    adjoint that follows then takes one thread per sightline on them.  Cotangent on every 24th pixel, oracle over those;
    the stand-alone adjoint (8 lanes, own pre-pass) must agree too."""
    import torch
    import paper_2410_01136_b200 as sx
    w4 = wl.config(4)
    w = wl.Workload("cfg4_mid", w4.kind, nside, n_los, w4.s_max, np.array(freqs), w4.params, w4.aux, cot_seed=3305)
    pix = np.arange(3, w.npix, 24)
    full = w.cotangents()
    cots_h = tuple(np.zeros_like(c) for c in full)
    for c, f in zip(cots_h, full):
        c[..., pix] = f[..., pix]
    ref = parity.oracle_vjp(w, tuple(np.ascontiguousarray(c[..., pix]) for c in cots_h), pix=pix)
    ref_maps = parity.oracle_forward(w, pix=pix)
    plan, model, params = parity.gpu_objects(w)
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    g_alone = _grad(plan, model, params, cots)
    maps = sx.forward(plan, model, params)
    torch.cuda.synchronize()
    if nside == 64:
        assert 0.02 * w.npix < plan.stats()["escalated"] < 0.9 * w.npix, plan.stats()     # split mode
    parity.assert_maps_close(tuple(m.cpu().numpy()[..., pix] for m in maps), ref_maps, what="mid-size forward")
    g_after = _grad(plan, model, params, cots)
    for g, what in ((g_alone, "stand-alone"), (g_after, "after the forward")):
        assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref)), (what, np.abs(g - ref) / np.abs(ref))
    assert np.array_equal(g_after, _grad(plan, model, params, cots))
    plan.close()


def test_mid_size_batch_of_three_with_lanes_then_one_thread_adjoint():
    """As above with three parameter vectors (82,944 sightlines; 12 frequencies: two frequency blocks): the stored totals and
    tile bases are indexed by batch element x pixel, written by an 8-lane forward, read by a one-thread adjoint."""
    import torch
    import paper_2410_01136_b200 as sx
    w4 = wl.config(4)
    p = np.repeat(w4.params, 3, axis=0) * (1.0 + 0.03 * np.arange(3, dtype=np.float32))[:, None]
    w = wl.Workload("cfg4_mid_b3", w4.kind, 48, 500, w4.s_max, np.geomspace(0.408e9, 30e9, 12), p.astype(np.float32), w4.aux,
                    cot_seed=3306)
    pix = np.arange(11, w.npix, 48)
    full = w.cotangents()
    cots_h = tuple(np.zeros_like(c) for c in full)
    for c, f in zip(cots_h, full):
        c[..., pix] = f[..., pix]
    ref = parity.oracle_vjp(w, tuple(np.ascontiguousarray(c[..., pix]) for c in cots_h), pix=pix)
    plan, model, params = parity.gpu_objects(w)
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    sx.forward(plan, model, params)
    g = _grad(plan, model, params, cots)
    assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref)), np.abs(g - ref) / np.abs(ref)
    plan.set_option("use_forward_totals", 0)
    g0 = _grad(plan, model, params, cots)
    assert np.all(np.abs(g0 - ref) <= parity.GRAD_TOL * np.abs(ref)), np.abs(g0 - ref) / np.abs(ref)
    plan.close()
