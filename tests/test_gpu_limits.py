"""Maximum sizes and robustness of the CUDA path (all through the C ABI): n_los = 65536, a large nside on sampled
pixels, batches beyond the 65535 grid.y limit, two plans on two streams, NaN parameters."""
import numpy as np
import pytest

import oracle
from harness import parity
from harness import workloads as wl

pytestmark = pytest.mark.gpu


def test_max_samples_per_sightline():
    w = wl.config(1).scaled(nside=1, n_los=65536)
    maps, _ = parity.gpu_forward(w)
    parity.assert_maps_close(maps, parity.oracle_forward(w), what="n_los = 65536")
    cots = w.cotangents()
    g, ref = parity.gpu_vjp(w, cots), parity.oracle_vjp(w, cots)
    assert np.all(np.abs(g - ref) <= parity.GRAD_TOL * np.abs(ref))


def test_large_nside_on_sampled_pixels():
    """nside = 2048 (50,331,648 sightlines, full launch); the oracle recomputes every 100,003rd pixel."""
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(0).scaled(nside=2048, n_los=4)
    plan, model, params = parity.gpu_objects(w)
    assert plan.npix == 12 * 2048 * 2048
    I, Q, U = sx.forward(plan, model, params)
    torch.cuda.synchronize()
    pix = np.arange(7, plan.npix, 100003)
    idx = torch.from_numpy(pix).cuda()
    sub = tuple(t[..., idx].cpu().numpy().astype(np.float64) for t in (I, Q, U))
    assert all(bool(torch.isfinite(t).all()) for t in (I, Q, U))
    plan.close()
    ref = parity.oracle_forward(w, pix=pix)
    parity.assert_maps_close(sub, ref, what="nside = 2048 (sampled pixels)")


def test_batch_beyond_grid_y_limit():
    """70,000 parameter vectors: the VJP launches in chunks of 65,535 batch elements."""
    base = wl.config(2).scaled(nside=1, n_los=16, batch=1)
    rng = np.random.Generator(np.random.PCG64(70))
    p = base.params.astype(np.float64) * (1.0 + 0.1 * rng.uniform(-1, 1, (70000, 16)))
    w = wl.Workload("big_batch", "full16", 1, 16, 20.0, base.freqs, p.astype(np.float32), None, cot_seed=71)
    maps, _ = parity.gpu_forward(w)
    cots = w.cotangents()
    g = parity.gpu_vjp(w, cots)
    assert np.all(np.isfinite(g))
    for b in (0, 65534, 65535, 69999):
        wb = wl.Workload("b", "full16", 1, 16, 20.0, base.freqs, w.params[b:b + 1], None)
        parity.assert_maps_close(tuple(m[b:b + 1] for m in maps), parity.oracle_forward(wb), what=f"batch element {b}")
        gb = parity.oracle_vjp(wb, tuple(c[b:b + 1] for c in cots))
        assert np.all(np.abs(g[b:b + 1] - gb) <= parity.GRAD_TOL * np.abs(gb)), b


def test_batch_times_npix_limit_is_an_error():
    import torch
    import paper_2410_01136_b200 as sx
    plan = sx.Plan(256, 4, 20.0, [23e9])                      # npix = 786,432: batch 4096 -> 3.2e9 sightlines >= 2^31
    params = torch.zeros((4096, 16), device="cuda")
    I = torch.zeros(8, device="cuda")
    with pytest.raises(sx.SynaxError, match="INVALID_ARG"):
        sx.forward(plan, sx.Model("full16"), params, out=(I, I, I))
    plan.close()


def test_two_plans_on_two_streams_match_serial_results():
    import torch
    import paper_2410_01136_b200 as sx
    wa, wb = wl.config(1).scaled(nside=32, n_los=128), wl.config(4).scaled(nside=16, n_los=256)
    pa, ma, xa = parity.gpu_objects(wa)
    pb, mb, xb = parity.gpu_objects(wb)
    ra = [t.clone() for t in sx.forward(pa, ma, xa)]
    rb = [t.clone() for t in sx.forward(pb, mb, xb)]
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for _ in range(3):
        with torch.cuda.stream(s1):
            oa = sx.forward(pa, ma, xa)
        with torch.cuda.stream(s2):
            ob = sx.forward(pb, mb, xb)
    s1.synchronize(); s2.synchronize()
    assert all(torch.equal(a, b) for a, b in zip(ra, oa)) and all(torch.equal(a, b) for a, b in zip(rb, ob))
    pa.close(); pb.close()


def test_nan_parameters_give_nan_maps_not_a_fault():
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(0)
    plan, model, params = parity.gpu_objects(w)
    params[0, 0] = float("nan")
    I, Q, U = sx.forward(plan, model, params)
    g = sx.vjp(plan, model, params, *[torch.from_numpy(c).cuda() for c in w.cotangents()])
    torch.cuda.synchronize()
    assert bool(torch.isnan(I).any()) and bool(torch.isnan(g).any())
    params[0, 0] = 6.0                                          # the plan and the library are still usable
    I2, _, _ = sx.forward(plan, model, params)
    assert bool(torch.isfinite(I2).all())
    plan.close()


def test_forward_and_vjp_are_cuda_graph_capturable():
    """No call synchronises or allocates outside the stream-ordered pool: a whole step can be captured once and
    replayed (the launch-bound regime of config 0: 9 launches per step)."""
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(0)
    plan, model, params = parity.gpu_objects(w)
    cots = [torch.from_numpy(c).cuda() for c in w.cotangents()]
    out = sx.forward(plan, model, params)
    g = sx.vjp(plan, model, params, *cots)
    torch.cuda.synchronize()
    ref_out, ref_g = [t.clone() for t in out], g.clone()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):                                   # warm-up on the capture stream
        sx.forward(plan, model, params, out=out)
        sx.vjp(plan, model, params, *cots, out=g)
    s.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        sx.forward(plan, model, params, out=out)
        sx.vjp(plan, model, params, *cots, out=g)
    for t in out:
        t.zero_()
    g.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert all(torch.equal(a, b) for a, b in zip(out, ref_out)) and torch.equal(g, ref_g)
    params.mul_(1.1)                                             # same graph, new parameter values
    graph.replay()
    torch.cuda.synchronize()
    eager = sx.forward(plan, model, params)
    torch.cuda.synchronize()
    assert all(torch.equal(a, b) for a, b in zip(out, eager))
    plan.close()


@pytest.mark.gpu
def test_adjoint_pair_on_two_streams_is_graph_capturable_and_ordered():
    """Long calls run the adjoint's per-CTA pair on two streams (fork after vjp_classify_kernel, join before the
    reduction).  The fork / join must be capturable in a CUDA graph and ordered with the caller's stream: the
    gradient read right after the call on the caller's stream is complete and bit-identical on replay."""
    import torch
    import paper_2410_01136_b200 as sx
    w4 = wl.config(4)
    w = wl.Workload("cfg4_pair", w4.kind, 256, 64, w4.s_max, w4.freqs, w4.params, w4.aux, cot_seed=2104)
    plan, model, params = parity.gpu_objects(w)
    cots = [torch.from_numpy(c).cuda() for c in w.cotangents()]
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        g = sx.vjp(plan, model, params, *cots)
        g_host = g.cpu()                                         # stream-ordered read right behind the call
        sx.vjp(plan, model, params, *cots, out=g)
    s.synchronize()
    assert torch.equal(g.cpu(), g_host) and bool(torch.isfinite(g_host).all())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        sx.vjp(plan, model, params, *cots, out=g)
    g.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(g.cpu(), g_host)
    plan.set_option("precision", 2)                               # float64 angles everywhere: within the bound of it
    gp = sx.vjp(plan, model, params, *cots)
    torch.cuda.synchronize()
    rel = ((gp.cpu() - g_host).abs() / gp.cpu().abs()).max().item()
    assert rel <= 1e-3, rel
    plan.close()


def test_pool_release_threshold_keyword():
    """Plan(pool_release_threshold_mb=...) sets the option of that name (process-wide, opt-in: include/synax.h); results are
    those of a plan without it, whether or not the caller synchronises between the calls."""
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(1).scaled(nside=16, n_los=96)
    plan0, model, params = parity.gpu_objects(w)
    ref = [t.clone() for t in sx.forward(plan0, model, params)]
    plan0.close()
    plan = sx.Plan(w.nside, w.n_los, w.s_max, w.freqs, pool_release_threshold_mb=64)
    for _ in range(3):
        out = sx.forward(plan, model, params)
        torch.cuda.synchronize()
        assert all(torch.equal(a, b) for a, b in zip(out, ref))
    with pytest.raises(sx.SynaxError):
        plan.set_option("pool_release_threshold_mb", -1.0)
    plan.close()


def test_workspace_growth_and_reuse_across_call_sizes():
    """The plan's scratch workspace (include/synax.h "Scratch"): calls of growing and shrinking batch on ONE plan -- the call
    that outgrows the buffer takes the excess from the pool, the next one reallocates -- give what fresh plans give, with and
    without a synchronisation between the calls; gridded model too (repacked grid + accumulation buffer in the workspace)."""
    import torch
    import paper_2410_01136_b200 as sx
    base = wl.config(2).scaled(nside=8, n_los=128, batch=8)
    plan = sx.Plan(base.nside, base.n_los, base.s_max, base.freqs)
    model = sx.Model("full16")
    for sync in (True, False):
        for nb in (1, 8, 3, 8, 1):
            p = torch.from_numpy(base.params[:nb].copy()).cuda()
            cots = [torch.from_numpy(np.ascontiguousarray(c[:nb])).cuda() for c in base.cotangents()]
            fresh = sx.Plan(base.nside, base.n_los, base.s_max, base.freqs)
            ref = [t.clone() for t in sx.forward(fresh, model, p)]
            gref = sx.vjp(fresh, model, p, *cots).clone()
            fresh.close()
            out = sx.forward(plan, model, p)
            g = sx.vjp(plan, model, p, *cots)
            if sync:
                torch.cuda.synchronize()
            assert all(torch.equal(a, b) for a, b in zip(out, ref)), (sync, nb)
            assert bool(((g - gref).abs() <= 1e-5 * gref.abs().max()).all()), (sync, nb)
    plan.close()
    w = wl.config(3).scaled(nside=4, n_los=64)
    plan, model, params = parity.gpu_objects(w)
    cots = [torch.from_numpy(c).cuda() for c in w.cotangents()]
    ref = [t.clone() for t in sx.forward(plan, model, params)]
    gref = sx.vjp(plan, model, params, *cots).clone()
    for _ in range(3):
        out = sx.forward(plan, model, params)
        g = sx.vjp(plan, model, params, *cots)
        torch.cuda.synchronize()
        assert all(torch.equal(a, b) for a, b in zip(out, ref))
        assert bool(((g - gref).abs() <= 1e-5 * gref.abs().max()).all())
    plan.close()
