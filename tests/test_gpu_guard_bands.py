"""No entry point writes outside the buffers it is given (include/synax.h: "ownership"): outputs are carved out of one
allocation with sentinel bands before, between and after them; after the call the bands are untouched and the results are
those of the same call into buffers of their own.  Ragged sizes on purpose: pixel counts that fill no block, odd batches,
frequency counts that split into blocks with a remainder, every lane count, pixel shards.  (compute-sanitizer is not
available on the GPU pool; this is the bound check the tests can make themselves.)"""
import numpy as np
import pytest

from harness import parity
from harness import workloads as wl

pytestmark = pytest.mark.gpu

SENTINEL = -12345.678
BAND = 1024   # elements


def _carve(torch, sizes, dtype):
    """One allocation `band | buf0 | band | buf1 | ... | band`; returns (whole, [views], [band slices])."""
    total = BAND + sum(s + BAND for s in sizes)
    whole = torch.full((total,), SENTINEL, dtype=dtype, device="cuda")
    views, bands, at = [], [slice(0, BAND)], BAND
    for s in sizes:
        views.append(whole[at:at + s])
        bands.append(slice(at + s, at + s + BAND))
        at += s + BAND
    return whole, views, bands


def _bands_intact(whole, bands):
    return all(bool((whole[b] == SENTINEL).all()) for b in bands)


def _cases():
    c0 = wl.config(0)
    yield "full16 nside 5 batch 3 n_freq 9", wl.config(4).scaled(nside=5, n_los=77, batch=3), 9, {}
    yield "full16 nside 8 lanes 1", wl.config(4).scaled(nside=8, n_los=130), 2, {"lanes": 1}
    yield "full16 nside 8 lanes 8 batch_share 2", wl.config(2).scaled(nside=8, n_los=96, batch=5), 1, {"lanes": 8, "batch_share": 2}
    yield "full16 precision 2", wl.config(4).scaled(nside=6, n_los=64, batch=2), 3, {"precision": 2}
    yield "disc4 nside 7", wl.config(1).scaled(nside=7, n_los=33), 17, {}
    yield "stack16 nside 3", wl.stack16(nside=3, n_los=50, batch=2), 1, {"lanes": 32}
    yield "uniform nside 1", wl.uniform_toy(nside=1, n_los=5), 1, {}
    yield "grid_b nside 6", wl.config(3).scaled(nside=6, n_los=70), 5, {}
    yield "cfg 0", c0, c0.n_freq, {}


def _with_freqs(w, n_freq):
    if n_freq != w.n_freq:
        w.freqs = np.geomspace(0.4e9, 30e9, n_freq)
    return w


@pytest.mark.parametrize("name,w,n_freq,opts", list(_cases()), ids=[c[0] for c in _cases()])
def test_forward_and_vjp_stay_inside_their_buffers(name, w, n_freq, opts):
    import torch
    import paper_2410_01136_b200 as sx
    w = _with_freqs(w, n_freq)
    plan, model, params = parity.gpu_objects(w, **opts)
    n = w.batch * w.n_freq * w.npix
    ref = [t.clone() for t in sx.forward(plan, model, params)]
    whole, (I, Q, U), bands = _carve(torch, [n, n, n], torch.float32)
    shape = ref[0].shape
    sx.forward(plan, model, params, out=(I.view(shape), Q.view(shape), U.view(shape)))
    torch.cuda.synchronize()
    assert _bands_intact(whole, bands), name
    for a, b in zip((I, Q, U), ref):
        assert torch.equal(a.view(shape), b), name

    cots = [torch.from_numpy(c).cuda() for c in w.cotangents()]
    for after_forward in (True, False):
        if not after_forward:
            plan.set_option("use_forward_totals", 1)     # drops what the forward stored: the stand-alone routes
        gref = sx.vjp(plan, model, params, *cots).clone()
        gwhole, (g,), gbands = _carve(torch, [params.numel()], torch.float32)
        sx.vjp(plan, model, params, *cots, out=g.view(params.shape))
        torch.cuda.synchronize()
        assert _bands_intact(gwhole, gbands), (name, after_forward)
        # (atomics in the block sums: equal to rounding, not bit for bit)
        scale = gref.abs().max()
        assert bool(((g.view(params.shape) - gref).abs() <= 1e-5 * scale).all()), (name, after_forward)
        if after_forward:
            sx.forward(plan, model, params)
    plan.close()


def test_pixel_shards_stay_inside_their_buffers():
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(4).scaled(nside=6, n_los=60, batch=2)
    w.freqs = np.geomspace(0.4e9, 30e9, 3)
    for pix_range, stride in (((5, 101), 1), ((3, 61), 7)):
        plan, model, params = parity.gpu_objects(w, pix_range=pix_range, pix_stride=stride)
        n = w.batch * w.n_freq * plan.npix
        whole, (I, Q, U), bands = _carve(torch, [n, n, n], torch.float32)
        shape = (w.batch, w.n_freq, plan.npix)
        sx.forward(plan, model, params, out=(I.view(shape), Q.view(shape), U.view(shape)))
        torch.cuda.synchronize()
        assert _bands_intact(whole, bands), (pix_range, stride)
        assert bool(torch.isfinite(whole).all())
        plan.close()


def test_float64_entry_points_stay_inside_their_buffers():
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(4).scaled(nside=5, n_los=40, batch=3)
    w.freqs = np.geomspace(0.4e9, 30e9, 3)
    plan, model, params = parity.gpu_objects(w)
    p64 = params.double()
    n = w.batch * w.n_freq * w.npix
    shape = (w.batch, w.n_freq, w.npix)
    whole, (I, Q, U), bands = _carve(torch, [n, n, n], torch.float64)
    sx.forward_f64(plan, model, p64, out=(I.view(shape), Q.view(shape), U.view(shape)))
    cots = [torch.from_numpy(c).cuda().double() for c in w.cotangents()]
    gwhole, (g, g2), gbands = _carve(torch, [p64.numel(), p64.numel()], torch.float64)
    sx.vjp_f64(plan, model, p64, *cots, out=g.view(p64.shape))
    sx.vjp_f64_noalloc(plan, model, p64, *cots, out=g2.view(p64.shape))
    torch.cuda.synchronize()
    assert _bands_intact(whole, bands) and _bands_intact(gwhole, gbands)
    assert bool(torch.isfinite(g).all()) and bool(((g - g2).abs() <= 1e-12 * g.abs().max()).all())
    plan.close()


def test_host_calls_loglike_and_adam_stay_inside_their_buffers():
    import torch
    import paper_2410_01136_b200 as sx
    w = wl.config(4).scaled(nside=5, n_los=48, batch=3)
    w.freqs = np.geomspace(0.4e9, 30e9, 5)
    plan, model, params = parity.gpu_objects(w)
    n = w.batch * w.n_freq * w.npix
    shape = (w.batch, w.n_freq, w.npix)
    # host entry points: numpy buffers carved out of one array
    total = BAND + 3 * (n + BAND) + (params.numel() + BAND)
    host = np.full(total, SENTINEL, dtype=np.float32)
    at, views, bands = BAND, [], [slice(0, BAND)]
    for s in (n, n, n, params.numel()):
        views.append(host[at:at + s]); bands.append(slice(at + s, at + s + BAND)); at += s + BAND
    hp = w.params.astype(np.float32)
    sx.forward_host(plan, model, hp, out=tuple(v.reshape(shape) for v in views[:3]))
    sx.vjp_host(plan, model, hp, *w.cotangents(), out=views[3].reshape(hp.shape))
    assert all(np.all(host[b] == np.float32(SENTINEL)) for b in bands)
    ref = [t.cpu().numpy() for t in sx.forward(plan, model, params)]
    for v, r in zip(views[:3], ref):
        assert np.array_equal(v.reshape(shape), r)
    assert np.isfinite(views[3]).all()

    # fused likelihood + gradient, then ADAM on the parameters
    obs = [torch.from_numpy(np.ascontiguousarray(r[0])).cuda() for r in ref]
    lwhole, (ll,), lbands = _carve(torch, [w.batch], torch.float64)
    gwhole, (g, m, v, th), gbands = _carve(torch, [params.numel()] * 4, torch.float32)
    sx.loglike_vjp(plan, model, params, None, obs[1], obs[2], (0.0, 1.0e6, 1.0e6), out=(ll, g.view(params.shape)))
    m.zero_(); v.zero_(); th.copy_(params.reshape(-1))
    sx.adam_step(th, g, m, v, 1, lr=1e-3)
    torch.cuda.synchronize()
    assert _bands_intact(lwhole, lbands) and _bands_intact(gwhole, gbands)
    assert bool(torch.isfinite(ll).all()) and bool(torch.isfinite(th).all())
    assert float(ll[0]) >= float(ll.max())   # vector 0 generated the observation
    plan.close()
