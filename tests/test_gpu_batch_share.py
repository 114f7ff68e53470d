"""Batched calls share the sightline geometry between NB parameter vectors per thread (PAPER.md L13
"batch acceleration"): per vector the arithmetic is unchanged, so the maps equal the unshared path's to fp32 rounding (bit
for bit in most instantiations, e.g. the full cfg-2 launch) and the gradients agree to rounding of the block sums."""
import numpy as np
import pytest

from harness import parity
from harness import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kind,batch", [("full16", 7), ("full16", 8), ("disc4", 5), ("full16", 2)])
def test_shared_geometry_is_bit_identical_and_matches_oracle(kind, batch):
    if kind == "full16":
        w = wl.config(2).scaled(nside=8, n_los=200, batch=batch)
    else:
        w = wl.config(1).scaled(nside=8, n_los=200)
        w.freqs = np.array([23e9])
        rng = np.random.Generator(np.random.PCG64(77))
        w.params = (w.params[0][None, :] * (1.0 + 0.2 * rng.uniform(-1, 1, (batch, 4)))).astype(np.float32)
    ref_maps, _ = parity.gpu_forward(w, lanes=1, batch_share=1)
    cots = w.cotangents()
    g1 = parity.gpu_vjp(w, cots, lanes=1, batch_share=1)
    oracle_maps = parity.oracle_forward(w)
    oracle_grad = parity.oracle_vjp(w, cots)
    for nb in (0, 2, 4):
        maps, _ = parity.gpu_forward(w, lanes=1, batch_share=nb)
        for a, b in zip(maps, ref_maps):
            # per vector the arithmetic is the unshared kernel's; the compiler contracts a few multiply-adds differently in
            # some instantiations (last-bit differences: ~1e-8 of the map maximum), so "equal" means to fp32 rounding
            assert np.all(np.abs(a - b) <= 3e-7 * np.abs(b).max(axis=-1, keepdims=True)), (kind, batch, nb)
        parity.assert_maps_close(maps, oracle_maps, what=f"batch_share={nb}")
        g = parity.gpu_vjp(w, cots, lanes=1, batch_share=nb)
        # (the unshared adjoint sweeps backwards, the batched one forwards with the prefix form: same sums, other order)
        parity.assert_log_gradient_close(g, g1, w.params.astype(np.float64), what=f"batch_share={nb} vs 1")
        nz = oracle_grad != 0
        assert np.all(np.abs(g - oracle_grad)[nz] <= parity.GRAD_TOL * np.abs(oracle_grad)[nz]), nb


def test_cfg2_full_launch_shared_vs_unshared():
    """BASELINE.json configs[2] at full size (256 vectors x 12,288 sightlines): every map value equal to the unshared path."""
    w = wl.config(2)
    a, _ = parity.gpu_forward(w, batch_share=1)
    b, _ = parity.gpu_forward(w)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    cots = w.cotangents()
    g1, g = parity.gpu_vjp(w, cots, batch_share=1), parity.gpu_vjp(w, cots, batch_share=2)
    th = w.params.astype(np.float64)
    parity.assert_log_gradient_close(g, g1, th, what="cfg2 shared vs unshared")


def test_batch_share_with_alpha_not_three_and_low_frequency():
    """alpha != 3 (lg2/ex2 branch) and a call whose pilot sends it to the float64-angle variants: the batched kernels
    must stand aside (mode word) and the result must not depend on the option."""
    w = wl.config(2).scaled(nside=8, n_los=256, batch=6)
    p = w.params.copy(); p[:, 12] = [2.6, 2.8, 3.0, 3.1, 3.3, 3.4]
    w.params = p
    cots = w.cotangents()
    th = w.params.astype(np.float64)
    ref = parity.oracle_vjp(w, cots)
    for nb in (1, 4):
        g = parity.gpu_vjp(w, cots, lanes=1, batch_share=nb)
        parity.assert_log_gradient_close(g, ref, th, what=f"alpha != 3, batch_share={nb}")
    w.freqs = np.array([0.3e9])
    ref = parity.oracle_vjp(w, cots)
    refm = parity.oracle_forward(w)
    for nb in (1, 4):
        maps, _ = parity.gpu_forward(w, lanes=1, batch_share=nb)
        parity.assert_maps_close(maps, refm, what=f"300 MHz batch_share={nb}")
        g = parity.gpu_vjp(w, cots, lanes=1, batch_share=nb)
        parity.assert_log_gradient_close(g, ref, th, what=f"300 MHz, batch_share={nb}")


def test_batch_share_after_a_forward_that_left_tile_bases():
    """Long single-frequency call at 408 MHz (strong rotation: device mode "split") with batch_share = 2, the adjoint right
    after the forward of the same plan: the forward left tile bases, which only the lean vjp_kernel uses -- the shared
    kernel stands aside for it (before, every launch of that combination stood aside and the gradient was never written)."""
    import torch
    import paper_2410_01136_b200 as sx
    w2 = wl.config(2)
    p = np.repeat(wl.FULL16_NOMINAL[None, :], 6, axis=0).astype(np.float32)
    p *= (1.0 + 0.02 * np.arange(6, dtype=np.float32))[:, None]
    w = wl.Workload("full16_408_b6", "full16", 64, 1024, w2.s_max, np.array([0.408e9]), p, w2.aux, cot_seed=515)
    pix = np.arange(5, w.npix, 48)
    full = w.cotangents()
    cots_h = tuple(np.zeros_like(c) for c in full)
    for c, f in zip(cots_h, full):
        c[..., pix] = f[..., pix]
    ref = parity.oracle_vjp(w, tuple(np.ascontiguousarray(c[..., pix]) for c in cots_h), pix=pix)
    cots = [torch.from_numpy(c).cuda() for c in cots_h]
    th = w.params.astype(np.float64)
    for nb in (1, 2):
        plan, model, params = parity.gpu_objects(w, lanes=1, batch_share=nb)
        out = torch.full_like(params, float("nan"))
        sx.vjp(plan, model, params, *cots, out=out)                       # stand-alone
        torch.cuda.synchronize()
        parity.assert_log_gradient_close(out.cpu().numpy().astype(np.float64), ref, th, what=f"alone, batch_share={nb}")
        sx.forward(plan, model, params)
        out.fill_(float("nan"))
        sx.vjp(plan, model, params, *cots, out=out)                       # on the forward's totals and tile bases
        torch.cuda.synchronize()
        assert plan.stats()["escalated"] > 0.02 * w.npix * 6
        parity.assert_log_gradient_close(out.cpu().numpy().astype(np.float64), ref, th, what=f"after forward, batch_share={nb}")
        plan.close()
