"""synax_vjp_f64_noalloc: the float64 adjoint on the library's fixed scratch array (no cudaMalloc / cudaFree anywhere in the
call; include/synax.h) against the existing path, synax_vjp_f64, on the same inputs -- same kernels, same fixed-order
reduction, so the two agree far inside the float64-mode gradient bound of tests/test_gpu_f64_mode.py (1e-9 relative).
Every call shares the array and finds the last call's contents in it: the calls below run back to back, a large one first,
then a smaller one of another model and batch, then the first again.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from harness import workloads as wl

pytestmark = pytest.mark.gpu

GRAD_TOL_F64 = 1.0e-9   # tests/test_gpu_f64_mode.py


def _case(w, params64, lanes, seed):
    import torch
    import paper_2410_01136_b200 as sx
    plan = sx.Plan(w.nside, w.n_los, w.s_max, w.freqs, observer=w.observer)
    if lanes:
        plan.set_option("lanes", lanes)
    model = sx.Model(w.kind, aux=w.aux)
    p = torch.from_numpy(np.ascontiguousarray(params64)).cuda()
    rng = np.random.Generator(np.random.PCG64(seed))
    shape = (p.shape[0], len(w.freqs), plan.npix)
    cots = [torch.from_numpy(rng.standard_normal(shape)).cuda() for _ in range(3)]
    return sx, plan, model, p, cots


def _close(got, want, what):
    got, want = got.cpu().numpy(), want.cpu().numpy()
    assert np.all(np.isfinite(got)), what
    nz = want != 0
    rel = np.abs(got - want)[nz] / np.abs(want)[nz]
    assert rel.size and rel.max() <= GRAD_TOL_F64, (what, rel.max())
    assert np.all(got[~nz] == 0.0), what
    return rel.max()


def test_noalloc_vjp_matches_vjp_f64_on_calls_in_a_row():
    import torch
    wa = wl.config(4).scaled(nside=16, n_los=256)                       # FULL16, 8 frequencies, strong rotation
    pa = wl.FULL16_NOMINAL[None, :] * (1.0 + 1e-3 * np.linspace(-1, 1, 16))
    wb = wl.config(2).scaled(nside=4, n_los=100, batch=5)               # FULL16 batch 5, alpha != 3
    pb = wb.params.astype(np.float64)
    pb[:, 12] = [2.5, 2.8, 3.0, 3.2, 3.4]
    sx, plan_a, model_a, p_a, cots_a = _case(wa, pa, 8, 901)
    _, plan_b, model_b, p_b, cots_b = _case(wb, pb, 0, 902)
    want_a = sx.vjp_f64(plan_a, model_a, p_a, *cots_a)                  # the existing path (stream-ordered pool scratch)
    want_b = sx.vjp_f64(plan_b, model_b, p_b, *cots_b)
    got_a, got_b, got_a2 = torch.full_like(p_a, np.nan), torch.full_like(p_b, np.nan), torch.full_like(p_a, np.nan)
    sx.vjp_f64_noalloc(plan_a, model_a, p_a, *cots_a, out=got_a)        # back to back on one stream, no synchronisation
    sx.vjp_f64_noalloc(plan_b, model_b, p_b, *cots_b, out=got_b)
    sx.vjp_f64_noalloc(plan_a, model_a, p_a, *cots_a, out=got_a2)
    torch.cuda.synchronize()
    ra = _close(got_a, want_a, "first call")
    rb = _close(got_b, want_b, "second call (smaller, on the first call's leftovers)")
    ra2 = _close(got_a2, want_a, "third call")
    print(f"noalloc vs vjp_f64: {ra:.1e}, {rb:.1e}, {ra2:.1e} relative")
    # a missing cotangent (NULL = zeros) goes the same way through both entry points
    want_q = sx.vjp_f64(plan_b, model_b, p_b, None, cots_b[1], None)
    got_q = sx.vjp_f64_noalloc(plan_b, model_b, p_b, None, cots_b[1], None, out=torch.full_like(p_b, np.nan))
    torch.cuda.synchronize()
    _close(got_q, want_q, "dQ only")
    plan_a.close(); plan_b.close()


def test_noalloc_vjp_rejects_calls_beyond_the_array_and_recovers():
    import torch
    w = wl.config(2).scaled(nside=16, n_los=32, batch=48)               # 32 lanes: 768 CTAs x 128 B x 48 = 4.7 MB > 4 MiB
    sx, plan, model, p, cots = _case(w, w.params.astype(np.float64), 32, 903)
    out = torch.full_like(p, np.nan)
    with pytest.raises(sx.SynaxError) as ei:
        sx.vjp_f64_noalloc(plan, model, p, *cots, out=out)
    assert ei.value.status == 2 and "4194304" in str(ei.value)          # SYNAX_ERR_UNSUPPORTED, names the limit
    torch.cuda.synchronize()
    assert torch.isnan(out).all()                                       # nothing was launched
    plan.set_option("lanes", 8)                                         # 192 CTAs x 128 B x 48 = 1.2 MB: fits
    got = sx.vjp_f64_noalloc(plan, model, p, *cots, out=out)
    want = sx.vjp_f64(plan, model, p, *cots)
    torch.cuda.synchronize()
    _close(got, want, "after a rejected call")
    plan.close()
