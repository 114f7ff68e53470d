"""The C-ABI boundary: libsynax.so loads and exports every symbol include/synax.h declares (CPU check, no
compute), and -- on the GPU box -- every invalid call returns an error code without launching."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = ROOT / "include" / "synax.h"


def _declared_symbols():
    text = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(synax_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared_symbols()
    for need in ("synax_plan_create", "synax_plan_destroy", "synax_forward", "synax_vjp", "synax_last_error"):
        assert need in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2410_01136_b200 import build as b
    import paper_2410_01136_b200 as sx
    b.build()
    L = sx.load_library()
    declared = _declared_symbols()
    assert sorted(sx.exported_symbols) == declared
    for name in declared:
        assert getattr(L, name) is not None
    assert b"sm_100a" in L.synax_version()
    assert L.synax_last_error() is not None
    assert L.synax_plan_npix(None) == -1          # host-only call, no device needed
    assert L.synax_plan_destroy(None) == 0


def test_header_has_no_torch_or_cxx_types():
    text = HEADER.read_text()
    assert "torch" not in text and "std::" not in text and "at::" not in text
    assert 'extern "C"' in text


def test_binding_refuses_to_run_without_cuda(monkeypatch):
    import torch
    import paper_2410_01136_b200 as sx
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        sx.Plan(8, 64, 20.0, [23e9])


def test_product_does_not_import_the_oracle():
    for p in list((ROOT / "paper_2410_01136_b200").rglob("*.py")) + list((ROOT / "paper_2410_01136_b200").rglob("*.cu*")):
        t = p.read_text()
        assert "import oracle" not in t and "from oracle" not in t and "synax_oracle" not in t, p
    t = (ROOT / "oracle" / "__init__.py").read_text()
    assert "import paper_2410_01136_b200" not in t and "from paper_2410_01136_b200" not in t


# ------------------------------------------------------------------------------------------------
@pytest.mark.gpu
def test_invalid_arguments_return_codes():
    import torch
    import paper_2410_01136_b200 as sx
    L = sx.load_library()
    torch.zeros(1, device="cuda")
    dbl = ctypes.c_double
    obs = (dbl * 3)(-8.3, 0.0, 0.006)
    fr = (dbl * 1)(23e9)
    h = ctypes.c_void_p()
    INVALID = 1
    bad = [dict(nside=0), dict(nside=8193), dict(n_los=0), dict(n_los=65537), dict(s_max=0.0), dict(s_max=float("nan")),
           dict(n_freq=0), dict(n_freq=33)]
    for kw in bad:
        a = dict(nside=8, n_los=64, s_max=20.0, n_freq=1)
        a.update(kw)
        rc = L.synax_plan_create(a["nside"], a["n_los"], a["s_max"], fr, a["n_freq"], obs, ctypes.byref(h))
        assert rc == INVALID and not h.value, kw
        assert len(L.synax_last_error()) > 0
    assert L.synax_plan_create(8, 64, 20.0, None, 1, obs, ctypes.byref(h)) == INVALID
    assert L.synax_plan_create(8, 64, 20.0, fr, 1, None, ctypes.byref(h)) == INVALID
    assert L.synax_plan_create(8, 64, 20.0, (dbl * 1)(-1.0), 1, obs, ctypes.byref(h)) == INVALID
    assert L.synax_plan_create(8, 64, 20.0, fr, 1, (dbl * 3)(float("inf"), 0, 0), ctypes.byref(h)) == INVALID
    assert L.synax_plan_create(8, 64, 20.0, fr, 1, obs, None) == INVALID

    plan = sx.Plan(8, 64, 20.0, [23e9])
    launches0 = plan.stats()["launches"]
    aux = np.array([2.1e-4, 5, 1, 3, 0.03, 20, 1], dtype=np.float32)
    model = sx.Model("disc4", aux=aux)
    params = torch.zeros((1, 4), device="cuda")
    I = torch.zeros((1, 1, plan.npix), device="cuda")
    vp = lambda t: ctypes.c_void_p(t.data_ptr())  # noqa: E731
    m = ctypes.byref(model.c)
    assert L.synax_forward(None, m, vp(params), 1, vp(I), vp(I), vp(I), None) == INVALID
    assert L.synax_forward(plan.h, None, vp(params), 1, vp(I), vp(I), vp(I), None) == INVALID
    assert L.synax_forward(plan.h, m, None, 1, vp(I), vp(I), vp(I), None) == INVALID
    assert L.synax_forward(plan.h, m, vp(params), 0, vp(I), vp(I), vp(I), None) == INVALID
    assert L.synax_forward(plan.h, m, vp(params), 1, None, vp(I), vp(I), None) == INVALID
    assert L.synax_vjp(plan.h, m, vp(params), 1, vp(I), vp(I), vp(I), None, None) == INVALID
    wrong = sx.Model("disc4", aux=aux)
    wrong.c.n_params = 5
    assert L.synax_forward(plan.h, ctypes.byref(wrong.c), vp(params), 1, vp(I), vp(I), vp(I), None) == INVALID
    noaux = sx.Model("disc4", aux=None)
    assert L.synax_forward(plan.h, ctypes.byref(noaux.c), vp(params), 1, vp(I), vp(I), vp(I), None) == INVALID
    unk = sx.Model("disc4", aux=aux)
    unk.c.kind = 9
    assert L.synax_forward(plan.h, ctypes.byref(unk.c), vp(params), 1, vp(I), vp(I), vp(I), None) == INVALID
    grid = sx.Model("grid_b", aux=aux, grid_shape=(4, 4, 4), box=(40, 40, 8))
    gp = torch.zeros((4, 4, 4, 3), device="cuda")
    assert L.synax_forward(plan.h, ctypes.byref(grid.c), vp(gp), 2, vp(I), vp(I), vp(I), None) == INVALID
    small = sx.Model("grid_b", aux=aux, grid_shape=(1, 4, 4), box=(40, 40, 8))
    assert L.synax_forward(plan.h, ctypes.byref(small.c), vp(gp), 1, vp(I), vp(I), vp(I), None) == INVALID
    assert L.synax_plan_set_option(plan.h, b"nonsense", 1.0) == INVALID
    assert L.synax_plan_set_option(plan.h, b"lanes", 3.0) == INVALID
    assert plan.stats()["launches"] == launches0          # nothing was launched by any of the above
    with pytest.raises(sx.SynaxError, match="SYNAX_ERR_INVALID_ARG"):
        sx.forward(plan, noaux, params)               # the binding turns the status into an exception
    plan.close()


@pytest.mark.gpu
def test_calls_are_asynchronous_on_the_given_stream():
    import torch
    import paper_2410_01136_b200 as sx
    from harness import workloads as wl
    w = wl.config(1).scaled(nside=16, n_los=128)
    plan = sx.Plan(w.nside, w.n_los, w.s_max, w.freqs)
    model = sx.Model("disc4", aux=w.aux)
    params = torch.from_numpy(w.params).cuda()
    ref = [t.clone() for t in sx.forward(plan, model, params)]
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        out = sx.forward(plan, model, params)
    s.synchronize()
    assert all(torch.equal(a, b) for a, b in zip(ref, out))
    plan.close()
