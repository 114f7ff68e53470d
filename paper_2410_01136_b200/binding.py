"""ctypes binding of libsynax.so -- same names and argument order as include/synax.h.

PyTorch is used for device memory and streams only.  Nothing is computed here.
"""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Optional, Sequence

import numpy as np

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libsynax.so"

STATUS = {0: "SYNAX_OK", 1: "SYNAX_ERR_INVALID_ARG", 2: "SYNAX_ERR_UNSUPPORTED", 3: "SYNAX_ERR_CUDA",
          4: "SYNAX_ERR_ALLOC"}
KINDS = {"disc4": 0, "full16": 1, "grid_b": 2, "uniform": 3, "stack16": 4}

# every symbol include/synax.h declares
exported_symbols = ("synax_plan_create", "synax_plan_create_shard", "synax_plan_create_strided", "synax_plan_destroy", "synax_plan_npix", "synax_plan_set_box", "synax_plan_set_option",
                    "synax_plan_directions", "synax_forward", "synax_vjp", "synax_forward_f64", "synax_vjp_f64", "synax_vjp_f64_noalloc", "synax_forward_host", "synax_vjp_host", "synax_loglike_vjp", "synax_adam_step",
                    "synax_plan_stats", "synax_last_error", "synax_version")


class SynaxError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS.get(status, status)}: {message}")
        self.status = status


class _CModel(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("n_params", ctypes.c_int32), ("aux", ctypes.POINTER(ctypes.c_float)),
                ("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
                ("lx", ctypes.c_double), ("ly", ctypes.c_double), ("lz", ctypes.c_double),
                ("ne_grid", ctypes.c_void_p), ("ne_n", ctypes.c_int32 * 3), ("ne_l", ctypes.c_double * 3),
                ("n0_grid", ctypes.c_void_p), ("n0_n", ctypes.c_int32 * 3), ("n0_l", ctypes.c_double * 3)]


_lib = None


def load_library() -> ctypes.CDLL:
    """Load the in-tree CUDA library; raise loudly when it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2410_01136_b200.build` "
                          "(nvcc, sm_100a).  There is no CPU fallback.")
    L = ctypes.CDLL(str(_LIB_PATH))
    vp, i32, i64, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
    L.synax_plan_create.argtypes = [i32, i32, dbl, ctypes.POINTER(dbl), i32, ctypes.POINTER(dbl), ctypes.POINTER(vp)]
    L.synax_plan_create.restype = ctypes.c_int
    L.synax_plan_create_shard.argtypes = [i32, i32, dbl, ctypes.POINTER(dbl), i32, ctypes.POINTER(dbl), i64, i64,
                                          ctypes.POINTER(vp)]
    L.synax_plan_create_shard.restype = ctypes.c_int
    L.synax_plan_create_strided.argtypes = [i32, i32, dbl, ctypes.POINTER(dbl), i32, ctypes.POINTER(dbl), i64, i64, i64,
                                            ctypes.POINTER(vp)]
    L.synax_plan_create_strided.restype = ctypes.c_int
    L.synax_plan_destroy.argtypes = [vp]
    L.synax_plan_destroy.restype = ctypes.c_int
    L.synax_plan_npix.argtypes = [vp]
    L.synax_plan_npix.restype = i64
    L.synax_plan_set_box.argtypes = [vp, ctypes.POINTER(dbl)]
    L.synax_plan_set_box.restype = ctypes.c_int
    L.synax_plan_set_option.argtypes = [vp, ctypes.c_char_p, dbl]
    L.synax_plan_set_option.restype = ctypes.c_int
    L.synax_plan_directions.argtypes = [vp, vp, vp]
    L.synax_plan_directions.restype = ctypes.c_int
    L.synax_plan_stats.argtypes = [vp, ctypes.POINTER(i64)]
    L.synax_plan_stats.restype = ctypes.c_int
    fwd = [vp, ctypes.POINTER(_CModel), vp, i32, vp, vp, vp, vp]
    bwd = [vp, ctypes.POINTER(_CModel), vp, i32, vp, vp, vp, vp, vp]
    for name, at in (("synax_forward", fwd), ("synax_forward_host", fwd), ("synax_vjp", bwd), ("synax_vjp_host", bwd),
                     ("synax_forward_f64", fwd), ("synax_vjp_f64", bwd), ("synax_vjp_f64_noalloc", bwd)):
        getattr(L, name).argtypes = at
        getattr(L, name).restype = ctypes.c_int
    L.synax_loglike_vjp.argtypes = [vp, ctypes.POINTER(_CModel), vp, i32, vp, vp, vp, ctypes.POINTER(dbl), vp, vp, vp]
    L.synax_loglike_vjp.restype = ctypes.c_int
    L.synax_adam_step.argtypes = [vp, vp, vp, vp, i64, dbl, dbl, dbl, dbl, i32, i32, vp]
    L.synax_adam_step.restype = ctypes.c_int
    L.synax_last_error.restype = ctypes.c_char_p
    L.synax_version.restype = ctypes.c_char_p
    _lib = L
    return L


def _check(rc: int):
    if rc != 0:
        raise SynaxError(rc, load_library().synax_last_error().decode())


class Model:
    """Mirror of `synax_model`.  kind: 'disc4' | 'full16' | 'grid_b' | 'uniform'."""

    def __init__(self, kind: str, aux: Optional[Sequence[float]] = None, grid_shape=None, box=None,
                 ne_grid=None, ne_box=None, n0_grid=None, n0_box=None):
        """ne_grid / n0_grid: contiguous float32 CUDA tensors [nx][ny][nz] over boxes ne_box / n0_box (kpc), replacing the
        analytic n_e / N_0 discs of a 'disc4' or 'grid_b' model (kept alive by this object)."""
        self.kind = kind
        self._grids = (ne_grid, n0_grid)
        self._aux = None if aux is None else np.ascontiguousarray(np.asarray(aux, dtype=np.float32))
        c = _CModel()
        c.kind = KINDS[kind]
        if kind == "grid_b":
            c.nx, c.ny, c.nz = (int(v) for v in grid_shape)
            c.lx, c.ly, c.lz = (float(v) for v in box)
            c.n_params = c.nx * c.ny * c.nz * 3
        else:
            c.n_params = {"disc4": 4, "full16": 16, "uniform": 6, "stack16": 16}[kind]
        c.aux = None if self._aux is None else self._aux.ctypes.data_as(ctypes.POINTER(ctypes.c_float))
        for name, g, b in (("ne", ne_grid, ne_box), ("n0", n0_grid, n0_box)):
            if g is None:
                continue
            if not (g.is_cuda and g.is_contiguous() and g.dim() == 3 and str(g.dtype) == "torch.float32"):
                raise TypeError(f"{name}_grid must be a contiguous float32 CUDA tensor [nx][ny][nz]")
            setattr(c, f"{name}_grid", g.data_ptr())
            for a in range(3):
                getattr(c, f"{name}_n")[a] = int(g.shape[a])
                getattr(c, f"{name}_l")[a] = float(b[a])
        self.c = c

    @property
    def n_params(self) -> int:
        return int(self.c.n_params)


class Plan:
    """synax_plan_create / synax_plan_create_shard (pix_range=(begin, count)) / synax_plan_create_strided
    (pix_range=(begin, count), pix_stride=n: pixels begin + i * n) / synax_plan_destroy.
    pool_release_threshold_mb: option of the same name (include/synax.h).  Calls cut their scratch from a workspace the plan
    keeps; only what exceeds 256 MB (the host entry points' staging of large maps) and calls inside a stream capture go to the
    device's stream-ordered memory pool, whose default is to give everything back at a synchronisation (the next pool
    allocation then waits ~0.23 ms).  Process-wide for the device, hence opt-in."""

    def __init__(self, nside: int, n_los: int, s_max: float, freqs, observer=(-8.3, 0.0, 0.006), pix_range=None, pix_stride=1,
                 pool_release_threshold_mb=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("synax needs a CUDA device (B200); there is no CPU fallback")
        L = load_library()
        torch.cuda.current_stream()  # make sure the CUDA context of the current device exists
        torch.zeros(1, device="cuda")
        f = np.ascontiguousarray(np.asarray(freqs, dtype=np.float64).ravel())
        o = np.ascontiguousarray(np.asarray(observer, dtype=np.float64).ravel())
        h = ctypes.c_void_p()
        fp, op = f.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), o.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
        if pix_range is None:
            _check(L.synax_plan_create(int(nside), int(n_los), float(s_max), fp, int(f.size), op, ctypes.byref(h)))
        elif int(pix_stride) == 1:
            _check(L.synax_plan_create_shard(int(nside), int(n_los), float(s_max), fp, int(f.size), op,
                                             int(pix_range[0]), int(pix_range[1]), ctypes.byref(h)))
        else:
            _check(L.synax_plan_create_strided(int(nside), int(n_los), float(s_max), fp, int(f.size), op,
                                               int(pix_range[0]), int(pix_stride), int(pix_range[1]), ctypes.byref(h)))
        self.pix_range = None if pix_range is None else (int(pix_range[0]), int(pix_range[1]))
        self.pix_stride = int(pix_stride)
        self.device = int(torch.cuda.current_device())
        self.h = h
        self.nside, self.n_los, self.s_max, self.freqs = int(nside), int(n_los), float(s_max), f
        self.n_freq = int(f.size)
        self.npix = int(L.synax_plan_npix(h))
        if pool_release_threshold_mb is not None:
            self.set_option("pool_release_threshold_mb", float(pool_release_threshold_mb))

    def set_box(self, box):
        """synax_plan_set_box: integrate from the observer to the faces of a box (lx, ly, lz kpc); None = fixed s_max."""
        if box is None:
            _check(load_library().synax_plan_set_box(self.h, None))
        else:
            b = (ctypes.c_double * 3)(*[float(v) for v in box])
            _check(load_library().synax_plan_set_box(self.h, b))

    def set_option(self, key: str, value: float):
        _check(load_library().synax_plan_set_option(self.h, key.encode(), float(value)))

    def directions(self):
        import torch
        out = torch.empty((self.npix, 4), dtype=torch.float64, device="cuda")
        _check(load_library().synax_plan_directions(self.h, out.data_ptr(), _stream()))
        return out

    def stats(self):
        out = (ctypes.c_int64 * 2)()
        _check(load_library().synax_plan_stats(self.h, out))
        return {"launches": int(out[0]), "escalated": int(out[1])}

    def close(self):
        if getattr(self, "h", None):
            load_library().synax_plan_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev_f32(t, what, numel=None):
    """Pointer of a contiguous float32 CUDA tensor; the C ABI cannot check sizes, so the element count is checked here."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{what} must be a contiguous float32 CUDA tensor")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{what} has {t.numel()} elements, expected {numel}")
    return ctypes.c_void_p(t.data_ptr())


def _check_device(plan, *tensors):
    """The plan lives on the device that was current when it was created: every tensor and the current device must match."""
    import torch
    if torch.cuda.current_device() != plan.device:
        raise RuntimeError(f"the plan was created on cuda:{plan.device}, the current device is cuda:{torch.cuda.current_device()}")
    for t in tensors:
        if t is not None and t.device.index != plan.device:
            raise ValueError(f"tensor on {t.device}, the plan is on cuda:{plan.device}")


def _batch_of(model: Model, params) -> int:
    if model.kind == "grid_b":
        if params.numel() != model.n_params:
            raise ValueError("grid tensor does not match the model's grid shape")
        return 1
    if params.shape[-1] != model.n_params:
        raise ValueError(f"params last dim {params.shape[-1]} != n_params {model.n_params}")
    return int(params.numel() // model.n_params)


def forward(plan: Plan, model: Model, params, out=None):
    """synax_forward: params CUDA fp32 [batch][P] (or the grid) -> (I, Q, U) CUDA fp32 [batch][n_freq][npix]."""
    import torch
    batch = _batch_of(model, params)
    if out is None:
        out = tuple(torch.empty((batch, plan.n_freq, plan.npix), dtype=torch.float32, device=params.device) for _ in range(3))
    I, Q, U = out
    n = batch * plan.n_freq * plan.npix if batch * plan.npix < 2 ** 31 else None   # (the library rejects larger calls itself)
    _check_device(plan, params, I, Q, U)
    _check(load_library().synax_forward(plan.h, ctypes.byref(model.c), _dev_f32(params, "params"), batch,
                                        _dev_f32(I, "I", n), _dev_f32(Q, "Q", n), _dev_f32(U, "U", n), _stream()))
    return I, Q, U


def vjp(plan: Plan, model: Model, params, dI, dQ, dU, out=None):
    """synax_vjp: cotangent maps CUDA fp32 [batch][n_freq][npix] (None = zeros) -> grad CUDA fp32 like params."""
    import torch
    batch = _batch_of(model, params)
    if out is None:
        out = torch.empty_like(params)
    n = batch * plan.n_freq * plan.npix
    ptr = lambda t, w: ctypes.c_void_p(None) if t is None else _dev_f32(t, w, n)  # noqa: E731
    _check_device(plan, params, dI, dQ, dU, out)
    _check(load_library().synax_vjp(plan.h, ctypes.byref(model.c), _dev_f32(params, "params"), batch,
                                    ptr(dI, "dI"), ptr(dQ, "dQ"), ptr(dU, "dU"), _dev_f32(out, "grad", params.numel()), _stream()))
    return out


def _dev_f64(t, what, numel=None):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{what} must be a contiguous float64 CUDA tensor")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{what} has {t.numel()} elements, expected {numel}")
    return ctypes.c_void_p(t.data_ptr())


def forward_f64(plan: Plan, model: Model, params, out=None):
    """synax_forward_f64 (the paper's all-float64 arithmetic): params CUDA float64 [batch][P] -> (I, Q, U) CUDA float64."""
    import torch
    batch = _batch_of(model, params)
    n = batch * plan.n_freq * plan.npix
    if out is None:
        out = tuple(torch.empty((batch, plan.n_freq, plan.npix), dtype=torch.float64, device=params.device) for _ in range(3))
    I, Q, U = out
    _check(load_library().synax_forward_f64(plan.h, ctypes.byref(model.c), _dev_f64(params, "params"), batch,
                                            _dev_f64(I, "I", n), _dev_f64(Q, "Q", n), _dev_f64(U, "U", n), _stream()))
    return I, Q, U


def vjp_f64(plan: Plan, model: Model, params, dI, dQ, dU, out=None):
    """synax_vjp_f64: cotangent maps CUDA float64 [batch][n_freq][npix] (None = zeros) -> grad CUDA float64 like params."""
    import torch
    batch = _batch_of(model, params)
    n = batch * plan.n_freq * plan.npix
    if out is None:
        out = torch.empty_like(params)
    ptr = lambda t, w: ctypes.c_void_p(None) if t is None else _dev_f64(t, w, n)  # noqa: E731
    _check(load_library().synax_vjp_f64(plan.h, ctypes.byref(model.c), _dev_f64(params, "params"), batch,
                                        ptr(dI, "dI"), ptr(dQ, "dQ"), ptr(dU, "dU"), _dev_f64(out, "grad", params.numel()), _stream()))
    return out


def vjp_f64_noalloc(plan: Plan, model: Model, params, dI, dQ, dU, out):
    """synax_vjp_f64_noalloc: synax_vjp_f64 on the library's fixed scratch array -- no allocation anywhere, so `out` (CUDA
    float64 like params) is required.  SynaxError (SYNAX_ERR_UNSUPPORTED) when the call needs more than the 4 MiB array."""
    batch = _batch_of(model, params)
    n = batch * plan.n_freq * plan.npix
    ptr = lambda t, w: ctypes.c_void_p(None) if t is None else _dev_f64(t, w, n)  # noqa: E731
    _check(load_library().synax_vjp_f64_noalloc(plan.h, ctypes.byref(model.c), _dev_f64(params, "params"), batch,
                                                ptr(dI, "dI"), ptr(dQ, "dQ"), ptr(dU, "dU"),
                                                _dev_f64(out, "grad", params.numel()), _stream()))
    return out


def loglike_vjp(plan: Plan, model: Model, params, I_obs, Q_obs, U_obs, inv_var, out=None):
    """synax_loglike_vjp: observed maps CUDA fp32 [n_freq][npix] (None = not in the likelihood), inv_var = 3 weights
    1/sigma^2 -> (logL CUDA float64 [batch], grad CUDA fp32 like params)."""
    import torch
    batch = _batch_of(model, params)
    if out is None:
        out = (torch.empty((batch,), dtype=torch.float64, device=params.device), torch.empty_like(params))
    logL, grad = out
    if not (logL.is_cuda and logL.dtype == torch.float64 and logL.is_contiguous() and logL.numel() == batch):
        raise TypeError("logL must be a contiguous float64 CUDA tensor [batch]")
    w = (ctypes.c_double * 3)(*[float(v) for v in inv_var])
    ptr = lambda t, n: ctypes.c_void_p(None) if t is None else _dev_f32(t, n)  # noqa: E731
    for t in (I_obs, Q_obs, U_obs):
        if t is not None and t.numel() != plan.n_freq * plan.npix:
            raise ValueError("observed maps must have n_freq * npix elements")
    _check(load_library().synax_loglike_vjp(plan.h, ctypes.byref(model.c), _dev_f32(params, "params"), batch,
                                            ptr(I_obs, "I_obs"), ptr(Q_obs, "Q_obs"), ptr(U_obs, "U_obs"), w,
                                            ctypes.c_void_p(logL.data_ptr()), _dev_f32(grad, "grad"), _stream()))
    return logL, grad


def adam_step(theta, grad, m, v, t: int, lr=1e-3, beta1=0.9, beta2=0.999, eps=1e-8, maximize=False):
    """synax_adam_step: in-place ADAM update of the CUDA fp32 tensor `theta` (m, v: moment buffers, zero at t = 1)."""
    n = theta.numel()
    for x, name in ((grad, "grad"), (m, "m"), (v, "v")):
        if x.numel() != n:
            raise ValueError(f"{name} must have as many elements as theta")
    _check(load_library().synax_adam_step(_dev_f32(theta, "theta"), _dev_f32(grad, "grad"), _dev_f32(m, "m"), _dev_f32(v, "v"),
                                          n, float(lr), float(beta1), float(beta2), float(eps), int(t), int(bool(maximize)),
                                          _stream()))
    return theta


def _host_f32(a, what, size=None):
    if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags.c_contiguous):
        raise TypeError(f"{what} must be a C-contiguous float32 numpy array")
    if size is not None and a.size != size:
        raise ValueError(f"{what} has {a.size} elements, expected {size}")
    return ctypes.c_void_p(a.ctypes.data)


def forward_host(plan: Plan, model: Model, params: np.ndarray, out=None):
    """synax_forward_host: numpy float32 in, numpy float32 (I, Q, U) out; copies inside the call."""
    batch = 1 if model.kind == "grid_b" else int(params.size // model.n_params)
    if out is None:
        out = tuple(np.empty((batch, plan.n_freq, plan.npix), dtype=np.float32) for _ in range(3))
    I, Q, U = out
    n = batch * plan.n_freq * plan.npix
    _check(load_library().synax_forward_host(plan.h, ctypes.byref(model.c), _host_f32(params, "params", batch * model.n_params), batch,
                                             _host_f32(I, "I", n), _host_f32(Q, "Q", n), _host_f32(U, "U", n), _stream()))
    return I, Q, U


def vjp_host(plan: Plan, model: Model, params: np.ndarray, dI, dQ, dU, out=None):
    """synax_vjp_host: numpy float32 in/out; copies inside the call."""
    batch = 1 if model.kind == "grid_b" else int(params.size // model.n_params)
    if out is None:
        out = np.empty_like(params)
    n = batch * plan.n_freq * plan.npix
    ptr = lambda a, w: ctypes.c_void_p(None) if a is None else _host_f32(a, w, n)  # noqa: E731
    _check(load_library().synax_vjp_host(plan.h, ctypes.byref(model.c), _host_f32(params, "params", batch * model.n_params), batch,
                                         ptr(dI, "dI"), ptr(dQ, "dQ"), ptr(dU, "dU"), _host_f32(out, "grad", params.size), _stream()))
    return out
