"""ctypes wrapper around the float64 CPU oracle (oracle/synax_oracle.cpp).

TEST INFRASTRUCTURE ONLY: tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2410_01136_b200`` and the CUDA library imports nothing from here.

Every array crossing this boundary is float64 on the host.  Inputs generated as float32 (what the
GPU receives) are promoted to float64 here, never re-derived.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "synax_oracle.cpp"
_LIB = _HERE / "liboracle.so"

KINDS = {"disc4": 0, "full16": 1, "grid_b": 2, "uniform": 3, "stack16": 4}
N_PARAMS = {"disc4": 4, "full16": 16, "uniform": 6, "stack16": 16}


def build(force: bool = False) -> Path:
    """Compile liboracle.so with g++ -O2 -fopenmp (no fast-math)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-ffp-contract=off",
               "-o", str(tmp), str(_SRC)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(str(build()))
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


class Model:
    """kind: 'disc4' | 'full16' | 'grid_b' | 'uniform'.

    params: [batch][P] (or [P]); grid_b: array [nx][ny][nz][3].  aux: 7 values
    (C0,h_r,h_z,alpha,ne0,h_er,h_ez) for disc4/grid_b; uniform: optional [R0] toy-sphere radius.
    box: (lx,ly,lz) kpc for grid_b.
    """

    def __init__(self, kind, params, aux=None, box=None):
        self.kind = kind
        self.k = KINDS[kind]
        p = _f64(params)
        if kind == "grid_b":
            assert p.ndim == 4 and p.shape[3] == 3
            self.gdim = np.asarray(p.shape[:3], dtype=np.int64)
            self.gbox = _f64(box)
            self.batch = 1
            self.n_params = int(p.size)
            self.params = p.reshape(1, -1)
        else:
            self.gdim = None
            self.gbox = None
            self.params = np.atleast_2d(p)
            self.batch, self.n_params = self.params.shape
            assert self.n_params == N_PARAMS[kind]
        self.aux = None if aux is None else _f64(aux)
        if kind in ("disc4", "grid_b", "stack16"):
            assert self.aux is not None and self.aux.size == 7


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(ctypes.c_int(int(n)))


def pix2ang_ring(nside: int, pix):
    """RING pixel centres: returns (z=cos theta, phi) float64 arrays."""
    pix = np.atleast_1d(np.asarray(pix, dtype=np.int64))
    z = np.empty(pix.size)
    phi = np.empty(pix.size)
    zz, pp = ctypes.c_double(), ctypes.c_double()
    L = lib()
    for k, p in enumerate(pix):
        rc = L.oracle_pix2ang_ring(ctypes.c_int64(nside), ctypes.c_int64(int(p)), ctypes.byref(zz), ctypes.byref(pp))
        if rc:
            raise ValueError("bad nside/pix")
        z[k], phi[k] = zz.value, pp.value
    return z, phi


def constants(nu, btrans_gauss, n0, alpha):
    """dict: K_F per kpc, j_I, j_P (CGS), T_RJ, digamma(alpha), dlnjI/dalpha, dlnjP/dalpha."""
    out = np.zeros(7)
    lib().oracle_constants(ctypes.c_double(nu), ctypes.c_double(btrans_gauss), ctypes.c_double(n0),
                           ctypes.c_double(alpha), _p(out))
    return dict(K_F=out[0], j_I=out[1], j_P=out[2], T_RJ=out[3], digamma=out[4], dlnjI=out[5], dlnjP=out[6])


def eval_fields(model: Model, r, observer=(-8.3, 0.0, 0.006), b=0):
    r = _f64(r).reshape(-1, 3)
    n = r.shape[0]
    B = np.zeros((n, 3)); N0 = np.zeros(n); ne = np.zeros(n); al = np.zeros(n)
    obs = _f64(observer)
    lib().oracle_eval_fields(ctypes.c_int(model.k), _p(model.params[b]), _p(model.aux), _p(model.gdim),
                             _p(model.gbox), _p(obs), ctypes.c_int64(n), _p(r), _p(B), _p(N0), _p(ne), _p(al))
    return B, N0, ne, al


class scalar_grids:
    """Context manager: n_e and / or N_0 of the DISC4 and GRID_B models come from regular grids [nx][ny][nz] over
    boxes (lx, ly, lz) centred on the Galactic centre, trilinear, zero outside."""

    def __init__(self, ne=None, ne_box=None, n0=None, n0_box=None):
        self.items = []
        for which, g, b in ((0, ne, ne_box), (1, n0, n0_box)):
            if g is not None:
                g = _f64(g)
                assert g.ndim == 3
                self.items.append((which, g, np.asarray(g.shape, dtype=np.int64), _f64(b)))

    def __enter__(self):
        for which, g, dim, box in self.items:
            if lib().oracle_set_scalar_grid(ctypes.c_int(which), _p(g), _p(dim), _p(box)):
                raise ValueError("bad scalar grid")
        return self

    def __exit__(self, *a):
        for which, *_ in self.items:
            lib().oracle_set_scalar_grid(ctypes.c_int(which), None, None, None)


class _clip:
    """Context manager: integrate from the observer to the faces of `box` (lx, ly, lz kpc, centred on the Galactic
    centre) instead of over the fixed [0, s_max]."""

    def __init__(self, box, observer):
        self.box = None if box is None else _f64(box)
        self.obs = _f64(observer)

    def __enter__(self):
        if self.box is not None and lib().oracle_set_clip_box(_p(self.box), _p(self.obs)):
            raise ValueError("observer must be strictly inside the clip box")

    def __exit__(self, *a):
        lib().oracle_set_clip_box(None, None)


def exit_distance(observer, l, b, box):
    lib().oracle_exit_distance.restype = ctypes.c_double
    return float(lib().oracle_exit_distance(_p(_f64(observer)), ctypes.c_double(l), ctypes.c_double(b), _p(_f64(box))))


def forward_dir(model: Model, l, b, n_los, s_max, freqs, observer=(-8.3, 0.0, 0.006), batch_index=0, clip_box=None):
    """I,Q,U [n_freq] (K) of one sightline towards Galactic (l,b) [rad]."""
    freqs = _f64(freqs).ravel()
    obs = _f64(observer)
    with _clip(clip_box, observer):
        return _forward_dir(model, l, b, n_los, s_max, freqs, obs, batch_index)


def _forward_dir(model, l, b, n_los, s_max, freqs, obs, batch_index):
    I = np.zeros(freqs.size); Q = np.zeros(freqs.size); U = np.zeros(freqs.size)
    lib().oracle_forward_dir(ctypes.c_int(model.k), _p(model.params[batch_index]), _p(model.aux), _p(model.gdim),
                             _p(model.gbox), ctypes.c_double(l), ctypes.c_double(b), ctypes.c_int64(n_los),
                             ctypes.c_double(s_max), _p(freqs), ctypes.c_int(freqs.size), _p(obs), _p(I), _p(Q), _p(U))
    return I, Q, U


def forward(model: Model, nside, n_los, s_max, freqs, observer=(-8.3, 0.0, 0.006), pix=None, clip_box=None):
    """I,Q,U maps float64 [batch][n_freq][n_out] in Kelvin; pix=None -> all 12 nside^2 pixels."""
    with _clip(clip_box, observer):
        return _forward(model, nside, n_los, s_max, freqs, observer, pix)


def _forward(model, nside, n_los, s_max, freqs, observer, pix):
    freqs = _f64(freqs).ravel()
    obs = _f64(observer)
    if pix is not None:
        pix = np.ascontiguousarray(np.asarray(pix, dtype=np.int64))
    n_out = 12 * nside * nside if pix is None else pix.size
    shape = (model.batch, freqs.size, n_out)
    I = np.zeros(shape); Q = np.zeros(shape); U = np.zeros(shape)
    rc = lib().oracle_forward(ctypes.c_int(model.k), _p(model.params), ctypes.c_int64(model.n_params), _p(model.aux),
                              _p(model.gdim), _p(model.gbox), ctypes.c_int64(model.batch), ctypes.c_int64(nside),
                              ctypes.c_int64(n_los), ctypes.c_double(s_max), _p(freqs), ctypes.c_int(freqs.size),
                              _p(obs), _p(pix), ctypes.c_int64(0 if pix is None else pix.size), _p(I), _p(Q), _p(U))
    if rc:
        raise ValueError("oracle_forward: invalid argument")
    return I, Q, U


def vjp(model: Model, nside, n_los, s_max, freqs, dI, dQ, dU, observer=(-8.3, 0.0, 0.006), pix=None, clip_box=None):
    """grad float64 [batch][P] (grid_b: [nx][ny][nz][3]) for cotangent maps [batch][n_freq][n_out]."""
    with _clip(clip_box, observer):
        return _vjp(model, nside, n_los, s_max, freqs, dI, dQ, dU, observer, pix)


def _vjp(model, nside, n_los, s_max, freqs, dI, dQ, dU, observer, pix):
    freqs = _f64(freqs).ravel()
    obs = _f64(observer)
    if pix is not None:
        pix = np.ascontiguousarray(np.asarray(pix, dtype=np.int64))
    n_out = 12 * nside * nside if pix is None else pix.size
    shape = (model.batch, freqs.size, n_out)
    cots = []
    for c in (dI, dQ, dU):
        if c is None:
            cots.append(None)
        else:
            c = _f64(c)
            assert c.size == int(np.prod(shape)), (c.shape, shape)
            cots.append(c)
    grad = np.zeros((model.batch, model.n_params))
    rc = lib().oracle_vjp(ctypes.c_int(model.k), _p(model.params), ctypes.c_int64(model.n_params), _p(model.aux),
                          _p(model.gdim), _p(model.gbox), ctypes.c_int64(model.batch), ctypes.c_int64(nside),
                          ctypes.c_int64(n_los), ctypes.c_double(s_max), _p(freqs), ctypes.c_int(freqs.size),
                          _p(obs), _p(pix), ctypes.c_int64(0 if pix is None else pix.size),
                          _p(cots[0]), _p(cots[1]), _p(cots[2]), _p(grad))
    if rc:
        raise ValueError("oracle_vjp: invalid argument")
    if model.kind == "grid_b":
        return grad.reshape(tuple(model.gdim) + (3,))
    return grad


def loglike_vjp(model: Model, nside, n_los, s_max, freqs, I_obs, Q_obs, U_obs, inv_var, observer=(-8.3, 0.0, 0.006)):
    """Gaussian pixel log-likelihood of Eq.(15) and its gradient, written out as the
    composition it is: maps = forward(theta); logL[b] = -1/2 sum_k w_k sum_{f,p} (X_k - X_k_obs)^2 over the Stokes
    maps k with an observation (None = not in the likelihood; the paper uses Q and U with w = 1/sigma^2,
    sigma = 1 mK); d logL / d theta = VJP with cotangent -w_k (X_k - X_k_obs).  Observations [n_freq][npix] are
    shared by all batch elements.  Returns (logL float64 [batch], grad like vjp())."""
    maps = forward(model, nside, n_los, s_max, freqs, observer=observer)
    logL = np.zeros(model.batch)
    cots = []
    for X, obs, w in zip(maps, (I_obs, Q_obs, U_obs), inv_var):
        if obs is None or w == 0.0:
            cots.append(None)
            continue
        r = X - _f64(obs).reshape((1,) + X.shape[1:])
        logL += -0.5 * float(w) * np.sum(r * r, axis=(1, 2))
        cots.append(-float(w) * r)
    grad = vjp(model, nside, n_los, s_max, freqs, cots[0], cots[1], cots[2], observer=observer)
    return logL, grad


def adam_step(theta, grad, m, v, t, lr=1e-3, beta1=0.9, beta2=0.999, eps=1e-8, maximize=False):
    """ADAM update of Kingma & Ba (2015), Algorithm 1, as used for the paper's field-level fits:
    returns (theta, m, v) after step t (float64; inputs untouched)."""
    g = -_f64(grad) if maximize else _f64(grad)
    m = beta1 * _f64(m) + (1.0 - beta1) * g
    v = beta2 * _f64(v) + (1.0 - beta2) * g * g
    mhat = m / (1.0 - beta1 ** t)
    vhat = v / (1.0 - beta2 ** t)
    return _f64(theta) - lr * mhat / (np.sqrt(vhat) + eps), m, v
