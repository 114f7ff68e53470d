"""Seeded synthetic inputs for the five BASELINE.json workloads.

This module holds NONE of the method's arithmetic (no emissivity, no Faraday depth, no
integration): it only draws numbers and lays them out.  The tests and bench.py hand the SAME
float32 arrays to the CUDA library and (promoted to float64) to the oracle; neither side imports
the other.  RNG = numpy.random.Generator(PCG64(seed)); values are generated in float64 and
rounded ONCE to float32.

The paper measures on mock skies built from WMAP B / N_0 fields plus the YMW16 n_e model and on the
Haslam map; neither is available here, so these inputs take the paper's
shapes (NSIDE 64..256, N_int 256..1024, a 128x128x32 B grid, 4- and 16-parameter models) and stand
in for them.

The config-3 grid is "Gaussian random field + logarithmic-spiral pattern" (BASELINE.json); the
spiral pattern is written out here as a data recipe (`spiral_pattern`) so that both sides receive
the finished grid as opaque input.
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np

OBSERVER = (-8.3, 0.0, 0.006)  # kpc

DEG = np.pi / 180.0

# DISC4 nominal parameters (b0 [uG], psi0, psi1, chi0 [rad]) -- BASELINE.json config 0
DISC4_NOMINAL = np.array([6.0, 27.0 * DEG, 0.9 * DEG, 25.0 * DEG])
# aux = (C0, h_r, h_z, alpha, ne0, h_er, h_ez) -- SURVEY.md 8(d), C-2 #9
AUX_NOMINAL = np.array([2.1038000728e-4, 5.0, 1.0, 3.0, 0.03, 20.0, 1.0])
# FULL16 nominal, order of SURVEY.md App. C
FULL16_NOMINAL = np.array([
    6.0, 27.0 * DEG, 0.9 * DEG, 25.0 * DEG, 10.0,   # disc: b0 psi0 psi1 chi0 h_b
    2.0, 1.5, 4.0, 0.4,                             # halo: B_h z_h0 r_h w_h
    2.1038000728e-4, 5.0, 1.0, 3.0,                 # CR: n0 h_r h_z p
    0.03, 20.0, 1.0,                                # n_e: ne0 h_er h_ez
])
FULL16_NAMES = ("b0", "psi0", "psi1", "chi0", "h_b", "B_h", "z_h0", "r_h", "w_h",
                "n0", "h_r", "h_z", "p", "ne0", "h_er", "h_ez")
DISC4_NAMES = ("b0", "psi0", "psi1", "chi0")
# The paper's own 16-parameter model: Table 3, (b0 [uG], psi0, psi1, chi0 [rad]) x 4 spirals,
# stacked by Eq. (16)
STACK16_TABLE3 = np.array([1.20, 0.4712, 0.0157, 0.4363,
                           3.50, 0.6457, 0.5393, 0.6108,
                           7.70, 1.1693, 1.0629, 1.1344,
                           5.70, 1.6930, 1.5865, 1.6580])


@dataclasses.dataclass
class Workload:
    name: str
    kind: str                    # 'disc4' | 'full16' | 'grid_b' | 'uniform'
    nside: int
    n_los: int
    s_max: float                 # kpc
    freqs: np.ndarray            # float64 [n_freq], Hz
    params: np.ndarray           # float32 [batch][P]  or grid [nx][ny][nz][3]
    aux: Optional[np.ndarray]    # float32 [7] or None
    box: Optional[tuple] = None  # grid_b: (lx, ly, lz) kpc
    cot_seed: int = 0
    observer: tuple = OBSERVER
    clip_box: Optional[tuple] = None  # (lx, ly, lz) kpc: integrate observer -> box face instead of [0, s_max]
    ne_grid: Optional[np.ndarray] = None   # float32 [nx][ny][nz]: gridded n_e replacing the analytic disc (disc4 / grid_b)
    ne_box: Optional[tuple] = None
    n0_grid: Optional[np.ndarray] = None   # the same for the CR density N_0
    n0_box: Optional[tuple] = None

    @property
    def npix(self) -> int:
        return 12 * self.nside * self.nside

    @property
    def batch(self) -> int:
        return 1 if self.kind == "grid_b" else int(self.params.shape[0])

    @property
    def n_freq(self) -> int:
        return int(self.freqs.size)

    @property
    def los_samples(self) -> int:
        """LoS samples per call = npix * n_los * batch (frequencies not multiplied in)."""
        return self.npix * self.n_los * self.batch

    def cotangents(self, ones: bool = False):
        """(dI, dQ, dU), each float32 [batch][n_freq][npix]; drawn as [batch][f][Stokes][pix]."""
        shape = (self.batch, self.n_freq, 3, self.npix)
        if ones:
            c = np.ones(shape, dtype=np.float32)
        else:
            rng = np.random.Generator(np.random.PCG64(self.cot_seed))
            c = rng.standard_normal(shape).astype(np.float32)
        return (np.ascontiguousarray(c[:, :, 0]), np.ascontiguousarray(c[:, :, 1]),
                np.ascontiguousarray(c[:, :, 2]))

    def scaled(self, nside: Optional[int] = None, n_los: Optional[int] = None, batch: Optional[int] = None,
               name: Optional[str] = None) -> "Workload":
        """Same model/frequencies at a smaller map, sample count or batch (parity-test sizes)."""
        w = dataclasses.replace(self)
        if nside is not None:
            w.nside = nside
        if n_los is not None:
            w.n_los = n_los
        if batch is not None and self.kind != "grid_b":
            w.params = np.ascontiguousarray(self.params[:batch])
        w.name = name or f"{self.name}@nside{w.nside}x{w.n_los}x{w.batch}"
        return w


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))


def spiral_pattern(x, y, z, b0, psi0, psi1, chi0):
    """Logarithmic-spiral vector pattern used only to fill the config-3 grid (data recipe)."""
    rho = np.hypot(x, y)
    inside = (rho > 3.0) & (rho < 20.0)
    safe = np.where(rho > 0, rho, 1.0)
    psi = psi0 + psi1 * np.log(safe / 8.0)
    chi = chi0 * np.tanh(z)
    brho = b0 * np.cos(psi) * np.cos(chi)
    bphi = b0 * np.sin(psi) * np.cos(chi)
    bx = (brho * x - bphi * y) / safe
    by = (brho * y + bphi * x) / safe
    bz = b0 * np.sin(chi) * np.ones_like(safe)
    out = np.stack([bx, by, bz], axis=-1)
    return np.where(inside[..., None], out, 0.0)


def gaussian_random_field(shape, box, seed, rms=3.0, slope=-11.0 / 3.0):
    """Three independent Cartesian components, power ~ k^slope, total rms sqrt<|dB|^2> = rms."""
    rng = np.random.Generator(np.random.PCG64(seed))
    nx, ny, nz = shape
    k = np.meshgrid(*[2 * np.pi * np.fft.fftfreq(n, d=l / n) for n, l in zip(shape, box)], indexing="ij")
    kk = np.sqrt(k[0] ** 2 + k[1] ** 2 + k[2] ** 2)
    amp = np.zeros_like(kk)
    amp[kk > 0] = kk[kk > 0] ** (slope / 2.0)
    comps = []
    for _ in range(3):
        re = rng.standard_normal(shape)
        im = rng.standard_normal(shape)
        comps.append(np.fft.ifftn((re + 1j * im) * amp).real)
    f = np.stack(comps, axis=-1)
    f *= rms / np.sqrt(np.mean(np.sum(f * f, axis=-1)))
    return f


def grid_nodes(shape, box):
    ax = [np.linspace(-l / 2.0, l / 2.0, n) for n, l in zip(shape, box)]
    return np.meshgrid(*ax, indexing="ij")


def clumpy_disc_grid(shape, box, amp, h_r, h_z, seed, contrast=0.3):
    """Data recipe for a gridded scalar field standing in for the paper's YMW16 n_e grid (not in the
    container): an exponential disc amp * exp(-rho/h_r) / cosh^2(z/h_z) at the nodes, modulated by exp(contrast * g)
    with g a unit-variance Gaussian random field (k^-11/3), rounded once to float32."""
    X, Y, Z = grid_nodes(shape, box)
    g = gaussian_random_field(shape, box, seed, rms=np.sqrt(3.0))[..., 0]
    v = amp * np.exp(-np.hypot(X, Y) / h_r) / np.cosh(Z / h_z) ** 2 * np.exp(contrast * g)
    return _f32(v)


def config(i: int) -> Workload:
    """BASELINE.json configs[i], i = 0..4, at full size."""
    if i == 0:
        return Workload("cfg0_tiny_disc4", "disc4", 8, 64, 20.0, np.array([23e9]),
                        _f32(DISC4_NOMINAL)[None, :], _f32(AUX_NOMINAL), cot_seed=1000)
    if i == 1:
        rng = np.random.Generator(np.random.PCG64(1001))
        p = np.array([rng.uniform(3, 9), rng.uniform(15, 35) * DEG, rng.uniform(0, 2) * DEG,
                      rng.uniform(10, 40) * DEG])
        return Workload("cfg1_mid_disc4", "disc4", 64, 256, 20.0, np.array([2.4e9, 23e9, 30e9]),
                        _f32(p)[None, :], _f32(AUX_NOMINAL), cot_seed=2001)
    if i == 2:
        rng = np.random.Generator(np.random.PCG64(1002))
        u = rng.uniform(-1.0, 1.0, size=(256, 16))
        p = FULL16_NOMINAL[None, :] * (1.0 + 0.2 * u)
        return Workload("cfg2_batched_full16", "full16", 32, 256, 20.0, np.array([23e9]),
                        _f32(p), None, cot_seed=2002)
    if i == 3:
        shape, box = (128, 128, 32), (40.0, 40.0, 8.0)
        X, Y, Z = grid_nodes(shape, box)
        g = gaussian_random_field(shape, box, 1003) + spiral_pattern(X, Y, Z, *DISC4_NOMINAL)
        return Workload("cfg3_grid_b", "grid_b", 64, 512, 20.0, np.array([408e6]),
                        _f32(g), _f32(AUX_NOMINAL), box=box, cot_seed=2003)
    if i == 4:
        return Workload("cfg4_large_full16", "full16", 256, 1024, 30.0, np.geomspace(0.408e9, 30e9, 8),
                        _f32(FULL16_NOMINAL)[None, :], None, cot_seed=2004)
    raise ValueError("config index 0..4")


def stack16(nside=32, n_los=256, s_max=20.0, freqs=(2.4e9,), batch=1, seed=1016) -> Workload:
    """The paper's section 4.3 model (Eq. 16, Table 3): batch > 1 draws each vector within +-10 % of Table 3."""
    p = np.tile(STACK16_TABLE3, (batch, 1))
    if batch > 1:
        rng = np.random.Generator(np.random.PCG64(seed))
        p[1:] *= 1.0 + 0.1 * rng.uniform(-1.0, 1.0, size=(batch - 1, 16))
    return Workload("stack16_table3", "stack16", nside, n_los, s_max, np.asarray(freqs, dtype=np.float64), _f32(p),
                    _f32(AUX_NOMINAL), cot_seed=3016)


def uniform_toy(bvec=(6.0, 0.0, 0.0), n0=4.01e-5, ne=0.01, alpha=3.0, nside=8, n_los=64, s_max=4.0,
                freqs=(2.4e9,)) -> Workload:
    """Homogeneous toy of PAPER.md L123 (section 2.4): the closed-form test model."""
    p = np.array([bvec[0], bvec[1], bvec[2], n0, ne, alpha])
    return Workload("uniform_toy", "uniform", nside, n_los, s_max, np.asarray(freqs, dtype=np.float64),
                    _f32(p)[None, :], None, cot_seed=999)


# PAPER.md section 3.1 (L175-180): WMAP B with the paper's true values, WMAP N_0, n_e on a (256, 256, 64) grid (the paper's
# is the YMW16 model, not in the container: a seeded clumpy exponential disc stands in for it), NSIDE 64, N_int 512,
# 2.4 GHz (Fig. 3), integration from the observer to the faces of the (40, 40, 10) kpc box of section 2.4.
SECTION31_B = np.array([1.2, 0.4712, 0.0157, 0.4363])
SECTION31_BOX = (40.0, 40.0, 10.0)


def paper_section31(nside=64, n_los=512, ne_shape=(256, 256, 64), freqs=(2.4e9,), seed=3101) -> Workload:
    w = Workload("paper_section31", "disc4", nside, n_los, 30.0, np.asarray(freqs, dtype=np.float64),
                 _f32(SECTION31_B)[None, :], _f32(AUX_NOMINAL), cot_seed=3102, clip_box=SECTION31_BOX)
    w.ne_grid, w.ne_box = clumpy_disc_grid(ne_shape, SECTION31_BOX, 0.03, 20.0, 1.0, seed=seed), SECTION31_BOX
    return w


def section31_gridded_b(n_x, base: Workload) -> Workload:
    """The same model with B given on a (n_x, n_x, n_x / 4) grid filled from the analytic spiral at the nodes (Fig. 6
    lower panel)."""
    shape = (n_x, n_x, n_x // 4)
    X, Y, Z = grid_nodes(shape, SECTION31_BOX)
    g = spiral_pattern(X, Y, Z, *base.params[0].astype(np.float64))
    w = dataclasses.replace(base, name=f"paper_section31_gridB{n_x}", kind="grid_b", params=_f32(g), box=SECTION31_BOX)
    return w


# ------------------------------------------------------------------------------------------------
# Seeded random draws beyond the BASELINE configs (tests/test_gpu_fuzz.py, python -m harness.random_sweeps)
# ------------------------------------------------------------------------------------------------
def random_mid(seed: int):
    """Mid-size maps (12,288 ... 393,216 sightlines: every lane count and forward strategy the library picks by size), random
    model kind, batch 1-3, 40-1400 samples, 1-12 frequencies from 0.3 (or 2) to 40 GHz, a box-clipped extent now and then."""
    rng = np.random.Generator(np.random.PCG64(seed))
    kind = rng.choice(["full16", "full16", "disc4", "stack16"])
    nside = int(rng.choice([32, 45, 48, 52, 64, 90, 96, 112, 114, 128, 148, 150, 160]))
    batch = int(rng.choice([1, 1, 2, 3]))
    if 12 * nside * nside * batch > 400000:
        batch = 1
    n_los = int(rng.integers(40, 1400))
    nf = int(rng.integers(1, 13))
    lo = rng.choice([0.3e9, 0.3e9, 2e9])
    freqs = np.sort(np.exp(rng.uniform(np.log(lo), np.log(40e9), nf)))
    s_max = float(rng.uniform(15.0, 35.0))
    if kind == "full16":
        p = FULL16_NOMINAL * np.exp(rng.uniform(-np.log(1.4), np.log(1.4), (batch, 16)))
        p[:, 12] = rng.uniform(2.5, 3.3, batch)
        if rng.random() < 0.3:
            p[:, 12] = 3.0
        aux = None
    elif kind == "disc4":
        p = DISC4_NOMINAL * np.exp(rng.uniform(-np.log(1.4), np.log(1.4), (batch, 4)))
        aux = AUX_NOMINAL.astype(np.float32)
    else:
        w0 = stack16()
        p = np.repeat(w0.params.astype(np.float64), batch, axis=0) * np.exp(rng.uniform(-0.2, 0.2, (batch, 16)))
        aux = w0.aux
    w = Workload(f"mid{seed}_{kind}", kind, nside, n_los, s_max, freqs, p.astype(np.float32), aux, cot_seed=seed)
    if rng.random() < 0.25:
        w.clip_box = (40.0, 40.0, 10.0)
    return w


def random_grid(seed: int):
    """GRID_B: non-cubic grids over boxes of arbitrary float64 lengths, a random field of 0.3-3 x cfg 3's amplitude on a spiral,
    n_e x 0.5-3, alpha 3 or random, 1-9 frequencies from 0.3 (or 1) GHz, nside 8-48, 40-900 samples."""
    rng = np.random.Generator(np.random.PCG64(seed))
    shape = (int(rng.choice([24, 32, 48, 64, 96])), int(rng.choice([24, 32, 48, 64, 96])), int(rng.choice([8, 12, 16, 32])))
    box = (float(rng.uniform(24, 44)), float(rng.uniform(24, 44)), float(rng.uniform(4, 12)))
    X, Y, Z = grid_nodes(shape, box)
    amp = float(rng.uniform(0.3, 3.0))
    g = amp * gaussian_random_field(shape, box, seed) + spiral_pattern(X, Y, Z, *DISC4_NOMINAL) * float(rng.uniform(0.5, 2.0))
    nside = int(rng.choice([8, 16, 24, 32, 48]))
    n_los = int(rng.integers(40, 900))
    nf = int(rng.integers(1, 10))
    freqs = np.sort(np.exp(rng.uniform(np.log(rng.choice([0.3e9, 1e9])), np.log(30e9), nf)))
    aux = AUX_NOMINAL.astype(np.float32).copy()
    aux[4] *= float(rng.uniform(0.5, 3.0))
    aux[3] = float(rng.choice([3.0, rng.uniform(2.5, 3.3)]))
    w = Workload(f"grid{seed}", "grid_b", nside, n_los, float(rng.uniform(15, 30)), freqs, g.astype(np.float32), aux, box=box,
                    cot_seed=seed)
    if rng.random() < 0.25:
        w.clip_box = box
    return w


def random_options(seed: int):
    """Small maps with everything else random: model kind (UNIFORM included), batch 1-8, 1 / 2 / 3 / 31 ... 65 or up to 600 samples,
    1-32 frequencies (every frequency-block split), box clip, gridded n_e / N_0, and the options lanes, precision, batch_share."""
    rng = np.random.Generator(np.random.PCG64(seed))
    kind = rng.choice(["full16", "disc4", "stack16", "uniform", "disc4"])
    nside = int(rng.choice([1, 2, 3, 4, 8, 12, 16, 24, 32]))
    batch = int(rng.choice([1, 1, 2, 3, 5, 8]))
    n_los = int(rng.choice([1, 2, 3, 31, 32, 33, 63, 64, 65, int(rng.integers(66, 600))]))
    nf = int(rng.choice([1, 2, 3, 4, 5, 7, 8, 9, 12, 13, 16, 17, 31, 32]))
    freqs = np.sort(np.exp(rng.uniform(np.log(rng.choice([0.3e9, 1e9, 5e9])), np.log(40e9), nf)))
    s_max = float(rng.uniform(10.0, 40.0))
    aux = None
    if kind == "full16":
        p = FULL16_NOMINAL * np.exp(rng.uniform(-np.log(1.4), np.log(1.4), (batch, 16)))
        p[:, 12] = rng.uniform(2.5, 3.3, batch)
        if rng.random() < 0.3:
            p[:, 12] = 3.0
    elif kind == "disc4":
        p = DISC4_NOMINAL * np.exp(rng.uniform(-np.log(1.4), np.log(1.4), (batch, 4)))
        aux = AUX_NOMINAL.astype(np.float32).copy()
        if rng.random() < 0.5:
            aux[3] = float(rng.uniform(2.5, 3.3))
    elif kind == "stack16":
        w0 = stack16()
        p = np.repeat(w0.params.astype(np.float64), batch, axis=0) * np.exp(rng.uniform(-0.2, 0.2, (batch, 16)))
        aux = w0.aux
    else:
        w0 = uniform_toy(bvec=(2.0, -3.0, 1.5))
        p = np.repeat(w0.params.astype(np.float64), batch, axis=0) * np.exp(rng.uniform(-0.3, 0.3, (batch, w0.params.shape[1])))
        if rng.random() < 0.5:
            p[:, 5] = rng.uniform(2.5, 3.3, batch)
        aux = w0.aux
    w = Workload(f"opt{seed}_{kind}", kind, nside, n_los, s_max, freqs, p.astype(np.float32), aux, cot_seed=seed)
    if rng.random() < 0.3:
        w.clip_box = (float(rng.uniform(30, 50)), float(rng.uniform(30, 50)), float(rng.uniform(6, 14)))
    if kind in ("disc4", "stack16") and rng.random() < 0.4:
        shp = (int(rng.choice([8, 16, 24])), int(rng.choice([8, 16, 24])), int(rng.choice([4, 8, 12])))
        bx = (float(rng.uniform(30, 50)), float(rng.uniform(30, 50)), float(rng.uniform(6, 14)))
        w.ne_grid, w.ne_box = clumpy_disc_grid(shp, bx, 0.03 * float(rng.uniform(0.5, 2)), 20.0, 1.0, seed=seed), bx
        if rng.random() < 0.5:
            w.n0_grid, w.n0_box = clumpy_disc_grid(shp, bx, 2.1e-4, 5.0, 1.0, seed=seed + 1), bx
    opts = {}
    if rng.random() < 0.5:
        opts["lanes"] = int(rng.choice([1, 8, 32]))
    if rng.random() < 0.25:
        opts["precision"] = 2
    if rng.random() < 0.3:
        opts["batch_share"] = int(rng.choice([1, 2, 4]))
    return w, opts
