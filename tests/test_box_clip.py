"""The paper's integration extent (Fig. 1 L97): observer -> box face, n_los equal segments per
sightline.  Oracle pins on CPU (closed forms), GPU parity through synax_plan_set_box."""
import numpy as np
import pytest

import oracle
from harness import parity
from conftest import load_golden
from harness import workloads as wl

BOX = (40.0, 40.0, 10.0)          # the paper's box
OBS = (-8.3, 0.0, 0.006)


def test_exit_distance_closed_forms():
    assert abs(oracle.exit_distance(OBS, 0.0, 0.0, BOX) - 28.3) < 1e-12            # +x face at 20
    assert abs(oracle.exit_distance(OBS, np.pi, 0.0, BOX) - 11.7) < 1e-12          # -x face at -20
    assert abs(oracle.exit_distance(OBS, 0.5 * np.pi, 0.0, BOX) - 20.0) < 1e-12    # +y face
    assert abs(oracle.exit_distance(OBS, 0.0, 0.5 * np.pi, BOX) - 4.994) < 1e-12   # +z face at 5
    assert abs(oracle.exit_distance(OBS, 0.0, -0.5 * np.pi, BOX) - 5.006) < 1e-12
    rng = np.random.Generator(np.random.PCG64(3))
    for _ in range(200):                                                           # the exit point lies ON the box surface
        l, b = rng.uniform(0, 2 * np.pi), np.arcsin(rng.uniform(-1, 1))
        L = oracle.exit_distance(OBS, l, b, BOX)
        n = np.array([np.cos(b) * np.cos(l), np.cos(b) * np.sin(l), np.sin(b)])
        q = np.abs(np.array(OBS) + L * n) / (0.5 * np.array(BOX))
        assert abs(q.max() - 1.0) < 1e-12 and L > 0
    assert oracle.exit_distance((25.0, 0, 0), 0.0, 0.0, BOX) < 0                    # observer outside


def test_uniform_field_in_box_gives_j_times_path_length():
    """Eq. 10 with the box as the emitting volume: I = j_I L_i for every sightline, any n_los."""
    gold = load_golden("constants.txt")
    m = oracle.Model("uniform", [0.0, 0.0, 6.0, 4.01e-5, 0.0, 3.0])                # B along z: B_perp = 6 uG at b = 0
    for l in (0.0, 1.0, 2.5, np.pi):
        for n_los in (1, 7, 64):
            I, Q, U = oracle.forward_dir(m, l, 0.0, n_los, 1.0, [2.4e9], clip_box=BOX)
            L = oracle.exit_distance(OBS, l, 0.0, BOX)
            assert abs(I[0] / (gold["toy_I_kelvin_per_kpc"] * L) - 1) < 1e-9
    with pytest.raises(ValueError):
        oracle.forward(m, 1, 4, 1.0, [2.4e9], observer=(30.0, 0, 0), clip_box=BOX)


def test_clipped_map_equals_per_pixel_fixed_length_runs():
    """Clipping only changes each sightline's s_max: pixel p of the clipped map = a fixed-s_max run with s_max = L_p."""
    w = wl.config(4).scaled(nside=2, n_los=32)
    w.clip_box = BOX
    I, Q, U = parity.oracle_forward(w)
    m = parity.oracle_model(w)
    for p in (0, 13, 20, 47):
        z, phi = oracle.pix2ang_ring(w.nside, [p])
        L = oracle.exit_distance(OBS, phi[0], np.arcsin(z[0]), BOX)
        Ip, Qp, Up = oracle.forward(m, w.nside, w.n_los, L, w.freqs, pix=[p])
        assert np.allclose(Ip[0, :, 0], I[0, :, p], rtol=1e-11) and np.allclose(Qp[0, :, 0], Q[0, :, p], rtol=1e-9, atol=1e-18)


def test_clipped_gradient_matches_finite_differences():
    w = wl.config(2).scaled(nside=2, n_los=40, batch=1)
    w.clip_box = BOX
    cots = w.cotangents()
    g = parity.oracle_vjp(w, cots)[0]
    base = w.params.astype(np.float64)
    for j in (0, 2, 4, 6, 10, 12, 14):
        h = 1e-6 * abs(base[0, j])
        vals = []
        for sgn in (1, -1):
            q = base.copy(); q[0, j] += sgn * h
            I, Q, U = oracle.forward(oracle.Model("full16", q), w.nside, w.n_los, w.s_max, w.freqs, clip_box=BOX)
            vals.append((I * cots[0]).sum() + (Q * cots[1]).sum() + (U * cots[2]).sum())
        fd = (vals[0] - vals[1]) / (2 * h)
        assert abs(fd - g[j]) <= 2e-5 * abs(g[j]), (j, fd, g[j])


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["disc4", "full16_f64", "full16_f64_256", "full16_batch", "grid", "uniform"])
def test_gpu_box_clipped_parity(case):
    if case == "disc4":
        w = wl.config(1).scaled(nside=16, n_los=128)
    elif case == "full16_f64":
        w = wl.config(4).scaled(nside=16, n_los=1024)         # 408 MHz: float64 Faraday chain
    elif case == "full16_f64_256":
        # under-resolved (256 samples at 408 MHz): the w_h component was 1.1e-2 off with the single-sweep T - P_m form of
        # the reverse scan (cancellation); the prefix form of DESIGN.md section 5 keeps it inside the bound
        w = wl.config(4).scaled(nside=16, n_los=256)
    elif case == "full16_batch":
        w = wl.config(2).scaled(nside=8, n_los=100, batch=6)
    elif case == "grid":
        w = wl.config(3).scaled(nside=8, n_los=200)
    else:
        w = wl.uniform_toy(nside=4, n_los=33, freqs=(1.4e9, 2.4e9))
    w.clip_box = (40.0, 40.0, 8.0) if case == "grid" else BOX
    maps, _ = parity.gpu_forward(w)
    parity.assert_maps_close(maps, parity.oracle_forward(w), what=f"box-clipped forward {case}")
    cots = w.cotangents()
    g, ref = parity.gpu_vjp(w, cots), parity.oracle_vjp(w, cots)
    if case == "grid":
        rms = np.sqrt(np.mean(ref[ref != 0] ** 2))
        assert np.all(np.abs(g - ref) <= 1e-3 * np.abs(ref) + 1e-4 * rms)
        assert np.array_equal(ref == 0.0, g == 0.0)
    else:
        nz = ref != 0
        assert np.all(np.abs(g - ref)[nz] <= parity.GRAD_TOL * np.abs(ref)[nz])


@pytest.mark.gpu
def test_gpu_set_box_errors_and_reset():
    import paper_2410_01136_b200 as sx
    w = wl.config(0)
    ref_maps, _ = parity.gpu_forward(w)
    plan, model, params = parity.gpu_objects(w)
    with pytest.raises(sx.SynaxError):
        plan.set_box((10.0, 40.0, 10.0))                      # observer at x = -8.3 is outside a 10-kpc box
    with pytest.raises(sx.SynaxError):
        plan.set_box((40.0, 40.0, 0.0))
    plan.set_box(BOX)
    clipped = [t.cpu().numpy() for t in sx.forward(plan, model, params)]
    plan.set_box(None)                                        # back to the fixed [0, s_max]
    again = [t.cpu().numpy().astype(np.float64) for t in sx.forward(plan, model, params)]
    plan.close()
    assert all(np.array_equal(a, b) for a, b in zip(again, ref_maps))
    assert not np.array_equal(clipped[0], again[0])
