"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Tolerances are BASELINE.json's: max|gpu-ref|/max|ref| <= 1e-10 per
field in fp64, <= 1e-4 on u and phi in fp32."""
import numpy as np
import pytest

from paper_2501_00846_b200 import inputs as I
from parity_util import compare, rel_err, run_gpu, run_oracle

pytestmark = pytest.mark.gpu

PATHS = {"naive": 1, "tiled": 0}            # TSLB_FLAG_NAIVE or the production kernels
TOL64, TOL32 = 1e-10, 1e-4


def _small_case(name):
    """Droplet centres are kept off the lattice nodes and off their periodic antipodes: a node
    where grad(phi) vanishes by symmetry while phi(1-phi) is not small makes the normal
    grad(phi)/sqrt(|grad(phi)|^2 + eps^2) (R13, eps = 1e-12) a ratio of rounding noise to eps,
    which no two summation orders reproduce."""
    if name == "ragged_periodic":            # several tiles in x and y plus a ragged tail
        shape = (19, 21, 37)
        prm = I.base_params()
        phi = I.sphere_profile(shape, (16.3, 9.1, 7.7), 6.0, 4.0, prm["bc"])
        u = I.noise_u(shape, 1e-3, 21)
        steps = [1, 2, 50]
    elif name == "bubble_walls_z":           # configs[2] in miniature: gravity + bounce-back
        cfg = I.rising_bubble(nx=20, ny=12, nz=26, radius=5.0, height=9.0)
        cfg["u"] = I.noise_u(cfg["shape"], 1e-4, 22)
        return cfg, [1, 60]
    elif name == "train_walls_z":            # NEXT-2 in miniature: droplets falling onto a wall,
        shape = (30, 12, 20)                 # gravity on the LIQUID (R20b, TSLB_FLAG_BODY_HEAVY)
        prm = I.base_params(rho_g=1.0 / 800.0, mu_l=1.0 / 300.0, mu_g=1.0 / 15000.0, sigma=8e-4,
                            bc=(0, 0, 1), body_accel=(1e-6, 0.0, -2e-5), body_heavy=True)
        phi = I.sphere_profile(shape, (9.6, 5.7, 5.2), 4.0, 4.0, prm["bc"])
        phi += I.sphere_profile(shape, (9.6, 5.7, 17.3), 4.0, 4.0, prm["bc"])
        u = I.noise_u(shape, 1e-4, 27)
        u[2] -= 0.05 * phi
        steps = [1, 60]
    elif name == "walls_all":                # droplet touching a corner, walls on every axis
        shape = (8, 9, 10)
        prm = I.base_params(bc=(1, 1, 1), body_accel=(1e-5, -2e-5, 3e-5))
        phi = I.sphere_profile(shape, (2.0, 2.5, 1.5), 3.0, 4.0, prm["bc"])
        u = I.noise_u(shape, 1e-3, 23)
        steps = [1, 40]
    elif name == "walls_xy":                 # walls on the tile axes, periodic marching axis
        shape = (12, 7, 35)
        prm = I.base_params(bc=(1, 1, 0), body_accel=(0.0, 0.0, 2e-5))
        phi = I.sphere_profile(shape, (30.3, 3.2, 5.6), 4.0, 4.0, prm["bc"])
        u = I.noise_u(shape, 1e-3, 24)
        steps = [1, 40]
    elif name == "min_periodic":             # smallest legal periodic box
        shape = (4, 4, 4)
        prm = I.base_params()
        phi = I.sphere_profile(shape, (1.5, 1.5, 1.5), 1.2, 4.0, prm["bc"])
        u = I.noise_u(shape, 1e-3, 25)
        steps = [1, 30]
    elif name == "min_walls":                # smallest legal box with walls everywhere
        shape = (2, 2, 2)
        prm = I.base_params(bc=(1, 1, 1))
        phi = I.sphere_profile(shape, (0.0, 0.0, 0.0), 0.8, 4.0, prm["bc"])
        u = I.noise_u(shape, 1e-3, 26)
        steps = [1, 30]
    else:
        raise KeyError(name)
    return dict(name=name, shape=shape, params=prm, phi=phi, u=u), steps


@pytest.mark.parametrize("path", PATHS)
def test_config0_static_droplet_fp64(ref, path):
    """BASELINE.json configs[0]: 32^3, 200 steps, fp64, error reported against step count."""
    cfg = I.static_droplet(32, 8.0, seed=1)
    steps = [1, 10, 100, 200]
    want = run_oracle(ref, cfg, steps)
    got, _ = run_gpu(cfg, steps, "f64", PATHS[path])
    for n, g, r in zip(steps, got, want):
        errs, bad = compare(ref, cfg, g, r, TOL64, state_tol=1e-9)
        print(f"[{path}] step {n}: " + " ".join(f"{k}={v:.2e}" for k, v in errs.items()))
        assert not bad, (n, bad)


@pytest.mark.parametrize("path", PATHS)
def test_config0_static_droplet_fp32(ref, path):
    cfg = I.static_droplet(32, 8.0, seed=1)
    steps = [1, 200]
    want = run_oracle(ref, cfg, steps)
    got, _ = run_gpu(cfg, steps, "f32", PATHS[path])
    for n, g, r in zip(steps, got, want):
        errs, bad = compare(ref, cfg, g, r, TOL32, fields=("u", "phi"))
        print(f"[{path}] fp32 step {n}: " + " ".join(f"{k}={v:.2e}" for k, v in errs.items()))
        assert not bad, (n, bad)
        assert rel_err(g["rho"], r["rho"]) < 1e-3


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("case", ["ragged_periodic", "bubble_walls_z", "train_walls_z", "walls_all",
                                  "walls_xy", "min_periodic", "min_walls"])
def test_small_cases_fp64(ref, path, case):
    cfg, steps = _small_case(case)
    want = run_oracle(ref, cfg, steps)
    got, _ = run_gpu(cfg, steps, "f64", PATHS[path])
    for n, g, r in zip(steps, got, want):
        errs, bad = compare(ref, cfg, g, r, TOL64, state_tol=1e-9)
        print(f"[{path}/{case}] step {n}: " + " ".join(f"{k}={v:.2e}" for k, v in errs.items()))
        assert not bad, (case, n, bad)


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("case", ["ragged_periodic", "bubble_walls_z", "train_walls_z", "walls_all"])
def test_small_cases_fp32(ref, path, case):
    cfg, steps = _small_case(case)
    want = run_oracle(ref, cfg, steps)
    got, _ = run_gpu(cfg, steps, "f32", PATHS[path])
    for n, g, r in zip(steps, got, want):
        errs, bad = compare(ref, cfg, g, r, TOL32, fields=("u", "phi"))
        print(f"[{path}/{case}] fp32 step {n}: " + " ".join(f"{k}={v:.2e}" for k, v in errs.items()))
        assert not bad, (case, n, bad)


@pytest.mark.parametrize("path", PATHS)
def test_laplace_128_short_fp64(ref, path):
    """configs[1] geometry (128^3, R = 16) for a few steps: many tiles, many z chunks."""
    cfg = I.static_droplet(128, 16.0, seed=16)
    steps = [1, 4]
    want = run_oracle(ref, cfg, steps)
    got, _ = run_gpu(cfg, steps, "f64", PATHS[path])
    for n, g, r in zip(steps, got, want):
        errs, bad = compare(ref, cfg, g, r, TOL64, state_tol=1e-9)
        print(f"[{path}] 128^3 step {n}: " + " ".join(f"{k}={v:.2e}" for k, v in errs.items()))
        assert not bad, (n, bad)


def _check_both_precisions(ref, cfg, steps, flags, tag):
    want = run_oracle(ref, cfg, steps)
    for prec, tol, fields in (("f64", TOL64, ("rho", "p", "u", "phi")), ("f32", TOL32, ("u", "phi"))):
        got, _ = run_gpu(cfg, steps, prec, flags)
        for n, g, r in zip(steps, got, want):
            errs, bad = compare(ref, cfg, g, r, tol, fields=fields,
                                state_tol=1e-9 if prec == "f64" else None)
            print(f"[{tag} {prec}] step {n}: " + " ".join(f"{k}={v:.2e}" for k, v in errs.items()))
            assert not bad, (tag, prec, n, bad)


# validation selectors of include/tslb.h: every one forces another CORRECT kernel of the product
SELECTORS = {"auto": 0, "generic": 2, "k2_cpasync": 4, "k2_tma": 8, "k1_flux": 16,
             "k2_tma+k1_flux": 8 | 16, "k2_cpasync+k1_flux": 4 | 16}


@pytest.mark.parametrize("sel", list(SELECTORS))
def test_kernel_selectors(ref, sel):
    """Every selectable kernel meets the same bar on a box of 3 x 5 tiles of 32 x 8, two z
    chunks, ragged in every direction (nx = 70: the TMA selector falls back to cp.async)."""
    cfg, _ = _small_case("ragged_periodic")
    cfg["shape"] = (40, 37, 70)
    cfg["phi"] = I.sphere_profile(cfg["shape"], (30.3, 16.1, 19.7), 9.0, 4.0)
    cfg["u"] = I.noise_u(cfg["shape"], 1e-3, 31)
    _check_both_precisions(ref, cfg, [1, 12], SELECTORS[sel], sel)


@pytest.mark.parametrize("sel", ["auto", "k1_flux"])
def test_interface_kernels_on_wide_rows(ref, sel):
    """Row kernel of the interface update (several nodes per thread) and its one-node-per-thread
    fallback: two x tiles in fp32 (128 + 8 columns), three in fp64 (64 + 64 + 8), ragged in y, z."""
    cfg, _ = _small_case("ragged_periodic")
    cfg["shape"] = (36, 19, 136)
    cfg["phi"] = I.sphere_profile(cfg["shape"], (128.3, 9.1, 16.7), 7.0, 4.0)
    cfg["u"] = I.noise_u(cfg["shape"], 1e-3, 41)
    _check_both_precisions(ref, cfg, [1, 10], SELECTORS[sel], f"wide rows/{sel}")


def test_odd_row_length_uses_the_flux_kernel(ref):
    """nx = 37 is not a multiple of the 128-bit vector width: the library itself falls back to
    the one-node-per-thread interface kernel (flags = 0)."""
    cfg, steps = _small_case("ragged_periodic")
    _check_both_precisions(ref, cfg, [1, 8], 0, "nx=37")


@pytest.mark.parametrize("nx", [64, 96, 128])
def test_tma_staged_kernel(ref, nx):
    """Stream-collide kernel with TMA tensor staging (production in fp64 on deep grids, forced
    here by TSLB_FLAG_K2_TMA in both precisions): x tiles that wrap on the left, on the right,
    and not at all; the wrapped row / corner boxes; ragged in y and z, 70 planes = two chunks
    with a ragged tail."""
    cfg, _ = _small_case("ragged_periodic")
    cfg["shape"] = (70, 19, nx)
    cfg["phi"] = I.sphere_profile(cfg["shape"], (nx - 2.7, 9.1, 30.7), 7.0, 4.0)
    cfg["u"] = I.noise_u(cfg["shape"], 1e-3, 43)
    _check_both_precisions(ref, cfg, [1, 10], SELECTORS["k2_tma"], f"tma nx={nx}")


@pytest.mark.parametrize("sel", ["auto", "k2_tma", "k2_cpasync", "generic"])
def test_z_walls_on_the_lean_pair(ref, sel):
    """Walls on the marching axis (configs[2]: no-slip floor and lid, periodic sides) run the lean
    periodic pair with bounce-back ghost planes; the wall-capable pair is the cross-check.  Gas
    bubble touching the floor, a liquid film... two tiles in x, three in y, 70 planes = chunks
    with a ragged tail, gravity on."""
    shape = (70, 19, 64)                                         # (nz, ny, nx)
    prm = I.base_params(bc=(0, 0, 1), body_accel=(1e-6, 0.0, -2e-5))
    phi = 1.0 - I.sphere_profile(shape, (20.3, 9.1, 4.6), 7.0, 4.0, prm["bc"])     # at the floor
    phi -= I.sphere_profile(shape, (50.2, 5.7, 66.1), 6.0, 4.0, prm["bc"])          # at the lid
    cfg = dict(name="z_walls", shape=shape, params=prm, phi=phi, u=I.noise_u(shape, 1e-3, 47))
    _check_both_precisions(ref, cfg, [1, 2, 14], SELECTORS[sel], f"z walls/{sel}")


@pytest.mark.parametrize("precision,tol", [("f64", 1e-12), ("f32", 1e-5)])
def test_resume_from_a_state_dump(precision, tol):
    """tslb_get_state -> tslb_set_state on a NEW solver -> step continues the run: equal to the
    uninterrupted run to rounding (the flux handed between the two kernels is rebuilt with another
    summation order).  Periodic lean pair and a box with walls."""
    from paper_2501_00846_b200 import binding as B
    for name in ("ragged_periodic", "bubble_walls_z"):
        cfg, _ = _small_case(name)
        nz, ny, nx = cfg["shape"]
        a = B.Solver(nx, ny, nz, cfg["params"], precision=precision)
        a.init(cfg["phi"], cfg["u"])
        a.step(17)
        dump = {k: v.clone() for k, v in a.get_state().items()}
        a.step(13)
        want = {k: v.clone() for k, v in a.get().items()}
        a.close()
        b = B.Solver(nx, ny, nz, cfg["params"], precision=precision)
        b.set_state(dump)
        b.step(13)
        got = b.get()
        for k in want:
            err = float((got[k] - want[k]).abs().max() / want[k].abs().max())
            assert err <= tol, (name, k, err)
        b.close()


@pytest.mark.parametrize("bc", [(1, 0, 0), (0, 1, 0), (1, 1, 0), (1, 1, 1), (0, 1, 1)])
@pytest.mark.parametrize("sel", ["auto", "generic"])
def test_side_walls_on_the_lean_kernel(ref, bc, sel):
    """Walls on the tile axes x / y: the lean stream-collide kernel with the bounce accounting of
    the wall-adjacent receivers (wall_bounce) + the wall-capable interface kernel; the
    wall-capable pair is the cross-check.  Three x tiles, five y tiles, two z chunks, ragged;
    droplets sitting in a corner, on an edge and on a face, gravity oblique to every wall."""
    shape = (40, 37, 72)                                         # (nz, ny, nx); nx % 4 == 0: row kernel
    prm = I.base_params(bc=bc, body_accel=(1e-5, -2e-5, 1.5e-5))
    phi = I.sphere_profile(shape, (2.3, 1.8, 3.1), 7.0, 4.0, bc)            # low corner
    phi += I.sphere_profile(shape, (69.2, 18.4, 37.6), 6.0, 4.0, bc)        # high x face / top
    phi += I.sphere_profile(shape, (35.5, 35.1, 20.3), 5.0, 4.0, bc)        # high y face
    cfg = dict(name="side_walls", shape=shape, params=prm, phi=np.minimum(phi, 1.0),
               u=I.noise_u(shape, 1e-3, 59))
    _check_both_precisions(ref, cfg, [1, 2, 12], SELECTORS[sel], f"side walls {bc}/{sel}")


@pytest.mark.parametrize("sel", ["generic", "k2_cpasync"])
def test_heavy_phase_body_force_on_every_pair(ref, sel):
    """R20b: the body-force reference density is part of the problem, not of a kernel: the
    wall-capable pair and the lean pair give the oracle's fields with it too, and the fields
    differ from the default R20 run (so the bit cannot be silently dropped)."""
    cfg, steps = _small_case("train_walls_z")
    _check_both_precisions(ref, cfg, steps, SELECTORS[sel], f"train/{sel}")
    other = dict(cfg, params=dict(cfg["params"], body_heavy=False))
    a, _ = run_gpu(cfg, [10], "f64", SELECTORS[sel])
    b, _ = run_gpu(other, [10], "f64", SELECTORS[sel])
    assert rel_err(a[0]["u"], b[0]["u"]) > 1e-3


def test_stray_flag_bits_are_rejected():
    from paper_2501_00846_b200 import binding as B
    cfg = I.static_droplet(16, 4.0, seed=2)
    for flags in (64, 1 << 8, 59 << 8, 1 << 16, 1 << 30):
        with pytest.raises(B.TslbError):
            B.Solver(16, 16, 16, cfg["params"], flags=flags)


def test_host_api_matches_device_api(ref):
    """tslb_init_host / tslb_get_host (the e2e calls of bench.py) give the same fields."""
    cfg, steps = _small_case("bubble_walls_z")
    dev, _ = run_gpu(cfg, steps, "f64", 0)
    host, _ = run_gpu(cfg, steps, "f64", 0, host_api=True)
    for d, h in zip(dev, host):
        for k in ("rho", "p", "u", "phi"):
            assert np.array_equal(d[k], h[k]), k


def test_step_zero_and_reinit():
    from paper_2501_00846_b200 import binding as B
    cfg = I.static_droplet(16, 4.0, seed=2)
    s = B.Solver(16, 16, 16, cfg["params"])
    s.init(cfg["phi"], cfg["u"])
    a = {k: v.clone() for k, v in s.get().items()}
    n0 = s.launches
    s.step(0)
    assert s.launches == n0
    s.step(7)
    b = {k: v.clone() for k, v in s.get().items()}
    s.init(cfg["phi"], cfg["u"])                 # restart
    c = s.get()
    s.step(7)
    d = s.get()
    s.synchronize()
    for k in a:
        assert bool((a[k] == c[k]).all()) and bool((b[k] == d[k]).all()), k
    s.close()
