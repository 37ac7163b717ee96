#!/usr/bin/env python
"""Write long-horizon expected values with the CPU ORACLE ONLY (never the CUDA path).

Usage:  python tests/golden/make_golden.py [--twin | --twin-only [--perturb-u]] [case ...]
        (no case = every case; --twin also records the conditioning run for the large cases,
        doubling their cost; --twin-only keeps the stored expected values of an existing file and
        adds sens_<cp> from one perturbed ORACLE run, measured on the stored sample nodes;
        --perturb-u also perturbs the input velocity by 1e-21 (absolute, the size of the
        one-step rounding differences between two summation orders), which reaches the gas
        phase where a relative perturbation of phi ~ 1e-9 is no perturbation at all;
        --twin-fma [case ...]: instead of perturbing the input, run the SAME input through the
        oracle source built with FMA contraction on (oracle/tslb_ref.py, TSLB_REF_FMA=1) and
        store fma_<cp> = its distance from the stored expected values: two correct roundings of
        one program, differing at every multiply-add of every step, which is what a CUDA kernel
        with another summation order is too);
        --twin-rev [case ...]: the same with the oracle source built to take every sum over the
        27 directions in reverse order (TSLB_REF_REV=1): stores rev_<cp>)

For each case the oracle runs the seeded input of paper_2501_00846_b200.inputs for the
config's full step count and stores, at the checkpoints {1, 10, 100, 1000, ..., final}:
  * rho, p, u, phi at NSAMPLE seeded node positions (element-by-element parity on samples),
  * per-field max|.| over the whole lattice (the denominators of the parity norm),
  * the diagnostics sum(phi), sum(p*), and for droplets the Laplace ratio of pin P9,
  * (small cases) sens_<cp>: the same norm between this run and a second ORACLE run whose phi
    input was perturbed by one part in 1e15 -- the conditioning of the trajectory itself.  Where
    the flow amplifies round-off (a rising bubble shedding its wake), no two summation orders
    can agree better than this, and the parity test widens its bar to 10 x sens.
Files: tests/golden/<case>.npz (a few hundred kB each).  tests/test_golden_gpu.py replays the
same inputs through the C ABI and compares.

Cases: tests/golden/cases.py (one per BASELINE.json config at the config's own grid, plus the
reduced-size long horizons).  The oracle advances ~2.5 M nodes per second on 8 cores: 256^3 to
step 100 takes ~12 min, a 128^3 Laplace case to step 1000 ~15 min, 384^3 to step 10 ~5 min and
~45 GB of host memory.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

if "--twin-fma" in sys.argv:
    os.environ["TSLB_REF_FMA"] = "1"                   # before the oracle library is loaded
if "--twin-rev" in sys.argv:
    os.environ["TSLB_REF_REV"] = "1"
from oracle import tslb_ref as R                      # noqa: E402
from paper_2501_00846_b200 import inputs as I          # noqa: E402

NSAMPLE = 2048
HERE = os.environ.get("TSLB_GOLDEN_DIR", os.path.dirname(os.path.abspath(__file__)))


def cases():
    from cases import CASES                            # tests/golden/cases.py: recipes only
    return CASES


def sample_index(shape, seed=12345):
    rng = np.random.Generator(np.random.PCG64(seed))
    n = int(np.prod(shape))
    return np.sort(rng.choice(n, size=min(NSAMPLE, n), replace=False))


def laplace_ratio(p, phi, sigma):
    inside, outside = phi > 0.99, phi < 0.01
    if not inside.any() or not outside.any():
        return np.nan
    dp = p[inside].mean() - p[outside].mean()
    r_eff = (3.0 * phi.sum() / (4.0 * np.pi)) ** (1.0 / 3.0)
    return dp * r_eff / (2.0 * sigma)


def run(name):
    make, checkpoints = cases()[name]
    cfg = make()
    nz, ny, nx = cfg["shape"]
    idx = sample_index(cfg["shape"])
    sim = R.RefSim(nx, ny, nz, R.make_params(**cfg["params"]))
    sim.init(cfg["phi"], cfg["u"])
    twin = None
    if nx * ny * nz <= 64 ** 3 or "--twin" in sys.argv:   # conditioning run (costs a second run)
        rng = np.random.Generator(np.random.PCG64(99))
        twin = R.RefSim(nx, ny, nz, R.make_params(**cfg["params"]))
        twin.init(cfg["phi"] * (1.0 + 1e-15 * rng.uniform(-1.0, 1.0, cfg["shape"])), cfg["u"])
    out = {"checkpoints": np.array(checkpoints), "sample_index": idx,
           "shape": np.array(cfg["shape"])}
    done, t0 = 0, time.time()
    for cp in checkpoints:
        sim.step(cp - done)
        if twin is not None:
            twin.step(cp - done)
        done = cp
        rho, p, u, phi = sim.get()
        if twin is not None:
            out[f"sens_{cp}"] = np.array([np.abs(a - b).max() / np.abs(a).max()
                                          for a, b in zip((rho, p, u, phi), twin.get())])
        ps = sim.get_state()[0]
        out[f"rho_{cp}"] = rho.ravel()[idx]
        out[f"p_{cp}"] = p.ravel()[idx]
        out[f"phi_{cp}"] = phi.ravel()[idx]
        out[f"u_{cp}"] = u.reshape(3, -1)[:, idx]
        out[f"max_{cp}"] = np.array([np.abs(rho).max(), np.abs(p).max(), np.abs(u).max(),
                                     np.abs(phi).max()])
        out[f"diag_{cp}"] = np.array([phi.sum(), ps.sum(),
                                      laplace_ratio(p, phi, cfg["params"]["sigma"]),
                                      float(np.isfinite(u).all())])
        print(f"{name}: step {cp} done after {time.time() - t0:.0f} s, max|u| = "
              f"{np.abs(u).max():.3e}, sum(phi) drift = {phi.sum() / cfg['phi'].sum() - 1:.1e}",
              flush=True)
        del rho, p, u, phi, ps
        # written after every checkpoint (a long run that is cut off keeps what it has)
        out["checkpoints"] = np.array([c for c in checkpoints if c <= cp])
        np.savez_compressed(os.path.join(HERE, name + ".npz"), **out)
    sim.close()
    if twin is not None:
        twin.close()


def run_twin_fma(name, key="fma"):
    """Add fma_<cp> (or rev_<cp>) to an existing golden file (the expected values are left
    untouched): the distance of a differently ROUNDED build of the same oracle source."""
    assert os.environ.get("TSLB_REF_FMA") == "1" or os.environ.get("TSLB_REF_REV") == "1"
    make, checkpoints = cases()[name]
    path = os.path.join(HERE, name + ".npz")
    cfg = make()
    nz, ny, nx = cfg["shape"]
    idx = np.load(path)["sample_index"]
    twin = R.RefSim(nx, ny, nz, R.make_params(**cfg["params"]))
    twin.init(cfg["phi"], cfg["u"])
    done, t0 = 0, time.time()
    for cp in checkpoints:
        twin.step(cp - done)
        done = cp
        rho, p, u, phi = twin.get()
        out = dict(np.load(path))                    # re-read: another twin may be writing too
        got = (rho.ravel()[idx], p.ravel()[idx], u.reshape(3, -1)[:, idx], phi.ravel()[idx])
        want = (out[f"rho_{cp}"], out[f"p_{cp}"], out[f"u_{cp}"], out[f"phi_{cp}"])
        out[f"{key}_{cp}"] = np.array([np.abs(a - b).max() / m
                                       for a, b, m in zip(got, want, out[f"max_{cp}"])])
        print(f"{name}: {key} twin step {cp} after {time.time() - t0:.0f} s, drift = "
              f"{out[f'{key}_{cp}']}", flush=True)
        np.savez_compressed(path, **out)
    twin.close()


def run_twin_only(name):
    """Add sens_<cp> to an existing golden file: one perturbed oracle run against the stored
    sample values (the expected values themselves are left untouched)."""
    make, checkpoints = cases()[name]
    path = os.path.join(HERE, name + ".npz")
    out = dict(np.load(path))
    cfg = make()
    nz, ny, nx = cfg["shape"]
    idx = out["sample_index"]
    rng = np.random.Generator(np.random.PCG64(99))
    twin = R.RefSim(nx, ny, nz, R.make_params(**cfg["params"]))
    phi0 = cfg["phi"] * (1.0 + 1e-15 * rng.uniform(-1.0, 1.0, cfg["shape"]))
    u0 = cfg["u"]
    if "--perturb-u" in sys.argv:
        u0 = u0 + 1e-21 * rng.uniform(-1.0, 1.0, u0.shape)
        out["sens_perturb_u"] = np.array(1e-21)
    twin.init(phi0, u0)
    done, t0 = 0, time.time()
    for cp in checkpoints:
        twin.step(cp - done)
        done = cp
        rho, p, u, phi = twin.get()
        got = (rho.ravel()[idx], p.ravel()[idx], u.reshape(3, -1)[:, idx], phi.ravel()[idx])
        want = (out[f"rho_{cp}"], out[f"p_{cp}"], out[f"u_{cp}"], out[f"phi_{cp}"])
        out[f"sens_{cp}"] = np.array([np.abs(a - b).max() / m
                                      for a, b, m in zip(got, want, out[f"max_{cp}"])])
        print(f"{name}: twin step {cp} after {time.time() - t0:.0f} s, sens = {out[f'sens_{cp}']}",
              flush=True)
        np.savez_compressed(path, **out)
    twin.close()


if __name__ == "__main__":
    names = [a for a in sys.argv[1:] if not a.startswith("--")]
    for nm in (names or list(cases())):
        if "--twin-fma" in sys.argv:
            run_twin_fma(nm)
        elif "--twin-rev" in sys.argv:
            run_twin_fma(nm, key="rev")
        elif "--twin-only" in sys.argv:
            run_twin_only(nm)
        else:
            run(nm)
