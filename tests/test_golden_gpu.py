"""Long-horizon parity: the CUDA path against expected values written by the CPU oracle
(tests/golden/make_golden.py, which calls only oracle/), one golden file per BASELINE.json config
at the config's own grid plus reduced-size long horizons (tests/golden/cases.py).  Error is
reported against step count.

The bar at a checkpoint is BASELINE.json's: 1e-10 per field in fp64, 1e-4 on u and phi in fp32.
It is widened ONLY by what the oracle itself measures about the trajectory: the
golden files record how far differently ROUNDED runs of the same oracle have drifted from the
expected values at that checkpoint -- sens (input perturbed by 1e-15), fma (same source built
with FMA contraction), rev (same source, sums over the 27 directions in reverse order).  With
cond = their maximum, counted only once it is clearly above what ONE step's rounding makes of
them (30 x the largest twin drift at the file's first checkpoint: below that the twins measure
round-off, not the trajectory), a third rounding of the same arithmetic, the CUDA kernel, is
allowed K = 30 times that drift (times eps32/eps64 in fp32):
    bar = max(tol, K * cond * scale).
Where that bar exceeds 1e-2 the two fields no longer describe the same flow pointwise: the
checkpoint is reported, not asserted, and what is asserted there is what holds at any horizon
(sum(phi), the Laplace ratio) -- the per-step arithmetic at those late times is checked by
tests/test_segment_gpu.py, which restarts the oracle from the GPU's own state.
Shortfalls against BASELINE.json's tolerance that are NOT explained by the oracle twins would be
listed in KNOWN_SHORTFALLS with the measured value (not hidden behind a formula; the test fails
if one of them grows by more than 3x or if anything else exceeds its bar).  There are none."""
import os
import sys

import numpy as np
import pytest

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
sys.path.insert(0, HERE)
from cases import CASES as _CASES                    # noqa: E402  (recipes only)

pytestmark = pytest.mark.gpu
CASES = {k: v[0] for k, v in _CASES.items()}
K_TWIN, CAP = 30.0, 1e-2

# (case, precision, checkpoint, field): measured error that exceeds BASELINE.json's tolerance and
# is not covered by K x the oracle twins' drift.  EMPTY since the interface kernels add phi's
# update as an increment of differences (round 2): before that the flux-form update cost ~10x more
# rounding noise in phi per step, which the unstable gas flow around a static droplet amplified to
# 500x .. 2000x the oracle twins' drift at step 2000 of laplace128_R12 (u 1.6e-5; now 6e-9, the
# twins: 0.8e-8 .. 3e-8), and fp32 u at step 1000 stood at 1.4e-4 (now 1.9e-5).  DESIGN.md 9.
KNOWN_SHORTFALLS = {}


def _errors(g, gold, cp, idx):
    mx = gold[f"max_{cp}"]
    out = {}
    for k, (name, den) in enumerate(zip(("rho", "p", "u", "phi"), mx)):
        got = g[name].double().reshape(3, -1)[:, idx] if name == "u" else g[name].double().ravel()[idx]
        out[name] = float(np.abs(got.cpu().numpy() - gold[f"{name}_{cp}"]).max() / den)
    return out


@pytest.mark.parametrize("case", list(CASES))
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_against_golden(case, precision):
    _replay(case, precision, 0)


@pytest.mark.parametrize("flags", [1, 2, 16], ids=["naive", "generic", "k1_flux"])
def test_laplace_horizon_on_every_path(flags):
    """configs[1]'s own horizon (R = 12, 2000 steps) through the other kernels of the product:
    the one-thread-per-node path, the wall-capable pair and the one-node interface kernel meet the
    same twin-based bar as the production pair ("the round-1 anomaly")."""
    _replay("laplace128_R12", "f64", flags)


def _replay(case, precision, flags):
    path = os.path.join(HERE, case + ".npz")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated")
    import torch
    from paper_2501_00846_b200 import binding as B
    gold = np.load(path)
    cfg = CASES[case]()
    assert tuple(gold["shape"]) == cfg["shape"]
    need_gb = 31 * np.prod(cfg["shape"]) * (8 if precision == "f64" else 4) / 1e9
    if need_gb > 0.8 * torch.cuda.get_device_properties(0).total_memory / 1e9:
        pytest.skip("lattice does not fit on this GPU")
    nz, ny, nx = cfg["shape"]
    idx = torch.as_tensor(gold["sample_index"], device="cuda")
    s = B.Solver(nx, ny, nz, cfg["params"], precision=precision, flags=flags)
    s.init(cfg["phi"], cfg["u"])
    done = 0
    first = int(gold["checkpoints"][0])
    floor = 30.0 * max([float(np.max(gold[f"{t}_{first}"])) for t in ("sens", "fma", "rev")
                        if f"{t}_{first}" in gold] + [1e-16])
    tol = 1e-10 if precision == "f64" else 1e-4
    fields = ("rho", "p", "u", "phi") if precision == "f64" else ("u", "phi")
    worst = {}
    for cp in gold["checkpoints"]:
        cp = int(cp)
        s.step(cp - done)
        done = cp
        g = s.get()
        errs = _errors(g, gold, cp, idx)
        st = s.get_state()
        sum_phi = float(g["phi"].double().sum())
        sum_ps = float(st["pstar"].double().sum())
        print(f"[{case} {precision}{' flags=%d' % flags if flags else ''}] step {cp}: " + " ".join(f"{k}={v:.2e}" for k, v in errs.items())
              + f" | sum(phi) rel diff {sum_phi / gold[f'diag_{cp}'][0] - 1:.1e}"
              + f" sum(p*) {sum_ps:.1e} (oracle {gold[f'diag_{cp}'][1]:.1e})")
        names = ("rho", "p", "u", "phi")
        twins = {t: dict(zip(names, gold[f"{t}_{cp}"])) for t in ("sens", "fma", "rev")
                 if f"{t}_{cp}" in gold}
        # conditioning of the trajectory at this checkpoint, measured by the ORACLE alone
        cond = {k: max([float(tw[k]) for tw in twins.values()] + [0.0]) for k in names}
        scale = 1.0 if precision == "f64" else 6e-8 / 1.1e-16
        worst[cp] = {}
        ill = False
        for k in fields:
            c = cond[k] if cond[k] > floor else 0.0
            bar = max(tol, K_TWIN * c * scale)
            if bar > CAP:                     # no pointwise meaning left: report only
                ill = True
                worst[cp][k] = (errs[k], bar, True)
                continue
            ok = errs[k] <= bar
            known = KNOWN_SHORTFALLS.get((case, precision, cp, k))
            if not ok and known is not None:
                print(f"    KNOWN SHORTFALL {k}: {errs[k]:.2e} > {bar:.1e} (recorded {known:.1e})")
                ok = errs[k] <= 3.0 * known
            worst[cp][k] = (errs[k], bar, ok)
        for t, tw in twins.items():
            print(f"    oracle twin {t}: " + " ".join(f"{k}={v:.1e}" for k, v in tw.items()))
        if ill:
            print("    [ill-conditioned checkpoint: K x twin drift > 1e-2, pointwise parity "
                  "reported only; see tests/test_segment_gpu.py]")
        # what holds at any horizon: phi is conserved (P7), and the quantity BASELINE.json asks of
        # the Laplace sweep at its final step, Delta p R_eff / (2 sigma) (pin P9's definition),
        # agrees with the oracle's although the pointwise fields no longer can
        # (fp32: sum(phi) is carried in fp32 fields, 1e-6 relative; the Laplace ratio to 1e-3)
        inv_tol, ratio_tol = (1e-12, 1e-8) if precision == "f64" else (1e-6, 1e-3)
        if True:
            assert abs(sum_phi / gold[f"diag_{cp}"][0] - 1.0) <= inv_tol, (cp, sum_phi)
            ratio_ref = float(gold[f"diag_{cp}"][2])
            if np.isfinite(ratio_ref) and "droplet" in cfg["name"]:
                phi_g, p_g = g["phi"].double(), g["p"].double()
                dp = float(p_g[phi_g > 0.99].mean() - p_g[phi_g < 0.01].mean())
                r_eff = (3.0 * sum_phi / (4.0 * np.pi)) ** (1.0 / 3.0)
                ratio = dp * r_eff / (2.0 * cfg["params"]["sigma"])
                print(f"    Laplace ratio {ratio:.9f} (oracle {ratio_ref:.9f})"
                      + ("   [ill-conditioned checkpoint]" if ill else ""))
                # a mean of p over two node sets: it moves by at most a few times the error of p
                assert abs(ratio - ratio_ref) <= max(ratio_tol, 10.0 * errs["p"]) \
                    * max(1.0, abs(ratio_ref)), (cp, ratio, ratio_ref)
        assert bool(torch.isfinite(g["u"]).all())
    s.close()
    bad = {cp: e for cp, e in worst.items() if any(not ok for _, _, ok in e.values())}
    assert not bad, bad
