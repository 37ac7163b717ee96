"""BASELINE.json configs[1] as stated: the Laplace sweep, 128^3, R in {12, 16, 24, 32}, 2000 steps,
fp64 and fp32, "check Delta p R / (2 sigma)".  A physics check of the CUDA path on its own (the
oracle's version of it is pin P9): Laplace's law Delta p = 2 sigma / R_eff, with
R_eff = (3 sum(phi) / 4 pi)^(1/3), p = p* rho cs^2 averaged over phi > 0.99 and phi < 0.01, all read
through the on-device diagnostics (tslb_diag, no field comes back to the host).

The pressure jump must be TIME-AVERAGED: the p* = 0 start (R9) leaves an undamped breathing mode,
the instantaneous ratio swings between 0.2 and 1.7 even in the last 250 steps and its period grows
with R, so SURVEY.md's window 1751-2000 is shorter than one period for R >= 16 (its mean there:
0.985, 0.93, 0.97, 0.90).  The window used is steps 1010-2000, sampled every 10 steps: measured
means 0.985, 0.975, 0.972, 0.976 (both precisions).  Asserted: within 5 % of 1 (the diffuse
interface is 4 nodes wide on droplets of 12-32), and fp32 within 1e-3 of fp64."""
import numpy as np
import pytest

from paper_2501_00846_b200 import inputs as I

pytestmark = pytest.mark.gpu


def _window_mean(radius, precision):
    from paper_2501_00846_b200 import binding as B
    cfg = I.static_droplet(128, float(radius), seed=int(radius))
    s = B.Solver(128, 128, 128, cfg["params"], precision=precision)
    s.init(cfg["phi"], cfg["u"])
    sigma = cfg["params"]["sigma"]
    d0 = s.diag()
    s.step(1000)
    ratios = []
    for _ in range(100):
        s.step(10)
        d = s.diag()
        dp = d["sum_p_in"] / d["n_in"] - d["sum_p_out"] / d["n_out"]
        r_eff = (3.0 * d["sum_phi"] / (4.0 * np.pi)) ** (1.0 / 3.0)
        ratios.append(dp * r_eff / (2.0 * sigma))
    s.close()
    assert np.isfinite(d["max_u"]) and d["max_u"] < 1e-3          # still a static droplet
    assert abs(d["sum_phi"] / d0["sum_phi"] - 1.0) <= (1e-12 if precision == "f64" else 1e-6)
    return float(np.mean(ratios)), float(np.min(ratios)), float(np.max(ratios)), r_eff


@pytest.mark.parametrize("radius", [12, 16, 24, 32])
def test_laplace_law_over_the_sweep(radius):
    m64, lo, hi, r_eff = _window_mean(radius, "f64")
    m32, _, _, _ = _window_mean(radius, "f32")
    print(f"[laplace sweep R={radius}] R_eff={r_eff:.3f}  mean Delta p R_eff/(2 sigma) over steps "
          f"1010..2000: fp64 {m64:.4f}, fp32 {m32:.4f}  (instantaneous {lo:.2f} .. {hi:.2f})")
    assert abs(m64 - 1.0) <= 0.05, m64
    assert abs(m32 - m64) <= 1e-3, (m32, m64)
