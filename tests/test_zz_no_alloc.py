"""tslb_diag_static, the allocation-free entry point (include/tslb.h): same result as tslb_diag,
whose partial sums live in the caller's workspace, although its scratch is a static device array
shared by every call.  Collected last on purpose (pytest -x would hide what follows a failure).
Passes alone in a fresh process and after the other tests."""
import ctypes as C

import numpy as np
import pytest

from paper_2501_00846_b200 import inputs as I


def test_rejects_lattices_beyond_the_static_scratch():
    """Size check comes first and needs no GPU: 384^3 > TSLB_DIAG_STATIC_MAX_NODES."""
    from paper_2501_00846_b200 import build, binding as B
    build.build_cuda()
    lib = B.load()
    prm = B.make_params(rho_l=1.0, rho_g=1e-3, mu_l=1 / 60, mu_g=1 / 6000, sigma=1e-3, delta=4.0,
                        mobility=0.05)
    h = C.c_void_p()
    fake = C.c_void_p(1 << 20)                        # never dereferenced by tslb_create
    assert lib.tslb_create(384, 384, 384, C.byref(prm), fake, None, C.byref(h)) == 0
    assert lib.tslb_diag_static(h, fake) == -1
    msg = lib.tslb_last_error().decode()
    assert "exceeds the static scratch" in msg and str(4096 * 8192) in msg
    lib.tslb_destroy(h)
    assert lib.tslb_create(320, 320, 320, C.byref(prm), fake, None, C.byref(h)) == 0
    assert lib.tslb_diag_static(h, fake) == -4        # fits; but not initialised yet
    assert lib.tslb_diag_static(h, None) == -1
    lib.tslb_destroy(h)


@pytest.mark.gpu
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_static_scratch_matches_workspace_scratch_twice(precision):
    """Two calls in a row on lattices of DIFFERENT size (the second, smaller one finds the first
    one's rows in the shared array and must not read them), each against tslb_diag on the same
    state.  Same kernels and reduction order, so the bar is equality; the tests' fp64 tolerance
    (1e-10) is asserted as well for the record."""
    import torch
    from paper_2501_00846_b200 import binding as B
    big = I.head_on_collision(n=48, radius=7.0, half_sep=11.0, noise=1e-4)      # 14 rows
    small = I.static_droplet(24, 6.0, seed=9, noise=1e-4)                        # 2 rows
    out = torch.full((B.NDIAG,), float("nan"), dtype=torch.float64, device="cuda:0")
    for cfg, steps in ((big, 6), (small, 9), (big, 3)):
        nz, ny, nx = cfg["shape"]
        s = B.Solver(nx, ny, nz, cfg["params"], precision=precision)
        s.init(cfg["phi"], cfg["u"])
        s.step(steps)
        want = s.diag_device().cpu().numpy()
        got = s.diag_static(out).cpu().numpy().copy()
        s.step(1)                                     # the state moves on; call again
        want2 = s.diag_device().cpu().numpy()
        got2 = s.diag_static(out).cpu().numpy().copy()
        s.close()
        for g, w in ((got, want), (got2, want2)):
            assert np.isfinite(g).all() and g[0] > 0
            assert np.all(np.abs(g - w) <= 1e-10 * (np.abs(w) + 1e-3 * np.abs(w).max()))
            assert np.array_equal(g, w), (g, w)
        assert not np.array_equal(got, got2)
