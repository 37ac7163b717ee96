"""Host-side checks of the C-ABI boundary (no GPU needed): the library builds, loads, exports
every symbol include/tslb.h declares, and validates its arguments as the header states."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2501_00846_b200 import build, binding
    build.build_cuda()
    binding.load()
    return binding


def good(B, **kw):
    d = dict(rho_l=1.0, rho_g=1e-3, mu_l=1 / 60, mu_g=1 / 6000, sigma=1e-3, delta=4.0,
             mobility=0.05)
    d.update(kw)
    return B.make_params(**d)


def test_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "tslb.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(tslb_[a-z_]+)\s*\(", hdr))
    assert declared == set(B.SYMBOLS)
    lib = B.load()
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_layout_matches_header(B):
    # 10 doubles, 3 + 1 + 1 ints
    assert C.sizeof(B.tslb_params) == 10 * 8 + 5 * 4 + 4
    assert B.tslb_params.bc.offset == 80 and B.tslb_params.precision.offset == 92


def test_workspace_bytes(B):
    p64, p32 = good(B), good(B, precision=B.F32)
    n = 32 ** 3
    # 2 x 14 state planes + 3 flux planes + the tslb_diag rows (one row of 16 doubles per 8192
    # nodes plus one result row, rounded up to 256 bytes)
    diag = lambda nodes: (((nodes + 8191) // 8192 + 1) * 128 + 255) // 256 * 256
    assert B.tslb_workspace_bytes(32, 32, 32, p64) == 31 * n * 8 + diag(n)
    assert B.tslb_workspace_bytes(32, 32, 32, p32) == 31 * n * 4 + diag(n)
    # planes are padded to 256 bytes
    assert B.tslb_workspace_bytes(5, 5, 5, p64) == 31 * 1024 + 256
    assert B.tslb_workspace_bytes(32, 32, 32, good(B, flags=B.FLAG_NAIVE)) == 31 * n * 8 + diag(n)
    assert B.tslb_workspace_bytes(0, 32, 32, p64) == 0
    assert B.tslb_workspace_bytes(3, 32, 32, p64) == 0            # periodic axis needs >= 4
    assert B.tslb_workspace_bytes(2, 32, 32, good(B, bc=(1, 0, 0))) > 0
    assert B.tslb_workspace_bytes(32, 32, 32, good(B, rho_g=0.0)) == 0
    assert B.tslb_workspace_bytes(32, 32, 32, good(B, precision=7)) == 0


def test_create_argument_errors(B):
    lib = B.load()
    h = C.c_void_p()
    fake = C.c_void_p(1 << 20)                                     # never dereferenced by create
    assert lib.tslb_create(32, 32, 32, C.byref(good(B)), fake, None, C.byref(h)) == 0
    assert lib.tslb_step(h, 1) == -4                               # before init
    assert b"before tslb_init" in lib.tslb_last_error()
    assert lib.tslb_step(h, -1) == -1
    assert lib.tslb_get(h, None, None, None, None) == -4
    assert lib.tslb_launch_count(h) == 0
    lib.tslb_destroy(h)
    assert lib.tslb_create(32, 32, 32, C.byref(good(B)), C.c_void_p((1 << 20) + 8), None,
                           C.byref(h)) == -2
    assert lib.tslb_create(32, 32, 32, C.byref(good(B)), None, None, C.byref(h)) == -2
    assert lib.tslb_create(32, 32, 32, C.byref(good(B, mu_l=-1.0)), fake, None, C.byref(h)) == -1
    assert lib.tslb_create(32, 32, 32, C.byref(good(B, bc=(0, 2, 0))), fake, None, C.byref(h)) == -1
    assert lib.tslb_create(32, 32, 32, C.byref(good(B)), fake, None, None) == -1
    # flags: only the documented validation selectors; a stray bit never selects anything
    for ok in (0, 1, 2, 4, 8, 16, 8 | 16):
        assert lib.tslb_create(32, 32, 32, C.byref(good(B, flags=ok)), fake, None, C.byref(h)) == 0
        lib.tslb_destroy(h)
    for stray in (64, 1 << 8, 59 << 8, 1 << 16, 1 << 23):
        assert lib.tslb_create(32, 32, 32, C.byref(good(B, flags=stray)), fake, None,
                               C.byref(h)) == -1
    assert lib.tslb_step(None, 1) == -1
    lib.tslb_destroy(None)


def test_solver_fails_loudly_without_gpu(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        B.Solver(8, 8, 8, dict(rho_l=1.0, rho_g=1e-3, mu_l=1 / 60, mu_g=1 / 6000, sigma=1e-3,
                               delta=4.0, mobility=0.05))
