"""ctypes loader for the CPU ORACLE (oracle/tslb_ref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from
paper_2501_00846_b200 and holds no arithmetic of the method (argument marshalling only).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tslb_ref.c")
_LIB = os.path.join(_HERE, "libtslb_ref.so")
# Conditioning twin (R22, section 9): the SAME source built with FMA contraction on, i.e.
# another rounding at every multiply-add of every node and step.  Selected by the environment
# variable TSLB_REF_FMA=1 before the first call; used only by tests/golden/make_golden.py
# --twin-fma to measure how far two correct roundings of this oracle drift apart.  Expected
# values always come from the contraction-off build.
_LIB_FMA = os.path.join(_HERE, "libtslb_ref_fma.so")
# Second conditioning twin: the same source with every sum over the 27 directions taken in
# reverse order (TSLB_REF_REV=1, -DTSLB_REF_REVERSE_SUMS, make_golden.py --twin-rev).
_LIB_REV = os.path.join(_HERE, "libtslb_ref_rev.so")

PERIODIC, WALL = 0, 1


def build_lib(force=False, fma=False, rev=False):
    """gcc -O3, contraction off (R22), OpenMP over nodes.  No -march flag: the .so travels.
    fma=True builds the conditioning twin (contraction on, -mfma) next to it."""
    hdr = os.path.join(_HERE, "tslb_ref.h")
    out = _LIB_FMA if fma else (_LIB_REV if rev else _LIB)
    if (not force and os.path.exists(out)
            and os.path.getmtime(out) >= max(os.path.getmtime(_SRC), os.path.getmtime(hdr))):
        return out
    tmp = out + f".{os.getpid()}.tmp"        # build aside, then rename: a process that has the
    flags = ["-ffp-contract=fast", "-mfma"] if fma else ["-ffp-contract=off"]
    if rev:
        flags.append("-DTSLB_REF_REVERSE_SUMS")
    subprocess.check_call(["gcc", "-O3"] + flags + ["-fopenmp", "-fPIC", "-shared",
                           "-Wall", "-o", tmp, _SRC, "-lm"])       # old library mapped keeps it
    os.replace(tmp, out)
    return out


class Params(C.Structure):
    _fields_ = [("rho_l", C.c_double), ("rho_g", C.c_double),
                ("mu_l", C.c_double), ("mu_g", C.c_double),
                ("sigma", C.c_double), ("delta", C.c_double), ("mobility", C.c_double),
                ("body_accel", C.c_double * 3), ("bc", C.c_int * 3),
                ("body_heavy", C.c_int)]


def make_params(rho_l, rho_g, mu_l, mu_g, sigma, delta, mobility,
                body_accel=(0.0, 0.0, 0.0), bc=(0, 0, 0), body_heavy=False):
    p = Params()
    p.rho_l, p.rho_g, p.mu_l, p.mu_g = rho_l, rho_g, mu_l, mu_g
    p.sigma, p.delta, p.mobility = sigma, delta, mobility
    p.body_accel[:] = [float(v) for v in body_accel]
    p.bc[:] = [int(v) for v in bc]
    p.body_heavy = 1 if body_heavy else 0
    return p


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_lib(fma=os.environ.get("TSLB_REF_FMA") == "1",
                                rev=os.environ.get("TSLB_REF_REV") == "1"))
        _lib.tslb_ref_create.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(Params),
                                         C.POINTER(C.c_void_p)]
        _lib.tslb_ref_init.argtypes = [C.c_void_p, _dp, _dp]
        _lib.tslb_ref_step.argtypes = [C.c_void_p, C.c_int]
        _lib.tslb_ref_get.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
        _lib.tslb_ref_get_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
        _lib.tslb_ref_set_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
        _lib.tslb_ref_diag.argtypes = [C.c_void_p, _dp]
        _lib.tslb_ref_destroy.argtypes = [C.c_void_p]
        _lib.tslb_ref_destroy.restype = None
        _lib.tslb_ref_omega.argtypes = [C.POINTER(Params), C.c_double]
        _lib.tslb_ref_omega.restype = C.c_double
        for name in ("tslb_ref_lattice", "tslb_ref_feq", "tslb_ref_fneq", "tslb_ref_forcing",
                     "tslb_ref_gradient", "tslb_ref_laplacian", "tslb_ref_divergence"):
            getattr(_lib, name).restype = None
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class RefSim:
    """Whole-lattice oracle.  Arrays are numpy fp64 shaped (nz, ny, nx) (x fastest); vectors
    (3, nz, ny, nx); the stress tensor (6, nz, ny, nx) in the order xx,yy,zz,xy,xz,yz."""

    def __init__(self, nx, ny, nz, params):
        self.nx, self.ny, self.nz = nx, ny, nz
        self.shape = (nz, ny, nx)
        self.params = params
        self._h = C.c_void_p()
        rc = lib().tslb_ref_create(nx, ny, nz, C.byref(params), C.byref(self._h))
        if rc != 0:
            raise ValueError(f"tslb_ref_create failed: {rc}")

    def init(self, phi, u):
        phi, u = _f64(phi), _f64(u)
        assert phi.shape == self.shape and u.shape == (3,) + self.shape
        rc = lib().tslb_ref_init(self._h, _p(phi), _p(u))
        assert rc == 0, rc

    def step(self, n=1):
        rc = lib().tslb_ref_step(self._h, int(n))
        if rc != 0:
            raise RuntimeError(f"tslb_ref_step failed: {rc}")

    def get(self):
        rho = np.empty(self.shape); p = np.empty(self.shape)
        u = np.empty((3,) + self.shape); phi = np.empty(self.shape)
        rc = lib().tslb_ref_get(self._h, _p(rho), _p(p), _p(u), _p(phi))
        assert rc == 0, rc
        return rho, p, u, phi

    def get_state(self):
        ps = np.empty(self.shape); u = np.empty((3,) + self.shape)
        A = np.empty((6,) + self.shape); a = np.empty((3,) + self.shape)
        phi = np.empty(self.shape)
        rc = lib().tslb_ref_get_state(self._h, _p(ps), _p(u), _p(A), _p(a), _p(phi))
        assert rc == 0, rc
        return ps, u, A, a, phi

    def set_state(self, pstar, u, A, a, phi):
        """Replace the whole state (a2_neq itself in A); copies only (segment-parity restarts)."""
        arrs = [_f64(x) for x in (pstar, u, A, a, phi)]
        want = [self.shape, (3,) + self.shape, (6,) + self.shape, (3,) + self.shape, self.shape]
        assert [x.shape for x in arrs] == want
        rc = lib().tslb_ref_set_state(self._h, *[_p(x) for x in arrs])
        assert rc == 0, rc

    def diag(self):
        """tslb_ref_diag: the 16 box reductions, in the order of include/tslb.h's TSLB_D_*."""
        out = np.empty(16)
        rc = lib().tslb_ref_diag(self._h, _p(out))
        assert rc == 0, rc
        return out

    def close(self):
        if self._h:
            lib().tslb_ref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lattice():
    c = (C.c_int * 3 * 27)(); w = (C.c_double * 27)(); opp = (C.c_int * 27)()
    lib().tslb_ref_lattice(c, w, opp)
    return (np.array([[c[i][k] for k in range(3)] for i in range(27)]),
            np.array(list(w)), np.array(list(opp)))


def _node27(fn, *args):
    out = np.empty(27)
    fn(*args, _p(out))
    return out


def feq(pstar, u):
    return _node27(lib().tslb_ref_feq, C.c_double(pstar), _p(_f64(u)))


def fneq(u, A):
    return _node27(lib().tslb_ref_fneq, _p(_f64(u)), _p(_f64(A)))


def forcing(u, a):
    return _node27(lib().tslb_ref_forcing, _p(_f64(u)), _p(_f64(a)))


def omega(params, phi):
    return lib().tslb_ref_omega(C.byref(params), float(phi))


def _bc3(bc):
    return (C.c_int * 3)(*[int(b) for b in bc])


def gradient(psi, bc=(0, 0, 0)):
    psi = _f64(psi); nz, ny, nx = psi.shape
    out = np.empty((3, nz, ny, nx))
    lib().tslb_ref_gradient(_p(psi), nx, ny, nz, _bc3(bc), _p(out))
    return out


def laplacian(psi, bc=(0, 0, 0)):
    psi = _f64(psi); nz, ny, nx = psi.shape
    out = np.empty((nz, ny, nx))
    lib().tslb_ref_laplacian(_p(psi), nx, ny, nz, _bc3(bc), _p(out))
    return out


def divergence(G, bc=(0, 0, 0), ghost_rule=0):
    G = _f64(G); _, nz, ny, nx = G.shape
    out = np.empty((nz, ny, nx))
    lib().tslb_ref_divergence(_p(G), nx, ny, nz, _bc3(bc), int(ghost_rule), _p(out))
    return out
