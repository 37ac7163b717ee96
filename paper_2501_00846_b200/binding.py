"""Thin Python binding of the C ABI in include/tslb.h (same names, argument marshalling only).

PyTorch supplies device memory and streams; every step of the path runs in the CUDA kernels of
libtslb.so.  There is no CPU fallback: a missing library or a missing GPU raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtslb.so")

BC_PERIODIC, BC_WALL = 0, 1
F32, F64 = 0, 1
FLAG_NAIVE, FLAG_GENERIC, FLAG_K2_CPASYNC, FLAG_K2_TMA, FLAG_K1_FLUX = 1, 2, 4, 8, 16
FLAG_BODY_HEAVY = 32        # body force (rho - rho_g) g instead of (rho - rho_l) g
NDIAG = 16
DIAG_NAMES = ("sum_phi", "sum_pstar", "max_u", "sum_phi_x", "sum_phi_y", "sum_phi_z",
              "sum_phi_ux", "sum_phi_uy", "sum_phi_uz", "sum_ux", "sum_uy", "sum_uz",
              "sum_p_in", "n_in", "sum_p_out", "n_out")

SYMBOLS = ("tslb_workspace_bytes", "tslb_create", "tslb_init", "tslb_step", "tslb_get",
           "tslb_get_state", "tslb_set_state", "tslb_init_host", "tslb_get_host", "tslb_step_timed",
           "tslb_launch_count", "tslb_diag", "tslb_diag_host", "tslb_diag_static", "tslb_fma_peak",
           "tslb_halo_bytes", "tslb_halo_pack", "tslb_halo_unpack",
           "tslb_slab_set_ends", "tslb_slab_step_faces", "tslb_slab_step_interior",
           "tslb_destroy", "tslb_last_error")


class tslb_params(C.Structure):
    _fields_ = [("rho_l", C.c_double), ("rho_g", C.c_double),
                ("mu_l", C.c_double), ("mu_g", C.c_double),
                ("sigma", C.c_double), ("delta", C.c_double), ("mobility", C.c_double),
                ("body_accel", C.c_double * 3), ("bc", C.c_int * 3),
                ("precision", C.c_int), ("flags", C.c_int)]


def make_params(rho_l, rho_g, mu_l, mu_g, sigma, delta, mobility, body_accel=(0.0, 0.0, 0.0),
                bc=(0, 0, 0), precision=F64, flags=0, body_heavy=False):
    p = tslb_params()
    p.rho_l, p.rho_g, p.mu_l, p.mu_g = rho_l, rho_g, mu_l, mu_g
    p.sigma, p.delta, p.mobility = sigma, delta, mobility
    p.body_accel[:] = [float(v) for v in body_accel]
    p.bc[:] = [int(v) for v in bc]
    p.precision = int(precision)
    p.flags = int(flags) | (FLAG_BODY_HEAVY if body_heavy else 0)
    return p


_lib = None


def load():
    """dlopen libtslb.so and declare the prototypes.  Raises if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run __graft_entry__.build() "
                           "(python -m paper_2501_00846_b200.build); there is no CPU fallback")
    lib = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    lib.tslb_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(tslb_params)]
    lib.tslb_workspace_bytes.restype = C.c_size_t
    lib.tslb_create.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(tslb_params), vp, vp,
                                C.POINTER(vp)]
    lib.tslb_init.argtypes = [vp, vp, vp]
    lib.tslb_step.argtypes = [vp, C.c_int]
    lib.tslb_get.argtypes = [vp, vp, vp, vp, vp]
    lib.tslb_get_state.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.tslb_set_state.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.tslb_init_host.argtypes = [vp, vp, vp]
    lib.tslb_get_host.argtypes = [vp, vp, vp, vp, vp]
    lib.tslb_step_timed.argtypes = [vp, C.c_int, C.POINTER(C.c_float)]
    lib.tslb_diag.argtypes = [vp, vp]
    lib.tslb_diag_host.argtypes = [vp, C.POINTER(C.c_double)]
    lib.tslb_diag_static.argtypes = [vp, vp]
    lib.tslb_fma_peak.argtypes = [C.c_int, vp, C.POINTER(C.c_double)]
    lib.tslb_halo_bytes.argtypes = [vp]
    lib.tslb_halo_bytes.restype = C.c_size_t
    lib.tslb_halo_pack.argtypes = [vp, C.c_int, vp]
    lib.tslb_halo_unpack.argtypes = [vp, C.c_int, vp]
    lib.tslb_slab_set_ends.argtypes = [vp, C.c_int, C.c_int]
    lib.tslb_slab_step_faces.argtypes = [vp]
    lib.tslb_slab_step_interior.argtypes = [vp]
    lib.tslb_launch_count.argtypes = [vp]
    lib.tslb_launch_count.restype = C.c_longlong
    lib.tslb_destroy.argtypes = [vp]
    lib.tslb_destroy.restype = None
    lib.tslb_last_error.restype = C.c_char_p
    _lib = lib
    return lib


class TslbError(RuntimeError):
    pass


def _check(rc, what):
    if rc != 0:
        raise TslbError(f"{what} failed ({rc}): {load().tslb_last_error().decode()}")


def tslb_workspace_bytes(nx, ny, nz, params):
    return int(load().tslb_workspace_bytes(nx, ny, nz, C.byref(params)))


def tslb_fma_peak(precision="f64", stream=None):
    """Measured FMA throughput (TFLOP/s) of the plain ALUs on the current device."""
    out = C.c_double()
    _check(load().tslb_fma_peak(F64 if precision == "f64" else F32,
                                stream.cuda_stream if stream is not None else None,
                                C.byref(out)), "tslb_fma_peak")
    return float(out.value)


class Solver:
    """tslb_create / tslb_init / tslb_step / tslb_get on torch device memory.

    Fields are torch tensors shaped (nz, ny, nx) (x fastest), vectors (3, nz, ny, nx), in the
    solver's precision, on the solver's device.  The workspace tensor is owned here."""

    def __init__(self, nx, ny, nz, params, precision="f64", flags=0, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("tslb needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.lib = load()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.device = torch.device(device)
        self.dtype = torch.float64 if precision == "f64" else torch.float32
        self.np_dtype = np.float64 if precision == "f64" else np.float32
        prm = dict(params)
        prm["precision"] = F64 if precision == "f64" else F32
        prm["flags"] = flags
        self.params = make_params(**prm)
        nbytes = tslb_workspace_bytes(nx, ny, nz, self.params)
        if nbytes == 0:
            raise TslbError("tslb_workspace_bytes: bad size or parameters")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        assert self.workspace.data_ptr() % 256 == 0
        self._h = C.c_void_p()
        _check(self.lib.tslb_create(nx, ny, nz, C.byref(self.params), self.workspace.data_ptr(),
                                    self.stream.cuda_stream, C.byref(self._h)), "tslb_create")

    # -- helpers -------------------------------------------------------------------------
    def _call(self, name, *args):
        """One ABI call with the solver's device current (launch attributes, the static scratch
        of tslb_diag_static and the stream all belong to a device)."""
        with self.torch.cuda.device(self.device):
            _check(getattr(self.lib, name)(self._h, *args), name)

    def _dev(self, a, shape):
        t = self.torch.as_tensor(a)
        t = t.to(device=self.device, dtype=self.dtype).contiguous()
        assert tuple(t.shape) == shape, (tuple(t.shape), shape)
        return t

    def _empty(self, *lead):
        return self.torch.empty(tuple(lead) + self.shape, dtype=self.dtype, device=self.device)

    # -- the ABI calls -------------------------------------------------------------------
    def init(self, phi, u):
        """tslb_init from device tensors (host arrays are copied to the device by torch first)."""
        phi = self._dev(phi, self.shape)
        u = self._dev(u, (3,) + self.shape)
        self._call("tslb_init", phi.data_ptr(), u.data_ptr())
        self.stream.synchronize()          # phi, u may be temporaries

    def init_host(self, phi, u):
        """tslb_init_host from host arrays/tensors of the solver's precision (pinned = async)."""
        phi, u = self._host_ptr(phi, self.shape), self._host_ptr(u, (3,) + self.shape)
        self._call("tslb_init_host", phi[1], u[1])
        self.stream.synchronize()
        return self

    def step(self, n=1):
        self._call("tslb_step", int(n))

    def step_timed(self, n=1):
        """tslb_step_timed: returns {kernel kind: total ms over the n steps} (synchronises)."""
        ms = (C.c_float * 4)()
        self._call("tslb_step_timed", int(n), ms)
        names = ("normal", "allen_cahn", "stream_collide", "reserved")
        return {k: float(v) for k, v in zip(names, ms) if v > 0.0}

    def get(self, want=("rho", "p", "u", "phi")):
        out = {k: (self._empty(3) if k == "u" else self._empty()) for k in want}
        ptr = lambda k: out[k].data_ptr() if k in out else None
        self._call("tslb_get", ptr("rho"), ptr("p"), ptr("u"), ptr("phi"))
        return out

    def get_state(self):
        out = dict(pstar=self._empty(), u=self._empty(3), A=self._empty(6), a=self._empty(3),
                   phi=self._empty())
        self._call("tslb_get_state", out["pstar"].data_ptr(), out["u"].data_ptr(),
                   out["A"].data_ptr(), out["a"].data_ptr(), out["phi"].data_ptr())
        return out

    def set_state(self, state):
        """tslb_set_state from a dict as get_state returns it (restart / resume)."""
        t = {"pstar": self._dev(state["pstar"], self.shape), "u": self._dev(state["u"], (3,) + self.shape),
             "A": self._dev(state["A"], (6,) + self.shape), "a": self._dev(state["a"], (3,) + self.shape),
             "phi": self._dev(state["phi"], self.shape)}
        self._call("tslb_set_state", t["pstar"].data_ptr(), t["u"].data_ptr(), t["A"].data_ptr(),
                   t["a"].data_ptr(), t["phi"].data_ptr())
        self.stream.synchronize()          # the arrays may be temporaries

    def halo_buffer(self):
        """A device tensor of tslb_halo_bytes for tslb_halo_pack / tslb_halo_unpack."""
        n = int(self.lib.tslb_halo_bytes(self._h))
        es = 8 if self.dtype == self.torch.float64 else 4
        return self.torch.empty(n // es, dtype=self.dtype, device=self.device)

    def halo_pack(self, face, buf):
        self._call("tslb_halo_pack", int(face), buf.data_ptr())

    def halo_unpack(self, face, buf):
        self._call("tslb_halo_unpack", int(face), buf.data_ptr())

    def slab_set_ends(self, ghost_low, ghost_high):
        """Which z ends carry two ghost planes (the others are walls of the global box)."""
        self._call("tslb_slab_set_ends", int(bool(ghost_low)), int(bool(ghost_high)))

    def slab_step_faces(self):
        """First stage of a slab's step: afterwards halo_pack packs the NEW face planes."""
        self._call("tslb_slab_step_faces")

    def slab_step_interior(self):
        self._call("tslb_slab_step_interior")

    def diag(self):
        """tslb_diag_host: dict of the TSLB_D_* box reductions (synchronises the stream)."""
        out = (C.c_double * NDIAG)()
        self._call("tslb_diag_host", out)
        return dict(zip(DIAG_NAMES, out))

    def diag_device(self):
        """tslb_diag into a device tensor of NDIAG doubles (no synchronisation)."""
        out = self.torch.empty(NDIAG, dtype=self.torch.float64, device=self.device)
        self._call("tslb_diag", out.data_ptr())
        return out

    def diag_static(self, out=None):
        """tslb_diag_static (no workspace scratch, no allocation inside the library) into the
        caller's device tensor `out` of NDIAG doubles (made here if None); no synchronisation."""
        if out is None:
            out = self.torch.empty(NDIAG, dtype=self.torch.float64, device=self.device)
        assert out.dtype == self.torch.float64 and out.numel() == NDIAG and out.is_contiguous()
        assert out.device == self.device
        self._call("tslb_diag_static", out.data_ptr())
        return out

    def get_host(self, out):
        """tslb_get_host into a dict of host arrays/tensors {rho,p,u,phi} (any subset)."""
        ptrs = {k: self._host_ptr(v, ((3,) if k == "u" else ()) + self.shape)[1]
                for k, v in out.items()}
        self._call("tslb_get_host", ptrs.get("rho"), ptrs.get("p"), ptrs.get("u"),
                   ptrs.get("phi"))
        return out

    def _host_ptr(self, a, shape):
        if isinstance(a, np.ndarray):
            assert a.dtype == self.np_dtype and a.flags.c_contiguous and a.shape == shape
            return a, a.ctypes.data
        assert a.device.type == "cpu" and a.dtype == self.dtype and a.is_contiguous()
        assert tuple(a.shape) == shape
        return a, a.data_ptr()

    @property
    def launches(self):
        return int(self.lib.tslb_launch_count(self._h))

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        if getattr(self, "_h", None):
            self.stream.synchronize()
            self.lib.tslb_destroy(self._h)
            self._h = C.c_void_p()
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
