"""Thin ctypes binding over include/lb.h -- argument marshalling only.

Every function here has the name and meaning of the C entry point it wraps; every step
of the lattice-Boltzmann path runs in the CUDA kernels behind them.  There is no
fallback: if the shared library is missing the import of `lib()` raises, and if no CUDA
device is present `lb_create*` raises with the library's own message.

This module never imports anything from `oracle/`.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

LB_OK, LB_EINVAL, LB_ENOMEM, LB_ECUDA, LB_ESTATE = 0, -1, -2, -3, -4
LB_F64, LB_F32 = 0, 1
LB_KERNEL_AUTO, LB_KERNEL_TWOPASS, LB_KERNEL_ONEPASS, LB_KERNEL_TMA, LB_KERNEL_HALO, LB_KERNEL_NODE = 0, 1, 2, 3, 4, 5
LB_OPT_ZC, LB_OPT_DIAG, LB_OPT_BALANCE = 1, 2, 3
LB_MODEL_SHAN_CHEN, LB_MODEL_COLOUR_GRADIENT = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "_lib", "liblb_b200.so")

# every symbol include/lb.h declares
SYMBOLS = (
    "lb_create", "lb_create_ex", "lb_destroy", "lb_set_fields", "lb_set_solid_mask",
    "lb_set_populations", "lb_step", "lb_get_populations", "lb_get_moments",
    "lb_get_link_mask", "lb_get_diagnostics", "lb_diagnostics_noalloc", "lb_set_kernel", "lb_get_kernel", "lb_launch_count",
    "lb_set_option", "lb_get_option", "lb_sync", "lb_last_error", "lb_last_error_code", "lb_version",
    "lb_set_colour_gradient", "lb_set_shan_chen", "lb_set_spheres", "lb_get_sphere_forces",
    "lb_export_planes", "lb_import_planes", "lb_plane_buffer_bytes",
    "lbs_create", "lbs_destroy", "lbs_set_fields", "lbs_set_populations", "lbs_step", "lbs_get_populations",
    "lbs_get_moments", "lbs_sync", "lbs_launch_count",
)

_dp = C.POINTER(C.c_double)
_lib = None


class LBError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"lb error {code}: {msg}")
        self.code = code


def lib() -> C.CDLL:
    """Load the CUDA library (built by paper_2112_08264_b200.build); raise if it is not there."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2112_08264_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.lb_create.restype = C.c_void_p
    L.lb_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]
    L.lb_create_ex.restype = C.c_void_p
    L.lb_create_ex.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int, C.c_void_p]
    L.lb_destroy.restype = None
    L.lb_destroy.argtypes = [C.c_void_p]
    L.lb_set_fields.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
    L.lb_set_solid_mask.argtypes = [C.c_void_p, C.POINTER(C.c_ubyte)]
    L.lb_set_populations.argtypes = [C.c_void_p, _dp]
    L.lb_step.argtypes = [C.c_void_p, C.c_int]
    L.lb_get_populations.argtypes = [C.c_void_p, _dp]
    L.lb_get_moments.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
    L.lb_get_link_mask.argtypes = [C.c_void_p, C.POINTER(C.c_uint)]
    L.lb_get_diagnostics.argtypes = [C.c_void_p, _dp, _dp]
    L.lb_diagnostics_noalloc.argtypes = [C.c_void_p, C.c_void_p]
    L.lb_set_kernel.argtypes = [C.c_void_p, C.c_int]
    L.lb_launch_count.restype = C.c_longlong
    L.lb_launch_count.argtypes = [C.c_void_p]
    L.lb_get_kernel.argtypes = [C.c_void_p]
    L.lb_set_option.argtypes = [C.c_void_p, C.c_int, C.c_longlong]
    L.lb_get_option.restype = C.c_longlong
    L.lb_get_option.argtypes = [C.c_void_p, C.c_int]
    L.lb_sync.argtypes = [C.c_void_p]
    L.lb_last_error.restype = C.c_char_p
    L.lb_version.restype = C.c_char_p
    L.lb_set_colour_gradient.argtypes = [C.c_void_p, C.c_double, C.c_double]
    L.lb_set_shan_chen.argtypes = [C.c_void_p]
    L.lb_set_spheres.argtypes = [C.c_void_p, C.c_int, _dp, C.c_double, _dp, _dp]
    L.lb_get_sphere_forces.argtypes = [C.c_void_p, _dp, _dp]
    L.lb_export_planes.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
    L.lb_import_planes.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
    L.lb_plane_buffer_bytes.restype = C.c_longlong
    L.lb_plane_buffer_bytes.argtypes = [C.c_void_p, C.c_int]
    L.lbs_create.restype = C.c_void_p
    L.lbs_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, C.c_void_p]
    L.lbs_destroy.restype = None
    L.lbs_destroy.argtypes = [C.c_void_p]
    L.lbs_set_fields.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
    L.lbs_set_populations.argtypes = [C.c_void_p, _dp]
    L.lbs_step.argtypes = [C.c_void_p, C.c_int]
    L.lbs_get_populations.argtypes = [C.c_void_p, _dp]
    L.lbs_get_moments.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
    L.lbs_sync.argtypes = [C.c_void_p]
    L.lbs_launch_count.restype = C.c_longlong
    L.lbs_launch_count.argtypes = [C.c_void_p]
    _lib = L
    return L


def lb_last_error() -> str:
    return lib().lb_last_error().decode()


def lb_version() -> str:
    return lib().lb_version().decode()


def _chk(rc):
    if rc != LB_OK:
        raise LBError(rc, lb_last_error())


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _host_f64(a, n, name):
    """A caller array as a contiguous float64 host buffer of n elements (no copy if it already is)."""
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=np.float64).reshape(-1)
    if a.size != n:
        raise ValueError(f"{name}: expected {n} elements, got {a.size}")
    return a


def lb_last_error_code() -> int:
    return int(lib().lb_last_error_code())


def lb_create(nx, ny, nz, tau_r, tau_b, G):
    h = lib().lb_create(nx, ny, nz, tau_r, tau_b, G)
    if not h:
        raise LBError(lb_last_error_code(), lb_last_error())
    return h


def lb_create_ex(nx, ny, nz, tau_r, tau_b, G, dtype=LB_F64, cuda_stream=None):
    h = lib().lb_create_ex(nx, ny, nz, tau_r, tau_b, G, dtype, cuda_stream)
    if not h:
        raise LBError(lb_last_error_code(), lb_last_error())
    return h


def lb_destroy(h):
    lib().lb_destroy(h)


def lb_set_fields(h, n, rho_r, rho_b, ux=None, uy=None, uz=None):
    a = [_host_f64(v, n, nm) for v, nm in zip((rho_r, rho_b, ux, uy, uz), ("rho_r", "rho_b", "ux", "uy", "uz"))]
    _chk(lib().lb_set_fields(h, *[_d(v) for v in a]))


def lb_set_solid_mask(h, n, mask):
    m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
    if m.size != n:
        raise ValueError(f"mask: expected {n} bytes, got {m.size}")
    _chk(lib().lb_set_solid_mask(h, m.ctypes.data_as(C.POINTER(C.c_ubyte))))


def lb_set_populations(h, n, f):
    _chk(lib().lb_set_populations(h, _d(_host_f64(f, 38 * n, "f"))))


def lb_step(h, nsteps):
    _chk(lib().lb_step(h, nsteps))


def lb_get_populations(h, n, out=None):
    f = np.empty(38 * n, dtype=np.float64) if out is None else out
    _chk(lib().lb_get_populations(h, _d(f)))
    return f


def lb_get_moments(h, n, out=None):
    o = [np.empty(n, dtype=np.float64) for _ in range(5)] if out is None else out
    _chk(lib().lb_get_moments(h, *[_d(v) for v in o]))
    return o


def lb_get_link_mask(h, n):
    m = np.empty(n, dtype=np.uint32)
    _chk(lib().lb_get_link_mask(h, m.ctypes.data_as(C.POINTER(C.c_uint))))
    return m


def lb_get_diagnostics(h):
    mass, mom = np.empty(2), np.empty(3)
    _chk(lib().lb_get_diagnostics(h, _d(mass), _d(mom)))
    return mass, mom


def lb_diagnostics_noalloc(h, out_dev_ptr):
    """out_dev_ptr: address of 5 doubles of DEVICE memory (e.g. tensor.data_ptr()); asynchronous on the context's stream."""
    _chk(lib().lb_diagnostics_noalloc(h, C.c_void_p(out_dev_ptr)))


def lb_set_kernel(h, kind):
    _chk(lib().lb_set_kernel(h, kind))


KERNEL_NAMES = {LB_KERNEL_TWOPASS: "twopass", LB_KERNEL_ONEPASS: "onepass", LB_KERNEL_TMA: "tma", LB_KERNEL_HALO: "halo", LB_KERNEL_NODE: "node"}


def lb_kernel_name(h) -> str:
    return KERNEL_NAMES.get(int(lib().lb_get_kernel(h)), "?")


def lb_set_option(h, option, value):
    _chk(lib().lb_set_option(h, option, value))


def lb_get_option(h, option) -> int:
    return int(lib().lb_get_option(h, option))


def lb_launch_count(h) -> int:
    return int(lib().lb_launch_count(h))


def lb_sync(h):
    _chk(lib().lb_sync(h))


class Box:
    """Convenience owner of one lb_ctx (same calls, `n` filled in)."""

    def __init__(self, nx, ny, nz, tau_r=1.0, tau_b=1.0, G=1.2, dtype=LB_F64, cuda_stream=None):
        self.nx, self.ny, self.nz = nx, ny, nz
        self.N = nx * ny * nz
        self.dtype = dtype
        self.h = lb_create_ex(nx, ny, nz, tau_r, tau_b, G, dtype, cuda_stream)

    def close(self):
        if getattr(self, "h", None):
            lb_destroy(self.h)
            self.h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_fields(self, rho_r, rho_b, ux=None, uy=None, uz=None):
        lb_set_fields(self.h, self.N, rho_r, rho_b, ux, uy, uz)

    def set_solid_mask(self, mask):
        lb_set_solid_mask(self.h, self.N, mask)

    def set_populations(self, f):
        lb_set_populations(self.h, self.N, f)

    def step(self, nsteps=1):
        lb_step(self.h, nsteps)

    def get_populations(self):
        return lb_get_populations(self.h, self.N).reshape(2, 19, self.nz, self.ny, self.nx)

    def get_moments(self):
        return lb_get_moments(self.h, self.N)

    def get_link_mask(self):
        return lb_get_link_mask(self.h, self.N)

    def get_diagnostics(self):
        return lb_get_diagnostics(self.h)

    def diagnostics_noalloc(self, out_dev_ptr):
        lb_diagnostics_noalloc(self.h, out_dev_ptr)

    def set_kernel(self, kind):
        lb_set_kernel(self.h, kind)

    def set_colour_gradient(self, sigma, beta):
        _chk(lib().lb_set_colour_gradient(self.h, sigma, beta))

    def set_shan_chen(self):
        _chk(lib().lb_set_shan_chen(self.h))

    def set_spheres(self, centres, radius, vel=None, omega=None):
        c = np.ascontiguousarray(centres, dtype=np.float64).reshape(-1, 3)
        self.nsph = c.shape[0]
        v = None if vel is None else _host_f64(vel, 3 * self.nsph, "vel")
        w = None if omega is None else _host_f64(omega, 3 * self.nsph, "omega")
        _chk(lib().lb_set_spheres(self.h, self.nsph, _d(c.reshape(-1)), radius, _d(v), _d(w)))

    def export_planes(self, z0, nplanes, device_ptr):
        _chk(lib().lb_export_planes(self.h, z0, nplanes, device_ptr))

    def plane_buffer_bytes(self, nplanes):
        return int(lib().lb_plane_buffer_bytes(self.h, nplanes))

    def import_planes(self, z0, nplanes, device_ptr):
        _chk(lib().lb_import_planes(self.h, z0, nplanes, device_ptr))

    def get_sphere_forces(self):
        F, T = np.zeros(3 * self.nsph), np.zeros(3 * self.nsph)
        _chk(lib().lb_get_sphere_forces(self.h, _d(F), _d(T)))
        return F.reshape(-1, 3), T.reshape(-1, 3)

    def set_option(self, option, value):
        lb_set_option(self.h, option, value)

    def get_option(self, option):
        return lb_get_option(self.h, option)

    def launch_count(self):
        return lb_launch_count(self.h)

    def sync(self):
        lb_sync(self.h)


class SingleBox:
    """Convenience owner of one lbs_ctx: the single-fluid calibration path (lbs_* calls)."""

    def __init__(self, nx, ny, nz, tau=1.0, dtype=LB_F64, cuda_stream=None):
        self.nx, self.ny, self.nz = nx, ny, nz
        self.N = nx * ny * nz
        self.h = lib().lbs_create(nx, ny, nz, tau, dtype, cuda_stream)
        if not self.h:
            raise LBError(lb_last_error_code(), lb_last_error())

    def close(self):
        if getattr(self, "h", None):
            lib().lbs_destroy(self.h)
            self.h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_fields(self, rho, ux=None, uy=None, uz=None):
        a = [_host_f64(v, self.N, nm) for v, nm in zip((rho, ux, uy, uz), ("rho", "ux", "uy", "uz"))]
        _chk(lib().lbs_set_fields(self.h, *[_d(v) for v in a]))

    def set_populations(self, f):
        _chk(lib().lbs_set_populations(self.h, _d(_host_f64(f, 19 * self.N, "f"))))

    def step(self, nsteps=1):
        _chk(lib().lbs_step(self.h, nsteps))

    def get_populations(self):
        f = np.empty(19 * self.N, dtype=np.float64)
        _chk(lib().lbs_get_populations(self.h, _d(f)))
        return f.reshape(19, self.nz, self.ny, self.nx)

    def get_moments(self):
        o = [np.empty(self.N, dtype=np.float64) for _ in range(4)]
        _chk(lib().lbs_get_moments(self.h, *[_d(v) for v in o]))
        return o

    def sync(self):
        _chk(lib().lbs_sync(self.h))

    def launch_count(self):
        return int(lib().lbs_launch_count(self.h))
