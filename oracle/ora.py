"""ctypes loader for the CPU oracle (oracle/lb_oracle.cpp).

TEST INFRASTRUCTURE ONLY: import this from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs, never from the product package.
It does not import paper_2112_08264_b200 and shares nothing with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lb_oracle.cpp")
_OUT = os.path.join(_HERE, "_build")

# name -> g++ flags.  "ref" is THE oracle; "fma" is the same source with FMA
# contraction, used only to measure the fp64 rounding-noise floor.
_VARIANTS = {
    "ref": ["-O2", "-ffp-contract=off"],
    "fma": ["-O2", "-ffp-contract=fast", "-mfma"],
}


def lib_path(variant: str = "ref") -> str:
    return os.path.join(_OUT, f"liblb_oracle_{variant}.so")


def build(variant: str = "ref", force: bool = False) -> str:
    out = lib_path(variant)
    if (not force and os.path.exists(out)
            and os.path.getmtime(out) >= os.path.getmtime(_SRC)):
        return out
    os.makedirs(_OUT, exist_ok=True)
    tmp = out + f".tmp{os.getpid()}"
    cmd = ["g++", "-std=c++17", "-shared", "-fPIC", *_VARIANTS[variant], "-o", tmp, _SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)
    return out


def host_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("flags"):
                    return " fma " in line + " "
    except OSError:
        pass
    return False


_dp = C.POINTER(C.c_double)
_libs: dict[str, C.CDLL] = {}


def _load(variant: str) -> C.CDLL:
    if variant in _libs:
        return _libs[variant]
    lib = C.CDLL(build(variant))
    lib.ora_create.restype = C.c_void_p
    lib.ora_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]
    lib.ora_destroy.restype = None
    lib.ora_destroy.argtypes = [C.c_void_p]
    lib.ora_set_forcing.argtypes = [C.c_void_p, C.c_int]
    lib.ora_set_fields.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
    lib.ora_set_solid_mask.argtypes = [C.c_void_p, C.POINTER(C.c_ubyte)]
    lib.ora_set_populations.argtypes = [C.c_void_p, _dp]
    lib.ora_step.argtypes = [C.c_void_p, C.c_int]
    lib.ora_get_populations.argtypes = [C.c_void_p, _dp]
    lib.ora_get_moments.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
    lib.ora_get_link_mask.argtypes = [C.c_void_p, C.POINTER(C.c_uint)]
    lib.ora_get_diagnostics.argtypes = [C.c_void_p, _dp, _dp]
    lib.ora_get_force.argtypes = [C.c_void_p, _dp, _dp]
    lib.ora_feq.restype = None
    lib.ora_feq.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, _dp]
    lib.ora_lattice.restype = None
    lib.ora_lattice.argtypes = [C.POINTER(C.c_int), _dp]
    lib.ora_set_colour_gradient.argtypes = [C.c_void_p, C.c_double, C.c_double]
    lib.ora_get_phase_field.argtypes = [C.c_void_p, _dp, _dp]
    lib.ora_cg_perturbation.restype = None
    lib.ora_cg_perturbation.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, _dp]
    lib.ora_set_spheres.argtypes = [C.c_void_p, C.c_int, _dp, C.c_double, _dp, _dp]
    lib.ora_get_sphere_forces.argtypes = [C.c_void_p, _dp, _dp]
    lib.ora_get_solid_mask.argtypes = [C.c_void_p, C.POINTER(C.c_ubyte)]
    _libs[variant] = lib
    return lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a, n):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=np.float64).reshape(-1)
    if a.size != n:
        raise ValueError(f"expected {n} elements, got {a.size}")
    return a


def feq(rho, ux, uy, uz, variant: str = "ref"):
    out = np.empty(19)
    _load(variant).ora_feq(rho, ux, uy, uz, _d(out))
    return out


def cg_perturbation(A, gx, gy, gz, variant: str = "ref"):
    out = np.empty(19)
    _load(variant).ora_cg_perturbation(A, gx, gy, gz, _d(out))
    return out


def lattice(variant: str = "ref"):
    c = np.empty((19, 3), dtype=np.int32)
    w = np.empty(19)
    _load(variant).ora_lattice(c.ctypes.data_as(C.POINTER(C.c_int)), _d(w))
    return c, w


class Oracle:
    """Thin object wrapper; arrays are flat float64, dense [..][z][y][x]."""

    def __init__(self, nx, ny, nz, tau_r=1.0, tau_b=1.0, G=1.2, variant="ref"):
        self._lib = _load(variant)
        self.nx, self.ny, self.nz = nx, ny, nz
        self.N = nx * ny * nz
        self._h = self._lib.ora_create(nx, ny, nz, tau_r, tau_b, G)
        if not self._h:
            raise ValueError("ora_create rejected the arguments")

    def close(self):
        if self._h:
            self._lib.ora_destroy(self._h)
            self._h = None

    __del__ = close

    def _chk(self, rc):
        if rc != 0:
            raise RuntimeError(f"oracle call failed with code {rc}")

    def set_colour_gradient(self, sigma, beta):
        self._chk(self._lib.ora_set_colour_gradient(self._h, sigma, beta))

    def get_phase_field(self):
        th, g = np.empty(self.N), np.empty(3 * self.N)
        self._chk(self._lib.ora_get_phase_field(self._h, _d(th), _d(g)))
        return th, g.reshape(3, self.N)

    def set_spheres(self, centres, radius, vel=None, omega=None):
        c = np.ascontiguousarray(centres, dtype=np.float64).reshape(-1, 3)
        self.nsph = c.shape[0]
        v = None if vel is None else _f64(vel, 3 * self.nsph)
        w = None if omega is None else _f64(omega, 3 * self.nsph)
        self._chk(self._lib.ora_set_spheres(self._h, self.nsph, _d(c.reshape(-1)), radius, _d(v), _d(w)))

    def get_sphere_forces(self):
        F, T = np.empty(3 * self.nsph), np.empty(3 * self.nsph)
        self._chk(self._lib.ora_get_sphere_forces(self._h, _d(F), _d(T)))
        return F.reshape(-1, 3), T.reshape(-1, 3)

    def get_solid_mask(self):
        m = np.empty(self.N, dtype=np.uint8)
        self._chk(self._lib.ora_get_solid_mask(self._h, m.ctypes.data_as(C.POINTER(C.c_ubyte))))
        return m

    def set_forcing(self, mode):
        self._chk(self._lib.ora_set_forcing(self._h, mode))

    def set_fields(self, rho_r, rho_b, ux=None, uy=None, uz=None):
        a = [_f64(v, self.N) for v in (rho_r, rho_b, ux, uy, uz)]
        self._chk(self._lib.ora_set_fields(self._h, *[_d(v) for v in a]))

    def set_solid_mask(self, mask):
        m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1)
        assert m.size == self.N
        self._chk(self._lib.ora_set_solid_mask(self._h, m.ctypes.data_as(C.POINTER(C.c_ubyte))))

    def set_populations(self, f):
        f = _f64(f, 38 * self.N)
        self._chk(self._lib.ora_set_populations(self._h, _d(f)))

    def step(self, n=1):
        self._chk(self._lib.ora_step(self._h, n))

    def get_populations(self):
        f = np.empty(38 * self.N)
        self._chk(self._lib.ora_get_populations(self._h, _d(f)))
        return f.reshape(2, 19, self.nz, self.ny, self.nx)

    def get_moments(self):
        out = [np.empty(self.N) for _ in range(5)]
        self._chk(self._lib.ora_get_moments(self._h, *[_d(v) for v in out]))
        return out

    def get_link_mask(self):
        m = np.empty(self.N, dtype=np.uint32)
        self._chk(self._lib.ora_get_link_mask(self._h, m.ctypes.data_as(C.POINTER(C.c_uint))))
        return m

    def get_diagnostics(self):
        mass, mom = np.empty(2), np.empty(3)
        self._chk(self._lib.ora_get_diagnostics(self._h, _d(mass), _d(mom)))
        return mass, mom

    def get_force(self):
        fr, fb = np.empty(3 * self.N), np.empty(3 * self.N)
        self._chk(self._lib.ora_get_force(self._h, _d(fr), _d(fb)))
        return fr.reshape(3, -1), fb.reshape(3, -1)
