"""Seeded synthetic inputs for the two-component D3Q19 workloads.

This module is the ONE piece of code that serves both the CPU oracle (`oracle/`)
and the CUDA path: it only draws random numbers and lays out input arrays
(densities, sphere centres, the solid byte mask).  It holds none of the method's
arithmetic (no equilibrium, no moments, no force, no streaming) and imports
neither side.

Recipe (SURVEY.md §8(d) "Synthetic inputs"; DESIGN.md §"Input recipe"):

* counter-based generator, all arithmetic mod 2^64::

      mix(x):  x += 0x9E3779B97F4A7C15
               x = (x ^ x>>30) * 0xBF58476D1CE4E5B9
               x = (x ^ x>>27) * 0x94D049BB133111EB
               return x ^ x>>31
      u01(seed, c) = (mix(seed + c*0x9E3779B97F4A7C15) >> 11) * 2^-53

* node index n = x + nx*(y + ny*z); arrays are dense [z][y][x], x fastest.
* random 50/50 mixture (stands in for the paper's case 2, §5, with
  BASELINE.json's +-1 % noise):  rho_r(n) = 1 + 0.01*(2*u01(s,2n)-1),
  rho_b(n) = 1 + 0.01*(2*u01(s,2n+1)-1), u = 0.
* colloid-like packing (stands in for case 3c, §5.3: radius 5.5,
  random positions): candidate m has centre (nx*u01(t,3m), ny*u01(t,3m+1),
  nz*u01(t,3m+2)); it is accepted iff its minimum-image distance to every centre
  accepted so far is >= min_dist; a node is solid iff its minimum-image squared
  distance to some centre is <= R^2.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

_GOLD = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def mix(x):
    """splitmix64 finaliser on uint64 scalars/arrays (wrapping arithmetic)."""
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = x + _GOLD
        x = (x ^ (x >> np.uint64(30))) * _M1
        x = (x ^ (x >> np.uint64(27))) * _M2
        return x ^ (x >> np.uint64(31))


def u01(seed: int, c):
    """Uniform double in [0,1) for counter(s) `c` under `seed` (53 random bits)."""
    c = np.asarray(c, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = mix(np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + c * _GOLD)
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def mixture_fields(nx: int, ny: int, nz: int, seed: int, amp: float = 0.01,
                   chunk: int = 1 << 24):
    """rho_r, rho_b as flat float64 arrays of N = nx*ny*nz (dense [z][y][x])."""
    n_nodes = nx * ny * nz
    rho_r = np.empty(n_nodes, dtype=np.float64)
    rho_b = np.empty(n_nodes, dtype=np.float64)
    for lo in range(0, n_nodes, chunk):
        hi = min(n_nodes, lo + chunk)
        n = np.arange(lo, hi, dtype=np.uint64)
        rho_r[lo:hi] = 1.0 + amp * (2.0 * u01(seed, np.uint64(2) * n) - 1.0)
        rho_b[lo:hi] = 1.0 + amp * (2.0 * u01(seed, np.uint64(2) * n + np.uint64(1)) - 1.0)
    return rho_r, rho_b


def _min_image(d, n):
    d = np.abs(d)
    return np.minimum(d, n - d)


def sphere_centres(nx: int, ny: int, nz: int, seed: int, count: int,
                   min_dist: float = 11.0, max_candidates: int = 10_000_000):
    """Random sequential addition of non-overlapping sphere centres.

    Returns (centres[count,3] float64, candidates_drawn)."""
    centres = np.empty((count, 3), dtype=np.float64)
    n_acc = 0
    m = 0
    box = np.array([nx, ny, nz], dtype=np.float64)
    md2 = min_dist * min_dist
    while n_acc < count:
        if m >= max_candidates:
            raise RuntimeError("sphere packing did not finish")
        c = box * u01(seed, np.arange(3 * m, 3 * m + 3, dtype=np.uint64))
        m += 1
        if n_acc:
            d = _min_image(centres[:n_acc] - c, box)
            if np.any(np.einsum("ij,ij->i", d, d) < md2):
                continue
        centres[n_acc] = c
        n_acc += 1
    return centres, m


def solid_mask_from_spheres(nx: int, ny: int, nz: int, centres, radius: float = 5.5):
    """uint8 mask [z][y][x] (flat): 1 iff min-image squared distance to a centre <= R^2."""
    mask = np.zeros((nz, ny, nx), dtype=np.uint8)
    r2 = radius * radius
    reach = int(np.floor(radius)) + 1
    for cx, cy, cz in np.asarray(centres, dtype=np.float64).reshape(-1, 3):
        xs = np.arange(int(np.floor(cx)) - reach, int(np.floor(cx)) + reach + 2)
        ys = np.arange(int(np.floor(cy)) - reach, int(np.floor(cy)) + reach + 2)
        zs = np.arange(int(np.floor(cz)) - reach, int(np.floor(cz)) + reach + 2)
        dx = _min_image(np.mod(xs, nx) - cx, nx)
        dy = _min_image(np.mod(ys, ny) - cy, ny)
        dz = _min_image(np.mod(zs, nz) - cz, nz)
        d2 = dz[:, None, None] ** 2 + dy[None, :, None] ** 2 + dx[None, None, :] ** 2
        zz, yy, xx = np.nonzero(d2 <= r2)
        mask[np.mod(zs, nz)[zz], np.mod(ys, ny)[yy], np.mod(xs, nx)[xx]] = 1
    return mask.reshape(-1)


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config (or a parity box) as seeded inputs."""
    name: str
    nx: int
    ny: int
    nz: int
    tau_r: float = 1.0
    tau_b: float = 1.0
    G: float = 1.2
    dtype: str = "f64"
    seed: int = 0
    steps: int = 100
    n_spheres: int = 0
    sphere_seed: int = 0

    @property
    def n_nodes(self) -> int:
        return self.nx * self.ny * self.nz

    def fields(self):
        return mixture_fields(self.nx, self.ny, self.nz, self.seed)

    def solid_mask(self):
        if self.n_spheres == 0:
            return None
        centres, _ = sphere_centres(self.nx, self.ny, self.nz, self.sphere_seed,
                                    self.n_spheres)
        return solid_mask_from_spheres(self.nx, self.ny, self.nz, centres)


# BASELINE.json "configs", in order (seeds: SURVEY.md §8(d) table).
CONFIGS = (
    Workload("config0_32c_f64", 32, 32, 32, seed=2112082640, steps=100),
    Workload("config1_256c_f64", 256, 256, 256, seed=2112082641, steps=1000),
    Workload("config2_512c_f64", 512, 512, 512, seed=2112082642, steps=200),
    Workload("config3_512c_f32", 512, 512, 512, dtype="f32", seed=2112082642, steps=200),
    Workload("config4_256c_spheres_f64", 256, 256, 256, seed=2112082644, steps=500,
             n_spheres=2000, sphere_seed=2112082654),
)
