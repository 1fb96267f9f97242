"""Seeded synthetic workloads (the five BASELINE.json configs).

This module holds NO arithmetic of the spectral Ewald method: it only draws
positions and forces.  It is the one piece shared by the oracle-side tests and
the CUDA-side tests/bench (neither `oracle/` nor the CUDA binding imports it
themselves; callers pass the arrays in).

Recipe (stand-in for the paper's U(0,1) and sphere-surface
workloads, App. B):
  rng = numpy.random.default_rng(190590 + cfg)          (PCG64)
  cfg 1-4: x = rng.random((N,3))*L ; f = rng.standard_normal((N,3)) ; f -= f.mean(0)
           cfg 4 casts x and f to float32 (the oracle consumes the rounded values).
  cfg 5  : 1024 sphere centres c ~ U[0,1)^3, unit quaternions q ~ N(0,1)^4 normalised
           -> rotation R_s; 4096-point Fibonacci lattice p_i on the unit sphere;
           x = (c_s + 0.02 R_s p_i) mod 1, sphere-major; f as above; one
           rng.permutation(N) applied to x and f.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

SEED_BASE = 190590


@dataclass(frozen=True)
class Config:
    cfg: int
    N: int
    L: float
    xi: float
    rc: float
    M: int
    P: int
    precision: str  # "fp64" | "fp32"
    kind: str       # "uniform" | "spheres"
    label: str
    window: str = "gaussian"   # "gaussian" | "kb" (Kaiser-Bessel, eq. (2.8))


CONFIGS = {
    1: Config(1, 1_000, 1.0, 18.0, 0.25, 56, 24, "fp64", "uniform", "cfg1 N=1e3 uniform fp64"),
    2: Config(2, 65_536, 1.0, 50.0, 0.09, 144, 24, "fp64", "uniform", "cfg2 N=65536 uniform fp64"),
    3: Config(3, 1_048_576, 1.0, 126.0, 0.0357, 360, 24, "fp64", "uniform", "cfg3 N=1048576 uniform fp64"),
    4: Config(4, 4_194_304, 1.0, 142.0, 0.0225, 320, 12, "fp32", "uniform", "cfg4 N=4194304 uniform fp32"),
    5: Config(5, 4_194_304, 1.0, 200.0, 0.0225, 576, 24, "fp64", "spheres", "cfg5 N=4194304 clustered fp64"),
}


def np_dtype(precision: str):
    return np.float64 if precision == "fp64" else np.float32


def _forces(rng: np.random.Generator, N: int) -> np.ndarray:
    f = rng.standard_normal((N, 3))
    f -= f.mean(axis=0)
    return f


def uniform_cloud(seed: int, N: int, L: float = 1.0):
    """x ~ U[0,L)^3, f ~ N(0,1) mean-subtracted.  Returns float64 (x, f)."""
    rng = np.random.default_rng(seed)
    x = rng.random((N, 3)) * L
    f = _forces(rng, N)
    return x, f


def _quat_to_rot(q: np.ndarray) -> np.ndarray:
    """Unit quaternions (S,4) [w,x,y,z] -> rotation matrices (S,3,3)."""
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((q.shape[0], 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z)
    R[:, 0, 1] = 2 * (x * y - z * w)
    R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w)
    R[:, 1, 1] = 1 - 2 * (x * x + z * z)
    R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w)
    R[:, 2, 1] = 2 * (y * z + x * w)
    R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def sphere_cloud(seed: int, n_spheres: int = 1024, n_per: int = 4096,
                 radius: float = 0.02, L: float = 1.0):
    """Clustered workload: Fibonacci-lattice points on randomly rotated spheres."""
    rng = np.random.default_rng(seed)
    c = rng.random((n_spheres, 3)) * L
    q = rng.standard_normal((n_spheres, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    R = _quat_to_rot(q)
    i = np.arange(n_per, dtype=np.float64)
    z = 1.0 - (2.0 * i + 1.0) / n_per
    th = i * np.pi * (3.0 - np.sqrt(5.0))
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    p = np.stack([s * np.cos(th), s * np.sin(th), z], axis=1)          # (n_per, 3)
    x = c[:, None, :] + radius * np.einsum("sab,ib->sia", R, p)         # (S, n_per, 3)
    x = np.mod(x.reshape(-1, 3), L)
    x[x >= L] = 0.0
    N = x.shape[0]
    f = _forces(rng, N)
    perm = rng.permutation(N)
    return np.ascontiguousarray(x[perm]), np.ascontiguousarray(f[perm])


def make(cfg: int, N: int | None = None):
    """(Config, x, f) for BASELINE config `cfg`; arrays in the config's dtype.

    `N` overrides the particle count (uniform configs only) — used by tests that
    need the config's parameters at a size the oracle finishes quickly.
    """
    c = CONFIGS[cfg]
    if N is not None and N != c.N:
        if c.kind != "uniform":
            raise ValueError("N override only for uniform configs")
        c = replace(c, N=int(N))
    if c.kind == "uniform":
        x, f = uniform_cloud(SEED_BASE + cfg, c.N, c.L)
    else:
        x, f = sphere_cloud(SEED_BASE + cfg, L=c.L)
    dt = np_dtype(c.precision)
    return c, np.ascontiguousarray(x.astype(dt)), np.ascontiguousarray(f.astype(dt))


def scaled(cfg: int, N: int, seed: int | None = None):
    """A small problem with config `cfg`'s *dimensionless* parameters.

    Keeps xi*rc, pi*M/(2 xi L) and P of the config but picks rc so that the mean
    number of in-range neighbours matches the config, and M accordingly (even).
    Used for parity cases that span several tiles/cells yet finish in seconds.
    """
    c = CONFIGS[cfg]
    dens_c = c.N / c.L ** 3
    nb = dens_c * 4.0 / 3.0 * np.pi * c.rc ** 3          # neighbours within rc
    rc = (nb / (N * 4.0 / 3.0 * np.pi)) ** (1.0 / 3.0) * c.L
    rc = min(rc, c.L / 3.0)
    xi = c.xi * c.rc / rc
    M = int(round(c.M * (xi / c.xi)))
    M += M & 1
    M = max(M, c.P)
    cc = replace(c, N=int(N), rc=float(rc), xi=float(xi), M=M,
                 label=f"cfg{cfg}-scaled N={N}")
    x, f = uniform_cloud(SEED_BASE + 100 * cfg + 7 if seed is None else seed, N, c.L)
    dt = np_dtype(c.precision)
    return cc, np.ascontiguousarray(x.astype(dt)), np.ascontiguousarray(f.astype(dt))


def smooth_grid(seed: int, M: int, ncomp: int = 3):
    """Synthetic band-limited real grid (ncomp, M, M, M) for stand-alone G2P tests."""
    rng = np.random.default_rng(seed)
    g = np.arange(M) / M
    out = np.zeros((ncomp, M, M, M))
    for c in range(ncomp):
        for _ in range(4):
            k = rng.integers(-3, 4, size=3)
            ph = rng.random() * 2 * np.pi
            amp = rng.standard_normal()
            out[c] += amp * np.cos(2 * np.pi * (k[0] * g[:, None, None] + k[1] * g[None, :, None]
                                                 + k[2] * g[None, None, :]) + ph)
    return out


def random_spectrum(seed: int, M: int, ncomp: int = 3):
    """Synthetic complex half-spectrum (ncomp, M, M, M//2+1) for stand-alone SCALE tests."""
    rng = np.random.default_rng(seed)
    shp = (ncomp, M, M, M // 2 + 1)
    return (rng.standard_normal(shp) + 1j * rng.standard_normal(shp)).astype(np.complex128)


# ---- index-defined synthetic fields (full-size stand-alone K4 / K5 parity) ------------------------
# Closed-form functions of the integer grid indices, so that the same field can be written on the device
# (xp = torch) and evaluated on the host (xp = numpy) at any size without storing or moving it.  No
# arithmetic of the method: plain cosines of index combinations.
def index_grid(xp, c, i, j, k, M):
    """Smooth real grid value of component c at (i, j, k): a few low wavenumbers of the periodic box,
    written as products of 1-D factors so that broadcasting index arrays keeps the cosines one-dimensional."""
    w = 2.0 * np.pi / M
    return (xp.cos(w * 2.0 * i + 0.3 * c) * xp.cos(w * j) * xp.cos(w * 3.0 * k)
            + 0.5 * xp.cos(w * i - 0.7 * c) * xp.sin(w * 2.0 * j)
            + 0.25 * xp.cos(w * 2.0 * i) * xp.cos(w * 3.0 * k + 1.1))


def index_spectrum(xp, c, i, j, k):
    """Complex half-spectrum value of component c at mode indices (i, j, k): (re, im), O(1) everywhere."""
    re = xp.cos(0.37 * i + 0.5 * c) * xp.cos(0.11 * j) + 0.5 * xp.cos(0.73 * k + 0.2)
    im = xp.cos(0.23 * i + 1.3) * xp.cos(0.19 * k + 0.9 * c) - 0.5 * xp.cos(0.41 * j)
    return re, im
