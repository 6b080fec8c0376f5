"""Seeded synthetic input generators for the five BASELINE.json configs.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path: it produces the host arrays (phi0, F) both sides consume.  It holds none
of the method's arithmetic (no differences, no cut-off, no band logic) — only
signed-distance / analytic initial fields and a counter-based PRNG.

Recipe:
  * grid points sit at cell centres x_i = (i + 1/2) dx, dx = 1/n        (R4)
  * everything is evaluated in float64 on the host and rounded ONCE to the
    field dtype
  * layout is dense, x fastest: array shape (nz, ny, nx), C-contiguous, so the
    flat index is (k*ny + j)*nx + i
  * random numbers: u(seed, n) = (splitmix64(seed + n) >> 11) * 2^-53 with n
    the flat point index — order independent, reproducible anywhere.

The paper measures on no public data set (its 101^3 / 201^3 runs state neither
the initial front nor F), so these synthetic shapes stand in.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

_U64 = np.uint64
_MASK64 = (1 << 64) - 1


# --------------------------------------------------------------------------
# counter-based PRNG
# --------------------------------------------------------------------------
def splitmix64(x: np.ndarray) -> np.ndarray:
    """Vectorised splitmix64 finaliser on uint64 (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = x.astype(np.uint64, copy=True)
        z += _U64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> _U64(27))) * _U64(0x94D049BB133111EB)
        z = z ^ (z >> _U64(31))
    return z


def uniform01(seed: int, start: int, count: int) -> np.ndarray:
    """u(seed, n) for n = start .. start+count-1, float64 in [0, 1)."""
    with np.errstate(over="ignore"):
        n = np.arange(start, start + count, dtype=np.uint64) + _U64(seed & _MASK64)
    return (splitmix64(n) >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# --------------------------------------------------------------------------
# workload description
# --------------------------------------------------------------------------
@dataclass
class Workload:
    """One config: host fields + the parameters of the step loop."""

    name: str
    nx: int
    ny: int
    nz: int
    dtype: np.dtype
    dx: float
    dt: float
    dtau: float
    beta: float
    gamma: float
    iters: int
    n_steps: int
    phi: np.ndarray = field(repr=False)      # (nz, ny, nx)
    F: np.ndarray | None = field(repr=False, default=None)
    mode: str = "band"                       # "band" | "dense" | "reinit_tol"
    tol: float = 0.0
    note: str = ""

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def n_points(self) -> int:
        return self.nx * self.ny * self.nz


def _centres(n: int, dx: float) -> np.ndarray:
    return (np.arange(n, dtype=np.float64) + 0.5) * dx


def sphere_sdf(n: int, r: float, centre=(0.5, 0.5, 0.5), dtype=np.float32,
               z_range: tuple[int, int] | None = None) -> np.ndarray:
    """phi = |x - c| - r on an n^3 cell-centred unit cube (cfg 1, cfg 2)."""
    dx = 1.0 / n
    x = _centres(n, dx)
    k0, k1 = z_range if z_range is not None else (0, n)
    X2 = (x - centre[0]) ** 2
    Y2 = (x - centre[1]) ** 2
    Z2 = (x[k0:k1] - centre[2]) ** 2
    out = np.empty((k1 - k0, n, n), dtype=dtype)
    xy = Y2[:, None] + X2[None, :]
    for k in range(k1 - k0):
        out[k] = np.sqrt(xy + Z2[k]) - r
    return out


def torus_sdf(n: int, R: float = 0.3, r: float = 0.1, dtype=np.float32,
              z_range: tuple[int, int] | None = None) -> np.ndarray:
    """phi = sqrt((sqrt((x-.5)^2+(y-.5)^2) - R)^2 + (z-.5)^2) - r  (cfg 4)."""
    dx = 1.0 / n
    x = _centres(n, dx)
    k0, k1 = z_range if z_range is not None else (0, n)
    rho = np.sqrt((x[:, None] - 0.5) ** 2 + (x[None, :] - 0.5) ** 2) - R  # [j, i]
    rho2 = rho * rho
    out = np.empty((k1 - k0, n, n), dtype=dtype)
    tmp = np.empty_like(rho2)
    for k in range(k0, k1):
        np.add(rho2, (x[k] - 0.5) ** 2, out=tmp)
        np.sqrt(tmp, out=tmp)
        np.subtract(tmp, r, out=tmp)
        out[k - k0] = tmp
    return out


def multi_sphere_sdf(n: int, n_spheres: int = 32, seed: int = 3001,
                     dtype=np.float32) -> np.ndarray:
    """phi = min over seeded sphere SDFs (cfg 3). Centres U[0.1,0.9]^3, radii U[0.03,0.12]."""
    dx = 1.0 / n
    x = _centres(n, dx)
    u = uniform01(seed, 0, 4 * n_spheres).reshape(n_spheres, 4)
    c = 0.1 + 0.8 * u[:, :3]
    rad = 0.03 + 0.09 * u[:, 3]
    out = np.empty((n, n, n), dtype=dtype)
    # z-slab chunks keep the float64 temporaries small
    chunk = max(1, min(n, (1 << 22) // (n * n) or 1))
    for k0 in range(0, n, chunk):
        k1 = min(n, k0 + chunk)
        best = np.full((k1 - k0, n, n), np.inf)
        for s in range(n_spheres):
            d2 = ((x[k0:k1, None, None] - c[s, 2]) ** 2
                  + (x[None, :, None] - c[s, 1]) ** 2
                  + (x[None, None, :] - c[s, 0]) ** 2)
            np.sqrt(d2, out=d2)
            d2 -= rad[s]
            np.minimum(best, d2, out=best)
        out[k0:k1] = best
    return out


def _box3_axis(a: np.ndarray, axis: int) -> np.ndarray:
    """(a[i-1] + a[i] + a[i+1]) / 3 along `axis`, edge replicate."""
    lo = np.concatenate([np.take(a, [0], axis=axis),
                         np.take(a, range(0, a.shape[axis] - 1), axis=axis)], axis=axis)
    hi = np.concatenate([np.take(a, range(1, a.shape[axis]), axis=axis),
                         np.take(a, [a.shape[axis] - 1], axis=axis)], axis=axis)
    return ((lo + a) + hi) / 3.0


def smoothed_noise_speed(n: int, seed: int = 3002, passes: int = 3,
                         dtype=np.float32) -> np.ndarray:
    """F = U[-1,1] per point, then `passes` separable 3x3x3 box filters (cfg 3, R24)."""
    f = (2.0 * uniform01(seed, 0, n * n * n) - 1.0).reshape(n, n, n)
    for _ in range(passes):
        f = _box3_axis(f, 2)   # x
        f = _box3_axis(f, 1)   # y
        f = _box3_axis(f, 0)   # z
    return f.astype(dtype)


def wavy_plane_noisy(n: int, seed: int = 5001, dtype=np.float64) -> np.ndarray:
    """(z - .5 - .05 sin6πx sin6πy) * U[0.8,1.2] per point (cfg 5; not an SDF)."""
    dx = 1.0 / n
    x = _centres(n, dx)
    wave = 0.05 * np.sin(6 * math.pi * x)[None, :] * np.sin(6 * math.pi * x)[:, None]  # [j,i]
    out = np.empty((n, n, n), dtype=dtype)
    plane = n * n
    for k in range(n):
        noise = 0.8 + 0.4 * uniform01(seed, k * plane, plane).reshape(n, n)
        out[k] = ((x[k] - 0.5) - wave) * noise
    return out


def sine_product_speed(n: int, dtype=np.float32,
                       z_range: tuple[int, int] | None = None) -> np.ndarray:
    """F = sin4πx sin4πy sin4πz (cfg 4)."""
    x = _centres(n, 1.0 / n)
    s = np.sin(4 * math.pi * x)
    k0, k1 = z_range if z_range is not None else (0, n)
    xy = s[:, None] * s[None, :]
    out = np.empty((k1 - k0, n, n), dtype=dtype)
    for k in range(k0, k1):
        out[k - k0] = xy * s[k]
    return out


def modulated_speed(n: int, dtype=np.float32) -> np.ndarray:
    """F = 1 + 0.5 sin(2πx) cos(2πy) in [0.5, 1.5] (cfg 2), constant in z."""
    x = _centres(n, 1.0 / n)
    xy = 1.0 + 0.5 * np.cos(2 * math.pi * x)[:, None] * np.sin(2 * math.pi * x)[None, :]
    return np.broadcast_to(xy.astype(dtype)[None], (n, n, n)).copy()


# --------------------------------------------------------------------------
# the five configs (BASELINE.json:configs, 1-based as in SURVEY.md)
# --------------------------------------------------------------------------
INF = float("inf")


def config(idx: int, n: int | None = None, n_steps: int | None = None) -> Workload:
    """Build config `idx` (1..5).  `n` overrides the grid edge (scaled-down parity
    cases keep every parameter in units of dx); `n_steps` overrides the step count."""
    if idx == 1:
        n = n or 64
        dx = 1.0 / n
        return Workload("cfg1_sphere_band", n, n, n, np.dtype(np.float32), dx,
                        dt=0.5 * dx, dtau=0.5 * dx, beta=3 * dx, gamma=6 * dx, iters=5,
                        n_steps=n_steps or 10,
                        phi=sphere_sdf(n, 0.3), F=np.ones((n, n, n), np.float32),
                        note="sphere r=0.3, F=1")
    if idx == 2:
        n = n or 256
        dx = 1.0 / n
        return Workload("cfg2_dense_advance", n, n, n, np.dtype(np.float32), dx,
                        dt=0.4 * dx, dtau=0.0, beta=INF, gamma=INF, iters=0,
                        n_steps=n_steps or 50, mode="dense",
                        phi=sphere_sdf(n, 0.35), F=modulated_speed(n),
                        note="full-domain advance, c=1")
    if idx == 3:
        n = n or 512
        dx = 1.0 / n
        return Workload("cfg3_multisphere_band", n, n, n, np.dtype(np.float32), dx,
                        dt=0.4 * dx, dtau=0.5 * dx, beta=3 * dx, gamma=6 * dx, iters=5,
                        n_steps=n_steps or 100,
                        phi=multi_sphere_sdf(n), F=smoothed_noise_speed(n),
                        note="32 seeded spheres, two-signed smoothed-noise F")
    if idx == 4:
        n = n or 1024
        dx = 1.0 / n
        return Workload("cfg4_torus_band", n, n, n, np.dtype(np.float32), dx,
                        dt=0.4 * dx, dtau=0.5 * dx, beta=3 * dx, gamma=6 * dx, iters=5,
                        n_steps=n_steps or 200,
                        phi=torus_sdf(n), F=sine_product_speed(n),
                        note="torus R=0.3 r=0.1, F=sin4πx sin4πy sin4πz")
    if idx == 5:
        n = n or 512
        dx = 1.0 / n
        return Workload("cfg5_reinit_fp64", n, n, n, np.dtype(np.float64), dx,
                        dt=0.0, dtau=0.3 * dx, beta=4 * dx, gamma=8 * dx, iters=0,
                        n_steps=n_steps or 1, mode="reinit_tol", tol=1e-10,
                        phi=wavy_plane_noisy(n), F=None,
                        note="noisy wavy plane, reinit to steady state")
    raise ValueError(f"config index {idx} not in 1..5")
