"""ctypes wrapper around the CPU oracle (oracle/ls_oracle.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  The product package
(paper_1612_04040_b200) never imports this module.

Arrays are numpy, shape (nz, ny, nx), C-contiguous (x fastest).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "ls_oracle.cpp"
_SO = _HERE / "liboracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle: plain -O2, no fast-math, FMA contraction off, OpenMP for the timed baseline."""
    if force or not _SO.exists() or _SO.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
               "-fPIC", "-shared", "-Wall", "-Wno-misleading-indentation", "-o", str(_SO), str(_SRC)]
        subprocess.run(cmd, check=True)
    return _SO


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(str(_SO))
        _declare(_lib)
    return _lib


_D = C.c_double
_I = C.c_int
_P = C.c_void_p
_L = C.c_int64


def _declare(L):
    for s in ("f32", "f64"):
        getattr(L, f"orc_cutoff_{s}").restype = _D
        getattr(L, f"orc_cutoff_{s}").argtypes = [_D, _D, _D]
        getattr(L, f"orc_upwind_q_{s}").restype = None
        getattr(L, f"orc_upwind_q_{s}").argtypes = [_P, _I, _I, _I, _I, _I, _I, _D, C.POINTER(_D), C.POINTER(_D)]
        getattr(L, f"orc_band_masks_{s}").restype = None
        getattr(L, f"orc_band_masks_{s}").argtypes = [_P, _I, _I, _I, _D, _P, _P]
        getattr(L, f"orc_advance_{s}").restype = None
        getattr(L, f"orc_advance_{s}").argtypes = [_P, _P, _P, _I, _I, _I, _D, _D, _D, _D, _P]
        getattr(L, f"orc_advance_point_{s}").restype = _D
        getattr(L, f"orc_advance_point_{s}").argtypes = [_P, _P, _I, _I, _I, _I, _I, _I, _D, _D, _D, _D]
        getattr(L, f"orc_reinit_iter_{s}").restype = _D
        getattr(L, f"orc_reinit_iter_{s}").argtypes = [_P, _P, _I, _I, _I, _D, _D, _P]
        getattr(L, f"orc_reinit_point_{s}").restype = _D
        getattr(L, f"orc_reinit_point_{s}").argtypes = [_P, _I, _I, _I, _I, _I, _I, _D, _D]
        getattr(L, f"orc_clamp_{s}").restype = None
        getattr(L, f"orc_clamp_{s}").argtypes = [_P, _L, _D]
        getattr(L, f"orc_advance_list_{s}").restype = None
        getattr(L, f"orc_advance_list_{s}").argtypes = [_P, _P, _P, _P, _L, _I, _I, _I, _D, _D, _D, _D, _P]
        getattr(L, f"orc_reinit_iter_list_{s}").restype = None
        getattr(L, f"orc_reinit_iter_list_{s}").argtypes = [_P, _P, _P, _L, _I, _I, _I, _D, _D, _P]
        getattr(L, f"orc_step_{s}").restype = _I
        getattr(L, f"orc_step_{s}").argtypes = [_P, _P, _I, _I, _I, _D, _D, _D, _D, _D, _I, _I, _I, C.POINTER(_L)]
        getattr(L, f"orc_reinit_tol_{s}").restype = _I
        getattr(L, f"orc_reinit_tol_{s}").argtypes = [_P, _P, _I, _I, _I, _D, _D, _D, _D, _I, _I,
                                                       C.POINTER(_D), C.POINTER(_I)]
    L.orc_brick_list.restype = _L
    L.orc_brick_list.argtypes = [_P, _I, _I, _I, _P, _P, _L, C.POINTER(_L)]
    L.orc_max_threads.restype = _I
    L.orc_set_threads.argtypes = [_I]


def _suf(a: np.ndarray) -> str:
    if a.dtype == np.float32:
        return "f32"
    if a.dtype == np.float64:
        return "f64"
    raise TypeError(f"oracle supports float32/float64, got {a.dtype}")


def _chk(a: np.ndarray, like: np.ndarray | None = None) -> np.ndarray:
    assert a.ndim == 3 and a.flags.c_contiguous, "need C-contiguous (nz, ny, nx) array"
    if like is not None:
        assert a.shape == like.shape and a.dtype == like.dtype
    return a


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_P)


def _dims(a):
    nz, ny, nx = a.shape
    return nx, ny, nz


def max_threads() -> int:
    return lib().orc_max_threads()


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


# ---- O4 -------------------------------------------------------------------
def cutoff(phi_c: float, beta: float, gamma: float, dtype=np.float64) -> float:
    """c(phi) of eq. 7, evaluated in `dtype`."""
    s = "f32" if np.dtype(dtype) == np.float32 else "f64"
    return getattr(lib(), f"orc_cutoff_{s}")(phi_c, beta, gamma)


# ---- O2/O3 ----------------------------------------------------------------
def upwind_q(phi: np.ndarray, i: int, j: int, k: int, dx: float):
    """(q+, q-) = ((nabla+)^2, (nabla-)^2) of eq. 4-5 at point (i, j, k)."""
    _chk(phi)
    qp, qm = _D(), _D()
    getattr(lib(), f"orc_upwind_q_{_suf(phi)}")(_ptr(phi), *_dims(phi), i, j, k, dx, C.byref(qp), C.byref(qm))
    return qp.value, qm.value


# ---- O5 -------------------------------------------------------------------
def band_masks(phi: np.ndarray, gamma: float):
    """Point masks (uint8 0/1) of tubes T (eq. 6) and N (eq. 11)."""
    _chk(phi)
    Tm = np.empty(phi.shape, np.uint8)
    Nm = np.empty(phi.shape, np.uint8)
    getattr(lib(), f"orc_band_masks_{_suf(phi)}")(_ptr(phi), *_dims(phi), gamma, _ptr(Tm), _ptr(Nm))
    return Tm, Nm


def brick_list(mask: np.ndarray):
    """Ascending ids (int32) + 8 uint64 words per brick of the 8^3 bricks that hold a mask point."""
    assert mask.dtype == np.uint8 and mask.ndim == 3 and mask.flags.c_contiguous
    n_pts = _L()
    nb = lib().orc_brick_list(_ptr(mask), *_dims(mask), None, None, 0, C.byref(n_pts))
    ids = np.empty(nb, np.int32)
    words = np.empty((nb, 8), np.uint64)
    lib().orc_brick_list(_ptr(mask), *_dims(mask), _ptr(ids), _ptr(words), nb, None)
    return ids, words, int(n_pts.value)


# ---- O6 -------------------------------------------------------------------
def advance(phi, F, Tmask, dt, dx, beta, gamma):
    """phi_bar (eq. 3/8).  Tmask=None: every point (full-domain mode)."""
    _chk(phi); _chk(F, phi)
    out = np.empty_like(phi)
    getattr(lib(), f"orc_advance_{_suf(phi)}")(_ptr(phi), _ptr(F), _ptr(Tmask), *_dims(phi),
                                               dt, dx, beta, gamma, _ptr(out))
    return out


def advance_point(phi, F, i, j, k, dt, dx, beta, gamma) -> float:
    return getattr(lib(), f"orc_advance_point_{_suf(phi)}")(_ptr(phi), _ptr(F), *_dims(phi), i, j, k,
                                                            dt, dx, beta, gamma)


def advance_list(phi, F, ids, words, dt, dx, beta, gamma, out):
    """List-driven O6: writes only listed points of `out`."""
    getattr(lib(), f"orc_advance_list_{_suf(phi)}")(_ptr(phi), _ptr(F), _ptr(ids), _ptr(words), len(ids),
                                                    *_dims(phi), dt, dx, beta, gamma, _ptr(out))
    return out


# ---- O7 -------------------------------------------------------------------
def reinit_iter(d, Nmask, dtau, dx):
    """One Jacobi iteration of eq. 12-13 on N. Returns (d_next, residual)."""
    _chk(d)
    out = np.empty_like(d)
    r = getattr(lib(), f"orc_reinit_iter_{_suf(d)}")(_ptr(d), _ptr(Nmask), *_dims(d), dtau, dx, _ptr(out))
    return out, r


def reinit_point(d, i, j, k, dtau, dx) -> float:
    return getattr(lib(), f"orc_reinit_point_{_suf(d)}")(_ptr(d), *_dims(d), i, j, k, dtau, dx)


def reinit_iter_list(d, ids, words, dtau, dx, out):
    getattr(lib(), f"orc_reinit_iter_list_{_suf(d)}")(_ptr(d), _ptr(ids), _ptr(words), len(ids),
                                                      *_dims(d), dtau, dx, _ptr(out))
    return out


def clamp(d, gamma):
    """eq. 10 on every point, in place."""
    getattr(lib(), f"orc_clamp_{_suf(d)}")(_ptr(d), d.size, gamma)
    return d


def reinit(phi_bar, Nmask, dtau, dx, gamma, iters):
    """`iters` x O7 from d0 = phi_bar, then eq. 10 everywhere."""
    d = phi_bar.copy()
    for _ in range(iters):
        d, _r = reinit_iter(d, Nmask, dtau, dx)
    return clamp(d, gamma)


# ---- O8 -------------------------------------------------------------------
def step(phi, F, dx, dt, dtau, beta, gamma, iters, n_steps=1, use_lists=False):
    """n_steps narrow-band steps. Returns (phi_new, band point-updates performed)."""
    _chk(phi); _chk(F, phi)
    out = phi.copy()
    upd = _L()
    rc = getattr(lib(), f"orc_step_{_suf(phi)}")(_ptr(out), _ptr(F), *_dims(phi), dx, dt, dtau, beta, gamma,
                                                 iters, n_steps, int(use_lists), C.byref(upd))
    if rc != 0:
        raise MemoryError("oracle step: allocation failed")
    return out, int(upd.value)


def reinit_tol(phi_bar, dtau, dx, gamma, tol, max_iters, check_every=1):
    """cfg 5: returns (d, iterations, residual, converged)."""
    _chk(phi_bar)
    d = np.empty_like(phi_bar)
    res, conv = _D(), _I()
    k = getattr(lib(), f"orc_reinit_tol_{_suf(phi_bar)}")(_ptr(phi_bar), _ptr(d), *_dims(phi_bar), dtau, dx,
                                                          gamma, tol, max_iters, check_every,
                                                          C.byref(res), C.byref(conv))
    return d, k, res.value, bool(conv.value)
