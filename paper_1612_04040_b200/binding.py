"""Thin ctypes binding of libls.so (include/ls.h).  Argument marshalling only.

Every function has the name and argument order of its C counterpart; device fields are torch CUDA
tensors (or raw integer device addresses), shape (nz, ny, nx), contiguous, dtype float32/float64.
PyTorch is used for device memory and the stream handle only.  There is NO fallback: if libls.so
is missing or fails to load, importing symbols from here raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
_SO = _PKG / "libls.so"

LS_OK, LS_ERR_ARG, LS_ERR_DIM, LS_ERR_DTYPE, LS_ERR_ALLOC, LS_ERR_CUDA, LS_ERR_CAPACITY, LS_NOT_CONVERGED, \
    LS_ERR_STATE = range(9)
LS_F32, LS_F64 = 0, 1
LS_REBUILD_FULL, LS_REBUILD_INCREMENTAL = 0, 1
LS_K_CLASSIFY, LS_K_BAND, LS_K_ADVANCE, LS_K_REINIT, LS_K_CLAMP, LS_K_COPY, LS_K_KINDS = range(7)
KERNEL_KINDS = ("classify", "band", "advance", "reinit", "clamp", "copy")

# every symbol include/ls.h declares (tests/test_abi.py checks the library exports them all)
SYMBOLS = (
    "ls_status_str", "ls_last_cuda_error", "ls_create", "ls_destroy", "ls_build_band", "ls_band_counts",
    "ls_band_export", "ls_advance", "ls_reinit", "ls_reinit_tol", "ls_step", "ls_step_host", "ls_stats",
    "ls_stats_reset", "ls_profile_enable", "ls_profile_read", "ls_profile_reset", "ls_selftest_math", "ls_step_snapshots",
    "ls_tile_threshold",
)
# every symbol include/ls_static.h declares (tests/test_zz_no_alloc.py checks them)
STATIC_SYMBOLS = ("ls_tube_static_setup", "ls_tube_static", "ls_tube_static_error")
LS_TUBE_STATIC_MAX_BRICKS = 65536


class ls_params(C.Structure):
    _fields_ = [("dx", C.c_double), ("dt", C.c_double), ("dtau", C.c_double), ("beta", C.c_double),
                ("gamma", C.c_double), ("iters", C.c_int32), ("rebuild", C.c_int32),
                ("chained", C.c_int32), ("fuse", C.c_int32)]


class LsError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().ls_status_str(status).decode()
        detail = lib().ls_last_cuda_error().decode() if status == LS_ERR_CUDA else ""
        super().__init__(f"{where}: {msg}" + (f" ({detail})" if detail else ""))


_lib = None
_P, _D, _I, _L = C.c_void_p, C.c_double, C.c_int32, C.c_int64


def lib() -> C.CDLL:
    """Load libls.so (built by paper_1612_04040_b200.build).  Raises if it is absent."""
    global _lib
    if _lib is None:
        if not _SO.exists():
            raise FileNotFoundError(
                f"{_SO} not found: run `python -m paper_1612_04040_b200.build` (nvcc, sm_100a). "
                "There is no CPU fallback.")
        L = C.CDLL(str(_SO))
        L.ls_status_str.restype = C.c_char_p
        L.ls_status_str.argtypes = [C.c_int]
        L.ls_last_cuda_error.restype = C.c_char_p
        L.ls_last_cuda_error.argtypes = []
        L.ls_create.argtypes = [_I, _I, _I, C.c_int, _P, C.POINTER(_P)]
        L.ls_destroy.argtypes = [_P]
        L.ls_build_band.argtypes = [_P, _P, _D, _D]
        L.ls_band_counts.argtypes = [_P, C.POINTER(_L), C.POINTER(_L), C.POINTER(_I), C.POINTER(_I)]
        L.ls_band_export.argtypes = [_P, _P, _P, _P, _P]
        L.ls_advance.argtypes = [_P, _P, _P, _D, _D, _D, _D, _P]
        L.ls_reinit.argtypes = [_P, _P, _P, _D, _D, _D, _I]
        L.ls_reinit_tol.argtypes = [_P, _P, _P, _D, _D, _D, _D, _I, _I, C.POINTER(_I), C.POINTER(_D)]
        L.ls_step.argtypes = [_P, _P, _P, C.POINTER(ls_params), _I]
        L.ls_step_host.argtypes = [_P, _P, _P, C.POINTER(ls_params), _I]
        L.ls_stats.argtypes = [_P, C.POINTER(_L), C.POINTER(_L), C.POINTER(_L)]
        L.ls_stats_reset.argtypes = [_P]
        L.ls_profile_enable.argtypes = [_P, _I]
        L.ls_profile_read.argtypes = [_P, _I, C.POINTER(_D), C.POINTER(_L)]
        L.ls_profile_reset.argtypes = [_P]
        L.ls_step_snapshots.argtypes = [_P, _P, _P, C.POINTER(ls_params), _I, _I, _P, C.POINTER(_I)]
        L.ls_tile_threshold.argtypes = [_P, _L]
        L.ls_selftest_math.argtypes = [_P, C.c_uint64, _L, _D, _D, _D, _D, C.POINTER(_L)]
        for name in SYMBOLS[2:]:
            getattr(L, name).restype = C.c_int
        L.ls_tube_static_setup.argtypes = []
        L.ls_tube_static_setup.restype = C.c_int
        L.ls_tube_static.argtypes = [_P, _I, _I, _I, C.c_int, _D, _P, _P, _P, _P]
        L.ls_tube_static.restype = C.c_int
        L.ls_tube_static_error.argtypes = []
        L.ls_tube_static_error.restype = C.c_char_p
        _lib = L
    return _lib


def _dev(t) -> int:
    """Device address of a torch CUDA tensor (checked) or a raw int."""
    if isinstance(t, int):
        return t
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return t.data_ptr()


def _host(a) -> int:
    """Host address of a numpy array / CPU torch tensor (contiguous) or a raw int."""
    if isinstance(a, int):
        return a
    if isinstance(a, np.ndarray):
        if not a.flags.c_contiguous:
            raise ValueError("expected a C-contiguous array")
        return a.ctypes.data
    if a.is_cuda or not a.is_contiguous():
        raise ValueError("expected a contiguous CPU tensor")
    return a.data_ptr()


def _ck(status: int, where: str, ok=(LS_OK,)) -> int:
    if status not in ok:
        raise LsError(status, where)
    return status


def ls_create(nx: int, ny: int, nz: int, dtype: int, cuda_stream: int = 0) -> int:
    """-> opaque ctx handle (int).  `cuda_stream` is e.g. torch.cuda.current_stream().cuda_stream."""
    out = _P()
    _ck(lib().ls_create(nx, ny, nz, dtype, _P(cuda_stream), C.byref(out)), "ls_create")
    return out.value


def ls_destroy(ctx: int) -> None:
    _ck(lib().ls_destroy(_P(ctx)), "ls_destroy")


def ls_build_band(ctx: int, phi, dx: float, gamma: float) -> None:
    _ck(lib().ls_build_band(_P(ctx), _P(_dev(phi)), dx, gamma), "ls_build_band")


def ls_band_counts(ctx: int):
    """-> (nT_points, nN_points, nT_bricks, nN_bricks)"""
    a, b, c, d = _L(), _L(), _I(), _I()
    _ck(lib().ls_band_counts(_P(ctx), C.byref(a), C.byref(b), C.byref(c), C.byref(d)), "ls_band_counts")
    return a.value, b.value, c.value, d.value


def ls_band_export(ctx: int):
    """-> (T_ids int32[nT], T_masks uint64[nT,8], N_ids int32[nN], N_masks uint64[nN,8]) as numpy arrays."""
    _, _, nT, nN = ls_band_counts(ctx)
    T_ids = np.empty(nT, np.int32)
    T_masks = np.empty((nT, 8), np.uint64)
    N_ids = np.empty(nN, np.int32)
    N_masks = np.empty((nN, 8), np.uint64)
    _ck(lib().ls_band_export(_P(ctx), _P(_host(T_ids)), _P(_host(T_masks)), _P(_host(N_ids)), _P(_host(N_masks))),
        "ls_band_export")
    return T_ids, T_masks, N_ids, N_masks


def ls_advance(ctx: int, phi, F, dt: float, dx: float, beta: float, gamma: float, out) -> None:
    _ck(lib().ls_advance(_P(ctx), _P(_dev(phi)), _P(_dev(F)), dt, dx, beta, gamma, _P(_dev(out))), "ls_advance")


def ls_reinit(ctx: int, d, phi_bar, dtau: float, dx: float, gamma: float, iters: int) -> None:
    _ck(lib().ls_reinit(_P(ctx), _P(_dev(d)), _P(_dev(phi_bar)), dtau, dx, gamma, iters), "ls_reinit")


def ls_reinit_tol(ctx: int, d, phi_bar, dtau: float, dx: float, gamma: float, tol: float, max_iters: int,
                  check_every: int = 1):
    """-> (iters_done, residual, converged)"""
    k, r = _I(), _D()
    st = _ck(lib().ls_reinit_tol(_P(ctx), _P(_dev(d)), _P(_dev(phi_bar)), dtau, dx, gamma, tol, max_iters,
                                 check_every, C.byref(k), C.byref(r)), "ls_reinit_tol", ok=(LS_OK, LS_NOT_CONVERGED))
    return k.value, r.value, st == LS_OK


def make_params(dx, dt, dtau, beta, gamma, iters, rebuild=LS_REBUILD_FULL, chained=0, fuse=0) -> ls_params:
    return ls_params(dx, dt, dtau, beta, gamma, iters, rebuild, chained, fuse)


def ls_step(ctx: int, phi, F, p: ls_params, n_steps: int) -> None:
    _ck(lib().ls_step(_P(ctx), _P(_dev(phi)), _P(_dev(F)), C.byref(p), n_steps), "ls_step")


def ls_step_host(ctx: int, phi_host, F_host, p: ls_params, n_steps: int) -> None:
    """F_host=None: reuse the F the last call with an F_host left on the device."""
    f = _P(None) if F_host is None else _P(_host(F_host))
    _ck(lib().ls_step_host(_P(ctx), _P(_host(phi_host)), f, C.byref(p), n_steps), "ls_step_host")


def ls_stats(ctx: int):
    """-> (point_updates, steps, kernel_launches)"""
    a, b, c = _L(), _L(), _L()
    _ck(lib().ls_stats(_P(ctx), C.byref(a), C.byref(b), C.byref(c)), "ls_stats")
    return a.value, b.value, c.value


def ls_stats_reset(ctx: int) -> None:
    _ck(lib().ls_stats_reset(_P(ctx)), "ls_stats_reset")


def ls_tile_threshold(ctx: int, min_cells: int) -> None:
    """0 = tiled kernels wherever they can run; negative = the library default (4 000 000 cells)."""
    _ck(lib().ls_tile_threshold(_P(ctx), min_cells), "ls_tile_threshold")


def ls_profile_enable(ctx: int, on: bool) -> None:
    _ck(lib().ls_profile_enable(_P(ctx), int(bool(on))), "ls_profile_enable")


def ls_profile_read(ctx: int, kind: int):
    """-> (ms_total, launches) of one ls_kernel_kind"""
    ms, n = _D(), _L()
    _ck(lib().ls_profile_read(_P(ctx), kind, C.byref(ms), C.byref(n)), "ls_profile_read")
    return ms.value, n.value


def ls_profile_reset(ctx: int) -> None:
    _ck(lib().ls_profile_reset(_P(ctx)), "ls_profile_reset")


def ls_selftest_math(seed: int, n: int, dx: float, dt: float, beta: float, gamma: float, cuda_stream: int = 0) -> int:
    """-> number of results (of 4n) where the packed fp32 pair arithmetic differs from the scalar IEEE path."""
    m = _L()
    _ck(lib().ls_selftest_math(_P(cuda_stream), C.c_uint64(seed), n, dx, dt, beta, gamma, C.byref(m)),
        "ls_selftest_math")
    return m.value


def ls_step_snapshots(ctx: int, phi, F, p: ls_params, n_steps: int, every: int, host_out) -> int:
    """-> number of snapshots written to `host_out` (numpy array / CPU tensor of >= n_steps//every fields)."""
    n = _I()
    _ck(lib().ls_step_snapshots(_P(ctx), _P(_dev(phi)), _P(_dev(F)), C.byref(p), n_steps, every,
                                _P(_host(host_out)) if host_out is not None else None, C.byref(n)),
        "ls_step_snapshots")
    return n.value


def ls_tube_static_setup() -> None:
    st = lib().ls_tube_static_setup()
    if st != LS_OK:
        raise LsError(st, "ls_tube_static_setup: " + lib().ls_tube_static_error().decode())


def ls_tube_static(phi, nx: int, ny: int, nz: int, dtype: int, gamma: float, cuda_stream: int, T_ids, T_masks, counts) -> None:
    """include/ls_static.h: T tube with no ctx and no allocation.  T_ids int32[nbricks], T_masks int64/uint64[8*nbricks],
    counts int64[2] are DEVICE tensors (or addresses) the caller owns; nothing is read back here."""
    st = lib().ls_tube_static(_P(_dev(phi)), nx, ny, nz, dtype, gamma, _P(cuda_stream), _P(_dev(T_ids)), _P(_dev(T_masks)),
                              _P(_dev(counts)))
    if st != LS_OK:
        raise LsError(st, "ls_tube_static: " + lib().ls_tube_static_error().decode())
