"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI, the oracle on the host."""
from __future__ import annotations

import numpy as np
import torch

from oracle import ls_oracle as orc
from paper_1612_04040_b200 import binding as ls

# north_star tolerances: elementwise max-abs error per step, in units of dx
TOL_F32 = 1e-5
TOL_F64 = 1e-12


def tol_for(dtype) -> float:
    return TOL_F32 if np.dtype(dtype) == np.float32 else TOL_F64


def dtype_code(dtype) -> int:
    return ls.LS_F32 if np.dtype(dtype) == np.float32 else ls.LS_F64


def to_dev(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class Ctx:
    """ctx bound to torch's current stream.  tile_min_cells = 0 (the default here): the tiled band kernels wherever they
    can run, so that the small parity shapes exercise them; None: the library's own threshold (small grids take the
    scalar kernels even when their rows are aligned)."""

    def __init__(self, shape, dtype, tile_min_cells=0):
        nz, ny, nx = shape
        self.h = ls.ls_create(nx, ny, nz, dtype_code(dtype), torch.cuda.current_stream().cuda_stream)
        if tile_min_cells is not None:
            ls.ls_tile_threshold(self.h, tile_min_cells)

    def __enter__(self):
        return self.h

    def __exit__(self, *exc):
        ls.ls_destroy(self.h)
        return False


def oracle_band(phi: np.ndarray, gamma: float):
    """-> (Tmask, Nmask, (T_ids, T_words, nT_pts), (N_ids, N_words, nN_pts)) from the oracle."""
    Tm, Nm = orc.band_masks(phi, gamma)
    return Tm, Nm, orc.brick_list(Tm), orc.brick_list(Nm)


def assert_band_equal(ctx: int, phi: np.ndarray, gamma: float):
    """Bit-exact comparison of the ctx's current band with the oracle's band of `phi`."""
    Tm, Nm, (T_ids, T_w, nT), (N_ids, N_w, nN) = oracle_band(phi, gamma)
    cT, cN, bT, bN = ls.ls_band_counts(ctx)
    assert (cT, cN, bT, bN) == (nT, nN, len(T_ids), len(N_ids)), \
        f"counts differ: gpu {(cT, cN, bT, bN)} oracle {(nT, nN, len(T_ids), len(N_ids))}"
    gT_ids, gT_w, gN_ids, gN_w = ls.ls_band_export(ctx)
    assert np.array_equal(gT_ids, T_ids), "T brick ids differ"
    assert np.array_equal(gT_w, T_w), "T mask words differ"
    assert np.array_equal(gN_ids, N_ids), "N brick ids differ"
    assert np.array_equal(gN_w, N_w), "N mask words differ"
    return Tm, Nm


def max_err_dx(a: np.ndarray, b: np.ndarray, dx: float) -> float:
    return float(np.max(np.abs(a.astype(np.float64) - b.astype(np.float64)))) / dx
