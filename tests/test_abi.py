"""CPU-side checks of the boundary: libls.so builds, loads without a GPU, exports every symbol that
include/ls.h declares, rejects bad arguments before touching CUDA, and fails loudly (no fallback)
when there is no device."""
import ctypes as C
import re
from pathlib import Path

import pytest

from paper_1612_04040_b200 import binding as ls
from paper_1612_04040_b200 import build as ls_build

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    ls_build.build()
    return ls.lib()


def _declared_in_header():
    text = (ROOT / "include" / "ls.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ls_[a-z_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    declared = _declared_in_header()
    assert declared == sorted(ls.SYMBOLS), "binding.SYMBOLS must list exactly what ls.h declares"
    for name in declared:
        assert getattr(lib, name) is not None


def test_status_strings(lib):
    names = ["LS_OK", "LS_ERR_ARG", "LS_ERR_DIM", "LS_ERR_DTYPE", "LS_ERR_ALLOC", "LS_ERR_CUDA", "LS_ERR_CAPACITY",
             "LS_NOT_CONVERGED", "LS_ERR_STATE"]
    for code, name in enumerate(names):
        assert lib.ls_status_str(code).decode() == name
    assert lib.ls_status_str(99).decode() == "LS_UNKNOWN"


def test_params_struct_layout():
    assert C.sizeof(ls.ls_params) == 56
    assert ls.ls_params.iters.offset == 40 and ls.ls_params.rebuild.offset == 44
    assert ls.ls_params.chained.offset == 48 and ls.ls_params.fuse.offset == 52


def test_bad_arguments_rejected_before_cuda(lib):
    out = C.c_void_p()
    assert lib.ls_create(0, 8, 8, ls.LS_F32, None, C.byref(out)) == ls.LS_ERR_DIM
    assert lib.ls_create(8, 8, -1, ls.LS_F32, None, C.byref(out)) == ls.LS_ERR_DIM
    assert lib.ls_create(8, 8, 8, 7, None, C.byref(out)) == ls.LS_ERR_DTYPE
    assert lib.ls_create(8, 8, 8, ls.LS_F32, None, None) == ls.LS_ERR_ARG
    assert lib.ls_create(1 << 14, 1 << 14, 1 << 14, ls.LS_F32, None, C.byref(out)) == ls.LS_ERR_DIM
    # null ctx
    p = ls.make_params(1.0, 0.1, 0.1, 1.0, 2.0, 1)
    assert lib.ls_step(None, None, None, C.byref(p), 1) == ls.LS_ERR_ARG
    assert lib.ls_build_band(None, None, 1.0, 1.0) == ls.LS_ERR_ARG
    assert lib.ls_destroy(None) == ls.LS_OK
    assert lib.ls_tile_threshold(None, 0) == ls.LS_ERR_ARG


def test_no_device_fails_loudly(lib):
    """On a box without a GPU the library must report LS_ERR_CUDA, never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    out = C.c_void_p()
    assert lib.ls_create(8, 8, 8, ls.LS_F32, None, C.byref(out)) == ls.LS_ERR_CUDA
    assert out.value is None
    assert lib.ls_last_cuda_error().decode() != ""
    with pytest.raises(ls.LsError):
        ls.ls_create(8, 8, 8, ls.LS_F32)


def test_product_does_not_import_oracle():
    """The product package never references oracle/ (the oracle is test infrastructure)."""
    pkg = ROOT / "paper_1612_04040_b200"
    for path in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.h")):
        text = path.read_text()
        assert "import oracle" not in text and "from oracle" not in text and "ls_oracle" not in text, path
        assert "liboracle" not in text, path


def test_packed_fp32_arithmetic_is_not_contracted():
    """The fp32 band kernels evaluate one item (4 cells) per lane as two packed pairs: FADD2 / FMUL2 / FFMA2.
    ptxas 12.9 contracts mul.rn.f32x2 + add.rn.f32x2 into one FFMA2 even under -fmad=false, which would break
    the arithmetic contract (R18: no FMA contraction); ls_math.cuh forms every product that feeds a sum as
    fma(a, b, +0) to prevent it.  The packed instruction mix per kernel is therefore fixed by the formulas:
      reinit sweep, per pair: 6 differences + 5 sums + den^2 + 2 sqrt seeds + (g - 1) + (c - dtau U) = 16 FADD2;
        6 scalings + 2x2 sqrt + U = 11 FMUL2; 6 squares + 2 (den^2) + 2x2 sqrt + 5 divide + dtau U = 18 FFMA2
      Advance, per pair: 16 FADD2, 13 FMUL2, 10 FFMA2
    and two pairs per item; the two-sweep kernels (temporal blocking) hold four copies of the sweep (three
    unrolled rounds of sweep 1 and sweep 2).  A different count means the toolchain fused (or split) something: fail here, on
    the CPU.  (The scalar slow path of the same kernels uses FADD / FMUL / FFMA, which are not counted.)"""
    import re
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not Path(cuobjdump).exists():
        pytest.skip("cuobjdump not available")
    from paper_1612_04040_b200 import build as ls_build
    so = ls_build.build()
    sass = subprocess.run([cuobjdump, "-sass", str(so)], capture_output=True, text=True, check=True).stdout
    counts, tma_ops, ldgsts = {}, {}, {}
    fn = None
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            fn = m.group(1)
            continue
        if not fn:
            continue
        for op in ("FFMA2", "FMUL2", "FADD2"):
            if re.search(r"\b" + op + r"\b", line):
                counts.setdefault(fn, {}).setdefault(op, 0)
                counts[fn][op] += 1
        if "UTMALDG" in line or "UBLKCP" in line:
            tma_ops[fn] = tma_ops.get(fn, 0) + 1
        if "LDGSTS" in line:
            ldgsts[fn] = ldgsts.get(fn, 0) + 1
    # mangled: k_band_tile<float, ADV, K, ...> -> "k_band_tileIfLb0ELi1E..." (one sweep), "...IfLb0ELi2E..." (two
    # sweeps), "...IfLb1ELi1E..." (advance)
    reinit_f32 = [f for f in counts if "k_band_tileIfLb0ELi1E" in f]
    reinit2_f32 = [f for f in counts if "k_band_tileIfLb0ELi2E" in f]
    advance_f32 = [f for f in counts if "k_band_tileIfLb1ELi1E" in f]
    assert len(reinit_f32) == 5 and len(reinit2_f32) == 5 and len(advance_f32) == 1, (reinit_f32, reinit2_f32, advance_f32)
    for f in reinit_f32:
        assert counts[f] == {"FFMA2": 36, "FMUL2": 22, "FADD2": 32}, (f, counts[f])
    for f in reinit2_f32:
        assert counts[f] == {"FFMA2": 144, "FMUL2": 88, "FADD2": 128}, (f, counts[f])
    assert counts[advance_f32[0]] == {"FFMA2": 20, "FMUL2": 26, "FADD2": 32}, counts[advance_f32[0]]
    # and the band kernels really use the asynchronous copy paths: the two-sweep kernels take whole boxes by TMA
    # (cp.async.bulk.tensor -> UTMALDG); the one-sweep kernels gather the sectors they need with cp.async (LDGSTS) and
    # take the item list by cp.async.bulk (UBLKCP)
    for f in reinit2_f32:
        assert tma_ops.get(f, 0) >= 2, f
    for f in reinit_f32 + advance_f32:
        assert tma_ops.get(f, 0) >= 1 and ldgsts.get(f, 0) >= 4, f
