"""include/ls_static.h — ls_tube_static, the one entry point that allocates nothing (its work memory is a file-scope
`static __device__` array of libls.so).  Collected LAST on purpose (the suite runs with pytest -x).

CPU part: the symbols are exported, sizes beyond LS_TUBE_STATIC_MAX_BRICKS and bad arguments are rejected before any
CUDA call, and the translation unit calls no allocating CUDA routine.
GPU part: its output against the existing path (ls_create + ls_build_band + ls_band_counts + ls_band_export), bit for
bit (integer work: the tolerance of every band test here is exact equality), on calls in a row that share the array —
larger grid, then smaller, then the first again — and against the oracle; free device memory does not move.
"""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest
import torch

from paper_1612_04040_b200 import binding as ls
from paper_1612_04040_b200 import build as ls_build
from paper_1612_04040_b200 import inputs

ROOT = Path(__file__).resolve().parent.parent
FAKE = 0x1000   # a non-null "pointer" for calls that must return before touching CUDA


@pytest.fixture(scope="module")
def lib():
    ls_build.build()
    return ls.lib()


def _call(lib, phi, nx, ny, nz, dtype, gamma, ids=FAKE, masks=FAKE, counts=FAKE):
    P = C.c_void_p
    return lib.ls_tube_static(P(phi), nx, ny, nz, dtype, gamma, None, P(ids), P(masks), P(counts))


def test_static_header_symbols_exported(lib):
    text = (ROOT / "include" / "ls_static.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = sorted(set(re.findall(r"\b(ls_[a-z_]+)\s*\(", text)))
    assert declared == sorted(ls.STATIC_SYMBOLS)
    for name in declared:
        assert getattr(lib, name) is not None
    m = re.search(r"#define\s+LS_TUBE_STATIC_MAX_BRICKS\s+(\d+)", text)
    assert int(m.group(1)) == ls.LS_TUBE_STATIC_MAX_BRICKS


def test_sizes_beyond_the_maximum_are_rejected_before_cuda(lib):
    # 41 x 40 x 40 = 65600 bricks > 65536; also a product that would overflow 32 bits
    for nx, ny, nz in [(328, 320, 320), (2 ** 31 - 1, 2 ** 31 - 1, 2 ** 31 - 1), (8 * 65536 + 1, 1, 1)]:
        assert _call(lib, FAKE, nx, ny, nz, ls.LS_F32, 1.0) == ls.LS_ERR_CAPACITY
        msg = lib.ls_tube_static_error().decode()
        assert "LS_TUBE_STATIC_MAX_BRICKS = 65536" in msg and "ls_build_band" in msg, msg


def test_bad_arguments_rejected_before_cuda(lib):
    assert _call(lib, None, 8, 8, 8, ls.LS_F32, 1.0) == ls.LS_ERR_ARG
    assert _call(lib, FAKE, 8, 8, 8, ls.LS_F32, 1.0, ids=None) == ls.LS_ERR_ARG
    assert _call(lib, FAKE, 8, 8, 8, ls.LS_F32, 1.0, masks=None) == ls.LS_ERR_ARG
    assert _call(lib, FAKE, 8, 8, 8, ls.LS_F32, 1.0, counts=None) == ls.LS_ERR_ARG
    assert _call(lib, FAKE, 8, 8, 8, ls.LS_F32, 0.0) == ls.LS_ERR_ARG
    assert _call(lib, FAKE, 8, 8, 8, ls.LS_F32, float("nan")) == ls.LS_ERR_ARG
    assert _call(lib, FAKE, 0, 8, 8, ls.LS_F32, 1.0) == ls.LS_ERR_DIM
    assert _call(lib, FAKE, 8, 8, -3, ls.LS_F64, 1.0) == ls.LS_ERR_DIM
    assert _call(lib, FAKE, 8, 8, 8, 7, 1.0) == ls.LS_ERR_DTYPE
    assert lib.ls_tube_static_error().decode() != ""


def test_no_device_fails_loudly(lib):
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    assert lib.ls_tube_static_setup() == ls.LS_ERR_CUDA
    assert _call(lib, FAKE, 256, 256, 512, ls.LS_F32, 1.0) == ls.LS_ERR_CUDA   # exactly the maximum: not a capacity error
    assert "ls_tube_static" in lib.ls_tube_static_error().decode()


def test_translation_unit_calls_no_allocating_routine():
    text = (ROOT / "paper_1612_04040_b200" / "csrc" / "ls_static.cu").read_text()
    code = re.sub(r"//[^\n]*", " ", re.sub(r"/\*.*?\*/", " ", text, flags=re.S))
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMemPool", "cuMemAlloc", "malloc(", "new ", "std::vector",
                   "cub::", "thrust::", "ls_internal.h"):
        assert banned not in code, banned
    assert re.search(r"static\s+__device__\s+__align__\(256\)\s+unsigned long long\s+g_tube_scratch\[", code)
    assert "cudaGetSymbolAddress((void**)&ptr, g_tube_scratch)" in code
    # the array's name appears in host code only as the argument of cudaGetSymbolAddress, never as a kernel argument
    assert len(re.findall(r"\bg_tube_scratch\b", code)) == 2


# ------------------------------------------------------------------------------------------------------------- GPU


def _field(shape, dtype, seed, dx):
    """Smooth two-signed field with |grad| ~ 1 (broadcast sums: cheap at 33 M cells) plus seeded noise on small grids."""
    nz, ny, nx = shape
    x = np.arange(nx, dtype=np.float64)[None, None, :]
    y = np.arange(ny, dtype=np.float64)[None, :, None]
    z = np.arange(nz, dtype=np.float64)[:, None, None]
    phi = dx * (4.0 * np.sin(0.37 * x + 0.2 + seed) + 3.0 * np.cos(0.29 * y) + 3.5 * np.sin(0.23 * z + 1.0))
    if nx * ny * nz <= 1 << 20:
        phi = phi + dx * 0.8 * (inputs.uniform01(seed, 0, nx * ny * nz).reshape(shape) - 0.5)
    return np.ascontiguousarray(phi.astype(dtype))


def _existing_path(phi_dev, shape, dtype, dx, gamma):
    nz, ny, nx = shape
    code = ls.LS_F32 if dtype == np.float32 else ls.LS_F64
    ctx = ls.ls_create(nx, ny, nz, code, torch.cuda.current_stream().cuda_stream)
    try:
        ls.ls_build_band(ctx, phi_dev, dx, gamma)
        nT_pts, _, nT_bricks, _ = ls.ls_band_counts(ctx)
        T_ids, T_w, _, _ = ls.ls_band_export(ctx)
    finally:
        ls.ls_destroy(ctx)
    return nT_pts, nT_bricks, T_ids, T_w


class _Out:
    """Caller-owned outputs, pre-filled with sentinels so that a write beyond the listed bricks shows."""

    def __init__(self, shape):
        nz, ny, nx = shape
        self.nbricks = -(-nx // 8) * -(-ny // 8) * -(-nz // 8)
        self.ids = torch.full((self.nbricks,), -7, dtype=torch.int32, device="cuda")
        self.masks = torch.full((self.nbricks, 8), 0x5A5A5A5A5A5A5A5A, dtype=torch.int64, device="cuda")
        self.counts = torch.full((2,), -1, dtype=torch.int64, device="cuda")

    def check(self, expect, what):
        nT_pts, nT_bricks, T_ids, T_w = expect
        counts = self.counts.cpu().numpy()
        assert (int(counts[0]), int(counts[1])) == (nT_pts, nT_bricks), (what, counts, nT_pts, nT_bricks)
        ids = self.ids.cpu().numpy()
        masks = self.masks.cpu().numpy().view(np.uint64)
        assert np.array_equal(ids[:nT_bricks], T_ids), what + ": T brick ids differ"
        assert np.array_equal(masks[:nT_bricks], T_w), what + ": T mask words differ"
        assert np.all(ids[nT_bricks:] == -7), what + ": id written beyond the list"
        assert np.all(masks[nT_bricks:] == np.uint64(0x5A5A5A5A5A5A5A5A)), what + ": mask written beyond the list"


def _static(phi_dev, shape, dtype, gamma, out):
    nz, ny, nx = shape
    code = ls.LS_F32 if dtype == np.float32 else ls.LS_F64
    ls.ls_tube_static(phi_dev, nx, ny, nz, code, gamma, torch.cuda.current_stream().cuda_stream, out.ids, out.masks,
                      out.counts)


@pytest.mark.gpu
def test_tube_static_equals_build_band_on_calls_in_a_row():
    """The calls share the static array, which keeps what the previous call left: large grid, small grid, the large one
    again with another gamma, ragged shapes, both dtypes, a misaligned field, the exact maximum size."""
    from oracle import ls_oracle as orc
    dx = 1.0 / 32
    ls.ls_tube_static_setup()
    cases = [
        ((64, 64, 64), np.float32, 3 * dx, 11),
        ((64, 64, 64), np.float32, 3 * dx, 11),        # two calls in a row on the same input
        ((9, 13, 20), np.float64, 2 * dx, 12),         # smaller grid: stale words of the larger one stay behind it
        ((64, 64, 64), np.float32, 1.5 * dx, 13),
        ((17, 8, 33), np.float32, 3 * dx, 14),
        ((4, 4, 4), np.float64, float("inf"), 15),     # every in-domain point in T; partial bricks only
        ((24, 40, 56), np.float64, 3 * dx, 16),
        ((1, 1, 2100), np.float32, 3 * dx, 17),        # one x-row of 263 bricks: nine segments, two compaction CTAs
        ((3, 1000, 5), np.float32, 1e-9, 18),          # (almost) empty tube
        ((512, 256, 256), np.float32, 3 * dx, 19),     # exactly LS_TUBE_STATIC_MAX_BRICKS bricks
        ((40, 24, 16), np.float32, 3 * dx, 20),
    ]
    for shape, dtype, gamma, seed in cases:
        what = f"{shape} {np.dtype(dtype).name} gamma {gamma}"
        phi = _field(shape, dtype, seed, dx)
        phi_dev = torch.from_numpy(phi).cuda()
        expect = _existing_path(phi_dev, shape, dtype, dx, gamma)
        out = _Out(shape)
        _static(phi_dev, shape, dtype, gamma, out)
        torch.cuda.synchronize()
        out.check(expect, what)
        if phi.size <= 1 << 18:   # and the oracle (eq. 6), where it finishes at once
            Tm, _ = orc.band_masks(phi, gamma)
            o_ids, o_w, o_pts = orc.brick_list(Tm)
            assert expect[0] == o_pts and np.array_equal(expect[2], o_ids) and np.array_equal(expect[3], o_w), what
    # a field that starts one element past a 256-byte boundary ("any alignment of the element type")
    shape, dtype, gamma = (17, 8, 33), np.float32, 3 * dx
    phi = _field(shape, dtype, 21, dx)
    aligned = torch.from_numpy(phi).cuda()
    buf = torch.empty(phi.size + 1, dtype=torch.float32, device="cuda")
    buf[1:].copy_(aligned.reshape(-1))
    out = _Out(shape)
    _static(buf[1:], shape, dtype, gamma, out)
    torch.cuda.synchronize()
    out.check(_existing_path(aligned, shape, dtype, dx, gamma), "misaligned field")


@pytest.mark.gpu
def test_tube_static_back_to_back_without_sync_and_no_allocation():
    """Calls queued on one stream with no synchronisation between them are ordered by the stream (the documented way to
    share the array); free device memory is the same before and after."""
    dx = 1.0 / 32
    ls.ls_tube_static_setup()
    work = []
    for i, (shape, dtype, gamma) in enumerate([((64, 64, 64), np.float32, 3 * dx), ((24, 40, 56), np.float64, 2 * dx),
                                               ((64, 64, 64), np.float32, 2 * dx), ((9, 13, 20), np.float32, 3 * dx)]):
        phi_dev = torch.from_numpy(_field(shape, dtype, 30 + i, dx)).cuda()
        work.append((shape, dtype, gamma, phi_dev, _existing_path(phi_dev, shape, dtype, dx, gamma), _Out(shape)))
    _static(work[0][3], work[0][0], work[0][1], work[0][2], work[0][5])   # warm: module loaded, address resolved
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        for shape, dtype, gamma, phi_dev, _, out in work:
            _static(phi_dev, shape, dtype, gamma, out)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, (free_before, free_after)
    for shape, dtype, gamma, _, expect, out in work:
        out.check(expect, f"{shape} queued back to back")


@pytest.mark.gpu
def test_tube_static_under_stream_capture():
    """What the entry point is for: it can be captured into a CUDA graph (a ctx call that allocates cannot) and replayed."""
    dx = 1.0 / 32
    shape, dtype, gamma = (40, 24, 16), np.float32, 3 * dx
    ls.ls_tube_static_setup()
    phi_dev = torch.from_numpy(_field(shape, dtype, 40, dx)).cuda()
    expect = _existing_path(phi_dev, shape, dtype, dx, gamma)
    out = _Out(shape)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        _static(phi_dev, shape, dtype, gamma, out)
    for _ in range(2):
        out.counts.fill_(-1)
        graph.replay()
        torch.cuda.synchronize()
        out.check(expect, "graph replay")
    # new contents in the same buffer, same graph
    phi2 = _field(shape, dtype, 41, dx)
    phi_dev.copy_(torch.from_numpy(phi2))
    expect2 = _existing_path(phi_dev, shape, dtype, dx, gamma)
    out.ids.fill_(-7)
    out.masks.fill_(0x5A5A5A5A5A5A5A5A)
    graph.replay()
    torch.cuda.synchronize()
    out.check(expect2, "graph replay on new contents")
