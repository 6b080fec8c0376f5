"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Band masks / brick lists bit-exact; fields within the north_star
tolerances (1e-5*dx per step fp32, 1e-12*dx fp64).  Sizes span several bricks and ragged tails.
"""
import numpy as np
import pytest
import torch

from oracle import ls_oracle as orc
from paper_1612_04040_b200 import binding as ls
from paper_1612_04040_b200 import inputs

from gpu_util import Ctx, assert_band_equal, max_err_dx, to_dev, tol_for

pytestmark = pytest.mark.gpu
INF = float("inf")


def _random_band_field(shape, dtype, seed, dx):
    """A smooth two-signed field with |grad| ~ 1 plus seeded noise: several disconnected band pieces
    that touch the domain boundary."""
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    u = inputs.uniform01(seed, 0, nx * ny * nz).reshape(shape)
    phi = dx * (4.0 * np.sin(0.37 * x + 0.2) + 3.0 * np.cos(0.29 * y) + 3.5 * np.sin(0.23 * z + 1.0)
                + 0.8 * (u - 0.5))
    F = 2.0 * inputs.uniform01(seed + 1, 0, nx * ny * nz).reshape(shape) - 1.0
    return phi.astype(dtype), F.astype(dtype)


SHAPES = [(4, 4, 4), (9, 13, 20), (17, 8, 33), (24, 40, 56), (64, 64, 64)]


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("shape", SHAPES)
def test_build_band_bit_exact(shape, dtype):
    dx = 1.0 / 32
    phi, _ = _random_band_field(shape, dtype, 11, dx)
    gamma = 3 * dx
    with Ctx(shape, dtype) as ctx:
        ls.ls_build_band(ctx, to_dev(phi), dx, gamma)
        assert_band_equal(ctx, phi, gamma)


def test_build_band_edge_cases():
    dx = 0.25
    shape = (10, 10, 10)
    with Ctx(shape, np.float32) as ctx:
        # empty band
        phi = np.full(shape, 5.0, np.float32)
        ls.ls_build_band(ctx, to_dev(phi), dx, 1.0)
        assert ls.ls_band_counts(ctx) == (0, 0, 0, 0)
        T_ids, T_w, N_ids, N_w = ls.ls_band_export(ctx)
        assert len(T_ids) == 0 and len(N_ids) == 0
        # |phi| == gamma is NOT in T (strict <, eq. 6)
        phi = np.full(shape, 1.0, np.float32)
        ls.ls_build_band(ctx, to_dev(phi), dx, 1.0)
        assert ls.ls_band_counts(ctx) == (0, 0, 0, 0)
        # single point: N is its 7-point star
        phi[3, 7, 8] = 0.5          # (k, j, i): sits at a brick corner in x (i = 8)
        ls.ls_build_band(ctx, to_dev(phi), dx, 1.0)
        assert_band_equal(ctx, phi, 1.0)
        assert ls.ls_band_counts(ctx)[:2] == (1, 7)
        # gamma = +inf: every point in T and N, all bricks listed
        ls.ls_build_band(ctx, to_dev(phi), dx, INF)
        nT, nN, bT, bN = ls.ls_band_counts(ctx)
        assert (nT, nN, bT, bN) == (1000, 1000, 8, 8)
        assert_band_equal(ctx, phi, INF)


def test_worked_4x4x4_masks():
    """SURVEY/DESIGN I13: T and N mask words of the 4^3 worked example (tests/golden/worked_4x4x4.txt)."""
    i, j, k = np.meshgrid(np.arange(4), np.arange(4), np.arange(4), indexing="ij")
    phi_ijk = 1.5 * i - 0.5 * j * j + 0.25 * j * k + k - 2.25
    phi = np.ascontiguousarray(phi_ijk.transpose(2, 1, 0)).astype(np.float64)  # (k, j, i)
    with Ctx((4, 4, 4), np.float64) as ctx:
        ls.ls_build_band(ctx, to_dev(phi), 1.0, 3.0)
        nT, nN, bT, bN = ls.ls_band_counts(ctx)
        assert (nT, nN, bT, bN) == (45, 60, 1, 1)
        _, T_w, _, N_w = ls.ls_band_export(ctx)
        assert [hex(int(w)) for w in T_w[0][:4]] == ["0x80e0f0f", "0xc0f0707", "0xe070707", "0x7030303"]
        assert [hex(int(w)) for w in N_w[0][:4]] == ["0xe0f0f0f", "0xf0f0f0f", "0xf0f0f0f", "0xf070707"]
        assert not T_w[0][4:].any() and not N_w[0][4:].any()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("shape", SHAPES[1:])
def test_advance_band_parity(shape, dtype):
    dx = 1.0 / 32
    phi, F = _random_band_field(shape, dtype, 21, dx)
    gamma, beta, dt = 4 * dx, 2 * dx, 0.4 * dx
    Tm, _ = orc.band_masks(phi, gamma)
    want = orc.advance(phi, F, Tm, dt, dx, beta, gamma)
    with Ctx(shape, dtype) as ctx:
        d_phi, d_F = to_dev(phi), to_dev(F)
        out = torch.empty_like(d_phi)
        ls.ls_build_band(ctx, d_phi, dx, gamma)
        ls.ls_advance(ctx, d_phi, d_F, dt, dx, beta, gamma, out)
        got = out.cpu().numpy()
    assert max_err_dx(got, want, dx) <= tol_for(dtype)
    assert np.array_equal(got, want), "advance is expected to be bit-identical to the oracle (exact mode)"


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("shape", [(9, 13, 20), (32, 32, 32), (40, 24, 72), (5, 6, 7), (3, 9, 130)])
def test_advance_dense_parity(shape, dtype):
    dx = 1.0 / 32
    phi, F = _random_band_field(shape, dtype, 31, dx)
    dt = 0.4 * dx
    want = orc.advance(phi, F, None, dt, dx, INF, INF)
    with Ctx(shape, dtype) as ctx:
        d_phi, d_F = to_dev(phi), to_dev(F)
        out = torch.empty_like(d_phi)
        ls.ls_advance(ctx, d_phi, d_F, dt, dx, INF, INF, out)   # no band needed in full-domain mode
        got = out.cpu().numpy()
    assert max_err_dx(got, want, dx) <= tol_for(dtype)
    assert np.array_equal(got, want)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("iters", [0, 1, 2, 5])
def test_reinit_parity(iters, dtype):
    shape = (24, 40, 56)
    dx = 1.0 / 32
    phi, _ = _random_band_field(shape, dtype, 41, dx)
    gamma, dtau = 4 * dx, 0.5 * dx
    _, Nm = orc.band_masks(phi, gamma)
    want = orc.reinit(phi, Nm, dtau, dx, gamma, iters)
    with Ctx(shape, dtype) as ctx:
        d_phi = to_dev(phi)
        d = torch.empty_like(d_phi)
        ls.ls_build_band(ctx, d_phi, dx, gamma)
        ls.ls_reinit(ctx, d, d_phi, dtau, dx, gamma, iters)
        got = d.cpu().numpy()
    assert max_err_dx(got, want, dx) <= tol_for(dtype) * max(iters, 1)
    assert np.array_equal(got, want)
    assert np.all(np.abs(got) <= np.asarray(gamma, dtype))          # eq. 10 everywhere


def test_reinit_zero_stays_zero():
    """I11: points with d == 0 never move (S = 0, R12)."""
    shape = (16, 16, 16)
    dx = 1.0 / 16
    phi, _ = _random_band_field(shape, np.float32, 51, dx)
    phi[4:12, 5, 3:9] = 0.0
    with Ctx(shape, np.float32) as ctx:
        d_phi = to_dev(phi)
        d = torch.empty_like(d_phi)
        ls.ls_build_band(ctx, d_phi, dx, 3 * dx)
        ls.ls_reinit(ctx, d, d_phi, 0.5 * dx, dx, 3 * dx, 7)
        got = d.cpu().numpy()
    assert np.all(got[4:12, 5, 3:9] == 0.0)


def _run_steps(w, n_steps, rebuild, chunks=1, chained=0):
    """GPU free-running: n_steps split into `chunks` ls_step calls."""
    with Ctx(w.shape, w.dtype) as ctx:
        d_phi, d_F = to_dev(w.phi), to_dev(w.F)
        p = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, chained)
        per = n_steps // chunks
        for c in range(chunks):
            ls.ls_step(ctx, d_phi, d_F, p, per if c < chunks - 1 else n_steps - per * (chunks - 1))
        updates, steps, launches = ls.ls_stats(ctx)
        band = ls.ls_band_export(ctx)
        return d_phi.cpu().numpy(), updates, steps, band


@pytest.mark.parametrize("rebuild", [ls.LS_REBUILD_FULL, ls.LS_REBUILD_INCREMENTAL])
def test_step_cfg1_free_running(rebuild):
    """cfg 1 (64^3 sphere, F = 1, 10 steps x 5 reinit): final field, update count, last band."""
    w = inputs.config(1)
    want, upd = orc.step(w.phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, w.n_steps)
    got, updates, steps, band = _run_steps(w, w.n_steps, rebuild)
    assert steps == w.n_steps and updates == upd
    assert max_err_dx(got, want, w.dx) <= TOL * w.n_steps
    assert np.array_equal(got, want), "exact mode: free-running field is bit-identical"
    # the band the last step used is the band of phi^{n_steps-1}
    prev, _ = orc.step(w.phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, w.n_steps - 1)
    Tm, Nm = orc.band_masks(prev, w.gamma)
    T_ids, T_w, _ = orc.brick_list(Tm)
    N_ids, N_w, _ = orc.brick_list(Nm)
    assert np.array_equal(band[0], T_ids) and np.array_equal(band[1], T_w)
    assert np.array_equal(band[2], N_ids) and np.array_equal(band[3], N_w)


TOL = 1e-5


@pytest.mark.parametrize("rebuild", [ls.LS_REBUILD_FULL, ls.LS_REBUILD_INCREMENTAL])
@pytest.mark.parametrize("iters", [0, 1, 2, 5])
def test_step_teacher_forced_cfg3(iters, rebuild):
    """cfg 3 shape at 96^3 (spheres cross the boundary, two-signed F): every step restarts from the
    oracle's phi^n; the band and phi^{n+1} are compared each step."""
    w = inputs.config(3, n=96)
    phi = w.phi
    with Ctx(w.shape, w.dtype) as ctx:
        d_F = to_dev(w.F)
        p = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, iters, rebuild)
        for s in range(4):
            d_phi = to_dev(phi)
            ls.ls_step(ctx, d_phi, d_F, p, 1)
            assert_band_equal(ctx, phi, w.gamma)
            want, _ = orc.step(phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, iters, 1)
            got = d_phi.cpu().numpy()
            assert max_err_dx(got, want, w.dx) <= TOL, f"step {s}"
            assert np.array_equal(got, want), f"step {s}"
            phi = want


@pytest.mark.parametrize("rebuild", [ls.LS_REBUILD_FULL, ls.LS_REBUILD_INCREMENTAL])
@pytest.mark.parametrize("cfg,n,steps", [(3, 96, 12), (4, 128, 12), (1, 40, 6)])
def test_step_free_running_multi(cfg, n, steps, rebuild):
    """Several steps inside one ls_step call and across two calls (scratch-buffer consistency)."""
    w = inputs.config(cfg, n=n)
    want, upd = orc.step(w.phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, steps)
    for chunks, chained in ((1, 0), (2, 0), (2, 1), (5, 1)):
        got, updates, nsteps, _ = _run_steps(w, steps, rebuild, chunks, chained)
        assert nsteps == steps and updates == upd
        assert max_err_dx(got, want, w.dx) <= TOL * steps
        assert np.array_equal(got, want)
        assert np.all(np.abs(got) <= np.float32(w.gamma))


def test_step_chained_falls_back_when_phi_differs():
    """chained = 1 with a different phi buffer (or after another band call) must run the unchained path."""
    w = inputs.config(1, n=40)
    want, _ = orc.step(w.phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 2)
    p = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, ls.LS_REBUILD_INCREMENTAL, 1)
    with Ctx(w.shape, w.dtype) as ctx:
        d_F = to_dev(w.F)
        a = to_dev(w.phi)
        ls.ls_step(ctx, a, d_F, p, 2)          # first call: nothing to chain to
        assert np.array_equal(a.cpu().numpy(), want)
        b = to_dev(w.phi)                      # another buffer: the promise cannot hold
        ls.ls_step(ctx, b, d_F, p, 2)
        assert np.array_equal(b.cpu().numpy(), want)
        ls.ls_build_band(ctx, b, w.dx, w.gamma)   # a band call in between invalidates the chain
        want4, _ = orc.step(want, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 2)
        ls.ls_step(ctx, b, d_F, p, 2)
        assert np.array_equal(b.cpu().numpy(), want4)


@pytest.mark.parametrize("fuse,reinit_launches", [(1, 15), (2, 9), (0, 15)])
def test_profile_counts_launches(fuse, reinit_launches):
    """Per-kernel event brackets: 3 steps of 5 sweeps are 15 launches with one sweep per launch and 9 with two
    (2 + 2 + 1, an odd number of launches so that the last one lands in phi)."""
    w = inputs.config(1, n=32)
    p = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, ls.LS_REBUILD_INCREMENTAL, 0, fuse)
    with Ctx(w.shape, w.dtype) as ctx:
        d_phi, d_F = to_dev(w.phi), to_dev(w.F)
        ls.ls_profile_enable(ctx, True)
        ls.ls_step(ctx, d_phi, d_F, p, 3)
        got = {name: ls.ls_profile_read(ctx, k) for k, name in enumerate(ls.KERNEL_KINDS)}
        ls.ls_profile_enable(ctx, False)
        assert got["reinit"][1] == reinit_launches and got["advance"][1] == 3 and got["band"][1] == 3
        assert got["classify"][1] == 1 and got["copy"][1] == 1 and got["clamp"][1] == 1
        assert all(ms > 0 for ms, n in got.values() if n)
        ls.ls_profile_reset(ctx)
        assert ls.ls_profile_read(ctx, ls.LS_K_REINIT) == (0.0, 0)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("shape", [(20, 13, 40), (33, 17, 64), (24, 40, 56), (64, 64, 64)])
def test_fused_sweeps_equal_single_sweeps(shape, dtype):
    """Temporal blocking (ls_params.fuse = 2: two eq. 12 iterations per staged tile) keeps Jacobi order
    exactly: free-running steps with fused sweeps equal the same steps with one launch per sweep AND the oracle, bit
    for bit, on ragged shapes whose band touches the domain boundary; iters = 5 (2 + 2 + 1) and 4 (2 + 1 + 1)."""
    dx = 1.0 / 32
    phi, F = _random_band_field(shape, dtype, 71, dx)
    F = (0.6 * F).astype(dtype)
    gamma, beta, dt, dtau = 4 * dx, 2 * dx, 0.4 * dx, 0.5 * dx
    for iters in (5, 4):
        want, _ = orc.step(phi, F, dx, dt, dtau, beta, gamma, iters, 3)
        got = {}
        for fuse in (1, 2):
            with Ctx(shape, dtype) as ctx:
                d_phi, d_F = to_dev(phi), to_dev(F)
                ls.ls_step(ctx, d_phi, d_F, ls.make_params(dx, dt, dtau, beta, gamma, iters, ls.LS_REBUILD_INCREMENTAL, 0, fuse), 3)
                got[fuse] = d_phi.cpu().numpy()
                launches = ls.ls_stats(ctx)[2]
            got[(fuse, "launches")] = launches
        assert got[(2, "launches")] < got[(1, "launches")]          # the fused path really ran
        assert np.array_equal(got[1], got[2])
        assert np.array_equal(got[2], want)


def test_step_ragged_fp64():
    """Non-multiple-of-8 dims (paper-shaped 101-style grid, scaled down), fp64, even and odd iters."""
    shape = (21, 37, 50)
    dx = 1.0 / 32
    phi, F = _random_band_field(shape, np.float64, 61, dx)
    F *= 0.5
    for iters in (2, 3):
        want, upd = orc.step(phi, F, dx, 0.4 * dx, 0.5 * dx, 2 * dx, 4 * dx, iters, 5)
        for rebuild in (ls.LS_REBUILD_FULL, ls.LS_REBUILD_INCREMENTAL):
            with Ctx(shape, np.float64) as ctx:
                d_phi, d_F = to_dev(phi), to_dev(F)
                ls.ls_step(ctx, d_phi, d_F, ls.make_params(dx, 0.4 * dx, 0.5 * dx, 2 * dx, 4 * dx, iters, rebuild), 5)
                got = d_phi.cpu().numpy()
                assert ls.ls_stats(ctx)[0] == upd
            assert max_err_dx(got, want, dx) <= 1e-12 * 5
            assert np.array_equal(got, want)


def test_step_host_matches_device():
    w = inputs.config(1, n=32)
    p = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters)
    want, _ = orc.step(w.phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 3)
    host_phi = w.phi.copy()
    with Ctx(w.shape, w.dtype) as ctx:
        with pytest.raises(ls.LsError):                     # no F on the device yet
            ls.ls_step_host(ctx, host_phi, None, p, 1)
        ls.ls_step_host(ctx, host_phi, w.F, p, 3)
        assert np.array_equal(host_phi, want)
        # F is static (R17): the following calls reuse the device copy
        want2, _ = orc.step(want, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 2)
        ls.ls_step_host(ctx, host_phi, None, p, 2)
        assert np.array_equal(host_phi, want2)


def _wide_band_field(shape, dtype, seed, dx):
    """As _random_band_field, by broadcasting (26 M cells): a front that crosses every z-slab cut, plus seeded noise."""
    nz, ny, nx = shape
    x = np.arange(nx, dtype=np.float64)[None, None, :]
    y = np.arange(ny, dtype=np.float64)[None, :, None]
    z = np.arange(nz, dtype=np.float64)[:, None, None]
    n = nx * ny * nz
    phi = dx * (4.0 * np.sin(0.37 * x + 0.2) + 3.0 * np.cos(0.29 * y) + 3.5 * np.sin(0.23 * z + 1.0)
                + 0.8 * (inputs.uniform01(seed, 0, n).reshape(shape) - 0.5))
    F = 2.0 * inputs.uniform01(seed + 1, 0, n).reshape(shape) - 1.0
    return np.ascontiguousarray(phi.astype(dtype)), np.ascontiguousarray(F.astype(dtype))


@pytest.mark.parametrize("shape,dtype,iters", [((100, 512, 512), np.float32, 5), ((100, 256, 512), np.float64, 4),
                                               ((100, 512, 512), np.float32, 0), ((70, 500, 601), np.float32, 3),
                                               ((90, 384, 512), np.float32, 1), ((90, 384, 512), np.float32, 2)])
def test_step_host_z_slab_pipeline(shape, dtype, iters):
    """ls_step_host on a field of >= 64 MiB, one step per call, runs as a pipeline of z-slabs (windows with iters + 1 halo
    layers on a child ctx; H2D / compute / D2H on three streams).  Bit-identical to the oracle on the whole grid and to the
    device-resident ls_step; the work counters count every grid point once; a second call (F reused) continues exactly.
    Shapes: five slabs of 24 layers with a ragged last one (iters 5, 4), seven of 16 (iters 0), a grid whose rows are
    not 16-byte multiples (scalar kernels), and 22-layer slabs with halos of 2 and 3 layers (iters 1, 2)."""
    dx = 1.0 / 32
    phi, F = _wide_band_field(shape, dtype, 77, dx)
    p = ls.make_params(dx, 0.4 * dx, 0.5 * dx, 3 * dx, 6 * dx, iters, ls.LS_REBUILD_INCREMENTAL)
    want1, upd1 = orc.step(phi, F, dx, 0.4 * dx, 0.5 * dx, 3 * dx, 6 * dx, iters, 1)
    want2, upd2 = orc.step(want1, F, dx, 0.4 * dx, 0.5 * dx, 3 * dx, 6 * dx, iters, 1)
    host = torch.from_numpy(phi.copy()).pin_memory()
    hF = torch.from_numpy(F).pin_memory()
    with Ctx(shape, dtype) as ctx:
        ls.ls_step_host(ctx, host.data_ptr(), hF.data_ptr(), p, 1)
        got1 = host.numpy().copy()
        assert np.array_equal(got1, want1), f"max err {max_err_dx(got1, want1, dx)} dx"
        assert ls.ls_stats(ctx)[:2] == (upd1, 1)
        ls.ls_step_host(ctx, host.data_ptr(), None, p, 1)       # F stays on the device
        assert np.array_equal(host.numpy(), want2)
        assert ls.ls_stats(ctx)[:2] == (upd1 + upd2, 2)
        # pageable host memory, and the unsliced multi-step call on the same ctx afterwards
        pageable = phi.copy()
        ls.ls_step_host(ctx, pageable, None, p, 1)
        assert np.array_equal(pageable, want1)
        ls.ls_step_host(ctx, pageable, None, p, 1)
        assert np.array_equal(pageable, want2)
        both = phi.copy()
        ls.ls_step_host(ctx, both, None, p, 2)                    # two steps in one call: not sliced
        assert np.array_equal(both, want2)
        ls.ls_band_counts(ctx)                                    # ... which leaves its band on the ctx
        if iters == 5:   # the windows honour the other step options too: paper-style full rebuild, two fused sweeps per launch
            p_alt = ls.make_params(dx, 0.4 * dx, 0.5 * dx, 3 * dx, 6 * dx, iters, ls.LS_REBUILD_FULL, 0, 2)
            pageable[...] = phi
            ls.ls_step_host(ctx, pageable, None, p_alt, 1)
            assert np.array_equal(pageable, want1)
        pageable[...] = phi
        ls.ls_step_host(ctx, pageable, None, p, 1)
        assert np.array_equal(pageable, want1)
        with pytest.raises(ls.LsError):                           # a sliced call leaves none (ls.h)
            ls.ls_band_counts(ctx)
    # and the device-resident path agrees (same library, other driver)
    with Ctx(shape, dtype) as ctx:
        d_phi, d_F = to_dev(phi), to_dev(F)
        ls.ls_step(ctx, d_phi, d_F, p, 1)
        assert np.array_equal(d_phi.cpu().numpy(), want1)


def test_step_host_pipeline_at_bench_size():
    """cfg 4 at its full 1024^3, the call bench.py's e2e leg times: ls_step_host (43 z-slabs in windows of 36 layers)
    against the device-resident ls_step on every point of the grid, both steps of two chained host calls, and the work
    counters; the device path itself is pinned to the oracle at this size by test_full_size_late_step_windowed."""
    w = inputs.config(4)
    p = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, ls.LS_REBUILD_INCREMENTAL, 0)
    host = torch.from_numpy(w.phi).clone().pin_memory()
    with Ctx(w.shape, w.dtype) as ctx:
        d_phi, d_F = to_dev(w.phi), to_dev(w.F)
        ls.ls_step(ctx, d_phi, d_F, p, 1)
        upd1 = ls.ls_stats(ctx)[0]
        ls.ls_stats_reset(ctx)
        ls.ls_step_host(ctx, host.data_ptr(), w.F, p, 1)
        assert ls.ls_stats(ctx)[:2] == (upd1, 1)
        assert torch.equal(host.cuda(), d_phi)
        ls.ls_step(ctx, d_phi, d_F, p, 1)
        ls.ls_step_host(ctx, host.data_ptr(), None, p, 1)
        assert torch.equal(host.cuda(), d_phi)


@pytest.mark.parametrize("n,dtype", [(32, np.float32), (64, np.float32), (64, np.float64), (48, np.float32)])
def test_library_kernel_choice_on_small_grids(n, dtype):
    """Ctx() in these tests forces the tiled band kernels so that the small shapes exercise them; the library's own
    choice (ls_tile_threshold default: scalar kernels below 4 M cells even on aligned rows) must give the same bits,
    step by step, in both rebuild modes, chained and not; switching the threshold between chained calls is allowed."""
    w = inputs.config(1, n=n)
    phi0, F0 = w.phi.astype(dtype), w.F.astype(dtype)
    want, upd = orc.step(phi0, F0, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 6)
    for rebuild in (ls.LS_REBUILD_INCREMENTAL, ls.LS_REBUILD_FULL):
        p0 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 0)
        p1 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 1)
        with Ctx(w.shape, dtype, tile_min_cells=None) as ctx:
            d_phi, d_F = to_dev(phi0), to_dev(F0)
            ls.ls_step(ctx, d_phi, d_F, p0, 2)
            ls.ls_step(ctx, d_phi, d_F, p1, 1)
            ls.ls_tile_threshold(ctx, 0)            # tiled from here on
            ls.ls_step(ctx, d_phi, d_F, p1, 1)
            ls.ls_tile_threshold(ctx, -1)           # and back to the default
            ls.ls_step(ctx, d_phi, d_F, p1, 2)
            assert np.array_equal(d_phi.cpu().numpy(), want)
            assert ls.ls_stats(ctx)[:2] == (upd, 6)


def test_dense_cfg2_steps():
    """cfg 2 at 64^3 and three steps at the full 256^3: ping-pong of full-domain advances."""
    for n, steps in ((64, 10), (256, 3)):
        w = inputs.config(2, n=n)
        a = w.phi
        for _ in range(steps):
            a = orc.advance(a, w.F, None, w.dt, w.dx, INF, INF)
        with Ctx(w.shape, w.dtype) as ctx:
            x, y, d_F = to_dev(w.phi), torch.empty_like(to_dev(w.phi)), to_dev(w.F)
            for _ in range(steps):
                ls.ls_advance(ctx, x, d_F, w.dt, w.dx, INF, INF, y)
                x, y = y, x
            got = x.cpu().numpy()
            assert ls.ls_stats(ctx)[0] == steps * n ** 3
        assert max_err_dx(got, a, w.dx) <= TOL * steps
        assert np.array_equal(got, a)


def test_cfg5_reinit_tol():
    """cfg 5 shape at 64^3 fp64: (i) trajectory parity over the first 300 iterations, (ii) the stopping
    rule (same iteration count and residual as the oracle for a loose tol), (iii) windowed parity
    from a GPU checkpoint, (iv) fixed-point certificate."""
    w = inputs.config(5, n=64)
    _, Nm = orc.band_masks(w.phi, w.gamma)
    with Ctx(w.shape, w.dtype) as ctx:
        d_phi = to_dev(w.phi)
        d = torch.empty_like(d_phi)
        ls.ls_build_band(ctx, d_phi, w.dx, w.gamma)
        assert_band_equal(ctx, w.phi, w.gamma)
        # (i)
        ls.ls_reinit(ctx, d, d_phi, w.dtau, w.dx, w.gamma, 300)
        want = orc.reinit(w.phi, Nm, w.dtau, w.dx, w.gamma, 300)
        got = d.cpu().numpy()
        assert max_err_dx(got, want, w.dx) <= 1e-12 * 300
        assert np.array_equal(got, want)
        # (ii)
        tol = 2e-4 * w.dx
        k, r, conv = ls.ls_reinit_tol(ctx, d, d_phi, w.dtau, w.dx, w.gamma, tol, 5000, 10)
        d_or, k_or, r_or, conv_or = orc.reinit_tol(w.phi, w.dtau, w.dx, w.gamma, tol, 5000, 10)
        assert conv and conv_or and k == k_or and r == r_or
        g_conv = d.cpu().numpy()
        assert np.array_equal(g_conv, d_or)
        # not converged path
        k2, r2, conv2 = ls.ls_reinit_tol(ctx, d, d_phi, w.dtau, w.dx, w.gamma, 1e-30, 37, 10)
        assert (k2, conv2) == (37, False)
        d37 = orc.reinit(w.phi, Nm, w.dtau, w.dx, w.gamma, 37)
        assert np.array_equal(d.cpu().numpy(), d37)
        # (iii) windowed: continue both sides for 50 iterations from the GPU state at k (unclamped
        # inside N; the clamp only touched points with |d| > gamma, so restart from the clamped field
        # on both sides with the ORIGINAL N)
        chk = d_or.copy()
        want50 = orc.reinit(chk, Nm, w.dtau, w.dx, w.gamma, 50)
        d2 = torch.empty_like(d_phi)
        ls.ls_reinit(ctx, d2, to_dev(chk), w.dtau, w.dx, w.gamma, 50)   # band in ctx is still N(phi0)
        assert np.array_equal(d2.cpu().numpy(), want50)
        # (iv) certificate: one oracle iteration on the GPU's converged state moves it by < tol
        # (checked away from the rim, where the final eq. 10 clamp has altered the iterate)
        nxt, _ = orc.reinit_iter(g_conv, Nm, w.dtau, w.dx)
        inner = (Nm != 0) & (np.abs(g_conv) < w.gamma - 2 * w.dx)
        assert np.max(np.abs(nxt - g_conv)[inner]) < tol


def test_selftest_packed_math_bit_identical():
    """ls_selftest_math: the packed two-point fp32 arithmetic of the TMA band kernels equals the scalar
    IEEE functions bit for bit on 3 x 2^24 random stencil pairs (band-like values, arbitrary bit
    patterns, zeros, flat patches), with a dyadic and a non-dyadic dx."""
    s = torch.cuda.current_stream().cuda_stream
    for seed, dx in ((1, 1.0 / 1024), (2, 1.0 / 512), (3, 0.0137)):
        bad = ls.ls_selftest_math(seed, 1 << 24, dx, 0.4 * dx, 3 * dx, 6 * dx, s)
        assert bad == 0, f"{bad} of {6 << 24} packed results differ (seed {seed}, dx {dx})"


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("shape", [(20, 13, 40), (9, 24, 8), (33, 17, 64)])
def test_tma_path_equals_oracle_exactly(shape, dtype):
    """TMA-addressable ragged grids (nx*sizeof(T) % 16 == 0; partial bricks in y and z; band touching
    the boundary): two free-running steps equal the oracle in every bit of every element (the contract
    is 1e-5*dx / 1e-12*dx; the implementation follows O2-O7's operation order exactly, so == holds)."""
    nz, ny, nx = shape
    dx = 1.0 / 32
    phi, F = _random_band_field(shape, dtype, 77, dx)
    want, upd = orc.step(phi, F, dx, 0.4 * dx, 0.5 * dx, 3 * dx, 6 * dx, 5, 2)
    for rebuild in (ls.LS_REBUILD_FULL, ls.LS_REBUILD_INCREMENTAL):
        with Ctx(shape, dtype) as ctx:
            d_phi, d_F = to_dev(phi), to_dev(F)
            ls.ls_step(ctx, d_phi, d_F, ls.make_params(dx, 0.4 * dx, 0.5 * dx, 3 * dx, 6 * dx, 5, rebuild), 2)
            got = d_phi.cpu().numpy()
            updates, _, _ = ls.ls_stats(ctx)
        assert updates == upd
        assert np.array_equal(got, want.astype(dtype)), f"max err {max_err_dx(got, want, dx)} dx"


# ---------------------------------------------------------------------------------------------
# Full BASELINE.json sizes, in the launch configuration bench.py times (one unchained step, then
# chained incremental steps).  The oracle cannot sweep 1024^3 in seconds, so it recomputes CROPS:
# a step reads at most 1 (Advance) + 5 (sweeps) + 2 (tube N around T) = 8 cells around a point, so
# after s steps a crop with a margin of 8 s cells reproduces the full-grid values in its interior
# exactly (where a crop face coincides with the domain boundary, edge replicate is the true rule and no
# margin is needed).  Interiors are brick aligned so band masks can be compared bit for bit too.
# ---------------------------------------------------------------------------------------------
def _crop_boxes(n, centres, size, margin):
    """-> list of (origin, interior lo, interior hi) per axis-tuple; origins multiples of 8, inside the grid."""
    boxes = []
    for c in centres:
        org = [int(np.clip((int(ci) - size // 2) // 8 * 8, 0, n - size)) for ci in c]   # (z, y, x)
        lo = [0 if o == 0 else margin for o in org]
        hi = [size if o + size == n else size - margin for o in org]
        boxes.append((org, lo, hi))
    return boxes


def _masks_from_export(ids, words, NB, org, lo, hi):
    """Point mask (bool) of the crop interior from a brick list export (ids ascending, words [n, 8])."""
    out = {}
    for b, w in zip(ids.tolist(), words):
        out[b] = w
    shape = tuple(h - l for l, h in zip(lo, hi))
    m = np.zeros(shape, bool)
    for bz in range((org[0] + lo[0]) // 8, (org[0] + hi[0]) // 8):
        for by in range((org[1] + lo[1]) // 8, (org[1] + hi[1]) // 8):
            for bx in range((org[2] + lo[2]) // 8, (org[2] + hi[2]) // 8):
                w = out.get((bz * NB + by) * NB + bx)
                if w is None:
                    continue
                bits = np.unpackbits(w.view(np.uint8), bitorder="little").reshape(8, 8, 8).astype(bool)
                z0, y0, x0 = bz * 8 - org[0] - lo[0], by * 8 - org[1] - lo[1], bx * 8 - org[2] - lo[2]
                m[z0:z0 + 8, y0:y0 + 8, x0:x0 + 8] = bits
    return m


@pytest.mark.parametrize("cfg", [4, 3])
def test_full_size_band_steps_sampled(cfg):
    w = inputs.config(cfg)
    n, steps, size = w.nx, 3, 112
    margin = 8 * steps
    if cfg == 4:   # torus R = 0.3, r = 0.1: outer / inner equator, top, and a diagonal point of the tube
        pts = [(0.5, 0.5, 0.9), (0.5, 0.7, 0.5), (0.6, 0.5, 0.8), (0.5 + 0.1 * 0.6, 0.5 + 0.38 * 0.6, 0.5 + 0.38 * 0.8)]
    else:          # cfg 3: +x pole of the first three seeded spheres, and the grid corner
        u = inputs.uniform01(3001, 0, 4 * 32).reshape(32, 4)
        pts = [(0.1 + 0.8 * u[s, 2], 0.1 + 0.8 * u[s, 1], 0.1 + 0.8 * u[s, 0] + 0.03 + 0.09 * u[s, 3]) for s in range(3)]
        pts.append((0.0, 0.0, 0.0))
    boxes = _crop_boxes(n, [[p * n for p in pt] for pt in pts], size, margin)
    p0 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, ls.LS_REBUILD_INCREMENTAL, 0)
    p1 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, ls.LS_REBUILD_INCREMENTAL, 1)
    with Ctx(w.shape, w.dtype) as ctx:
        d_phi, d_F = to_dev(w.phi), to_dev(w.F)
        # band of phi^0 at full size: |T| against torch's own count and (cfg 4) the closed form of I12
        ls.ls_build_band(ctx, d_phi, w.dx, w.gamma)
        nT0 = ls.ls_band_counts(ctx)[0]
        assert nT0 == int((d_phi.abs() < np.float32(w.gamma)).sum().item())
        if cfg == 4:
            assert abs(nT0 / n ** 3 - 4 * np.pi ** 2 * 0.3 * 0.1 * 12 * w.dx) < 0.01 * 0.0139
        ls.ls_step(ctx, d_phi, d_F, p0, 1)
        ls.ls_step(ctx, d_phi, d_F, p1, steps - 1)
        nT, nN, bT, bN = ls.ls_band_counts(ctx)      # band of the last step (built from phi^{steps-1})
        T_ids, T_w, N_ids, N_w = ls.ls_band_export(ctx)
        gamma32 = np.float32(w.gamma)
        assert float(d_phi.abs().max().item()) <= gamma32                       # eq. 10 everywhere (I4)
        got = d_phi.cpu().numpy()
    assert len(T_ids) == bT and len(N_ids) == bN and np.all(np.diff(N_ids) > 0) and np.all(np.diff(T_ids) > 0)
    assert int(np.unpackbits(T_w.view(np.uint8)).sum()) == nT and int(np.unpackbits(N_w.view(np.uint8)).sum()) == nN
    checked = 0
    for org, lo, hi in boxes:
        sl = tuple(slice(o, o + size) for o in org)
        inner = tuple(slice(l, h) for l, h in zip(lo, hi))
        phi_c, F_c = np.ascontiguousarray(w.phi[sl]), np.ascontiguousarray(w.F[sl])
        prev, _ = orc.step(phi_c, F_c, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, steps - 1)
        want, _ = orc.step(prev, F_c, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 1)
        g = got[sl][inner]
        assert np.array_equal(g, want[inner]), f"crop at {org}: max err {max_err_dx(g, want[inner], w.dx)} dx"
        Tm, Nm = orc.band_masks(prev, w.gamma)       # the band the last step used
        assert np.array_equal(_masks_from_export(T_ids, T_w, n // 8, org, lo, hi), Tm[inner] != 0)
        assert np.array_equal(_masks_from_export(N_ids, N_w, n // 8, org, lo, hi), Nm[inner] != 0)
        checked += int((Nm[inner] != 0).sum())
        # points off N hold exactly +-gamma after a step (I4)
        off = (Nm[inner] == 0)
        assert np.all(np.abs(g[off]) == gamma32)
    assert checked > 50000   # the crops really sit on the band


def test_full_size_cfg5_reinit_sampled():
    """cfg 5 at 512^3 fp64: 40 sweeps of ls_reinit on the band of phi^0, crops recomputed by the oracle
    (margin 40 + 2 cells), bit for bit; and the residual rule of ls_reinit_tol at full size."""
    w = inputs.config(5)
    n, iters, size = w.nx, 40, 128
    margin = 48
    pts = [(0.5, 0.25, 1 / 3), (0.5, 0.75, 2 / 3), (0.5, 0.0, 0.0)]   # nodes of the wave (z = 0.5); one at the domain edge
    boxes = _crop_boxes(n, [[p * n for p in pt] for pt in pts], size, margin)
    with Ctx(w.shape, w.dtype) as ctx:
        d_phi = to_dev(w.phi)
        d = torch.empty_like(d_phi)
        ls.ls_build_band(ctx, d_phi, w.dx, w.gamma)
        nT = ls.ls_band_counts(ctx)[0]
        assert nT == int((d_phi.abs() < w.gamma).sum().item())
        assert abs(nT / (16 * n * n) - 1.0) < 0.08          # 16 n^2 without the noise factor (I12), ~ +3 % with it
        ls.ls_reinit(ctx, d, d_phi, w.dtau, w.dx, w.gamma, iters)
        got = d.cpu().numpy()
        k, r, conv = ls.ls_reinit_tol(ctx, d, d_phi, w.dtau, w.dx, w.gamma, w.tol, 60, 20)
        assert (k, conv) == (60, False) and r > 100 * w.tol   # far from the 1e-10 steady state after 60 sweeps (R13)
    for org, lo, hi in boxes:
        sl = tuple(slice(o, o + size) for o in org)
        inner = tuple(slice(l, h) for l, h in zip(lo, hi))
        phi_c = np.ascontiguousarray(w.phi[sl])
        _, Nm = orc.band_masks(phi_c, w.gamma)
        want = orc.reinit(phi_c, Nm, w.dtau, w.dx, w.gamma, iters)
        assert np.array_equal(got[sl][inner], want[inner]), f"crop at {org}"
        assert (Nm[inner] != 0).sum() > 10000


@pytest.mark.parametrize("n", [101, 201])
def test_paper_shaped_grids(n):
    """the paper's own grid sizes, 101^3 and 201^3, 10 time steps
    (Tables 1-2).  Its front, F, gamma are not stated, so cfg 1's sphere set-up stands
    in.  Dimensions that are not multiples of 8 (partial bricks on every high face) nor of 4 (rows not
    16-byte aligned: the scalar band kernels run, not the TMA ones).  Free-running, both rebuild modes,
    band export and field compared bit for bit after the last step."""
    w = inputs.config(1, n=n)
    steps = 10 if n == 101 else 4      # the oracle sweeps the full 201^3 grid: keep the CPU side in seconds
    prev, _ = orc.step(w.phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, steps - 1)
    want, upd = orc.step(prev, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 1)
    upd_prev = orc.step(w.phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, steps - 1)[1]
    for rebuild in (ls.LS_REBUILD_FULL, ls.LS_REBUILD_INCREMENTAL):
        with Ctx(w.shape, w.dtype) as ctx:
            d_phi, d_F = to_dev(w.phi), to_dev(w.F)
            ls.ls_step(ctx, d_phi, d_F, ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild), steps)
            assert_band_equal(ctx, prev, w.gamma)      # the band of the last step
            assert ls.ls_stats(ctx)[0] == upd_prev + upd
            assert np.array_equal(d_phi.cpu().numpy(), want)


def test_step_snapshots_match_oracle_trajectory():
    """ls_step_snapshots (m-step batching, f-2): every 2nd of 7 steps returned to pinned host memory while
    the next steps compute; each snapshot equals the oracle's trajectory bit for bit, the final field equals
    the plain ls_step result, and a chained continuation still matches."""
    w = inputs.config(3, n=64)
    traj, cur = [], w.phi
    for s in range(9):
        cur, _ = orc.step(cur, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 1)
        traj.append(cur)
    for rebuild in (ls.LS_REBUILD_FULL, ls.LS_REBUILD_INCREMENTAL):
        host = torch.empty((3,) + w.shape, dtype=torch.float32).pin_memory()
        with Ctx(w.shape, w.dtype) as ctx:
            d_phi, d_F = to_dev(w.phi), to_dev(w.F)
            p = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild)
            assert ls.ls_step_snapshots(ctx, d_phi, d_F, p, 7, 2, host) == 3
            for k in range(3):
                assert np.array_equal(host[k].numpy(), traj[2 * k + 1]), f"snapshot {k}"
            assert np.array_equal(d_phi.cpu().numpy(), traj[6])
            p1 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 1)
            assert ls.ls_step_snapshots(ctx, d_phi, d_F, p1, 2, 5, host) == 0     # fewer steps than `every`
            assert np.array_equal(d_phi.cpu().numpy(), traj[8])
            assert ls.ls_stats(ctx)[1] == 9


# ---------------------------------------------------------------------------------------------
# Late steps at BASELINE.json's full sizes and lengths (windowed parity, SURVEY.md section 8(c) protocol 3-ii): the GPU runs
# N - 1 steps alone, the crops of phi^{N-1} are downloaded, one more step follows, and the oracle repeats that ONE step
# from the GPU's own phi^{N-1} crops.  The incremental rebuild's exactness argument (T^{n+1} inside N^n)
# is the kind of thing that breaks late (fronts merging in cfg 3, the band reaching the domain faces), not at step 3.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,total,rebuild", [(4, 200, ls.LS_REBUILD_INCREMENTAL), (4, 77, ls.LS_REBUILD_INCREMENTAL),
                                               (3, 100, ls.LS_REBUILD_INCREMENTAL),
                                               (3, 100, ls.LS_REBUILD_FULL)])
def test_full_size_late_step_windowed(cfg, total, rebuild):
    w = inputs.config(cfg)
    n, size, margin = w.nx, 112, 8
    p0 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 0)
    p1 = ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 1)
    with Ctx(w.shape, w.dtype) as ctx:
        d_phi, d_F = to_dev(w.phi), to_dev(w.F)
        ls.ls_step(ctx, d_phi, d_F, p0, 1)
        ls.ls_step(ctx, d_phi, d_F, p1, total - 2)           # phi^{N-1}
        _, _, N_ids, _ = ls.ls_band_export(ctx)              # band of step N-1: where the front is now
        NB = n // 8
        picks = [N_ids[int(q * (len(N_ids) - 1))] for q in (0.03, 0.27, 0.5, 0.74, 0.97)]
        bz, by, bx = np.unravel_index(N_ids, (NB, NB, NB))
        face = np.flatnonzero((np.minimum.reduce([bz, by, bx]) == 0) | (np.maximum.reduce([bz, by, bx]) == NB - 1))
        if len(face):                                        # a brick where the band touches a domain face (cfg 3)
            picks.append(N_ids[face[len(face) // 2]])
        centres = [[(c * 8 + 4) for c in np.unravel_index(int(b), (NB, NB, NB))] for b in picks]
        boxes = _crop_boxes(n, centres, size, margin)
        prev = [d_phi[tuple(slice(o, o + size) for o in org)].contiguous().cpu().numpy() for org, _, _ in boxes]
        upd0 = ls.ls_stats(ctx)[0]
        ls.ls_step(ctx, d_phi, d_F, p1, 1)                    # step N
        nT, nN, bT, bN = ls.ls_band_counts(ctx)
        assert ls.ls_stats(ctx)[0] - upd0 == nT + w.iters * nN
        T_ids, T_w, N_ids, N_w = ls.ls_band_export(ctx)
        got = [d_phi[tuple(slice(o, o + size) for o in org)].contiguous().cpu().numpy() for org, _, _ in boxes]
        gamma32 = np.float32(w.gamma)
        assert float(d_phi.abs().max().item()) <= gamma32
    checked = 0
    for (org, lo, hi), phi_c, g in zip(boxes, prev, got):
        sl = tuple(slice(o, o + size) for o in org)
        inner = tuple(slice(l, h) for l, h in zip(lo, hi))
        F_c = np.ascontiguousarray(w.F[sl])
        want, _ = orc.step(phi_c, F_c, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 1)
        assert np.array_equal(g[inner], want[inner]), f"crop at {org}: max err {max_err_dx(g[inner], want[inner], w.dx)} dx"
        Tm, Nm = orc.band_masks(phi_c, w.gamma)
        assert np.array_equal(_masks_from_export(T_ids, T_w, NB, org, lo, hi), Tm[inner] != 0)
        assert np.array_equal(_masks_from_export(N_ids, N_w, NB, org, lo, hi), Nm[inner] != 0)
        checked += int((Nm[inner] != 0).sum())
    assert checked > 50000


def test_cfg2_step_50_full_grid():
    """cfg 2 at its full size and length: 49 full-domain advances on the GPU alone, then the 50th compared with ONE
    oracle advance of the GPU's own phi^49, every point of the 256^3 grid, bit for bit."""
    w = inputs.config(2)
    with Ctx(w.shape, w.dtype) as ctx:
        a, d_F = to_dev(w.phi), to_dev(w.F)
        b = torch.empty_like(a)
        for _ in range(49):
            ls.ls_advance(ctx, a, d_F, w.dt, w.dx, INF, INF, b)
            a, b = b, a
        prev = a.cpu().numpy()
        ls.ls_advance(ctx, a, d_F, w.dt, w.dx, INF, INF, b)
        got = b.cpu().numpy()
    want = orc.advance(prev, w.F, None, w.dt, w.dx, INF, INF)
    assert np.array_equal(got, want)
    assert np.abs(prev - w.phi).max() > 10 * w.dx            # the front really moved (F >= 0.5, 49 x 0.4 dx)


@pytest.mark.parametrize("rebuild", [ls.LS_REBUILD_FULL, ls.LS_REBUILD_INCREMENTAL])
@pytest.mark.parametrize("cfg,n,steps", [(3, 128, 100), (4, 128, 200)])
def test_free_running_full_length(cfg, n, steps, rebuild):
    """BASELINE.json's step counts, free running, on grids the oracle can follow: |T| and |N| of every step and the
    final field must equal the oracle's (a single flipped band bit anywhere would show in the counts)."""
    w = inputs.config(cfg, n=n)
    want_counts = []
    phi = w.phi
    for _ in range(steps):
        Tm, Nm = orc.band_masks(phi, w.gamma)
        want_counts.append((int(Tm.sum()), int(Nm.sum())))
        phi, _ = orc.step(phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 1)
    got_counts = []
    with Ctx(w.shape, w.dtype) as ctx:
        d_phi, d_F = to_dev(w.phi), to_dev(w.F)
        for s in range(steps):
            ls.ls_step(ctx, d_phi, d_F, ls.make_params(w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, rebuild, 1 if s else 0), 1)
            got_counts.append(ls.ls_band_counts(ctx)[:2])
        got = d_phi.cpu().numpy()
    assert got_counts == want_counts
    assert np.array_equal(got, phi)
    assert want_counts[-1] != want_counts[0]


def test_cfg5_runs_to_its_stopping_rule():
    """cfg 5 as BASELINE.json states it: 512^3 fp64, reinit 'solved to steady state' (R13: max_N |d^k - d^{k-1}|
    < 1e-10).  The GPU iterates alone to the stopping rule; the oracle certifies the fixed point: ONE oracle iteration from
    crops of the converged state moves no well-inside band point by 1e-10 or more, and repeats the GPU's own next sweep bit
    for bit.  (About 2.5e5 sweeps, 20 s of GPU time.)  Writes iterations / residual / seconds to
    gpurun_out/cfg5_converged.json."""
    import json
    import os
    import time
    w = inputs.config(5)
    n, size = w.nx, 128
    with Ctx(w.shape, w.dtype) as ctx:
        d_phi = to_dev(w.phi)
        d = torch.empty_like(d_phi)
        ls.ls_build_band(ctx, d_phi, w.dx, w.gamma)
        nT, nN, _, _ = ls.ls_band_counts(ctx)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        k, r, conv = ls.ls_reinit_tol(ctx, d, d_phi, w.dtau, w.dx, w.gamma, w.tol, 6_000_000, 2000)
        torch.cuda.synchronize()
        secs = time.perf_counter() - t0
        os.makedirs("gpurun_out", exist_ok=True)
        with open("gpurun_out/cfg5_converged.json", "w") as f:
            json.dump({"workload": "cfg5 512^3 fp64", "tol": w.tol, "check_every": 2000, "iterations": k, "residual": r,
                       "converged": conv, "seconds": secs, "N_points": nN, "us_per_sweep": secs / max(k, 1) * 1e6}, f)
        assert conv and r < w.tol and k % 2000 == 0
        got = d.cpu().numpy()
        d2 = torch.empty_like(d)
        ls.ls_reinit(ctx, d2, d, w.dtau, w.dx, w.gamma, 1)      # the GPU's own next sweep from the converged state
        nxt = d2.cpu().numpy()
    boxes = _crop_boxes(n, [[0.5 * n, 0.25 * n, n / 3], [0.5 * n, 0.75 * n, 2 * n / 3], [0.5 * n, 0.0, 0.0]], size, 2)
    checked = 0
    for org, lo, hi in boxes:
        sl = tuple(slice(o, o + size) for o in org)
        inner = tuple(slice(l, h) for l, h in zip(lo, hi))
        _, Nm = orc.band_masks(np.ascontiguousarray(w.phi[sl]), w.gamma)       # the tube N of phi^0 (R25)
        c = np.ascontiguousarray(got[sl])
        one, _ = orc.reinit_iter(c, Nm, w.dtau, w.dx)
        # clamped rim values (eq. 10 ran at the end) feed their neighbours: certify two cells inside the clamp
        well = (Nm[inner] != 0) & (np.abs(c[inner]) < w.gamma - 2 * w.dx)
        assert np.abs(one[inner] - c[inner])[well].max() < w.tol
        assert np.array_equal(np.clip(one, -w.gamma, w.gamma)[inner][well], nxt[sl][inner][well])
        checked += int(well.sum())
    assert checked > 100000


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("shape", [(9, 13, 20), (17, 8, 33), (24, 40, 56)])
def test_no_write_outside_the_fields(shape, dtype):
    """compute-sanitizer is closed on the GPU pool, so out-of-bounds WRITES are looked for directly: phi, F and the
    output field sit inside larger buffers whose guard zones (4096 elements before and after, a NaN pattern) must come
    back untouched from every entry point, on the tile path and (nx % 4 != 0) on the scalar path, with bands that touch
    the domain faces.  (Out-of-bounds reads would show as parity failures elsewhere: every result is compared bit for bit.)"""
    G = 4096
    dx = 1.0 / 32
    phi, F = _random_band_field(shape, dtype, 91, dx)
    F = (0.6 * F).astype(dtype)
    n = phi.size
    tdt = torch.float32 if dtype == np.float32 else torch.float64

    def guarded(a):
        buf = torch.full((n + 2 * G,), float("nan"), dtype=tdt, device="cuda")
        view = buf[G:G + n].view(*shape)
        if a is not None:
            view.copy_(torch.from_numpy(a))
        return buf, view

    def intact(buf):
        return bool(torch.isnan(buf[:G]).all().item() and torch.isnan(buf[G + n:]).all().item())

    gamma, beta, dt, dtau = 4 * dx, 2 * dx, 0.4 * dx, 0.5 * dx
    bp, vp = guarded(phi)
    bF, vF = guarded(F)
    bo, vo = guarded(None)
    with Ctx(shape, dtype) as ctx:
        ls.ls_build_band(ctx, vp, dx, gamma)
        ls.ls_advance(ctx, vp, vF, dt, dx, beta, gamma, vo)
        ls.ls_reinit(ctx, vo, vp, dtau, dx, gamma, 3)
        ls.ls_reinit_tol(ctx, vo, vp, dtau, dx, gamma, 1e-3 * dx, 40, 5)
        for fuse in (1, 2):
            ls.ls_step(ctx, vp, vF, ls.make_params(dx, dt, dtau, beta, gamma, 5, ls.LS_REBUILD_INCREMENTAL, 0, fuse), 3)
        ls.ls_step(ctx, vp, vF, ls.make_params(dx, dt, dtau, beta, gamma, 4, ls.LS_REBUILD_FULL, 0), 2)
        ls.ls_advance(ctx, vp, vF, dt, dx, INF, INF, vo)
        torch.cuda.synchronize()
    assert intact(bp) and intact(bF) and intact(bo)
    assert bool(torch.isfinite(vp).all().item()) and bool(torch.isfinite(vo).all().item())


@pytest.mark.parametrize("iters", [5, 4])
@pytest.mark.parametrize("shape", [(24, 40, 56), (17, 8, 33)])
def test_advance_and_export_after_incremental_step(shape, iters):
    """ls.h: ls_advance and ls_band_export use 'the band last built', and the last step of ls_step counts as a build
    (the band of phi^{n-1}).  With LS_REBUILD_INCREMENTAL the launch that writes phi^n also emits the T masks of phi^n
    for the NEXT step; they go into the other half of a double buffer and must not be what ls_advance / ls_band_export
    see (round-1 advisor finding: they did).  Odd and even `iters` (last sweep / band copy emits), tile and scalar path."""
    dx = 1.0 / 32
    phi, F = _random_band_field(shape, np.float32, 55, dx)
    F = (0.6 * F).astype(np.float32)
    gamma, beta, dt, dtau = 4 * dx, 2 * dx, 0.4 * dx, 0.5 * dx
    phi1, _ = orc.step(phi, F, dx, dt, dtau, beta, gamma, iters, 1)
    phi2, _ = orc.step(phi1, F, dx, dt, dtau, beta, gamma, iters, 1)
    Tm1, _ = orc.band_masks(phi1, gamma)                      # the band the second step built
    want = orc.advance(phi2, F, Tm1, dt, dx, beta, gamma)     # eq. 8 on THAT T, applied to the current field
    with Ctx(shape, np.float32) as ctx:
        d_phi, d_F = to_dev(phi), to_dev(F)
        ls.ls_step(ctx, d_phi, d_F, ls.make_params(dx, dt, dtau, beta, gamma, iters, ls.LS_REBUILD_INCREMENTAL), 2)
        assert np.array_equal(d_phi.cpu().numpy(), phi2)
        assert_band_equal(ctx, phi1, gamma)
        out = torch.empty_like(d_phi)
        ls.ls_advance(ctx, d_phi, d_F, dt, dx, beta, gamma, out)
        got = out.cpu().numpy()
        assert_band_equal(ctx, phi1, gamma)                  # still the band last built
    assert np.array_equal(got, want)
    assert (Tm1 != orc.band_masks(phi2, gamma)[0]).any()      # the two bands do differ: the test can tell them apart


@pytest.mark.parametrize("seed", list(range(int(__import__("os").environ.get("LS_FUZZ", "12")))))
def test_random_shapes_and_parameters(seed):
    """Seeded random cases: shape (ragged; nx a multiple of 4 or not: tile or scalar path), dtype, gamma / beta / dt / dtau,
    iters (odd, even, 0), rebuild mode, sweeps per launch, chunking of the steps into chained calls — free running for a
    few steps, band export and field compared with the oracle bit for bit."""
    u = inputs.uniform01(7000 + seed, 0, 16)
    dtype = np.float32 if u[0] < 0.6 else np.float64
    nx = int(4 + u[1] * 70); nx = nx - nx % 4 if u[2] < 0.7 else nx | 1
    shape = (int(3 + u[3] * 40), int(3 + u[4] * 40), max(nx, 4))
    dx = 1.0 / 32
    gamma = (2.0 + 5.0 * u[5]) * dx
    beta = gamma * (0.3 + 0.5 * u[6])
    dt, dtau = (0.2 + 0.3 * u[7]) * dx, (0.2 + 0.3 * u[8]) * dx
    iters = int(u[9] * 7)
    rebuild = ls.LS_REBUILD_INCREMENTAL if u[10] < 0.6 else ls.LS_REBUILD_FULL
    fuse = 2 if u[11] < 0.4 else 1
    steps = 2 + int(u[12] * 4)
    first = 1 + int(u[13] * (steps - 1))
    phi, F = _random_band_field(shape, dtype, 7100 + seed, dx)
    F = (0.8 * F).astype(dtype)
    want, upd = orc.step(phi, F, dx, dt, dtau, beta, gamma, iters, steps)
    prev, _ = orc.step(phi, F, dx, dt, dtau, beta, gamma, iters, steps - 1)
    with Ctx(shape, dtype) as ctx:
        d_phi, d_F = to_dev(phi), to_dev(F)
        ls.ls_step(ctx, d_phi, d_F, ls.make_params(dx, dt, dtau, beta, gamma, iters, rebuild, 0, fuse), first)
        if steps > first:
            ls.ls_step(ctx, d_phi, d_F, ls.make_params(dx, dt, dtau, beta, gamma, iters, rebuild, 1, fuse), steps - first)
        got = d_phi.cpu().numpy()
        assert ls.ls_stats(ctx)[0] == upd
        assert_band_equal(ctx, prev, gamma)
    assert np.array_equal(got, want), (shape, dtype, iters, rebuild, fuse, max_err_dx(got, want, dx))
