"""Pins of the CPU oracle against what the paper and the mathematics fix (I1-I14).

None of these compares the oracle with itself re-typed: they use closed forms, exact special
cases, invariants, an exact-rational hand evaluation (tests/golden/) and numpy brute force on
small grids.  CPU only (-m "not gpu").
"""
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

from oracle import ls_oracle as orc
from paper_1612_04040_b200 import inputs

GOLDEN = Path(__file__).parent / "golden"
INF = float("inf")


def rnd(shape, seed, dtype):
    return (2 * inputs.uniform01(seed, 0, int(np.prod(shape))) - 1).reshape(shape).astype(dtype)


# ---------------------------------------------------------------- I2: eq. 7 closed forms
@pytest.mark.parametrize("dtype,ulp", [(np.float64, 2.3e-16), (np.float32, 1.2e-7)])
def test_cutoff_closed_forms(dtype, ulp):
    b, g = 3.0, 6.0
    assert orc.cutoff(b, b, g, dtype) == 1.0
    assert orc.cutoff(0.0, b, g, dtype) == 1.0
    assert orc.cutoff(-2.9, b, g, dtype) == 1.0
    assert orc.cutoff(g, b, g, dtype) == 0.0
    assert orc.cutoff(-g, b, g, dtype) == 0.0
    assert orc.cutoff(7.0, b, g, dtype) == 0.0
    assert abs(orc.cutoff(0.5 * (b + g), b, g, dtype) - 0.5) <= 2 * ulp
    assert abs(orc.cutoff(3.5, b, g, dtype) - 25.0 / 27.0) <= 2 * ulp      # (2.5^2 * 4)/27
    for a in np.linspace(b, g, 41):
        t = (a - b) / (g - b)
        want = 1 - 3 * t * t + 2 * t ** 3                                   # the same cubic, Hermite form
        assert abs(orc.cutoff(a, b, g, dtype) - want) <= 8 * ulp
        assert abs(orc.cutoff(-a, b, g, dtype) - want) <= 8 * ulp
    # full-domain mode: beta = gamma = +inf => c = 1
    assert orc.cutoff(1e30, INF, INF, dtype) == 1.0


# ---------------------------------------------------------------- I1, I3
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_zero_speed_leaves_phi_unchanged(dtype):
    phi = rnd((9, 10, 11), 11, dtype)
    F = np.zeros_like(phi)
    out = orc.advance(phi, F, None, 0.5, 1.0, 0.3, 0.6)
    assert np.array_equal(out, phi)
    Tm, Nm = orc.band_masks(phi, 0.6)
    assert np.array_equal(orc.advance(phi, F, Tm, 0.5, 1.0, 0.3, 0.6), phi)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_advance_outside_tube_is_identity(dtype):
    """c(phi) = 0 for |phi| >= gamma, so Advance on all points == Advance on T (I3)."""
    phi = rnd((12, 9, 13), 5, dtype)
    F = rnd(phi.shape, 6, dtype)
    g = 0.5
    Tm, _ = orc.band_masks(phi, g)
    a = orc.advance(phi, F, Tm, 0.1, 0.25, 0.2, g)
    b = orc.advance(phi, F, None, 0.1, 0.25, 0.2, g)
    assert np.array_equal(a, b)
    assert np.array_equal(a[Tm == 0], phi[Tm == 0])
    assert (a[Tm == 1] != phi[Tm == 1]).mean() > 0.9        # and it does move points inside T


# ---------------------------------------------------------------- I5 + brick layout (numpy brute force)
def np_dilate6(m):
    out = m.copy()
    out[1:] |= m[:-1]; out[:-1] |= m[1:]
    out[:, 1:] |= m[:, :-1]; out[:, :-1] |= m[:, 1:]
    out[:, :, 1:] |= m[:, :, :-1]; out[:, :, :-1] |= m[:, :, 1:]
    return out


def np_brick_list(mask):
    nz, ny, nx = mask.shape
    NBx, NBy, NBz = -(-nx // 8), -(-ny // 8), -(-nz // 8)
    pad = np.zeros((NBz * 8, NBy * 8, NBx * 8), np.uint8)
    pad[:nz, :ny, :nx] = mask
    v = pad.reshape(NBz, 8, NBy, 8, NBx, 8).transpose(0, 2, 4, 1, 3, 5)   # bz by bx lz ly lx
    bits = (v.reshape(NBz, NBy, NBx, 8, 64).astype(np.uint64) << np.arange(64, dtype=np.uint64)).sum(-1,
                                                                                                    dtype=np.uint64)
    flat = bits.reshape(-1, 8)
    ids = np.nonzero(flat.any(1))[0].astype(np.int32)
    return ids, flat[ids]


@pytest.mark.parametrize("shape", [(16, 16, 16), (13, 9, 21), (4, 4, 4), (8, 24, 40)])
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_band_masks_and_brick_lists(shape, dtype):
    phi = rnd(shape, 21, dtype) * 2
    g = 0.37
    Tm, Nm = orc.band_masks(phi, g)
    assert np.array_equal(Tm, (np.abs(phi) < dtype(g)).astype(np.uint8))        # eq. 6, strict
    assert np.array_equal(Nm, np_dilate6(Tm))                                   # eq. 11 (R6)
    assert np.all(Nm >= Tm)                                                     # T subset N
    assert np.all(np.abs(phi[(Nm == 1) & (Tm == 0)]) >= dtype(g))
    for m in (Tm, Nm):
        ids, words, npts = orc.brick_list(m)
        rid, rwords = np_brick_list(m)
        assert np.array_equal(ids, rid) and np.array_equal(words, rwords)
        assert npts == int(m.sum())
        assert np.all(np.diff(ids) > 0)


def test_band_threshold_is_strict_and_in_field_precision():
    g = 0.1                                # not representable: float32(0.1) > 0.1 > nextbelow
    g32 = np.float32(g)
    phi = np.array([g32, np.nextafter(g32, np.float32(0)), -g32, 0.0], np.float32).reshape(1, 1, 4)
    Tm, _ = orc.band_masks(phi, g)
    assert Tm.ravel().tolist() == [0, 1, 0, 1]


# ---------------------------------------------------------------- I13: the 4^3 worked example
def load_golden():
    txt = (GOLDEN / "worked_4x4x4.txt").read_text().splitlines()
    g = {"point": [], "reinit": [], "all": []}
    for ln in txt:
        t = ln.split()
        if not t or t[0] == "#":
            continue
        if t[0] == "count":
            g["n" + t[1]] = int(t[2])
        elif t[0] == "words":
            g["w" + t[1]] = [int(x, 16) for x in t[2:]]
        elif t[0] == "point":
            g["point"].append((tuple(map(int, t[1:4])), t[7], t[9], t[11], float(t[15])))
        elif t[0] == "reinit":
            g["reinit"].append((tuple(map(int, t[1:4])), float(t[5])))
        elif t[0] == "sum":
            g["sum_" + t[1]] = float(t[2])
        elif t[0] == "all":
            g["all"].append((tuple(map(int, t[1:4])), float(t[4]), float(t[5])))
    return g


def worked_inputs(dtype):
    k, j, i = np.meshgrid(np.arange(4.0), np.arange(4.0), np.arange(4.0), indexing="ij")
    phi = (1.5 * i - 0.5 * j * j + 0.25 * j * k + k - 2.25).astype(dtype)
    F = np.where((i + j + k) % 2 == 0, 1.0, -0.5).astype(dtype)
    return phi, F


def test_golden_file_matches_its_derivation_script():
    out = subprocess.run([sys.executable, str(GOLDEN / "derive_worked_4x4x4.py")], capture_output=True,
                         text=True, check=True).stdout
    assert out == (GOLDEN / "worked_4x4x4.txt").read_text()


@pytest.mark.parametrize("dtype,tol", [(np.float64, 4.5e-16), (np.float32, 2.4e-7)])
def test_worked_example_4x4x4(dtype, tol):
    from fractions import Fraction
    g = load_golden()
    phi, F = worked_inputs(dtype)
    dx, gamma, beta, dt, dtau = 1.0, 3.0, 1.5, 0.5, 0.5
    Tm, Nm = orc.band_masks(phi, gamma)
    assert int(Tm.sum()) == g["nT"] == 45 and int(Nm.sum()) == g["nN"] == 60
    for m, w in ((Tm, g["wT"]), (Nm, g["wN"])):
        ids, words, _ = orc.brick_list(m)
        assert ids.tolist() == [0]
        assert words[0, :4].tolist() == w and words[0, 4:].tolist() == [0, 0, 0, 0]
    bar = orc.advance(phi, F, Tm, dt, dx, beta, gamma)
    for (i, j, k), qp, qm, c, want in g["point"]:
        got_qp, got_qm = orc.upwind_q(phi, i, j, k, dx)
        assert got_qp == float(Fraction(qp)) and got_qm == float(Fraction(qm))      # dyadic => exact
        assert abs(orc.cutoff(float(phi[k, j, i]), beta, gamma, dtype) - float(Fraction(c))) <= tol
        assert abs(bar[k, j, i] - want) <= tol * max(1.0, abs(want))
        assert abs(orc.advance_point(phi, F, i, j, k, dt, dx, beta, gamma) - want) <= tol * max(1.0, abs(want))
    d1, _ = orc.reinit_iter(bar, Nm, dtau, dx)
    for (i, j, k), want in g["reinit"]:
        assert abs(d1[k, j, i] - want) <= 4 * tol * max(1.0, abs(want))
    for (i, j, k), wb, wd in g["all"]:
        assert abs(bar[k, j, i] - wb) <= 2 * tol * max(1.0, abs(wb))
        assert abs(d1[k, j, i] - wd) <= 8 * tol * max(1.0, abs(wd))
    assert abs(float(bar.astype(np.float64).sum()) - g["sum_bar"]) <= 64 * tol * 8
    assert abs(float(d1.astype(np.float64).sum()) - g["sum_d1"]) <= 64 * tol * 16


# ---------------------------------------------------------------- I6: planar fronts
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("Fc", [1.0, -0.75])
def test_axis_aligned_plane_moves_exactly(dtype, axis, Fc):
    """phi = s - s0 on a power-of-two grid, constant F, full-domain mode: exact F*dt per step
    away from the edge-replicate boundary (one polluted layer per step)."""
    n, steps = 16, 4
    dx = 1.0 / n
    dt = 0.5 * dx
    s = (np.arange(n) + 0.5) * dx
    shp = [1, 1, 1]; shp[axis] = n
    phi0 = np.broadcast_to((s - 0.40625).reshape(shp), (n, n, n)).astype(dtype).copy()
    F = np.full_like(phi0, Fc)
    phi = phi0
    for _ in range(steps):
        phi = orc.advance(phi, F, None, dt, dx, INF, INF)
    want = phi0 - dtype(Fc * dt * steps)               # |grad phi| = 1 exactly
    sl = [slice(None)] * 3
    sl[axis] = slice(steps + 1, n - steps - 1)
    assert np.array_equal(phi[tuple(sl)], want[tuple(sl)])
    lo = [slice(None)] * 3; lo[axis] = slice(0, 1)
    if Fc > 0:                                           # and the polluted boundary layer is really different
        assert not np.array_equal(phi[tuple(lo)], want[tuple(lo)])


@pytest.mark.parametrize("dtype,tol", [(np.float32, 2.4e-6), (np.float64, 3.6e-15)])
@pytest.mark.parametrize("Fc", [1.0, -1.0])
def test_oblique_plane(dtype, tol, Fc):
    """phi = a.x - b with a = (3,4,12)/13 (|a| = 1): every one-sided difference is exact up to
    rounding, so phi moves F*dt per step; checked away from the boundary, in units of dx."""
    n, steps = 32, 5
    dx = 1.0 / n
    dt = 0.5 * dx
    x = (np.arange(n) + 0.5) * dx
    a = np.array([3.0, 4.0, 12.0]) / 13.0
    phi0 = (a[0] * x[None, None, :] + a[1] * x[None, :, None] + a[2] * x[:, None, None] - 0.7)
    F = np.full((n, n, n), Fc, dtype)
    phi = phi0.astype(dtype)
    for _ in range(steps):
        phi = orc.advance(phi, F, None, dt, dx, INF, INF)
    inner = (slice(steps + 1, n - steps - 1),) * 3
    err = np.abs(phi[inner].astype(np.float64) - (phi0[inner] - Fc * dt * steps)).max()
    assert err <= tol * dx * steps


@pytest.mark.parametrize("mixed_sign", [False, True])
def test_upwind_selects_the_right_side(mixed_sign):
    """A kink phi = |x - x0| has D-x != D+x at the kink: eq. 4 must take max(D-,0), min(D+,0)."""
    n = 8
    x = np.arange(n, dtype=np.float64)
    phi = np.broadcast_to(np.abs(x - 3.0)[None, None, :], (n, n, n)).copy()
    if mixed_sign:
        phi = -phi
    qp, qm = orc.upwind_q(phi, 3, 4, 4, 1.0)
    # at the kink D-x = -1, D+x = +1 (or the reverse for -phi)
    assert (qp, qm) == ((2.0, 0.0) if mixed_sign else (0.0, 2.0))
    qp, qm = orc.upwind_q(phi, 5, 4, 4, 1.0)            # smooth side: both one-sided slopes equal
    assert (qp, qm) == (1.0, 1.0)


# ---------------------------------------------------------------- I8: expanding sphere (cfg 1)
@pytest.mark.parametrize("n", [32, 64])
def test_expanding_sphere_tracks_r0_plus_Ft(n):
    w = inputs.config(1, n=n)
    steps = n * 10 // 64                                  # same physical time t = 5/64
    phi, upd = orc.step(w.phi, w.F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, steps)
    t = steps * w.dt
    x = (np.arange(n) + 0.5) * w.dx
    r = np.sqrt((x[:, None, None] - 0.5) ** 2 + (x[None, :, None] - 0.5) ** 2 + (x[None, None, :] - 0.5) ** 2)
    near = np.abs(phi) < 0.75 * w.dx
    r_est = r[near] - phi[near]                           # phi ~ signed distance near the front
    err = (r_est - (0.3 + t)) / w.dx
    assert near.sum() > 100
    assert abs(err.mean()) < 0.5 and np.abs(err).max() < 0.6
    exact = r - (0.3 + t)
    inner = np.abs(exact) <= w.beta
    assert np.abs(phi[inner] - exact[inner]).max() < 0.5 * w.dx
    assert upd > 0


# ---------------------------------------------------------------- I9: reinit drives |grad d| to 1
def test_reinit_restores_unit_gradient():
    n = 48
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    X, Y, Z = x[None, None, :], x[None, :, None], x[:, None, None]
    sdf = np.sqrt((X - 0.5) ** 2 + (Y - 0.5) ** 2 + (Z - 0.5) ** 2) - 0.3
    d0 = sdf * (1.0 + 0.4 * np.sin(7 * X) * np.cos(5 * Y + 1) * np.sin(6 * Z + 2))   # same zero set, wrong slope
    gamma = 6 * dx
    _, Nm = orc.band_masks(d0, gamma)

    def grad_err(d):
        gz, gy, gx = np.gradient(d, dx)
        g = np.sqrt(gx ** 2 + gy ** 2 + gz ** 2)
        return np.abs(g - 1)[np.abs(sdf) <= 2 * dx].max()

    errs = [grad_err(d0)]
    d = d0
    for it in range(30):
        d, _ = orc.reinit_iter(d, Nm, 0.5 * dx, dx)
        if it + 1 in (5, 10, 20, 30):
            errs.append(grad_err(d))
    assert errs[0] > 0.3
    assert errs[0] > errs[1] > errs[2], errs              # monotone over the first 10 iterations
    assert max(errs[2:]) < 0.07, errs                      # then the first-order floor (curvature * dx)
    core = np.abs(sdf) <= 2 * dx
    assert np.abs(d - sdf)[core].max() < 0.25 * dx         # the zero level set stays put (first order)
    assert np.array_equal(np.sign(d), np.sign(sdf))        # and no point changes side


# ---------------------------------------------------------------- I11: d == 0 never moves
def test_zero_points_are_fixed_in_reinit():
    d = rnd((10, 10, 10), 77, np.float64)
    d[3, 4, 5] = 0.0; d[0, 0, 0] = 0.0; d[9, 9, 2] = 0.0
    Nm = np.ones(d.shape, np.uint8)
    out, _ = orc.reinit_iter(d, Nm, 0.3, 1.0)
    assert out[3, 4, 5] == 0.0 and out[0, 0, 0] == 0.0 and out[9, 9, 2] == 0.0
    flat = np.zeros((5, 5, 5))                               # 0/0 case (R12)
    out, r = orc.reinit_iter(flat, np.ones(flat.shape, np.uint8), 0.3, 1.0)
    assert np.array_equal(out, flat) and r == 0.0


def test_reinit_sign_and_direction_1d():
    """d = 2x (slope 2, d>0): |grad| = 2 > 1 so d must decrease; for d = -2x-like it must increase.
    S = d/sqrt(d^2 + 4): closed form of eq. 12-13 on a linear profile."""
    n = 9
    x = np.arange(n, dtype=np.float64) - 4
    d = np.broadcast_to((2 * x)[None, None, :], (n, n, n)).copy()
    out, _ = orc.reinit_iter(d, np.ones(d.shape, np.uint8), 0.25, 1.0)
    for i in (5, 6, 7):
        c = d[4, 4, i]
        want = c - 0.25 * (c / np.sqrt(c * c + 4.0)) * (2.0 - 1.0)
        assert abs(out[4, 4, i] - want) < 1e-15
    for i in (1, 2, 3):
        c = d[4, 4, i]
        want = c - 0.25 * (c / np.sqrt(c * c + 4.0)) * (2.0 - 1.0)
        assert abs(out[4, 4, i] - want) < 1e-15 and out[4, 4, i] > c


# ---------------------------------------------------------------- I4: clamp invariants, T^{n+1} in N^n
def test_step_invariants_two_signed_speed():
    n = 32
    w = inputs.config(1, n=n)
    x = (np.arange(n) + 0.5) * w.dx
    F = (np.sin(2 * np.pi * x)[None, None, :] * np.cos(2 * np.pi * x)[None, :, None]
         * np.ones(n)[:, None, None]).astype(np.float32)
    phi = w.phi
    g32 = np.float32(w.gamma)
    for s in range(6):
        Tm, Nm = orc.band_masks(phi, w.gamma)
        new, _ = orc.step(phi, F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 1)
        assert np.abs(new).max() <= g32                                  # eq. 10
        assert np.all(np.abs(new[Nm == 0]) == g32)                       # outside N exactly +-gamma
        assert np.array_equal(orc.clamp(new.copy(), w.gamma), new)       # idempotent
        T1, _ = orc.band_masks(new, w.gamma)
        assert np.all(Nm[T1 == 1] == 1)                                  # T^{n+1} subset N^n
        assert np.array_equal(np.sign(new[Nm == 0]), np.sign(phi[Nm == 0]))
        phi = new


# ---------------------------------------------------------------- I10: reflection symmetry, bit exact
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_reflection_symmetry_is_bit_exact(axis):
    n = 24
    w = inputs.config(1, n=n)
    x = (np.arange(n) + 0.5) * w.dx
    s = np.cos(2 * np.pi * x)                                             # symmetric about 0.5
    F = (s[None, None, :] * s[None, :, None] * s[:, None, None]).astype(np.float32)
    F = ((F + np.flip(F, axis)) * np.float32(0.5)).astype(np.float32)
    phi = ((w.phi + np.flip(w.phi, axis)) * np.float32(0.5)).astype(np.float32)
    out, _ = orc.step(phi, F, w.dx, w.dt, w.dtau, w.beta, w.gamma, w.iters, 5)
    assert np.array_equal(out, np.flip(out, axis))
    assert not np.array_equal(out, phi)


# ---------------------------------------------------------------- I12: band sizes with closed forms
def test_band_counts_match_closed_forms():
    w = inputs.config(1)
    Tm, Nm = orc.band_masks(w.phi, w.gamma)
    shell = 4.0 / 3.0 * np.pi * ((19.2 + 6) ** 3 - (19.2 - 6) ** 3)      # in cells
    assert abs(Tm.sum() - shell) / shell < 0.01
    assert Tm.sum() == 57584 and Nm.sum() == 66136                       # survey probe values
    # cfg 5 without the noise factor: 16 resp. 18 layers of 512^2 -> scaled to n = 64
    n = 64
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    wave = 0.05 * np.sin(6 * np.pi * x)[None, None, :] * np.sin(6 * np.pi * x)[None, :, None]
    phi = (x[:, None, None] - 0.5) - wave
    Tm, Nm = orc.band_masks(phi, 8 * dx)
    assert Tm.sum() == 16 * n * n
    assert Nm.sum() == 18 * n * n


def test_cfg4_band_fraction_closed_form():
    """|T0| ~ 4 pi^2 R r * 12 dx * n^3 for the torus (scaled-down n)."""
    n = 128
    phi = inputs.torus_sdf(n)
    Tm, _ = orc.band_masks(phi, 6.0 / n)
    want = 4 * np.pi ** 2 * 0.3 * 0.1 * (12.0 / n) * n ** 3
    assert abs(Tm.sum() - want) / want < 0.01


# ---------------------------------------------------------------- I14: list-driven == full-grid
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_list_driven_equals_full_grid(dtype):
    n = 28                                                               # ragged bricks (28 = 3*8 + 4)
    dx = 1.0 / n
    phi = inputs.sphere_sdf(n, 0.31, centre=(0.45, 0.55, 0.5), dtype=dtype)
    F = rnd((n, n, n), 9, dtype)
    a, ua = orc.step(phi, F, dx, 0.4 * dx, 0.5 * dx, 3 * dx, 6 * dx, 5, 4, use_lists=False)
    b, ub = orc.step(phi, F, dx, 0.4 * dx, 0.5 * dx, 3 * dx, 6 * dx, 5, 4, use_lists=True)
    assert np.array_equal(a, b) and ua == ub
    # and the standalone list calls against the masked calls
    Tm, Nm = orc.band_masks(phi, 6 * dx)
    ids, words, _ = orc.brick_list(Tm)
    ref = orc.advance(phi, F, Tm, 0.4 * dx, dx, 3 * dx, 6 * dx)
    got = orc.advance_list(phi, F, ids, words, 0.4 * dx, dx, 3 * dx, 6 * dx, phi.copy())
    assert np.array_equal(ref, got)
    ids, words, _ = orc.brick_list(Nm)
    ref2, _ = orc.reinit_iter(ref, Nm, 0.5 * dx, dx)
    got2 = orc.reinit_iter_list(ref, ids, words, 0.5 * dx, dx, ref.copy())
    assert np.array_equal(ref2, got2)


def test_point_functions_equal_grid_functions():
    phi = rnd((7, 8, 9), 3, np.float32)
    F = rnd((7, 8, 9), 4, np.float32)
    full = orc.advance(phi, F, None, 0.2, 0.5, 0.3, 0.6)
    re, _ = orc.reinit_iter(phi, np.ones(phi.shape, np.uint8), 0.2, 0.5)
    for (k, j, i) in [(0, 0, 0), (6, 7, 8), (3, 0, 8), (2, 5, 1)]:
        assert np.float32(orc.advance_point(phi, F, i, j, k, 0.2, 0.5, 0.3, 0.6)) == full[k, j, i]
        assert np.float32(orc.reinit_point(phi, i, j, k, 0.2, 0.5)) == re[k, j, i]


def test_reinit_tol_stops_on_the_residual_rule():
    n = 20
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    phi = np.broadcast_to(((x - 0.5) * 1.3)[:, None, None], (n, n, n)).copy()
    d, k, r, conv = orc.reinit_tol(phi, 0.3 * dx, dx, 8 * dx, 1e-9, 5000, check_every=10)
    assert conv and k % 10 == 0 and r < 1e-9
    mid = (slice(6, 14), slice(2, -2), slice(2, -2))
    gz = np.gradient(d, dx, axis=0)[mid]
    assert np.abs(np.abs(gz) - 1).max() < 1e-6               # a tilted plane relaxes to slope 1
    d2, k2, r2, conv2 = orc.reinit_tol(phi, 0.3 * dx, dx, 8 * dx, 1e-30, 7, check_every=1)
    assert not conv2 and k2 == 7


# ---------------------------------------------------------------- outputs the pins above do not reach
def _perturbed_sphere(n, dtype, amp=0.35):
    dx = 1.0 / n
    x = (np.arange(n) + 0.5) * dx
    X, Y, Z = x[None, None, :], x[None, :, None], x[:, None, None]
    sdf = np.sqrt((X - 0.5) ** 2 + (Y - 0.5) ** 2 + (Z - 0.5) ** 2) - 0.3
    return (sdf * (1.0 + amp * np.sin(9 * X + 1) * np.cos(7 * Y) * np.sin(8 * Z + 2))).astype(dtype), dx


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_reinit_iter_residual_is_max_abs_change_over_N(dtype):
    """Stopping rule of eq. 12 (R13): r = max_{x in N} |d^{k+1} - d^k|, an ABSOLUTE value taken
    over N only.  Two fields: one whose largest change is a DECREASE (slope 2, d > 0: eq. 12 lowers d), so a
    signed maximum would come out smaller or negative; one where a big change lies outside N and must not count."""
    n = 9
    x = np.arange(n, dtype=np.float64) - 4
    d = np.broadcast_to((3 * x + 13)[None, None, :], (n, n, n)).astype(dtype).copy()   # d > 0 everywhere, |grad| = 3
    Nm = np.ones(d.shape, np.uint8)
    out, r = orc.reinit_iter(d, Nm, 0.25, 1.0)
    diff = out.astype(np.float64) - d.astype(np.float64)
    # interior points move DOWN by ~0.5 (|grad| = 3 > 1); only the x = 0 face (edge replicate: upwind |grad| = 0)
    # moves up, by < 0.25: a signed maximum would report that face instead
    assert diff.min() < -0.45 and 0.0 < diff.max() < 0.26
    assert r == np.abs(diff).max() and r > 0.45
    # restricted to N: the steep half is outside N
    d2 = d.copy()
    d2[:, :, :4] = d2[:, :, 3:4] + (x[:4] - x[3])[None, None, :].astype(dtype)   # |grad| = 1 for x <= 3: nearly still
    Nm2 = np.zeros(d.shape, np.uint8)
    Nm2[:, :, :3] = 1
    out2, r2 = orc.reinit_iter(d2, Nm2, 0.25, 1.0)
    diff2 = np.abs(out2.astype(np.float64) - d2.astype(np.float64))
    assert np.array_equal(out2[Nm2 == 0], d2[Nm2 == 0])
    assert r2 == diff2[Nm2 == 1].max()
    full2, rfull = orc.reinit_iter(d2, Nm, 0.25, 1.0)
    assert rfull > r2                                          # the steep part would have dominated


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_reinit_tol_iterates_on_N_and_clamps_everywhere(dtype):
    """Step 3 runs "on the tube N" (eq. 11), not on T, and eq. 10 (R14) is
    applied at every point afterwards.  Built from the single-iteration function (pinned above) and numpy:
    k x reinit_iter on the N mask of numpy's own dilation, then numpy's clip."""
    n = 24
    phi, dx = _perturbed_sphere(n, dtype)
    gamma = 4 * dx
    phi[2, 3, 4] = dtype(11 * dx)                               # far outside N and beyond +-gamma: only eq. 10 moves them
    phi[20, 20, 3] = dtype(-9 * dx)
    Tm = (np.abs(phi) < dtype(gamma))
    Nm = np_dilate6(Tm).astype(np.uint8)
    k = 7
    d = phi.copy()
    for _ in range(k):
        d, r_last = orc.reinit_iter(d, Nm, 0.3 * dx, dx)
    moved_rim = (d != phi) & (Nm == 1) & ~Tm
    assert moved_rim.sum() > 50                                 # points of N \ T do move: T-only iteration differs
    on_T = phi.copy()
    for _ in range(k):
        on_T, _ = orc.reinit_iter(on_T, Tm.astype(np.uint8), 0.3 * dx, dx)
    want = np.clip(d, dtype(-gamma), dtype(gamma))
    assert not np.array_equal(np.clip(on_T, dtype(-gamma), dtype(gamma)), want)
    assert np.abs(d).max() > dtype(gamma)                       # and the clamp has something to do
    got, kk, r, conv = orc.reinit_tol(phi, 0.3 * dx, dx, gamma, 1e-30, k, check_every=1)
    assert kk == k and not conv and r == r_last
    assert np.array_equal(got, want)
    assert got[2, 3, 4] == dtype(gamma) and got[20, 20, 3] == dtype(-gamma)
    # a check that is not yet due must not stop the iteration: tol is met from the start, check_every = 5
    flat_ok, k5, _, conv5 = orc.reinit_tol(phi, 0.3 * dx, dx, gamma, 1e30, 12, check_every=5)
    assert conv5 and k5 == 5


@pytest.mark.parametrize("use_lists", [False, True])
def test_step_update_count_is_T_plus_iters_times_N(use_lists):
    """The metric's numerator: sum over steps of |T_s| + iters * |N_s|, with T_s, N_s the
    tubes of phi^s (Step 1) — recomputed here with numpy along the oracle's own trajectory."""
    n = 24
    w = inputs.config(1, n=n)
    F = rnd((n, n, n), 21, np.float32)
    iters = 3
    phi = w.phi
    total = 0
    for s in range(4):
        Tm = np.abs(phi) < np.float32(w.gamma)
        Nm = np_dilate6(Tm)
        assert Nm.sum() > Tm.sum() > 0
        total += int(Tm.sum()) + iters * int(Nm.sum())
        phi, u1 = orc.step(phi, F, w.dx, w.dt, w.dtau, w.beta, w.gamma, iters, 1, use_lists=use_lists)
        assert u1 == int(Tm.sum()) + iters * int(Nm.sum())
    _, u4 = orc.step(w.phi, F, w.dx, w.dt, w.dtau, w.beta, w.gamma, iters, 4, use_lists=use_lists)
    assert u4 == total
