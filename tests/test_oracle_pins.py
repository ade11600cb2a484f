"""Pins for the CPU oracle (oracle/mphv_oracle.c): it is checked here against what the
paper and the mathematics fix, not against itself. CPU only.

Pin names P1..P9 follow SURVEY.md sec. 8(c) / DESIGN.md "Oracle pins".
"""
from fractions import Fraction as Fr
from math import erf, pi, sqrt
from pathlib import Path

import numpy as np
import pytest

GOLDEN = Path(__file__).parent / "golden"
PER, OUT, WALL = 0, 1, 2


# ----------------------------------------------------------------------------------------
# Independent formulation used by P2/P3: the PFC piecewise-quadratic reconstruction of the
# cited method, with the positivity correctors in their published *division* form, integrated
# in exact rationals over the region swept through each face ("remap form"). Nothing of the
# oracle's division-free min/max flux formula (c1, c2 polynomials, index shift by k) is used.
# ----------------------------------------------------------------------------------------
def _poly_int(coeffs, a, b):
    """Exact integral over [a, b] of sum_k coeffs[k] xi^k."""
    return sum(c * (b ** (k + 1) - a ** (k + 1)) / (k + 1) for k, c in enumerate(coeffs))


def _value(f, idx, bc):
    n = len(f)
    if 0 <= idx < n:
        return f[idx]
    if bc == PER:
        return f[idx % n]
    if bc == OUT:
        return f[0] if idx < 0 else f[n - 1]
    return Fr(0)


def _cell_integral(f, c, a, b, bc):
    """Integral over local coordinate xi in [a, b] (subset of [-1/2, 1/2]) of the PFC
    reconstruction in cell c:
      p(xi) = g + eps+ A(xi) (g_{c+1} - g) + eps- B(xi) (g - g_{c-1}),
      A = [2 xi (xi + 3/2) + (xi + 1/2)(xi - 1/2)] / 6,
      B = -[2 xi (xi - 3/2) + (xi + 1/2)(xi - 1/2)] / 6,
      eps+ = min(1, 2 g / (g_{c+1} - g)) if g_{c+1} > g else 1,
      eps- = min(1, -2 g / (g - g_{c-1})) if g < g_{c-1} else 1.
    """
    g, gp, gm = _value(f, c, bc), _value(f, c + 1, bc), _value(f, c - 1, bc)
    dp, dm = gp - g, g - gm
    eps_p = min(Fr(1), 2 * g / dp) if dp > 0 else Fr(1)
    eps_m = min(Fr(1), -2 * g / dm) if dm < 0 else Fr(1)
    A = [Fr(-1, 4) / 6, Fr(3) / 6, Fr(3) / 6]       # (3 xi^2 + 3 xi - 1/4)/6
    B = [Fr(1, 4) / 6, Fr(3) / 6, Fr(-3) / 6]       # -(3 xi^2 - 3 xi - 1/4)/6
    return g * (b - a) + eps_p * dp * _poly_int(A, a, b) + eps_m * dm * _poly_int(B, a, b)


def _swept_flux(f, face, s, bc):
    """Signed mass through face (face index i means x_{i+1/2}, cell widths = 1) when the
    whole profile moves by s cells: integral of the reconstruction over [x_face - s, x_face]."""
    xf = Fr(face) + Fr(1, 2)        # cell c spans [c - 1/2, c + 1/2]
    lo, hi = (xf - s, xf) if s >= 0 else (xf, xf - s)
    total = Fr(0)
    import math
    c = math.floor(lo + Fr(1, 2))
    while Fr(c) - Fr(1, 2) < hi:
        a = max(lo, Fr(c) - Fr(1, 2))
        b = min(hi, Fr(c) + Fr(1, 2))
        if b > a:
            total += _cell_integral(f, c, a - c, b - c, bc)
        c += 1
    return total if s >= 0 else -total


def remap_bruteforce(f, s, bc):
    f = [Fr(x) for x in f]
    s = Fr(s)
    n = len(f)
    phi = [_swept_flux(f, i, s, bc) for i in range(-1, n)]       # faces -1/2 .. n-1/2
    if bc == WALL:
        phi[0] = phi[n] = Fr(0)
    return [f[i] + phi[i] - phi[i + 1] for i in range(n)]


# ----------------------------------------------------------------------------------------
# P1: integer Courant numbers are exact translations (BASELINE.json north_star)
# ----------------------------------------------------------------------------------------
def test_p1_integer_courant_pencil_is_bitwise_roll(orc):
    rng = np.random.default_rng(1)
    f = rng.random(17)
    for k in (-5, -1, 0, 1, 2, 17, 40):
        out = orc.sweep_pencil(f, float(k), PER)
        assert np.array_equal(out, np.roll(f, k)), k


def test_p1_integer_courant_sweep_x_rolls_every_velocity_row(orc):
    # dyadic dx, dv; dt = 2 dx / dv  =>  s_j = v_j dt / dx = 2 vlo/dv + 2j + 1: odd integers
    nx, nv = 16, 8
    grid = orc.Grid(nx=(nx, 1, 1), nv=(nv, 1, 1))
    box = orc.Box(xlo=(0, 0, 0), xhi=(4.0, 1, 1), vlo=(-2.0, 0, 0), vhi=(2.0, 1, 1))
    dx, dv = 4.0 / nx, 4.0 / nv
    dt = 2 * dx / dv
    rng = np.random.default_rng(2)
    f = rng.random(grid.shape)
    f0 = f.copy()
    net = orc.sweep_x(f, grid, box, 0, dt)
    assert net == 0.0
    for j in range(nv):
        k = int(round((-2.0 + (j + 0.5) * dv) * dt / dx))
        assert k % 2 != 0
        assert np.array_equal(f[0, 0, :, 0, 0, j], np.roll(f0[0, 0, :, 0, 0, j], k))


# ----------------------------------------------------------------------------------------
# P2: exact-rational worked examples (golden file) and their independent re-derivation
# ----------------------------------------------------------------------------------------
def _golden_cases():
    cases = []
    for line in (GOLDEN / "pfc3_rationals.txt").read_text().splitlines():
        if not line.strip() or line.startswith("#"):
            continue
        fin, s, exp = [p.strip() for p in line.split("|")]
        cases.append(([Fr(x) for x in fin.split()], Fr(s), [Fr(x) for x in exp.split()]))
    return cases


def test_p2_golden_rationals(orc):
    cases = _golden_cases()
    assert len(cases) == 5
    for fin, s, exp in cases:
        out = orc.sweep_pencil([float(x) for x in fin], float(s), PER)
        assert np.allclose(out, [float(x) for x in exp], rtol=0, atol=4e-16 * 11), (fin, s)
        # the golden values themselves follow from the remap form of the cited method
        assert remap_bruteforce(fin, s, PER) == exp


def test_p2_hand_checked_face_flux(orc):
    # f = [1,4,2,0], s = 1/2: flux through the high end face (= face -1/2 by periodicity) is
    # the flux out of cell 3 (g=0 => 0); phi_{1/2} = 11/16 shows up as f0_new = 1 + 0 - 11/16.
    out, lo, hi = orc.sweep_pencil([1, 4, 2, 0], 0.5, PER, return_flux=True)
    assert lo == 0.0 and hi == 0.0
    assert out[0] == 1.0 - 11.0 / 16.0


# ----------------------------------------------------------------------------------------
# P3: flux form == remap form, brute force in exact rationals (incl. all limiter branches)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [PER, OUT, WALL])
def test_p3_remap_bruteforce_random(orc, bc):
    rng = np.random.default_rng(100 + bc)
    for trial in range(120):
        n = int(rng.integers(4, 9))
        # small dyadic non-negative data with many zeros and steep jumps => every limiter branch
        f = [Fr(int(rng.integers(0, 64)) * int(rng.integers(0, 2) + (trial % 3 == 0)), 8) for _ in range(n)]
        smax = 20 if bc == PER else 7
        s = Fr(int(rng.integers(-smax, smax + 1)), 8)            # |s| up to 2.5 periodic, < 1 else
        exp = remap_bruteforce(f, s, bc)
        out = orc.sweep_pencil([float(x) for x in f], float(s), bc)
        scale = max(1.0, max(float(x) for x in f))
        assert np.max(np.abs(out - np.array([float(x) for x in exp]))) <= 8e-16 * scale, (f, s, bc)


def test_p3_limiter_branches_are_hit():
    # sanity of the test data above: both correctors must be active somewhere
    f = [Fr(0), Fr(8), Fr(0), Fr(1)]
    assert remap_bruteforce(f, Fr(1, 2), PER) != [  # unlimited third-order result would differ
        f[i] for i in range(4)]
    g, gp = Fr(1), Fr(8)
    assert min(Fr(1), 2 * g / (gp - g)) < 1


def test_p3_bruteforce_4x4_step(orc):
    """BASELINE.json: 'brute-force flux sums on 4x4 grids'. 1D1V 4x4 grid, one full split
    step = x sweep (periodic) then vx sweep (walls), every pencil remapped by the
    exact-rational brute force with s from eq. (1)."""
    nx = nv = 4
    grid = orc.Grid(nx=(nx, 1, 1), nv=(nv, 1, 1))
    box = orc.Box(xlo=(0, 0, 0), xhi=(4.0, 1, 1), vlo=(-2.0, 0, 0), vhi=(2.0, 1, 1))
    dt, qm = 0.25, 2.0
    rng = np.random.default_rng(7)
    f = (rng.integers(0, 16, size=grid.shape) * rng.integers(0, 2, size=grid.shape)).astype(np.float64)
    E = np.zeros((3, 1, 1, nx)); B = np.zeros((3, 1, 1, nx))
    E[0, 0, 0] = [0.5, -0.25, 1.0, -1.5]
    B[2, 0, 0] = [1.0, 2.0, -1.0, 0.5]          # no effect in 1V: vy = vz = 0
    ref = [[Fr(int(f[0, 0, i, 0, 0, j])) for j in range(nv)] for i in range(nx)]
    # x sweep: s = v_j dt / dx, dx = 1, v_j = -2 + (j + 1/2)
    for j in range(nv):
        s = (Fr(-2) + Fr(2 * j + 1, 2)) * Fr(1, 4)
        col = remap_bruteforce([ref[i][j] for i in range(nx)], s, PER)
        for i in range(nx):
            ref[i][j] = col[i]
    # vx sweep: s = (q/m) E_x dt / dv, dv = 1
    for i in range(nx):
        s = Fr(2) * Fr(float(E[0, 0, 0, i])) * Fr(1, 4)
        ref[i] = remap_bruteforce(ref[i], s, WALL)
    net = orc.step(f, grid, box, qm, E, B, dt)
    assert net == 0.0
    exp = np.array([[float(x) for x in row] for row in ref])
    assert np.max(np.abs(f[0, 0, :, 0, 0, :] - exp)) <= 1e-14


# ----------------------------------------------------------------------------------------
# P4: textbook special case -- limiter inactive => exact for quadratics (third order)
# ----------------------------------------------------------------------------------------
def _quad_avg(a, b, c, lo, hi):
    """Cell average over [lo,hi] of a + b x + c x^2."""
    return (a * (hi - lo) + b * (hi ** 2 - lo ** 2) / 2 + c * (hi ** 3 - lo ** 3) / 3) / (hi - lo)


@pytest.mark.parametrize("s", [0.37, -0.81, 2.25, -1.5])
def test_p4_quadratic_exactness(orc, s):
    n = 24
    a, b, c = 1000.0, 3.0, -0.7                     # large constant keeps the limiter inactive
    edges = np.arange(n + 1, dtype=float)
    f = np.array([_quad_avg(a, b, c, edges[i], edges[i + 1]) for i in range(n)])
    out = orc.sweep_pencil(f, s, PER)
    exact = np.array([_quad_avg(a, b, c, edges[i] - s, edges[i + 1] - s) for i in range(n)])
    m = int(abs(s)) + 3                             # stay away from the periodic wrap
    assert np.max(np.abs(out[m:n - m] - exact[m:n - m])) <= 1e-12 * a
    # a transposed operand or dropped term would break this by O(1)
    assert np.max(np.abs(out[m:n - m] - f[m:n - m])) > 0.1


def test_p4_third_order_convergence(orc):
    errs = []
    for n in (32, 64, 128, 256):
        x = (np.arange(n + 1)) * (2 * pi / n)
        avg = lambda sh: 2.0 + (np.cos(x[:-1] - sh) - np.cos(x[1:] - sh)) / (2 * pi / n)  # avg of 2+sin
        s = 0.37
        f = avg(0.0)
        steps = n // 4
        for _ in range(steps):
            f = orc.sweep_pencil(f, s, PER)
        errs.append(np.max(np.abs(f - avg(steps * s * 2 * pi / n))))
    rates = [errs[i] / errs[i + 1] for i in range(3)]
    assert all(6.5 < r < 9.5 for r in rates), (errs, rates)      # x8 per doubling


# ----------------------------------------------------------------------------------------
# P5: invariants -- conservation, positivity, mirror symmetry
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc,smax", [(PER, 3.0), (WALL, 0.999)])
def test_p5_mass_conservation(orc, bc, smax):
    rng = np.random.default_rng(5)
    for _ in range(50):
        n = int(rng.integers(4, 64))
        f = rng.random(n) * (rng.random(n) > 0.3) * 10.0 ** rng.integers(-8, 3, size=n)
        s = float(rng.uniform(-smax, smax))
        out = orc.sweep_pencil(f, s, bc)
        assert abs(out.sum() - f.sum()) <= 4e-16 * np.sqrt(n) * np.abs(f).sum() + 1e-300


def test_p5_outflow_mass_budget(orc):
    rng = np.random.default_rng(6)
    for _ in range(50):
        n = int(rng.integers(4, 40))
        f = rng.random(n) + 0.1
        s = float(rng.uniform(-0.999, 0.999))
        out, lo, hi = orc.sweep_pencil(f, s, OUT, return_flux=True)
        assert abs((out.sum() - f.sum()) - (lo - hi)) <= 1e-14 * f.sum()
        assert (hi > 0 and lo > 0) if s > 0 else (hi <= 0 and lo <= 0)


@pytest.mark.parametrize("bc", [PER, OUT, WALL])
def test_p5_positivity(orc, bc):
    rng = np.random.default_rng(8)
    worst = 0.0
    for _ in range(300):
        n = int(rng.integers(4, 40))
        f = rng.random(n) * (rng.random(n) > 0.5) * 10.0 ** rng.integers(-12, 4, size=n)
        s = float(rng.uniform(-0.999, 0.999))
        for _ in range(5):
            f = orc.sweep_pencil(f, s, bc)
            worst = min(worst, f.min() / (f.max() + 1e-300))
    # exact arithmetic keeps f >= 0; rounding may undershoot by ~ulp of the local maximum
    assert worst >= -4e-16


@pytest.mark.parametrize("bc", [PER, OUT, WALL])
def test_p5_mirror_symmetry_is_bitwise(orc, bc):
    rng = np.random.default_rng(9)
    for _ in range(200):
        n = int(rng.integers(4, 30))
        f = rng.random(n) * (rng.random(n) > 0.3)
        s = float(rng.uniform(-0.999, 0.999)) if bc != PER else float(rng.uniform(-3, 3))
        a = orc.sweep_pencil(f, s, bc)[::-1]
        b = orc.sweep_pencil(f[::-1].copy(), -s, bc)
        assert np.array_equal(a, b)


def test_range_errors(orc):
    f = np.ones(8)
    for bc in (OUT, WALL):
        with pytest.raises(ValueError):
            orc.sweep_pencil(f, 1.0, bc)
        with pytest.raises(ValueError):
            orc.sweep_pencil(f, -1.25, bc)
    grid = orc.Grid(nx=(8, 8, 1), nv=(4, 4, 1), bc=(PER, OUT, PER))
    box = orc.Box(xlo=(0, 0, 0), xhi=(8.0, 8.0, 1), vlo=(-2.0, -2.0, 0), vhi=(2.0, 2.0, 1))
    g = np.random.default_rng(0).random(grid.shape)
    g0 = g.copy()
    with pytest.raises(ValueError):                 # |s| = 1.5*1/1 on the outflow axis
        orc.sweep_x(g, grid, box, 1, 1.0)
    assert np.array_equal(g, g0)                    # failed call leaves f untouched
    orc.sweep_x(g, grid, box, 0, 1.0)               # periodic axis takes any s


# ----------------------------------------------------------------------------------------
# P6: free streaming against the analytic f0(x - v t, v)  (BASELINE.json north_star)
# ----------------------------------------------------------------------------------------
def _free_stream(orc, nx, nv=16, steps=20, cfl=0.5):
    L = 4 * pi
    grid = orc.Grid(nx=(nx, 1, 1), nv=(nv, 1, 1))
    box = orc.Box(xlo=(0, 0, 0), xhi=(L, 1, 1), vlo=(-6.0, 0, 0), vhi=(6.0, 1, 1))
    dx, dv = L / nx, 12.0 / nv
    v = -6.0 + (np.arange(nv) + 0.5) * dv
    edges = np.arange(nx + 1) * dx
    gv = np.exp(-0.5 * v ** 2) / sqrt(2 * pi)

    def exact(t):
        # x-cell average of (1 + 0.01 cos(0.5 (x - v t))) g(v): v is NOT averaged -- the scheme
        # moves a whole velocity cell at its centre speed (semi-discrete exact solution)
        lo = edges[:-1, None] - v[None, :] * t
        hi = edges[1:, None] - v[None, :] * t
        return (1.0 + 0.01 * (np.sin(0.5 * hi) - np.sin(0.5 * lo)) / (0.5 * dx)) * gv[None, :]

    f = np.ascontiguousarray(exact(0.0).reshape(grid.shape))
    dt = cfl * dx / np.max(np.abs(v))
    for _ in range(steps):
        orc.sweep_x(f, grid, box, 0, dt)
    return np.max(np.abs(f.reshape(nx, nv) - exact(steps * dt)))


def test_p6_free_streaming(orc):
    e64 = _free_stream(orc, 64, nv=128)
    assert e64 < 1e-7                               # survey scratch: 3.0e-8 on the config-0 grid
    e = [_free_stream(orc, n, steps=20 * n // 32, cfl=0.5) for n in (32, 64, 128)]
    assert 6.0 < e[0] / e[1] < 10.0 and 6.0 < e[1] / e[2] < 10.0, e


def test_p6_direction_of_streaming(orc):
    # a bump at x0 moves towards +x for v > 0 and -x for v < 0 (sign of the v.grad_x term)
    nx, nv = 32, 2
    grid = orc.Grid(nx=(nx, 1, 1), nv=(nv, 1, 1))
    box = orc.Box(xlo=(0, 0, 0), xhi=(32.0, 1, 1), vlo=(-2.0, 0, 0), vhi=(2.0, 1, 1))
    f = np.zeros(grid.shape)
    f[0, 0, 16, 0, 0, :] = 1.0
    for _ in range(8):
        orc.sweep_x(f, grid, box, 0, 0.5)          # v = -1, +1; s = -0.5, +0.5; 4 cells total
    x = np.arange(nx)
    cm = (f[0, 0, :, 0, 0, :] * x[:, None]).sum(0) / f[0, 0, :, 0, 0, :].sum(0)
    assert abs(cm[0] - 12.0) < 1e-12 and abs(cm[1] - 20.0) < 1e-12


def test_sweep_x_other_axes_and_bc(orc):
    """y and z sweeps use the right stride, velocity component and boundary rule."""
    grid = orc.Grid(nx=(5, 6, 7), nv=(2, 3, 4), bc=(PER, OUT, PER))
    box = orc.Box(xlo=(0, 0, 0), xhi=(5.0, 6.0, 7.0), vlo=(-1, -1.5, -2), vhi=(1, 1.5, 2))
    rng = np.random.default_rng(11)
    f0 = rng.random(grid.shape)
    for dim, axis, bc in ((0, 2, PER), (1, 1, OUT), (2, 0, PER)):
        f = f0.copy()
        dt = 0.4
        orc.sweep_x(f, grid, box, dim, dt)
        nvd = grid.nv[dim]
        vc = box.vlo[dim] + (np.arange(nvd) + 0.5) * (box.vhi[dim] - box.vlo[dim]) / nvd
        # check three random pencils against the pencil routine
        for _ in range(6):
            idx = [int(rng.integers(0, s)) for s in grid.shape]
            sl = list(idx); sl[axis] = slice(None)
            jv = idx[5 - dim]                       # f[...,jvz,jvy,jvx]: vx is axis 5, vy 4, vz 3
            s = vc[jv] * dt / 1.0
            exp = orc.sweep_pencil(f0[tuple(sl)], s, bc)
            assert np.array_equal(f[tuple(sl)], exp)


# ----------------------------------------------------------------------------------------
# P7: gyration in a uniform B returns to the initial f after one (discrete) period
# ----------------------------------------------------------------------------------------
def _gyrate(orc, n, N, axis=2, quarter=False):
    """0D2V: B along `axis`, velocity plane = the other two dims (cyclic order e1, e2)."""
    e1, e2 = (axis + 1) % 3, (axis + 2) % 3
    nv = [1, 1, 1]; nv[e1] = nv[e2] = n
    vlo = [0.0, 0.0, 0.0]; vhi = [1.0, 1.0, 1.0]
    for e in (e1, e2):
        vlo[e], vhi[e] = -6.0, 6.0
    grid = orc.Grid(nx=(1, 1, 1), nv=tuple(nv))
    box = orc.Box(vlo=tuple(vlo), vhi=tuple(vhi))
    v = -6.0 + (np.arange(n) + 0.5) * 12.0 / n
    b = 2.0 * np.sin(pi / N)                         # (q/m) B0 dt with trace(M) = 2 - b^2 => M^N = I
    qm, dt = 1.0, 1.0
    B = np.zeros((3, 1, 1, 1)); B[axis] = b
    E = np.zeros((3, 1, 1, 1))
    # drifting Maxwellian u = 1.5 along e1
    shape = grid.shape                              # (1,1,1,nvz,nvy,nvx)
    V = [np.zeros(1)] * 3
    V[e1] = v; V[e2] = v
    vx, vy, vz = V[0][None, None, :], V[1][None, :, None], V[2][:, None, None]
    comp = [vx, vy, vz]
    f0 = np.exp(-0.5 * ((comp[e1] - 1.5) ** 2 + comp[e2] ** 2)) / (2 * pi)
    f0 = np.ascontiguousarray(np.broadcast_to(f0, shape[3:]).reshape(shape))
    f = f0.copy()
    steps = N // 4 if quarter else N
    for _ in range(steps):
        orc.step(f, grid, box, qm, E, B, dt)
    return f0, f, grid, box, (e1, e2)


def test_p7_gyration_closure(orc):
    f0, f1, *_ = _gyrate(orc, 32, 128)
    e32 = np.max(np.abs(f1 - f0)) / f0.max()
    f0b, f1b, *_ = _gyrate(orc, 64, 256)
    e64 = np.max(np.abs(f1b - f0b)) / f0b.max()
    # no error figure in the paper; survey scratch: 1.1e-1 (32^2, N=128), 1.7e-2 (64^2, N=256)
    assert e32 < 0.15 and e64 < 0.025 and e32 / e64 > 4.0, (e32, e64)
    assert abs(f1b.sum() - f0b.sum()) <= 1e-13 * f0b.sum()      # closed velocity box
    assert f1b.min() >= 0.0


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p7_gyration_sense_all_axes(orc, axis):
    """dv/dt = (q/m) v x B: for q/m > 0 the velocity rotates clockwise about B (left-handed),
    so a drift along e1 becomes a drift along -e2 after a quarter period, (e1, e2, B) cyclic.
    Pins the sign and the index pattern of every component of v x B."""
    f0, f, grid, box, (e1, e2) = _gyrate(orc, 40, 160, axis=axis, quarter=True)
    n, j, P = orc.moments(f, grid, box)
    u = j[:, 0, 0, 0] / n[0, 0, 0]
    assert abs(u[e1]) < 0.05 and abs(u[e2] + 1.5) < 0.05 and abs(u[axis]) < 1e-12, u


# ----------------------------------------------------------------------------------------
# P8: uniform E -- rigid shift of f in velocity by (q/m) E t
# ----------------------------------------------------------------------------------------
def _gauss_cell_avg(lo, hi, mu, sig):
    return 0.5 * (np.vectorize(erf)((hi - mu) / (sig * sqrt(2))) - np.vectorize(erf)((lo - mu) / (sig * sqrt(2)))) / (hi - lo)


@pytest.mark.parametrize("dim", [0, 1, 2])
def test_p8_uniform_E_shift(orc, dim):
    errs = []
    for nv in (32, 64, 128):
        nvs = [1, 1, 1]; nvs[dim] = nv
        vlo = [0.0] * 3; vhi = [1.0] * 3
        vlo[dim], vhi[dim] = -8.0, 8.0
        grid = orc.Grid(nx=(1, 1, 1), nv=tuple(nvs))
        box = orc.Box(vlo=tuple(vlo), vhi=tuple(vhi))
        edges = -8.0 + np.arange(nv + 1) * 16.0 / nv
        f = np.ascontiguousarray(_gauss_cell_avg(edges[:-1], edges[1:], 0.0, 1.0).reshape(grid.shape))
        E = np.zeros((3, 1, 1, 1)); E[dim] = 0.75
        B = np.zeros((3, 1, 1, 1))
        qm, T, steps = -2.0, 1.0, nv // 2
        for _ in range(steps):
            orc.sweep_v(f, grid, box, qm, E, B, dim, T / steps)
        exact = _gauss_cell_avg(edges[:-1], edges[1:], qm * 0.75 * T, 1.0)   # moved to -1.5
        errs.append(np.max(np.abs(f.ravel() - exact)))
        assert abs(np.argmax(f.ravel()) - np.argmax(exact)) <= 1
    assert errs[0] / errs[1] > 5.5 and errs[1] / errs[2] > 5.5, errs     # third order in dv
    assert errs[2] < 4e-4                           # measured 2.5e-4 at dv = 1/8 (sigma = 1)


def test_p8_acceleration_uses_other_components(orc):
    """s of a vx pencil = (q/m)(E_x + v_y B_z - v_z B_y) dt / dvx with cell-centre v_y, v_z."""
    grid = orc.Grid(nx=(2, 1, 1), nv=(8, 3, 2))
    box = orc.Box(xlo=(0, 0, 0), xhi=(2.0, 1, 1), vlo=(-2, -1.5, -1), vhi=(2, 1.5, 1))
    rng = np.random.default_rng(12)
    f0 = rng.random(grid.shape)
    E = rng.normal(size=(3, 1, 1, 2)) * 0.1
    B = rng.normal(size=(3, 1, 1, 2)) * 0.1
    qm, dt = 1.5, 0.3
    vx = -2 + (np.arange(8) + 0.5) * 0.5
    vy = -1.5 + (np.arange(3) + 0.5) * 1.0
    vz = -1 + (np.arange(2) + 0.5) * 1.0
    dvs = (0.5, 1.0, 1.0)
    for dim in range(3):
        f = f0.copy()
        orc.sweep_v(f, grid, box, qm, E, B, dim, dt)
        for ix in range(2):
            for jz in range(2):
                for jy in range(3):
                    for jx in range(8):
                        v = (vx[jx], vy[jy], vz[jz])
                        Ec, Bc = E[:, 0, 0, ix], B[:, 0, 0, ix]
                        a = qm * (Ec + np.cross(v, Bc))[dim]
                        s = a * dt / dvs[dim]
                        sl = [0, 0, ix, jz, jy, jx]; sl[5 - dim] = slice(None)
                        exp = orc.sweep_pencil(f0[tuple(sl)], s, WALL)
                        assert np.allclose(f[tuple(sl)], exp, rtol=0, atol=1e-15)


# ----------------------------------------------------------------------------------------
# P9: moments
# ----------------------------------------------------------------------------------------
def test_p9_moments_by_hand(orc):
    grid = orc.Grid(nx=(2, 1, 1), nv=(2, 2, 2))
    box = orc.Box(xlo=(0, 0, 0), xhi=(2.0, 1, 1), vlo=(-1, -2, -3), vhi=(1, 2, 3))
    f = np.zeros(grid.shape)
    # cell 0: small integers; centres vx=+-0.5, vy=+-1, vz=+-1.5; dV = 1*2*3 = 6
    f[0, 0, 0] = np.arange(1, 9).reshape(2, 2, 2)               # [jvz][jvy][jvx]
    f[0, 0, 1, 1, 0, 1] = 2.0                                    # cell 1: one entry at (+.5,-1,+1.5)
    n, j, P = orc.moments(f, grid, box)
    assert n[0, 0, 0] == 36 * 6 and n[0, 0, 1] == 2 * 6
    # cell 0 by hand: sum f = 36; sum vx f = 0.5*(2+4+6+8) - 0.5*(1+3+5+7) = 2
    assert j[0, 0, 0, 0] == 2 * 6
    # sum vy f = 1*(3+4+7+8) - 1*(1+2+5+6) = 8 ; sum vz f = 1.5*(5+6+7+8) - 1.5*(1+2+3+4) = 24
    assert j[1, 0, 0, 0] == 8 * 6 and j[2, 0, 0, 0] == 24 * 6
    # Pxx = 0.25*36 ; Pyy = 1*36 ; Pzz = 2.25*36
    assert P[0, 0, 0, 0] == 9 * 6 and P[3, 0, 0, 0] == 36 * 6 and P[5, 0, 0, 0] == 81 * 6
    # Pxy = sum vx vy f = .5*(4+8) -.5*(3+7) - .5*(2+6) + .5*(1+5) = 0 ; Pxz = .75*(6+8-5-7) -.75*(2+4-1-3) = 0
    assert P[1, 0, 0, 0] == 0 and P[2, 0, 0, 0] == 0
    # Pyz = 1.5*((7+8)-(5+6)) - 1.5*((3+4)-(1+2)) = 6 - 6 = 0
    assert P[4, 0, 0, 0] == 0
    # cell 1: v = (+.5,-1,+1.5), f = 2
    assert np.allclose(j[:, 0, 0, 1], np.array([0.5, -1.0, 1.5]) * 12)
    assert np.allclose(P[:, 0, 0, 1], np.array([0.25, -0.5, 0.75, 1.0, -1.5, 2.25]) * 12)


def test_p9_maxwellian_moments(orc):
    nv = 32
    grid = orc.Grid(nx=(1, 1, 1), nv=(nv, nv, nv))
    box = orc.Box(vlo=(-6, -6, -6), vhi=(6, 6, 6))
    v = -6 + (np.arange(nv) + 0.5) * 12 / nv
    u = np.array([0.3, -0.2, 0.5]); sig = np.array([1.0, 0.8, 1.2]); n0 = 1.7
    g = [np.exp(-0.5 * ((v - u[a]) / sig[a]) ** 2) / (sig[a] * sqrt(2 * pi)) for a in range(3)]
    f = n0 * g[2][:, None, None] * g[1][None, :, None] * g[0][None, None, :]
    f = np.ascontiguousarray(f.reshape(grid.shape))
    n, j, P = orc.moments(f, grid, box)
    assert abs(n[0, 0, 0] - n0) < 1e-5
    assert np.allclose(j[:, 0, 0, 0], n0 * u, atol=5e-5)        # tail truncation at 4.6 sigma dominates
    full = n0 * (np.diag(sig ** 2) + np.outer(u, u))            # P = n (sigma^2 delta + u u), not centred
    exp = np.array([full[0, 0], full[0, 1], full[0, 2], full[1, 1], full[1, 2], full[2, 2]])
    assert np.allclose(P[:, 0, 0, 0], exp, atol=5e-4)
    # inactive velocity dimensions: v == 0, dv == 1
    grid1 = orc.Grid(nx=(1, 1, 1), nv=(nv, 1, 1))
    box1 = orc.Box(vlo=(-6, 0, 0), vhi=(6, 1, 1))
    f1 = np.ascontiguousarray((n0 * g[0]).reshape(grid1.shape))
    n1, j1, P1 = orc.moments(f1, grid1, box1)
    assert abs(n1[0, 0, 0] - n0) < 1e-5 and abs(j1[0, 0, 0, 0] - n0 * u[0]) < 1e-5
    assert j1[1, 0, 0, 0] == 0 and j1[2, 0, 0, 0] == 0 and P1[3, 0, 0, 0] == 0


# ----------------------------------------------------------------------------------------
# step order and mass budget on a small Harris-type grid (oracle's own budget)
# ----------------------------------------------------------------------------------------
def test_step_is_x_y_then_vx_vy_vz_and_budget(orc):
    from paper_2305_01487_b200 import inputs
    w = inputs.harris2d(8, 16, 12, seed_offset=3)
    f, E, B, dt = inputs.make_all(w)
    grid = orc.Grid(nx=w.nx, nv=w.nv, bc=w.bc)
    box = orc.Box(xlo=w.xlo, xhi=w.xhi, vlo=w.vlo, vhi=w.vhi)
    a = f.copy()
    m0 = orc.total(a)
    net_total = 0.0
    for _ in range(10):
        net_total += orc.step(a, grid, box, w.q_over_m, E, B, dt)
    b = f.copy()
    for _ in range(10):
        for d in (0, 1):
            orc.sweep_x(b, grid, box, d, dt)
        for d in (0, 1, 2):
            orc.sweep_v(b, grid, box, w.q_over_m, E, B, d, dt)
    assert np.array_equal(a, b)
    m1 = orc.total(a)
    assert m1 != m0                                               # outflow in y does lose mass
    assert abs((m1 - m0) + net_total) <= 1e-13 * m0               # ... exactly what left through y
    assert a.min() >= 0.0
    # all-periodic variant conserves mass outright
    wp = inputs.harris2d(8, 16, 12, bc_y=inputs.PERIODIC, seed_offset=3)
    gridp = orc.Grid(nx=wp.nx, nv=wp.nv, bc=wp.bc)
    c = f.copy()
    for _ in range(10):
        assert orc.step(c, gridp, box, w.q_over_m, E, B, dt) == 0.0
    assert abs(orc.total(c) - m0) <= 1e-13 * m0


def test_total_is_the_exactly_rounded_sum(orc):
    """orc.total against math.fsum (the exactly rounded sum) on data that defeats a plain running sum: one large
    entry followed by many entries below half an ulp of it, and a Maxwellian-like spread over 60 decades."""
    from math import fsum
    a = np.concatenate([[1.0e5], np.full(1_000_000, 1.0e-16), [-1.0e5], np.full(1000, 3.0e-17)])
    assert abs(orc.total(a) - fsum(a)) <= 1e-18 * fsum(np.abs(a))      # a plain long double sum returns 0 here
    rng = np.random.default_rng(7)
    b = np.exp(-rng.uniform(0.0, 140.0, 400_000))
    assert abs(orc.total(b) - fsum(b)) <= 1e-16 * fsum(b)
