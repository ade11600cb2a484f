"""Pins of the oracle's backsubstituted velocity update ("The velocity
space splitting is realized via backsubstitution [27]"; reading R15 of DESIGN.md). CPU only.

PAPER.md prints no formula for the method, so the pins are what the method has to achieve and what
the mathematics fixes:
  B1  the Boris map against its implicit (Cayley) definition in exact rationals, and against the
      analytic gyration (angle 2 atan(|t|), sense of dv/dt = (q/m) v x B);
  B2  the three foot maps compose to the exact characteristic foot R^-1 (v - c) (exact-rational solve);
  B3  B = 0 reduces to the plain sweeps V_vx, V_vy, V_vz;
  B4  the per-face flux form against the brute-force remap (integral of the PFC reconstruction
      between the displaced faces, exact rationals) and, for equal faces, bitwise against c-5;
  B5  gyration: the composition has no splitting error -- after a quarter period f is the rotated
      f0 up to interpolation error, third order in dv, where the plain sweeps are stuck at O(b);
  B6  conservation to round-off and positivity; B7 the three 1-D Jacobians multiply to 1.
"""
from fractions import Fraction as Fr

import numpy as np
import pytest

from test_oracle_pins import _swept_flux, WALL


def _cross_matrix(t):
    """Matrix of u -> u x t."""
    return [[0, t[2], -t[1]], [-t[2], 0, t[0]], [t[1], -t[0], 0]]


def _solve(A, b):
    """Gaussian elimination in exact rationals."""
    n = len(b)
    M = [[Fr(x) for x in row] + [Fr(b[i])] for i, row in enumerate(A)]
    for i in range(n):
        p = next(r for r in range(i, n) if M[r][i] != 0)
        M[i], M[p] = M[p], M[i]
        M[i] = [x / M[i][i] for x in M[i]]
        for r in range(n):
            if r != i:
                M[r] = [x - M[r][i] * y for x, y in zip(M[r], M[i])]
    return [M[i][n] for i in range(n)]


def _boris_exact(qm, E, B, dt):
    """Implicit definition of the Boris rotation, v+ - v- = (v+ + v-)/2 x (2t)  <=>
    (I - T) v+ = (I + T) v-, with the two half kicks around it; exact rationals."""
    h = Fr(qm) * Fr(dt) / 2
    t = [h * Fr(b) for b in B]
    T = _cross_matrix(t)
    ImT = [[(1 if i == j else 0) - T[i][j] for j in range(3)] for i in range(3)]
    IpT = [[(1 if i == j else 0) + T[i][j] for j in range(3)] for i in range(3)]
    R = [[None] * 3 for _ in range(3)]
    for j in range(3):
        col = _solve(ImT, [IpT[i][j] for i in range(3)])
        for i in range(3):
            R[i][j] = col[i]
    hE = [h * Fr(e) for e in E]
    c = [hE[i] + sum(R[i][k] * hE[k] for k in range(3)) for i in range(3)]
    return R, c


CASES = [
    (1, (Fr(1, 10), Fr(-1, 5), Fr(3, 10)), (Fr(1, 2), Fr(1, 3), Fr(-1, 5)), Fr(2, 5)),
    (-100, (Fr(1, 100), Fr(0), Fr(-1, 50)), (Fr(0), Fr(0), Fr(1)), Fr(1, 200)),
    (Fr(1, 2), (Fr(0), Fr(0), Fr(0)), (Fr(-3, 4), Fr(1, 8), Fr(1)), Fr(-1, 4)),
]


@pytest.mark.parametrize("qm,E,B,dt", CASES)
def test_b1_boris_map_is_the_cayley_rotation(orc, qm, E, B, dt):
    R, c = orc.boris_map(float(qm), [float(x) for x in E], [float(x) for x in B], float(dt))
    Rx, cx = _boris_exact(qm, E, B, dt)
    assert np.max(np.abs(R - np.array([[float(x) for x in r] for r in Rx]))) <= 4e-16
    assert np.max(np.abs(c - np.array([float(x) for x in cx]))) <= 4e-16 * max(1.0, float(max(abs(x) for x in cx)))


def test_b1_gyration_angle_and_sense(orc):
    # q/m > 0, B = B0 z: dvx/dt = Om vy, dvy/dt = -Om vx (clockwise); angle 2 atan(Om dt / 2)
    qm, B0, dt = 2.0, 0.75, 0.3
    R, c = orc.boris_map(qm, [0, 0, 0], [0, 0, B0], dt)
    th = 2 * np.arctan(qm * B0 * dt / 2)
    expect = np.array([[np.cos(th), np.sin(th), 0], [-np.sin(th), np.cos(th), 0], [0, 0, 1]])
    assert np.max(np.abs(R - expect)) <= 1e-15 and np.all(c == 0)
    # uniform E, no B: pure kick (q/m) E dt
    R, c = orc.boris_map(qm, [0.1, -0.2, 0.3], [0, 0, 0], dt)
    assert np.array_equal(R, np.eye(3)) and np.allclose(c, qm * dt * np.array([0.1, -0.2, 0.3]), rtol=1e-15)


@pytest.mark.parametrize("qm,E,B,dt", CASES)
def test_b2_three_foot_maps_compose_to_the_exact_foot(orc, qm, E, B, dt):
    Rx, cx = _boris_exact(qm, E, B, dt)
    R = np.array([[float(x) for x in r] for r in Rx])
    c = np.array([float(x) for x in cx])
    rng = np.random.default_rng(5)
    for _ in range(20):
        v = [Fr(int(k), 16) for k in rng.integers(-96, 97, 3)]        # dyadic points in [-6, 6]^3
        foot = _solve(Rx, [v[i] - cx[i] for i in range(3)])            # R V + c = v, exact
        vf = [float(x) for x in v]
        Z = orc.backsub_foot(R, c, 2, vf)                              # sweep 3 knows (vx, vy, vz)
        Y = orc.backsub_foot(R, c, 1, [vf[0], vf[1], Z])               # sweep 2 knows (vx, vy, Z)
        X = orc.backsub_foot(R, c, 0, [vf[0], Y, Z])                   # sweep 1 knows (vx, Y, Z)
        assert np.max(np.abs(np.array([X, Y, Z]) - np.array([float(x) for x in foot]))) <= 2e-14


@pytest.mark.parametrize("qm,E,B,dt", CASES)
def test_b7_jacobians_multiply_to_one(orc, qm, E, B, dt):
    R, c = orc.boris_map(float(qm), [float(x) for x in E], [float(x) for x in B], float(dt))
    jac = 1.0
    for d in range(3):
        a, b = [0.3, -0.2, 0.5], [0.3, -0.2, 0.5]
        b[d] += 1.0
        jac *= orc.backsub_foot(R, c, d, b) - orc.backsub_foot(R, c, d, a)     # affine: slope = difference
    assert abs(jac - 1.0) <= 1e-14


def _grid(orc, nv, vmax=6.0, nx=(1, 1, 1)):
    grid = orc.Grid(nx=nx, nv=nv)
    box = orc.Box(xlo=(0, 0, 0), xhi=(1, 1, 1), vlo=(-vmax,) * 3, vhi=(vmax,) * 3)
    return grid, box


def test_b3_zero_B_reduces_to_plain_sweeps(orc):
    grid, box = _grid(orc, (12, 10, 8))
    rng = np.random.default_rng(7)
    f = rng.random(grid.shape) * (rng.random(grid.shape) > 0.2)
    E = np.array([0.7, -1.1, 0.4]).reshape(3, 1, 1, 1)
    B = np.zeros((3, 1, 1, 1))
    dt = 0.5
    a, b = f.copy(), f.copy()
    for d in range(3):
        orc.sweep_v(a, grid, box, 1.0, E, B, d, dt)
        orc.sweep_v_backsub(b, grid, box, 1.0, E, B, d, dt)
        assert np.max(np.abs(a - b)) <= 1e-14, d


def test_b4_equal_faces_are_bitwise_the_plain_pencil(orc):
    rng = np.random.default_rng(8)
    g = rng.random(23) * (rng.random(23) > 0.3)
    for s in (0.37, -0.81, 0.0, 0.999):
        out = orc.sweep_pencil_faces(g, np.full(24, s))
        assert np.array_equal(out, orc.sweep_pencil(g, s, WALL)), s


def test_b4_displaced_faces_against_bruteforce_remap(orc):
    """new_i = g_i + phi_{i-1/2} - phi_{i+1/2} with phi = exact integral of the PFC reconstruction
    between the face and its foot; faces move by different amounts, signs change along the pencil."""
    rng = np.random.default_rng(9)
    for trial in range(12):
        n = int(rng.integers(4, 9))
        g = [Fr(int(k), 8) for k in rng.integers(0, 40, n)]
        if trial % 3 == 0:
            g[int(rng.integers(0, n))] = Fr(0)
        sf = [Fr(int(k), 16) for k in rng.integers(-15, 16, n + 1)]
        phi = [_swept_flux(g, i - 1, sf[i], WALL) for i in range(n + 1)]
        phi[0] = phi[n] = Fr(0)
        exact = [g[i] + phi[i] - phi[i + 1] for i in range(n)]
        out = orc.sweep_pencil_faces([float(x) for x in g], [float(x) for x in sf])
        assert np.max(np.abs(out - np.array([float(x) for x in exact]))) <= 1e-13


def test_b4_range_error(orc):
    with pytest.raises(ValueError):
        orc.sweep_pencil_faces(np.ones(6), np.array([0, 0.2, 1.0, 0.1, 0, 0, 0.0]))
    # the wall faces are never used: any value there is accepted
    orc.sweep_pencil_faces(np.ones(6), np.array([5.0, 0.2, 0.3, 0.1, 0, 0, -7.0]))


def _rotated_gaussian_avg(n, vmax, centre, sig, angle):
    """Cell averages (4x4 Gauss points per cell) of a Gaussian centred at Rot(angle) centre."""
    dv = 2 * vmax / n
    ctr = -vmax + (np.arange(n) + 0.5) * dv
    gp = np.array([-0.8611363115940526, -0.3399810435848563, 0.3399810435848563, 0.8611363115940526])
    gw = np.array([0.3478548451374538, 0.6521451548625461, 0.6521451548625461, 0.3478548451374538]) / 2
    cx = np.cos(angle) * centre[0] + np.sin(angle) * centre[1]      # clockwise for q/m B > 0
    cy = -np.sin(angle) * centre[0] + np.cos(angle) * centre[1]
    pts = (ctr[:, None] + 0.5 * dv * gp[None, :])
    ex = np.exp(-0.5 * ((pts - cx) / sig) ** 2) @ gw
    ey = np.exp(-0.5 * ((pts - cy) / sig) ** 2) @ gw
    return ey[:, None] * ex[None, :] / (2 * np.pi * sig ** 2)       # [vy][vx]


def _plane_to_cube(G, n, axis):
    """f [vz][vy][vx] (extent 4 along velocity axis `axis`) from G [b][a], the gyration plane of B along `axis`:
    a = (axis + 1) % 3, b = (axis + 2) % 3 (cyclic, so that dv_a/dt = +(q/m) B v_b, dv_b/dt = -(q/m) B v_a)."""
    a, b = (axis + 1) % 3, (axis + 2) % 3
    shape = [0, 0, 0]
    shape[2 - a], shape[2 - b], shape[2 - axis] = n, n, 4           # array index of velocity dim d is 2 - d
    idx = [None, None, None]
    idx[2 - a] = np.arange(n).reshape([n if k == 2 - a else 1 for k in range(3)])
    idx[2 - b] = np.arange(n).reshape([n if k == 2 - b else 1 for k in range(3)])
    return np.ascontiguousarray(np.broadcast_to(G[idx[2 - b], idx[2 - a]], shape))


def _quarter_turn_error(orc, n, N, backsub, axis=2):
    """Quarter gyration of an off-centre Gaussian about B = B0 e_axis in N steps; max error / max f."""
    vmax, sig, centre = 6.0, 1.0, (1.5, 0.0)
    nv = [n, n, n]
    nv[axis] = 4
    grid, box = _grid(orc, tuple(nv), vmax)
    th = (np.pi / 2) / N
    b = 2 * np.tan(th / 2)                                          # Boris angle per step = th exactly
    E, B = np.zeros((3, 1, 1, 1)), np.zeros((3, 1, 1, 1))
    B[axis] = b
    f0 = _plane_to_cube(_rotated_gaussian_avg(n, vmax, centre, sig, 0.0), n, axis)
    f = f0.reshape((1, 1, 1) + f0.shape).copy()
    for _ in range(N):
        for d in range(3):
            (orc.sweep_v_backsub if backsub else orc.sweep_v)(f, grid, box, 1.0, E, B, d, 1.0)
    exact = _plane_to_cube(_rotated_gaussian_avg(n, vmax, centre, sig, np.pi / 2), n, axis)
    assert np.all(f >= 0.0)
    assert abs(f.sum() - f0.sum()) <= 1e-12 * f0.sum()
    return float(np.max(np.abs(f[0, 0, 0] - exact)) / exact.max())


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_b5_quarter_gyration_has_no_splitting_error(orc, axis):
    # B along every axis in turn (the dim = 0, 1, 2 branches of the backsubstituted sweeps each take the
    # role of first, second and last sweep of the rotation once), mirroring P7's parametrisation.
    # the face displacement is |v| theta / dv < 1: N >= (6 / dv) pi/2 = 25 (n = 32), 50 (n = 64)
    e32 = _quarter_turn_error(orc, 32, 28, True, axis)
    e64 = _quarter_turn_error(orc, 64, 56, True, axis)
    e64_half_angle = _quarter_turn_error(orc, 64, 112, True, axis)
    plain64 = _quarter_turn_error(orc, 64, 56, False, axis)
    plain64_half_angle = _quarter_turn_error(orc, 64, 112, False, axis)
    assert e64 < e32 / 5 and e64 < 6e-3, (e32, e64)                # interpolation error only: ~third order in dv
    assert abs(e64_half_angle - e64) < 0.2 * e64                   # ... and independent of the angle per step
    assert plain64 > 3 * e64, (plain64, e64)                       # the plain sweeps add an O(b) splitting error
    assert plain64_half_angle < 0.65 * plain64                     # ... which falls with the angle per step


def test_b6_conservation_and_positivity_general_fields(orc):
    grid, box = _grid(orc, (10, 12, 8), 5.0, nx=(3, 2, 1))
    rng = np.random.default_rng(11)
    f = rng.random(grid.shape) * (rng.random(grid.shape) > 0.3)
    E = 0.3 * rng.standard_normal((3, 1, 2, 3))
    B = 0.6 * rng.standard_normal((3, 1, 2, 3))
    m0 = orc.total(f)
    for _ in range(3):
        for d in range(3):
            orc.sweep_v_backsub(f, grid, box, 1.0, E, B, d, 0.05)
    assert f.min() >= 0.0
    assert abs(orc.total(f) - m0) <= 1e-14 * m0


def test_step_backsub_is_x_sweeps_then_backsub_sweeps(orc):
    grid = orc.Grid(nx=(6, 5, 1), nv=(8, 6, 4), bc=(0, 1, 0))
    box = orc.Box(xlo=(0, 0, 0), xhi=(3, 2.5, 1), vlo=(-4,) * 3, vhi=(4,) * 3)
    rng = np.random.default_rng(12)
    f = rng.random(grid.shape)
    E = 0.2 * rng.standard_normal((3, 1, 5, 6))
    B = 0.5 * rng.standard_normal((3, 1, 5, 6))
    a, b = f.copy(), f.copy()
    dt = 0.05
    orc.step_backsub(a, grid, box, 1.0, E, B, dt)
    for d in (0, 1):
        orc.sweep_x(b, grid, box, d, dt)
    for d in range(3):
        orc.sweep_v_backsub(b, grid, box, 1.0, E, B, d, dt)
    assert np.array_equal(a, b)
