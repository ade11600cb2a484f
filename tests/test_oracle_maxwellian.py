"""Pins of the oracle's ten-moment Maxwellian and exchange of Maxwellians (
P:L185 "ten-moment Maxwellian ... (a multivariate normal distribution)", P:L187 sigma_1 = 2/3,
sigma_2 = 1/3; readings R16, R17 of DESIGN.md). CPU only.

  M1  isotropic case against the textbook closed form n (2 pi s^2)^(-3/2) exp(-|v-u|^2 / 2 s^2);
  M2  general covariance against scipy.stats.multivariate_normal (library routine);
  M3  the midpoint moments (c-8) of the filled distribution reproduce (n, j, P);
  M4  degenerate input (n <= 0, covariance not positive definite) gives 0; 1V and 2V grids;
  X1  exchange: the boundary cells carry the fluid moments; X2 the weights are 2/3 next to the
      interior and 1/3 in the outer cell, on either side; X3 interior cells are untouched and a
      Vlasov state that already is the fluid's Maxwellian gives exactly-ish that Maxwellian.
"""
import numpy as np
import pytest
from scipy.stats import multivariate_normal


def _grid(orc, nv=(24, 24, 24), vmax=8.0, nx=(1, 1, 1)):
    grid = orc.Grid(nx=nx, nv=nv, bc=(0, 0, 0))
    box = orc.Box(xlo=(0, 0, 0), xhi=(1, 1, 1), vlo=(-vmax,) * 3, vhi=(vmax,) * 3)
    return grid, box


def _centres(n, vmax):
    dv = 2 * vmax / n
    return -vmax + (np.arange(n) + 0.5) * dv


def _moments_from(n, u, C):
    u = np.asarray(u, float); C = np.asarray(C, float)
    S = n * (C + np.outer(u, u))
    return n, n * u, np.array([S[0, 0], S[0, 1], S[0, 2], S[1, 1], S[1, 2], S[2, 2]])


def test_m1_isotropic_closed_form(orc):
    grid, box = _grid(orc, (16, 12, 10), 6.0)
    n0, u, sg = 1.7, np.array([0.4, -0.3, 0.2]), 1.3
    n, j, P = _moments_from(n0, u, sg ** 2 * np.eye(3))
    f = orc.maxwellian(grid, box, [n], j.reshape(3, 1), P.reshape(6, 1))[0]
    vx, vy, vz = _centres(16, 6.0), _centres(12, 6.0), _centres(10, 6.0)
    r2 = (vz[:, None, None] - u[2]) ** 2 + (vy[None, :, None] - u[1]) ** 2 + (vx[None, None, :] - u[0]) ** 2
    expect = n0 * (2 * np.pi * sg ** 2) ** -1.5 * np.exp(-r2 / (2 * sg ** 2))
    assert np.max(np.abs(f - expect) / expect) <= 1e-12


def test_m2_general_covariance_against_scipy(orc):
    grid, box = _grid(orc, (14, 12, 10), 6.0)
    rng = np.random.default_rng(3)
    A = rng.standard_normal((3, 3))
    C = A @ A.T + 0.5 * np.eye(3)
    u = np.array([0.3, -0.6, 0.1])
    n, j, P = _moments_from(2.5, u, C)
    f = orc.maxwellian(grid, box, [n], j.reshape(3, 1), P.reshape(6, 1))[0]
    vx, vy, vz = _centres(14, 6.0), _centres(12, 6.0), _centres(10, 6.0)
    Z, Y, X = np.meshgrid(vz, vy, vx, indexing="ij")
    pdf = multivariate_normal(mean=u, cov=C).pdf(np.stack([X, Y, Z], axis=-1))
    assert np.max(np.abs(f - 2.5 * pdf) / (2.5 * pdf)) <= 1e-10


def test_m3_moments_are_reproduced(orc):
    grid, box = _grid(orc, (32, 32, 32), 9.0)
    C = np.array([[1.2, 0.3, -0.2], [0.3, 0.9, 0.1], [-0.2, 0.1, 1.5]])
    n, j, P = _moments_from(0.8, [0.5, -0.4, 0.3], C)
    f = orc.maxwellian(grid, box, [n], j.reshape(3, 1), P.reshape(6, 1))
    g1 = orc.Grid(nx=(1, 1, 1), nv=(32, 32, 32))
    n2, j2, P2 = orc.moments(np.ascontiguousarray(f.reshape(g1.shape)), g1, box)
    assert abs(n2[0, 0, 0] - n) <= 1e-9
    assert np.max(np.abs(j2.reshape(3) - j)) <= 1e-9 and np.max(np.abs(P2.reshape(6) - P)) <= 1e-8


def test_m4_degenerate_and_lower_dimensional(orc):
    grid, box = _grid(orc, (8, 8, 8), 5.0)
    n, j, P = _moments_from(1.0, [0, 0, 0], np.eye(3))
    assert np.all(orc.maxwellian(grid, box, [0.0], j.reshape(3, 1), P.reshape(6, 1)) == 0.0)
    assert np.all(orc.maxwellian(grid, box, [-1.0], j.reshape(3, 1), P.reshape(6, 1)) == 0.0)
    Pbad = P.copy(); Pbad[3] = -0.1                                  # C_yy < 0
    assert np.all(orc.maxwellian(grid, box, [1.0], j.reshape(3, 1), Pbad.reshape(6, 1)) == 0.0)
    # two cells in one call, second one shifted
    n2, j2, P2 = _moments_from(2.0, [1.0, 0, 0], np.eye(3))
    f = orc.maxwellian(grid, box, [1.0, 2.0], np.stack([j, j2], 1), np.stack([P, P2], 1))
    assert f.shape == (2, 8, 8, 8) and f[1].sum() > 1.9 * f[0].sum()
    # 1V grid: a 1-D normal in vx
    g1 = orc.Grid(nx=(1, 1, 1), nv=(16, 1, 1))
    b1 = orc.Box(xlo=(0, 0, 0), xhi=(1, 1, 1), vlo=(-6, 0, 0), vhi=(6, 1, 1))
    f1 = orc.maxwellian(g1, b1, [1.0], [[0.5], [0], [0]], [[1.25], [0], [0], [0], [0], [0]])[0, 0, 0]
    v = _centres(16, 6.0)
    assert np.allclose(f1, np.exp(-0.5 * (v - 0.5) ** 2) / np.sqrt(2 * np.pi), rtol=1e-13)


def _exchange_setup(orc, dim=1, nv=(26, 26, 26), vmax=11.0):
    nx = [1, 1, 1]; nx[dim] = 6; nx[(dim + 1) % 3] = 2
    grid = orc.Grid(nx=tuple(nx), nv=nv, bc=(0, 0, 0))
    box = orc.Box(xlo=(0, 0, 0), xhi=(1, 1, 1), vlo=(-vmax,) * 3, vhi=(vmax,) * 3)
    rng = np.random.default_rng(21)
    # Vlasov state: a two-beam (non-Maxwellian) distribution in every cell, cell-dependent weights
    nsp = grid.n_space
    n, ja, Pa = _moments_from(1.0, [1.5, 0, 0], 0.8 * np.eye(3))
    _, jb, Pb = _moments_from(1.0, [-1.2, 0.5, 0], 1.1 * np.eye(3))
    fa = orc.maxwellian(grid, box, [1.0], ja.reshape(3, 1), Pa.reshape(6, 1))[0]
    fb = orc.maxwellian(grid, box, [1.0], jb.reshape(3, 1), Pb.reshape(6, 1))[0]
    wts = 0.5 + rng.random(nsp)
    f = (wts[:, None, None, None] * fa + (1.5 - 0.5 * wts)[:, None, None, None] * fb).reshape(grid.shape)
    plane = nsp // grid.nx[dim]
    nf, jf, Pf = [], [], []
    for k in range(2 * plane):
        C = np.diag(0.8 + 0.4 * rng.random(3)); C[0, 1] = C[1, 0] = 0.1
        a, b, c = _moments_from(0.7 + 0.6 * rng.random(), 0.3 * rng.standard_normal(3), C)
        nf.append(a); jf.append(b); Pf.append(c)
    n_fl = np.array(nf).reshape(2, plane)
    j_fl = np.array(jf).T.reshape(3, 2, plane).copy()
    P_fl = np.array(Pf).T.reshape(6, 2, plane).copy()
    return grid, box, np.ascontiguousarray(f), n_fl, j_fl, P_fl


@pytest.mark.parametrize("dim", [0, 1, 2])
@pytest.mark.parametrize("side", [0, 1])
def test_x1_x2_boundary_cells_carry_fluid_moments_with_weights(orc, dim, side):
    grid, box, f, n_fl, j_fl, P_fl = _exchange_setup(orc, dim)
    f0 = f.copy()
    orc.exchange_maxwellian(f, grid, box, dim, side, n_fl, j_fl, P_fl)
    ax = {0: 2, 1: 1, 2: 0}[dim]
    nd = grid.nx[dim]
    layers = [nd - 2, nd - 1] if side else [0, 1]
    interior = nd - 3 if side else 2
    # X3: everything but the two boundary layers is untouched
    keep = [i for i in range(nd) if i not in layers]
    assert np.array_equal(np.take(f, keep, axis=ax), np.take(f0, keep, axis=ax))
    # X1: midpoint moments of the boundary cells = the fluid data (up to the quadrature defect of M)
    n2, j2, P2 = orc.moments(f, grid, box)
    for li, idx in enumerate(layers):
        assert np.max(np.abs(np.take(n2, idx, axis=ax).reshape(-1) - n_fl[li])) <= 1e-7
        assert np.max(np.abs(np.take(j2, idx, axis=ax + 1).reshape(3, -1) - j_fl[:, li])) <= 1e-7
        assert np.max(np.abs(np.take(P2, idx, axis=ax + 1).reshape(6, -1) - P_fl[:, li])) <= 1e-6
    # X2: ghost - M[fluid] = sigma (f_ext - M[mom f_ext]); the non-Maxwellian remainder of the cell next
    # to the interior is exactly twice that of the outer cell, and 2/3 of the interior cell's own
    near, far = (layers[0], layers[1]) if side else (layers[1], layers[0])
    lnear, lfar = (0, 1) if side else (1, 0)
    fext = np.take(f0, interior, axis=ax)
    sp = fext.shape[:2]
    ne, je, Pe = orc.moments(f0, grid, box)
    Mex = orc.maxwellian(grid, box, np.take(ne, interior, axis=ax).reshape(-1),
                         np.take(je, interior, axis=ax + 1).reshape(3, -1),
                         np.take(Pe, interior, axis=ax + 1).reshape(6, -1)).reshape(fext.shape)
    rem = fext - Mex
    assert np.max(np.abs(rem)) > 1e-3, "the test state must have a non-Maxwellian part"
    for idx, li, sigma in [(near, lnear, 2.0 / 3.0), (far, lfar, 1.0 / 3.0)]:
        Mfl = orc.maxwellian(grid, box, n_fl[li], j_fl[:, li], P_fl[:, li]).reshape(fext.shape)
        got = np.take(f, idx, axis=ax) - Mfl
        assert np.max(np.abs(got - sigma * rem)) <= 1e-15 * max(1.0, np.max(np.abs(fext)))


def test_x3_maxwellian_vlasov_state_gives_the_fluid_maxwellian(orc):
    grid, box, f, n_fl, j_fl, P_fl = _exchange_setup(orc, 0, nv=(26, 26, 26), vmax=11.0)
    n, j, P = _moments_from(1.0, [0.2, 0.1, -0.3], np.diag([1.0, 1.2, 0.9]))
    cube = orc.maxwellian(grid, box, [n], j.reshape(3, 1), P.reshape(6, 1))[0]
    f[...] = cube
    orc.exchange_maxwellian(f, grid, box, 0, 1, n_fl, j_fl, P_fl)
    for li, idx in enumerate([4, 5]):
        Mfl = orc.maxwellian(grid, box, n_fl[li], j_fl[:, li], P_fl[:, li]).reshape(f[:, :, idx].shape)
        assert np.max(np.abs(f[:, :, idx] - Mfl)) <= 1e-9        # f_ext - M[mom f_ext] = quadrature defect only


def test_r18_match_moments(orc):
    """f <- M[target] + (f - M[mom f]): the cell then carries the target moments (up to the quadrature
    defect of the two Maxwellians), its non-Maxwellian remainder is unchanged, matching to its own
    moments changes nothing, and matching is idempotent."""
    grid, box, f, n_fl, j_fl, P_fl = _exchange_setup(orc, 0)
    ns = grid.n_space
    rng = np.random.default_rng(41)
    tn, tj, tP = [], [], []
    for _ in range(ns):
        C = np.diag(0.8 + 0.5 * rng.random(3)); C[1, 2] = C[2, 1] = -0.15
        a, b, c = _moments_from(0.6 + rng.random(), 0.4 * rng.standard_normal(3), C)
        tn.append(a); tj.append(b); tP.append(c)
    n_t = np.array(tn).reshape(grid.shape[:3])
    j_t = np.array(tj).T.reshape((3,) + grid.shape[:3]).copy()
    P_t = np.array(tP).T.reshape((6,) + grid.shape[:3]).copy()
    f0 = f.copy()
    n0, j0, P0 = orc.moments(f0, grid, box)
    rem0 = f0 - orc.maxwellian(grid, box, n0.reshape(-1), j0.reshape(3, -1), P0.reshape(6, -1)).reshape(f0.shape)
    orc.match_moments(f, grid, box, n_t, j_t, P_t)
    n1, j1, P1 = orc.moments(f, grid, box)
    assert np.max(np.abs(n1 - n_t)) <= 1e-7 and np.max(np.abs(j1 - j_t)) <= 1e-7 and np.max(np.abs(P1 - P_t)) <= 1e-6
    rem1 = f - orc.maxwellian(grid, box, n_t.reshape(-1), j_t.reshape(3, -1), P_t.reshape(6, -1)).reshape(f.shape)
    assert np.max(np.abs(rem1 - rem0)) <= 1e-15
    g = f.copy()
    orc.match_moments(g, grid, box, n_t, j_t, P_t)                  # idempotent up to the quadrature defect
    assert np.max(np.abs(g - f)) <= 1e-7
    h = f0.copy()
    orc.match_moments(h, grid, box, n0, j0, P0)                     # own moments: nothing changes
    assert np.max(np.abs(h - f0)) <= 1e-15
