"""GPU parity of mphv_maxwellian and mphv_exchange_maxwellian (readings R16, R17) against
the oracle, element by element, through the C ABI. Tolerance: PER ELEMENT and relative,
|gpu - oracle| <= 1e-12 |oracle| + 1e-300 for a Maxwellian fill; for exchange and matching, whose result
M[a] + sigma (f - M[b]) is a difference that may cancel, 1e-12 of the sum of the magnitudes of its three terms
in that same cell (never the cube maximum)."""
import numpy as np
import pytest

from test_gpu_parity import small_workload, torch_cuda, mphv  # noqa: F401
from test_oracle_maxwellian import _moments_from

pytestmark = pytest.mark.gpu
TOL = 1e-12


def _worst(got, ref):
    """largest relative error over the elements above 1e-280 (for the assertion message)"""
    m = np.abs(ref) > 1e-280
    return float(np.max(np.abs(got - ref)[m] / np.abs(ref)[m])) if m.any() else 0.0


def _cell_maxwellians(orc, grid, box, f):
    """M[moments of f] per spatial cell, same shape as f (oracle calls only; used for error scales)."""
    n, j, P = orc.moments(f, grid, box)
    M = orc.maxwellian(grid, box, n.reshape(-1), j.reshape(3, -1), P.reshape(6, -1))
    return M.reshape(f.shape)


def _random_moments(rng, count):
    n, j, P = [], [], []
    for _ in range(count):
        A = 0.4 * rng.standard_normal((3, 3))
        C = A @ A.T + np.diag(0.6 + 0.6 * rng.random(3))
        a, b, c = _moments_from(0.3 + rng.random(), 0.8 * rng.standard_normal(3), C)
        n.append(a); j.append(b); P.append(c)
    return np.array(n), np.array(j).T.copy(), np.array(P).T.copy()


@pytest.mark.parametrize("nv", [(12, 10, 8), (9, 7, 5), (40, 40, 8), (16, 12, 1), (16, 1, 1)])
def test_maxwellian_matches_oracle(torch_cuda, mphv, orc, nv):
    torch = torch_cuda
    w = small_workload((4, 4, 1), nv)
    sim = mphv.Vlasov.from_workload(w)
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    rng = np.random.default_rng(31)
    n, j, P = _random_moments(rng, 7)
    n[2] = 0.0                      # degenerate cells give 0
    P[3, 4] = -1.0
    ref = orc.maxwellian(grid, box, n, j, P)
    out = sim.maxwellian(torch.from_numpy(n).cuda(), torch.from_numpy(j).cuda(), torch.from_numpy(P).cuda())
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.all(got[2] == 0.0) and (nv[1] == 1 or np.all(got[4] == 0.0))     # C_yy < 0 only matters if vy is active
    for c in range(7):
        assert np.all(np.abs(got[c] - ref[c]) <= TOL * np.abs(ref[c]) + 1e-300), (c, _worst(got[c], ref[c]))


@pytest.mark.parametrize("sigma", [0.05, 0.012, 0.3])
def test_cold_maxwellians_have_no_nan(torch_cuda, mphv, orc, sigma):
    """Thermal spread far below the cell width (dv = 0.31..1.25 here), centred near the box edge and in the middle:
    the vz recurrence would form 0 * inf; such blocks are evaluated cell by cell. No NaN, and every element within
    the relative bound (the oracle evaluates one exp per cell and underflows to 0 where the kernel must too)."""
    torch = torch_cuda
    w = small_workload((4, 4, 1), (16, 8, 32))
    sim = mphv.Vlasov.from_workload(w)
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    n, j, P = [], [], []
    for u in ((0.0, 0.0, 0.0), (0.0, 0.0, 0.02), (-0.01, 0.01, -0.03), (0.0, 0.02, 0.0)):      # small drifts: C = P/n - uu stays well conditioned
        a, b, c = _moments_from(1.0, np.array(u), np.diag([sigma ** 2, (2 * sigma) ** 2, sigma ** 2]))
        n.append(a); j.append(b); P.append(c)
    n, j, P = np.array(n), np.array(j).T.copy(), np.array(P).T.copy()
    ref = orc.maxwellian(grid, box, n, j, P)
    got = sim.maxwellian(torch.from_numpy(n).cuda(), torch.from_numpy(j).cuda(), torch.from_numpy(P).cuda()).cpu().numpy()
    assert np.isfinite(got).all()
    assert np.all(np.abs(got - ref) <= TOL * np.abs(ref) + 1e-300), _worst(got, ref)
    # and through the matching kernel, whose target moments come from the caller
    f = np.abs(np.random.default_rng(5).standard_normal((4,) + ref.shape[1:])) + 0.1
    wl = small_workload((4, 1, 1), (16, 8, 32))
    sim2 = mphv.Vlasov.from_workload(wl)
    fd = torch.from_numpy(f.reshape(wl.shape).copy()).cuda()
    sim2.bind_f(fd)
    sim2.match_moments(torch.from_numpy(n.reshape(1, 1, 4)).cuda(), torch.from_numpy(j.reshape(3, 1, 1, 4)).cuda(),
                       torch.from_numpy(P.reshape(6, 1, 1, 4)).cuda())
    assert bool(torch.isfinite(fd).all())


@pytest.mark.parametrize("nx,dim", [((6, 4, 1), 0), ((4, 6, 1), 1), ((4, 4, 5), 2)])
@pytest.mark.parametrize("side", [0, 1])
def test_exchange_maxwellian_matches_oracle(torch_cuda, mphv, orc, nx, dim, side):
    torch = torch_cuda
    from paper_2305_01487_b200 import inputs
    w = small_workload(nx, (12, 12, 8), (0, 0, 0))
    f0, _, _, _ = inputs.make_all(w)
    sim = mphv.Vlasov.from_workload(w)
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    plane = grid.n_space // w.nx[dim]
    rng = np.random.default_rng(32)
    n, j, P = _random_moments(rng, 2 * plane)
    n_fl, j_fl, P_fl = n.reshape(2, plane), j.reshape(3, 2, plane), P.reshape(6, 2, plane)
    ref = f0.copy()
    orc.exchange_maxwellian(ref, grid, box, dim, side, n_fl, j_fl, P_fl)
    f = torch.from_numpy(f0).cuda()
    sim.bind_f(f)
    sim.exchange_maxwellian(dim, side, torch.from_numpy(n_fl).cuda(), torch.from_numpy(j_fl).cuda(),
                            torch.from_numpy(P_fl).cuda())
    torch.cuda.synchronize()
    got = f.cpu().numpy()
    ax = {0: 2, 1: 1, 2: 0}[dim]
    nd = w.nx[dim]
    layers = [nd - 2, nd - 1] if side else [0, 1]
    keep = [i for i in range(nd) if i not in layers]
    assert np.array_equal(np.take(got, keep, axis=ax), np.take(f0, keep, axis=ax)), "interior untouched"
    # per-element scale: |M[fluid]| + sigma (|f_ext| + |M[moments of f_ext]|) in the same velocity cell
    M_fl = orc.maxwellian(grid, box, n, j, P).reshape((2, plane) + f0.shape[3:])
    ext = nd - 3 if side else 2
    f_ext = np.take(f0, [ext], axis=ax)
    M_ext = np.take(_cell_maxwellians(orc, grid, box, f0), [ext], axis=ax)
    for k, layer in enumerate(layers):
        sigma = (2.0 / 3.0) if abs(layer - ext) == 1 else (1.0 / 3.0)
        sc = np.abs(M_fl[k].reshape(f_ext.shape)) + sigma * (np.abs(f_ext) + np.abs(M_ext))
        d = np.abs(np.take(got, [layer], axis=ax) - np.take(ref, [layer], axis=ax))
        assert np.all(d <= TOL * sc + 1e-300), (layer, float(np.max(d / np.maximum(sc, 1e-300))))


@pytest.mark.parametrize("nx,nv", [((4, 4, 1), (12, 12, 8)), ((4, 1, 4), (9, 7, 5)), ((4, 4, 1), (40, 40, 8))])
def test_match_moments_matches_oracle(torch_cuda, mphv, orc, nx, nv):
    torch = torch_cuda
    from paper_2305_01487_b200 import inputs
    w = small_workload(nx, nv, (0, 0, 0))
    f0, _, _, _ = inputs.make_all(w)
    sim = mphv.Vlasov.from_workload(w)
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    ns = grid.n_space
    n, j, P = _random_moments(np.random.default_rng(33), ns)
    ref = f0.copy()
    orc.match_moments(ref, grid, box, n, j, P)
    f = torch.from_numpy(f0).cuda()
    sim.bind_f(f)
    sim.match_moments(torch.from_numpy(n).cuda(), torch.from_numpy(j).cuda(), torch.from_numpy(P).cuda())
    torch.cuda.synchronize()
    got = f.cpu().numpy()
    # per-element scale: |M[target]| + |f| + |M[moments of f]| in the same velocity cell
    sc = np.abs(orc.maxwellian(grid, box, n, j, P).reshape(f0.shape)) + np.abs(f0) + np.abs(_cell_maxwellians(orc, grid, box, f0))
    d = np.abs(got - ref)
    assert np.all(d <= TOL * sc + 1e-300), float(np.max(d / np.maximum(sc, 1e-300)))


def test_maxwellian_errors(torch_cuda, mphv, orc):
    w = small_workload((4, 4, 1), (8, 8, 8))
    sim = mphv.Vlasov.from_workload(w)
    with pytest.raises(mphv.MphvError) as e:
        mphv.mphv_maxwellian(sim.ctx, 3, None, None, None, None)
    assert e.value.code == mphv.ERR_ARG
    with pytest.raises(mphv.MphvError) as e:
        mphv.mphv_exchange_maxwellian(sim.ctx, 2, 0, None, None, None)      # z inactive
    assert e.value.code == mphv.ERR_ARG
