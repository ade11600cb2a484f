"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs. Bar: 1e-12 relative per sweep/step (BASELINE.json), bit-exact for
whole-cell shifts, mass to 1e-13. Run with ``-m gpu`` on a B200."""
import numpy as np
import pytest

from parity_util import TOL_MASS, TOL_SWEEP, moment_scales, moments_err, moments_worst, rel_err

pytestmark = pytest.mark.gpu

# f array axes: [iz, iy, ix, jvz, jvy, jvx]
AX_X = {0: 2, 1: 1, 2: 0}
AX_V = {0: 5, 1: 4, 2: 3}


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need a GPU"
    return torch


@pytest.fixture(scope="module")
def mphv():
    from paper_2305_01487_b200 import mphv as m
    m.lib()
    return m


def small_workload(nx, nv, bc=(0, 1, 0), seed_offset=0, kind=None):
    from paper_2305_01487_b200 import inputs
    kind = kind or ("harris3d" if nx[2] > 1 else "harris2d")
    return inputs.Workload(
        name="small", index=1, kind=kind, nx=tuple(nx), nv=tuple(nv), bc=tuple(bc),
        xlo=(0.0, -6.4, 0.0), xhi=(25.6, 6.4, 12.8), vlo=(-5.0,) * 3, vhi=(5.0,) * 3,
        steps=2, seed_offset=seed_offset)


class Pair:
    """Same inputs on both sides: oracle on numpy arrays, CUDA path on device tensors."""

    def __init__(self, torch, mphv, orc, w, with_scratch=False, fusion=True):
        from paper_2305_01487_b200 import inputs
        self.torch, self.orc, self.w = torch, orc, w
        self.f0, self.E, self.B, self.dt = inputs.make_all(w)
        self.grid = orc.Grid(w.nx, w.nv, w.bc)
        self.box = orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
        self.f_ref = self.f0.copy()
        self.sim = mphv.Vlasov.from_workload(w)
        self.sim.set_fusion(fusion)
        self.f_dev = torch.from_numpy(self.f0).cuda()
        self.scratch = torch.empty_like(self.f_dev) if with_scratch else None
        self.sim.bind_f(self.f_dev, self.scratch)
        self.E_dev, self.B_dev = torch.from_numpy(self.E).cuda(), torch.from_numpy(self.B).cuda()
        self.sim.set_fields(self.E_dev, self.B_dev)

    def gpu(self):
        self.torch.cuda.synchronize()
        return self.f_dev.cpu().numpy()

    def set_f(self, arr):
        self.f_ref = np.ascontiguousarray(arr, dtype=np.float64).copy()
        self.f_dev.copy_(self.torch.from_numpy(self.f_ref))


SHAPES = [
    # nx, nv, bc : even/odd inner (double2 vs scalar path), ragged vs block sizes, 3-D
    ((12, 10, 1), (12, 10, 8), (0, 1, 0)),
    ((8, 12, 1), (9, 7, 5), (1, 0, 0)),
    ((6, 5, 4), (8, 6, 4), (0, 1, 0)),
    ((5, 4, 6), (7, 4, 12), (1, 1, 1)),
    ((36, 8, 1), (40, 12, 6), (0, 1, 0)),
]


@pytest.mark.parametrize("nx,nv,bc", SHAPES)
@pytest.mark.parametrize("sign", [1.0, -1.0])
def test_each_sweep_matches_oracle(torch_cuda, mphv, orc, nx, nv, bc, sign):
    w = small_workload(nx, nv, bc)
    p = Pair(torch_cuda, mphv, orc, w)
    dt = sign * p.dt * 1.7          # CFL 0.85: exercises large fractional shifts, both signs
    for d in range(3):
        if w.nx[d] > 1:
            orc.sweep_x(p.f_ref, p.grid, p.box, d, dt)
            p.sim.sweep_x(d, dt)
            err = rel_err(p.gpu(), p.f_ref, AX_X[d])
            assert err <= TOL_SWEEP, f"sweep_x({d}) err {err:.3e}"
            p.set_f(p.f_ref)        # restart both sides from identical data
    for d in range(3):
        if w.nv[d] > 1:
            orc.sweep_v(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, d, dt)
            p.sim.sweep_v(d, dt)
            err = rel_err(p.gpu(), p.f_ref, AX_V[d])
            assert err <= TOL_SWEEP, f"sweep_v({d}) err {err:.3e}"
            p.set_f(p.f_ref)


@pytest.mark.parametrize("nx,nv,bc", SHAPES + [((4, 4, 1), (40, 40, 8), (0, 1, 0)), ((4, 4, 1), (20, 36, 4), (0, 0, 0)),
                                            ((4, 4, 1), (4, 4, 4), (0, 1, 0)), ((4, 4, 1), (64, 8, 1), (0, 1, 0)),
                                            ((4, 4, 1), (36, 36, 6), (0, 1, 0)), ((8, 4, 1), (16, 16, 16), (0, 1, 0))])
@pytest.mark.parametrize("fusion", [0, 1, 2, 3])
def test_full_step_and_moments_fused_and_unfused(torch_cuda, mphv, orc, nx, nv, bc, fusion):
    """mphv_step_moments (fused plane kernel vx+vy, fused vz+moments when fusion is on) against
    oracle step + oracle moments, ragged and odd shapes included (odd extents fall back to the
    unfused kernels inside the library)."""
    w = small_workload(nx, nv, bc)
    p = Pair(torch_cuda, mphv, orc, w, fusion=fusion)
    dt = 1.6 * p.dt
    out = None
    for _ in range(2):
        orc.step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, dt)
        out = p.sim.step_moments(dt)
    g = p.gpu()
    last_ax = AX_V[2] if w.nv[2] > 1 else (AX_V[1] if w.nv[1] > 1 else AX_V[0])
    assert rel_err(g, p.f_ref, last_ax) <= 2 * TOL_SWEEP
    n_r, j_r, P_r = orc.moments(p.f_ref, p.grid, p.box)
    n_g, j_g, P_g = (t.cpu().numpy() for t in out)
    scale = np.abs(P_r[0]) + np.abs(P_r[3]) + np.abs(P_r[5]) + np.abs(n_r)
    for a, b in [(n_g, n_r), (j_g, j_r), (P_g, P_r)]:
        assert np.max(np.abs(a - b) / scale) <= 1e-12


def test_limiter_active_data_matches_oracle(torch_cuda, mphv, orc):
    """Random non-negative data with exact zeros and spikes: every limiter branch fires."""
    w = small_workload((16, 12, 1), (12, 8, 8), (0, 1, 0), seed_offset=5)
    p = Pair(torch_cuda, mphv, orc, w)
    rng = np.random.default_rng(99)
    f = rng.uniform(0.0, 1.0, size=w.shape) ** 6
    f[rng.uniform(size=w.shape) < 0.3] = 0.0
    for d, fn_o, fn_g, ax in [(0, "x", "x", AX_X[0]), (1, "x", "x", AX_X[1]),
                              (0, "v", "v", AX_V[0]), (1, "v", "v", AX_V[1]), (2, "v", "v", AX_V[2])]:
        p.set_f(f)
        if fn_o == "x":
            orc.sweep_x(p.f_ref, p.grid, p.box, d, p.dt * 1.5)
            p.sim.sweep_x(d, p.dt * 1.5)
        else:
            orc.sweep_v(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, d, p.dt * 1.5)
            p.sim.sweep_v(d, p.dt * 1.5)
        g = p.gpu()
        assert g.min() >= 0.0, "positivity lost on the GPU"
        assert rel_err(g, p.f_ref, ax) <= TOL_SWEEP
    # the same data through the fused V stage
    p.set_f(f)
    for d in range(3):
        orc.sweep_v(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, d, p.dt * 1.5)
    p.sim.set_fusion(True)
    # mphv_step would also do the spatial sweeps: use a zero-extent trick instead -- run the
    # oracle's spatial sweeps too and compare the whole step
    p.set_f(f)
    orc.step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, p.dt * 1.5)
    p.sim.step(p.dt * 1.5)
    g = p.gpu()
    assert g.min() >= 0.0
    assert rel_err(g, p.f_ref, AX_V[2]) <= TOL_SWEEP


@pytest.mark.parametrize("fusion", [0, 1, 2, 3])
def test_config0_landau_20_steps_and_moments(torch_cuda, mphv, orc, fusion):
    from paper_2305_01487_b200 import inputs
    w = inputs.config(0)
    p = Pair(torch_cuda, mphv, orc, w, fusion=fusion)
    for _ in range(w.steps):
        orc.step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, p.dt)
        p.sim.step(p.dt)
    g = p.gpu()
    assert rel_err(g, p.f_ref, AX_V[0]) <= w.steps * TOL_SWEEP
    m_ref, m_gpu = orc.total(p.f_ref), orc.total(g)
    assert abs(m_gpu - m_ref) <= TOL_MASS * abs(m_ref)
    assert abs(m_gpu - orc.total(p.f0)) <= TOL_MASS * abs(m_ref), "all-periodic grid: mass is conserved"
    check_moments(p, orc, g)


def check_moments(p, orc, g):
    n_r, j_r, P_r = orc.moments(p.f_ref, p.grid, p.box)
    n_g, j_g, P_g = (t.cpu().numpy() for t in p.sim.moments())
    w = p.w
    vx, vy, vz = (w.v_centres(d) for d in range(3))
    dV = w.dv(0) * w.dv(1) * w.dv(2)
    fa = np.abs(p.f_ref)
    V = [vx[None, None, None, None, None, :], vy[None, None, None, None, :, None], vz[None, None, None, :, None, None]]
    assert moments_err(n_g, n_r, fa.sum(axis=(3, 4, 5)) * dV) <= 1e-13
    for a in range(3):
        assert moments_err(j_g[a], j_r[a], (fa * np.abs(V[a])).sum(axis=(3, 4, 5)) * dV) <= 1e-13
    k = 0
    for a in range(3):
        for b in range(a, 3):
            assert moments_err(P_g[k], P_r[k], (fa * np.abs(V[a] * V[b])).sum(axis=(3, 4, 5)) * dV) <= 1e-13
            k += 1


@pytest.mark.parametrize("fusion", [0, 1, 2, 3])
def test_config1_harris_steps_and_moments(torch_cuda, mphv, orc, fusion):
    from paper_2305_01487_b200 import inputs
    w = inputs.config(1)
    p = Pair(torch_cuda, mphv, orc, w, fusion=fusion)
    nsteps = 3
    for s in range(nsteps):
        orc.step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, p.dt)
        p.sim.step(p.dt)
        if s == 0:
            assert rel_err(p.gpu(), p.f_ref, AX_V[2]) <= TOL_SWEEP, "single step must meet 1e-12"
    g = p.gpu()
    assert rel_err(g, p.f_ref, AX_V[2]) <= nsteps * TOL_SWEEP
    assert g.min() >= 0.0
    m_ref, m_gpu = orc.total(p.f_ref), orc.total(g)
    assert abs(m_gpu - m_ref) <= TOL_MASS * abs(m_ref)
    assert abs(p.sim.sum_f() - m_ref) <= TOL_MASS * abs(m_ref), "device-side sum"
    check_moments(p, orc, g)


SXY_SHAPES = [
    # nx, nv, bc : nvel % 16 == 0 (128-byte chunks) and nvel % 16 == 8 (64-byte chunks), every
    # combination of periodic / outflow on x and y, ragged thread counts, 3-D (S_z stays a march)
    ((12, 10, 1), (12, 10, 8), (0, 1, 0)),
    ((12, 10, 1), (12, 10, 8), (1, 0, 0)),
    ((16, 9, 1), (6, 4, 1), (0, 0, 0)),
    ((16, 9, 1), (6, 4, 1), (1, 1, 0)),
    ((8, 4, 1), (4, 4, 4), (0, 1, 0)),
    ((36, 8, 1), (40, 12, 6), (0, 1, 0)),
    ((8, 6, 4), (8, 6, 4), (0, 1, 0)),
    ((64, 7, 1), (8, 4, 4), (0, 1, 0)),
    ((128, 6, 1), (4, 4, 1), (0, 0, 0)),
    ((256, 5, 1), (4, 4, 1), (0, 1, 0)),     # nx = 256: 64-byte chunks, 512 threads
]


@pytest.mark.parametrize("nx,nv,bc", SXY_SHAPES)
@pytest.mark.parametrize("sign", [1.0, -1.0])
def test_stage_x_fused_matches_oracle_sweeps(torch_cuda, mphv, orc, nx, nv, bc, sign):
    """mphv_stage_x at fusion level 3 (S_x and S_y in one pass, sxy_kernel) against the oracle's
    S_x, S_y, S_z in order (R5), both signs of dt, CFL 0.85."""
    w = small_workload(nx, nv, bc)
    p = Pair(torch_cuda, mphv, orc, w, fusion=3)
    dt = sign * 1.7 * p.dt
    for rep in range(2):
        last = 0
        for d in range(3):
            if w.nx[d] > 1:
                orc.sweep_x(p.f_ref, p.grid, p.box, d, dt)
                last = d
        n0 = p.sim.launches
        p.sim.stage_x(dt)
        assert p.sim.launches - n0 == (2 if w.nx[2] > 1 else 1), "the fused kernel must be the one that ran"
        g = p.gpu()
        assert rel_err(g, p.f_ref, AX_X[last]) <= 2 * TOL_SWEEP, f"rep {rep}"
        assert rel_err(g, p.f_ref, AX_X[0]) <= 2 * TOL_SWEEP
        p.set_f(p.f_ref)


def test_stage_x_then_stage_v_is_step(torch_cuda, mphv, orc):
    """Strang pieces: stage_x(dt/2), stage_v(dt), stage_x(dt/2) against the oracle's sweeps."""
    w = small_workload((12, 8, 1), (8, 8, 8))
    for fusion in (0, 3):
        p = Pair(torch_cuda, mphv, orc, w, fusion=fusion)
        for d in (0, 1):
            orc.sweep_x(p.f_ref, p.grid, p.box, d, 0.5 * p.dt)
        for d in range(3):
            orc.sweep_v(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, d, p.dt)
        for d in (0, 1):
            orc.sweep_x(p.f_ref, p.grid, p.box, d, 0.5 * p.dt)
        p.sim.stage_x(0.5 * p.dt); p.sim.stage_v(p.dt); p.sim.stage_x(0.5 * p.dt)
        assert rel_err(p.gpu(), p.f_ref, AX_X[1]) <= 3 * TOL_SWEEP


def test_step_moments_equals_step_then_moments(torch_cuda, mphv, orc):
    w = small_workload((8, 8, 1), (12, 10, 8))
    p = Pair(torch_cuda, mphv, orc, w)
    orc.step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, p.dt)
    n_g, j_g, P_g = (t.cpu().numpy() for t in p.sim.step_moments(p.dt))
    g = p.gpu()
    assert rel_err(g, p.f_ref, AX_V[2]) <= TOL_SWEEP
    n_r, j_r, P_r = orc.moments(p.f_ref, p.grid, p.box)
    scale = np.abs(P_r[0]) + np.abs(P_r[3]) + np.abs(P_r[5]) + np.abs(n_r)
    for a, b in [(n_g, n_r), (j_g, j_r), (P_g, P_r)]:
        assert np.max(np.abs(a - b) / scale) <= 1e-12


def test_3d3v_step_all_six_sweeps(torch_cuda, mphv, orc):
    w = small_workload((8, 6, 8), (8, 8, 8), (0, 1, 0))
    p = Pair(torch_cuda, mphv, orc, w)
    for _ in range(2):
        orc.step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, p.dt)
        p.sim.step(p.dt)
    g = p.gpu()
    assert rel_err(g, p.f_ref, AX_V[2]) <= 2 * TOL_SWEEP
    check_moments(p, orc, g)


def test_integer_courant_is_bitwise_roll(torch_cuda, mphv, orc):
    """P1 on the GPU: dyadic dx, dv and dt = 2 dx / dv give odd-integer Courant numbers; the
    sweep must equal the index-rolled input bit for bit (whole-cell shift path, needs scratch)."""
    from paper_2305_01487_b200 import inputs
    w = inputs.Workload(name="p1", index=0, kind="harris2d", nx=(16, 8, 1), nv=(8, 4, 4), bc=(0, 0, 0),
                        xlo=(0.0, 0.0, 0.0), xhi=(16.0, 8.0, 1.0), vlo=(-2.0, -1.0, -1.0), vhi=(2.0, 1.0, 1.0))
    p = Pair(torch_cuda, mphv, orc, w, with_scratch=True)
    rng = np.random.default_rng(3)
    f = rng.uniform(0.0, 1.0, size=w.shape)
    p.set_f(f)
    dt = 2.0 * 1.0 / 0.5            # s_j = v_j dt / dx = (j + 1/2) 0.5 * 4 - 8 = odd integers
    p.sim.sweep_x(0, dt)
    g = p.gpu()
    vx = w.v_centres(0)
    for j, v in enumerate(vx):
        k = int(round(v * dt / 1.0))
        assert k % 2 != 0
        assert np.array_equal(g[..., j], np.roll(f[..., j], k, axis=2))
    # fractional + whole-cell shift against the oracle, |s| up to 3.6
    p.set_f(f)
    orc.sweep_x(p.f_ref, p.grid, p.box, 0, 0.9 * dt)
    p.sim.sweep_x(0, 0.9 * dt)
    assert rel_err(p.gpu(), p.f_ref, AX_X[0]) <= TOL_SWEEP
    # zero time step: identity, bitwise, on every in-place kernel
    p.set_f(f)
    for d in (0, 1):
        p.sim.sweep_x(d, 0.0)
    for d in (0, 1, 2):
        p.sim.sweep_v(d, 0.0)
    assert np.array_equal(p.gpu(), f)


def test_mirror_symmetry_on_gpu(torch_cuda, mphv, orc):
    """reverse(sweep(f, dt)) == sweep(reverse(f), -dt) along a periodic axis (<= 1e-12)."""
    w = small_workload((16, 8, 1), (8, 8, 4), (0, 0, 0))
    p = Pair(torch_cuda, mphv, orc, w)
    f = p.f0.copy()
    p.sim.sweep_x(0, p.dt)
    a = p.gpu()
    # mirror x and vx together: v -> -v, x -> -x leaves v dt/dx unchanged in sign convention
    p.set_f(f[:, :, ::-1])
    p.sim.sweep_x(0, -p.dt)
    b = p.gpu()[:, :, ::-1]
    assert rel_err(a, b, AX_X[0]) <= TOL_SWEEP


def test_error_codes_on_gpu(torch_cuda, mphv, orc):
    torch = torch_cuda
    w = small_workload((8, 8, 1), (8, 8, 8))
    sim = mphv.Vlasov.from_workload(w)
    with pytest.raises(mphv.MphvError) as ei:
        sim.step(0.1)
    assert ei.value.code == mphv.ERR_STATE
    f = torch.zeros(w.shape, dtype=torch.float64, device="cuda")
    sim.bind_f(f)
    with pytest.raises(mphv.MphvError) as ei:
        sim.sweep_v(0, 0.1)
    assert ei.value.code == mphv.ERR_STATE
    E = torch.zeros((3,) + w.space_shape, dtype=torch.float64, device="cuda")
    B = torch.ones((3,) + w.space_shape, dtype=torch.float64, device="cuda")
    sim.set_fields(E, B)
    f.fill_(1.0)
    for call, code in [(lambda: sim.sweep_x(2, 0.1), mphv.ERR_ARG), (lambda: sim.sweep_x(3, 0.1), mphv.ERR_ARG),
                       (lambda: sim.sweep_x(0, float("nan")), mphv.ERR_ARG),
                       (lambda: sim.sweep_x(1, 10.0), mphv.ERR_RANGE),      # outflow axis, |s| >= 1
                       (lambda: sim.sweep_x(0, 10.0), mphv.ERR_RANGE),      # periodic, no scratch
                       (lambda: sim.sweep_v(0, 10.0), mphv.ERR_RANGE),
                       (lambda: sim.step(10.0), mphv.ERR_RANGE)]:
        with pytest.raises(mphv.MphvError) as ei:
            call()
        assert ei.value.code == code
    torch.cuda.synchronize()
    assert bool((f == 1.0).all()), "a failed call leaves f untouched"
    # the RANGE decision is the oracle's: |s| < 1 accepted right up to the bound
    vmax = float(np.max(np.abs(w.v_centres(0))))
    amax = 2.0 * vmax                       # |v_a B_b - v_b B_a| with B = (1,1,1)
    dt_ok = 0.999 * w.dv(0) / amax
    sim.sweep_v(0, dt_ok)
    with pytest.raises(mphv.MphvError):
        sim.sweep_v(0, 1.001 * w.dv(0) / amax)


def test_run_host_roundtrip(torch_cuda, mphv, orc):
    torch = torch_cuda
    w = small_workload((8, 8, 1), (8, 8, 8))
    p = Pair(torch, mphv, orc, w)
    fh = torch.from_numpy(p.f0.copy()).pin_memory()
    nh = torch.empty(w.space_shape, dtype=torch.float64).pin_memory()
    jh = torch.empty((3,) + w.space_shape, dtype=torch.float64).pin_memory()
    Ph = torch.empty((6,) + w.space_shape, dtype=torch.float64).pin_memory()
    p.sim.run_host(fh, 2, p.dt, nh, jh, Ph)
    for _ in range(2):
        orc.step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, p.dt)
    assert rel_err(fh.numpy(), p.f_ref, AX_V[2]) <= 2 * TOL_SWEEP
    n_r, j_r, P_r = orc.moments(p.f_ref, p.grid, p.box)
    assert np.max(np.abs(nh.numpy() - n_r) / np.abs(n_r)) <= 1e-12
    assert np.max(np.abs(Ph.numpy()[0] - P_r[0]) / np.abs(P_r[0])) <= 1e-12


@pytest.mark.parametrize("fusion,vmode", [(3, 0), (1, 0), (3, 1)])
def test_step_is_bitwise_reproducible(torch_cuda, mphv, orc, fusion, vmode):
    """Race check by determinism (compute-sanitizer is not available on the GPU pool): the fused kernels
    recycle shared-memory ring slots and update f in place; a missing wait or barrier would show as
    run-to-run differences. Config 1 (33.5 M cells: every SM busy, many CTAs per SM over time)."""
    from paper_2305_01487_b200 import inputs
    w = inputs.config(1)
    p = Pair(torch_cuda, mphv, orc, w, fusion=fusion)
    p.sim.set_vmode(vmode)
    dt = 0.9 * p.dt
    results = []
    for _ in range(3):
        p.f_dev.copy_(torch_cuda.from_numpy(p.f0))
        for _ in range(2):
            n, j, P = p.sim.step_moments(dt)
        torch_cuda.cuda.synchronize()
        results.append((p.f_dev.clone(), n.clone(), P.clone()))
    for r in results[1:]:
        assert torch_cuda.equal(r[0], results[0][0]) and torch_cuda.equal(r[1], results[0][1]) and torch_cuda.equal(r[2], results[0][2])


@pytest.mark.parametrize("fusion", [0, 3])
def test_negative_input_follows_the_formulas_as_written(torch_cuda, mphv, orc, fusion):
    """Reading R12: f >= 0 is a precondition, but the formulas are applied as written otherwise (no
    clamping): data with negative entries must still agree with the oracle on every kernel path."""
    w = small_workload((12, 8, 1), (12, 8, 8), (0, 1, 0), seed_offset=6)
    p = Pair(torch_cuda, mphv, orc, w, fusion=fusion)
    rng = np.random.default_rng(98)
    f = rng.uniform(-0.3, 1.0, size=w.shape) ** 3
    f[rng.uniform(size=w.shape) < 0.2] = 0.0
    assert (f < 0).mean() > 0.1
    p.set_f(f)
    for _ in range(2):
        orc.step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, p.dt * 1.5)
        p.sim.step(p.dt * 1.5)
    assert rel_err(p.gpu(), p.f_ref, AX_V[2]) <= 2 * TOL_SWEEP
    p.set_f(f)
    p.sim.set_vmode(mphv.V_BACKSUB)
    orc.step_backsub(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, p.dt)
    p.sim.step(p.dt)
    assert rel_err(p.gpu(), p.f_ref, AX_V[2]) <= TOL_SWEEP


def test_step_fields_host_coupled_step(torch_cuda, mphv, orc):
    """mphv_step_fields_host: host fields in, f resident, host moments out = oracle step + moments."""
    torch = torch_cuda
    w = small_workload((12, 8, 1), (8, 8, 8))
    p = Pair(torch, mphv, orc, w)
    Eh, Bh = torch.from_numpy(p.E).pin_memory(), torch.from_numpy(p.B).pin_memory()
    nh = torch.empty(w.space_shape, dtype=torch.float64).pin_memory()
    jh = torch.empty((3,) + w.space_shape, dtype=torch.float64).pin_memory()
    Ph = torch.empty((6,) + w.space_shape, dtype=torch.float64).pin_memory()
    for _ in range(2):
        orc.step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, p.dt)
        p.sim.step_fields_host(Eh, Bh, p.dt, nh, jh, Ph)
    assert rel_err(p.gpu(), p.f_ref, AX_V[2]) <= 2 * TOL_SWEEP
    n_r, j_r, P_r = orc.moments(p.f_ref, p.grid, p.box)
    scale = np.abs(P_r[0]) + np.abs(P_r[3]) + np.abs(P_r[5]) + np.abs(n_r)
    for a, b in [(nh.numpy(), n_r), (jh.numpy(), j_r), (Ph.numpy(), P_r)]:
        assert np.max(np.abs(a - b) / scale) <= 1e-12
    # its RANGE check is the deferred one: fields a thousand times larger are reported when the call returns
    big = torch.from_numpy(1e3 * p.E).pin_memory()
    with pytest.raises(mphv.MphvError) as ei:
        p.sim.step_fields_host(big, Bh, p.dt, nh, jh, Ph)
    assert ei.value.code == mphv.ERR_RANGE


@pytest.mark.parametrize("vmode", [0, 1])
def test_electron_species_negative_charge_36cubed(torch_cuda, mphv, orc, vmode):
    """The paper's electron setup (m_i/m_e = 100, electron velocities in [-20, 20] v_A, 36^3 cells):
    q/m = -100 reverses every acceleration and the sense of gyration; same parity bar, both V-stage modes."""
    from paper_2305_01487_b200 import inputs
    w = inputs.variant(small_workload((8, 4, 1), (36, 36, 8), (0, 1, 0)), q_over_m=-100.0,
                       vlo=(-20.0,) * 3, vhi=(20.0,) * 3)
    p = Pair(torch_cuda, mphv, orc, w, fusion=3)
    p.sim.set_vmode(vmode)
    dt = 0.8 * p.dt
    step = orc.step_backsub if vmode else orc.step
    for _ in range(2):
        step(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, dt)
        n, j, P = p.sim.step_moments(dt)
    g = p.gpu()
    # sigma = 1 on a +-20 box: neighbouring cells differ by up to e^-20, along EVERY velocity axis. Each of the
    # three velocity sweeps leaves a rounding error proportional to ITS stencil's largest value, so the scale of
    # the parity metric is the maximum over the 5x5x5 velocity neighbourhood, not over the last-swept axis only.
    from parity_util import local_scale
    scale = np.abs(p.f_ref)
    for ax in (AX_V[0], AX_V[1], AX_V[2]):
        scale = local_scale(scale, ax)
    assert np.max(np.abs(g - p.f_ref) / np.maximum(scale, 1e-300)) <= 2 * TOL_SWEEP
    n_r, j_r, P_r = orc.moments(p.f_ref, p.grid, p.box)
    scale = np.abs(P_r[0]) + np.abs(P_r[3]) + np.abs(P_r[5]) + np.abs(n_r)
    assert np.max(np.abs(j.cpu().numpy() - j_r) / scale) <= 1e-12


@pytest.mark.parametrize("nvz", [40, 14, 12, 8, 4])
@pytest.mark.parametrize("gen", [2, 3, 4])
def test_every_generation_of_the_whole_v_stage_kernel_on_40x40_planes(torch_cuda, mphv, orc, gen, nvz):
    """vstage_kernel, vstage2_kernel and vstage3_kernel (the default) on the velocity planes of the headline config:
    the V stage with moments against the oracle's three sweeps, every cell. The generation is chosen with mphv_set_vstage_generation.
    nvz = 14 / 12: 7 / 6 plane pairs per cube, either side of where vstage3_kernel starts to finish a cube's moments
    without a barrier; 4: the shortest cube (first and last pair only). 19 x 8 spatial cells: CTAs with one cube and with two."""
    torch = torch_cuda
    w = small_workload((19 if nvz < 40 else 8, 8, 1), (40, 40, nvz))
    p = Pair(torch, mphv, orc, w, fusion=3)
    p.sim.set_vstage_generation(gen)
    mom = p.sim.alloc_moments()
    l0 = p.sim.launches
    p.sim.stage_v(p.dt, mom)
    assert p.sim.launches - l0 == 1, "one fused kernel"
    for d in range(3):
        orc.sweep_v(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, d, p.dt)
    assert max(rel_err(p.gpu(), p.f_ref, ax) for ax in (3, 4, 5)) <= TOL_SWEEP
    # every component on its own absolute-sum scale: this is the kernel of the headline config
    assert moments_worst(mom, orc.moments(p.f_ref, p.grid, p.box), moment_scales(p.f_ref, w)) <= 1e-12


def test_a_later_smaller_context_does_not_break_an_earlier_one(torch_cuda, mphv, orc):
    """Contexts share the generic kernel instances, whose dynamic shared-memory limit is a property of the KERNEL:
    creating a second context on a smaller velocity grid must not lower it for the first (regression: the launch of
    the first context's fused V stage failed with 'invalid argument' once a smaller grid had been created)."""
    big = Pair(torch_cuda, mphv, orc, small_workload((8, 4, 1), (24, 20, 12)), fusion=3)
    small = Pair(torch_cuda, mphv, orc, small_workload((8, 4, 1), (12, 12, 8)), fusion=3)
    for p in (big, small, big):
        orc.step(p.f_ref, p.grid, p.box, p.w.q_over_m, p.E, p.B, p.dt)
        p.sim.step(p.dt)
    assert rel_err(big.gpu(), big.f_ref, AX_V[2]) <= 2 * TOL_SWEEP
    assert rel_err(small.gpu(), small.f_ref, AX_V[2]) <= TOL_SWEEP
