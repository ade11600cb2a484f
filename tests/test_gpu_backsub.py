"""GPU parity of the backsubstituted V stage (mphv_set_vmode(MPHV_V_BACKSUB), reading R15)
against the oracle's orc_sweep_v_backsub / orc_step_backsub, element by element, through the C ABI."""
import numpy as np
import pytest

from parity_util import rel_err, TOL_SWEEP, TOL_MASS
from test_gpu_parity import Pair, small_workload, AX_V, check_moments, torch_cuda, mphv  # noqa: F401

pytestmark = pytest.mark.gpu

SHAPES = [
    ((4, 4, 1), (12, 10, 8), (0, 1, 0)),     # even inner (double2 path), nvx % 4 == 0
    ((4, 1, 4), (9, 7, 5), (1, 0, 0)),       # odd extents: scalar paths everywhere
    ((4, 4, 1), (40, 12, 6), (0, 1, 0)),
    ((4, 5, 1), (6, 4, 4), (0, 0, 0)),       # nvx % 4 == 2
    ((4, 1, 1), (32, 32, 8), (0, 1, 0)),
]


@pytest.mark.parametrize("nx,nv,bc", SHAPES)
@pytest.mark.parametrize("sign", [1.0, -1.0])
def test_each_backsub_sweep_matches_oracle(torch_cuda, mphv, orc, nx, nv, bc, sign):
    w = small_workload(nx, nv, bc)
    p = Pair(torch_cuda, mphv, orc, w)
    p.sim.set_vmode(mphv.V_BACKSUB)
    dt = sign * 1.5 * p.dt
    for d in range(3):
        orc.sweep_v_backsub(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, d, dt)
        p.sim.sweep_v(d, dt)
        err = rel_err(p.gpu(), p.f_ref, AX_V[d])
        assert err <= TOL_SWEEP, f"backsub sweep_v({d}) err {err:.3e}"
        p.set_f(p.f_ref)


@pytest.mark.parametrize("nx,nv,bc", SHAPES)
@pytest.mark.parametrize("fusion", [0, 3])
def test_step_moments_backsub_matches_oracle(torch_cuda, mphv, orc, nx, nv, bc, fusion):
    w = small_workload(nx, nv, bc)
    p = Pair(torch_cuda, mphv, orc, w, fusion=fusion)
    p.sim.set_vmode(mphv.V_BACKSUB)
    dt = 1.4 * p.dt
    out = None
    for _ in range(2):
        orc.step_backsub(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, dt)
        out = p.sim.step_moments(dt)
    g = p.gpu()
    assert rel_err(g, p.f_ref, AX_V[2]) <= 2 * TOL_SWEEP
    n_r, j_r, P_r = orc.moments(p.f_ref, p.grid, p.box)
    n_g, j_g, P_g = (t.cpu().numpy() for t in out)
    scale = np.abs(P_r[0]) + np.abs(P_r[3]) + np.abs(P_r[5]) + np.abs(n_r)
    for a, b in [(n_g, n_r), (j_g, j_r), (P_g, P_r)]:
        assert np.max(np.abs(a - b) / scale) <= 1e-12


def test_config1_backsub_steps_mass_positivity(torch_cuda, mphv, orc):
    from paper_2305_01487_b200 import inputs
    w = inputs.config(1)
    p = Pair(torch_cuda, mphv, orc, w, fusion=3)
    p.sim.set_vmode(mphv.V_BACKSUB)
    dt = 0.9 * p.dt
    for s in range(2):
        orc.step_backsub(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, dt)
        p.sim.step(dt)
    g = p.gpu()
    assert rel_err(g, p.f_ref, AX_V[2]) <= 2 * TOL_SWEEP
    assert g.min() >= 0.0
    m_ref = orc.total(p.f_ref)
    assert abs(orc.total(g) - m_ref) <= TOL_MASS * abs(m_ref)
    check_moments(p, orc, g)


def test_backsub_differs_from_plain_and_plain_is_restored(torch_cuda, mphv, orc):
    w = small_workload((4, 4, 1), (12, 12, 8))
    p = Pair(torch_cuda, mphv, orc, w)
    p.sim.set_vmode(mphv.V_BACKSUB)
    p.sim.stage_v(p.dt)
    a = p.gpu().copy()
    p.set_f(p.f0)
    p.sim.set_vmode(mphv.V_PLAIN)
    p.sim.stage_v(p.dt)
    b = p.gpu()
    for d in range(3):
        orc.sweep_v(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, d, p.dt)
    assert rel_err(b, p.f_ref, AX_V[2]) <= TOL_SWEEP
    assert np.max(np.abs(a - b)) > 1e-6 * np.max(np.abs(b)), "the two modes must differ when B != 0"


def test_backsub_errors(torch_cuda, mphv, orc):
    w = small_workload((4, 4, 1), (8, 8, 8))
    p = Pair(torch_cuda, mphv, orc, w)
    with pytest.raises(mphv.MphvError) as e:
        mphv.mphv_set_vmode(p.sim.ctx, 7)
    assert e.value.code == mphv.ERR_ARG
    p.sim.set_vmode(mphv.V_BACKSUB)
    before = p.gpu().copy()
    with pytest.raises(mphv.MphvError) as e:
        p.sim.sweep_v(1, 500.0 * p.dt)           # |s_face| >= 1 (B is mostly along x: vy, vz rotate)
    assert e.value.code == mphv.ERR_RANGE
    with pytest.raises(mphv.MphvError) as e:
        p.sim.step(500.0 * p.dt)
    assert e.value.code == mphv.ERR_RANGE
    assert np.array_equal(p.gpu(), before), "a failed call leaves f untouched"
    # 2V grid: backsubstitution needs all three velocity dimensions
    w2 = small_workload((4, 4, 1), (8, 8, 1))
    sim2 = mphv.Vlasov.from_workload(w2)
    with pytest.raises(mphv.MphvError) as e:
        sim2.set_vmode(mphv.V_BACKSUB)
    assert e.value.code == mphv.ERR_ARG


def test_fused_backsub_kernel_is_the_one_that_runs(torch_cuda, mphv, orc):
    """At fusion level >= 2 the backsubstituted V stage is ONE kernel (vstage_bs_kernel) where the grid allows:
    stage_v = 1 launch (after the first call with this dt, which also runs the coefficient kernel)."""
    w = small_workload((4, 4, 1), (32, 32, 8), (0, 1, 0))
    p = Pair(torch_cuda, mphv, orc, w, fusion=3)
    p.sim.set_vmode(mphv.V_BACKSUB)
    p.sim.stage_v(p.dt)
    n0 = p.sim.launches
    mom = p.sim.alloc_moments()
    p.sim.stage_v(p.dt, mom)
    assert p.sim.launches - n0 == 1
    for _ in range(2):
        for d in range(3):
            orc.sweep_v_backsub(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, d, p.dt)
    assert rel_err(p.gpu(), p.f_ref, AX_V[2]) <= 2 * TOL_SWEEP
    p.sim.set_fusion(0)
    n0 = p.sim.launches
    p.sim.stage_v(p.dt, mom)
    assert p.sim.launches - n0 == 4, "three sweep kernels and the moments"


@pytest.mark.parametrize("nvz", [40, 12, 4])
@pytest.mark.parametrize("gen", [3, 4])
def test_backsub_whole_v_stage_kernels_on_40x40_planes(torch_cuda, mphv, orc, gen, nvz):
    """The velocity planes of the headline config in backsubstitution mode: vstage3_bs_kernel (warp-specialised, the
    default there) and vstage_bs_kernel (mphv_set_vstage_generation(3)) against the oracle's three backsubstituted sweeps, every
    cell, with the moments; long cubes, short cubes (moments finished behind a barrier) and the shortest."""
    w = small_workload((19 if nvz < 40 else 8, 8, 1), (40, 40, nvz))
    p = Pair(torch_cuda, mphv, orc, w, fusion=3)
    p.sim.set_vstage_generation(gen)
    p.sim.set_vmode(mphv.V_BACKSUB)
    mom = p.sim.alloc_moments()
    dt = 1.4 * p.dt
    p.sim.stage_v(dt, mom)
    l0 = p.sim.launches
    p.sim.stage_v(dt, mom)
    assert p.sim.launches - l0 == 1, "one fused kernel"
    for _ in range(2):
        for d in range(3):
            orc.sweep_v_backsub(p.f_ref, p.grid, p.box, w.q_over_m, p.E, p.B, d, dt)
    assert max(rel_err(p.gpu(), p.f_ref, ax) for ax in (3, 4, 5)) <= 2 * TOL_SWEEP
    n_r, j_r, P_r = orc.moments(p.f_ref, p.grid, p.box)
    sc = np.abs(P_r[0]) + np.abs(P_r[3]) + np.abs(P_r[5]) + np.abs(n_r)
    for a_g, a_r in zip(mom, (n_r, j_r, P_r)):
        assert np.max(np.abs(a_g.cpu().numpy() - a_r) / sc) <= 1e-12
