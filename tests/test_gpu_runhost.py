"""mphv_run_host (host buffers in, host buffers out) on grids large enough for its slab pipeline (copy in, sweeps
and copy out overlapped slab by slab along the outermost spatial axis): every cell and the moments against the
oracle, for an outflow slab axis (2D3V), a periodic one (3D3V: slab 0 goes last) and several steps per call."""
import numpy as np
import pytest

from parity_util import TOL_SWEEP, moments_err, rel_err

pytestmark = pytest.mark.gpu


def _run(orc, w, nsteps, dt_scale=1.0, with_scratch=False):
    import torch
    from paper_2305_01487_b200 import inputs, mphv
    f0, E, B, dt = inputs.make_all(w)
    dt *= dt_scale
    assert f0.nbytes >= 16 << 20, "below the pipeline's size threshold: the test would not test it"
    sim = mphv.Vlasov.from_workload(w)
    f = torch.empty(w.shape, dtype=torch.float64, device="cuda")
    sim.bind_f(f, torch.empty_like(f) if with_scratch else None)
    sim.set_fields(torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
    fh = torch.from_numpy(f0.copy()).pin_memory()
    nh = torch.empty(w.space_shape, dtype=torch.float64).pin_memory()
    jh = torch.empty((3,) + w.space_shape, dtype=torch.float64).pin_memory()
    Ph = torch.empty((6,) + w.space_shape, dtype=torch.float64).pin_memory()
    sim.run_host(fh, nsteps, dt, nh, jh, Ph)
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    ref = f0
    for _ in range(nsteps):
        orc.step(ref, grid, box, w.q_over_m, E, B, dt)
    n_r, j_r, P_r = orc.moments(ref, grid, box)
    got = fh.numpy()
    assert max(rel_err(got, ref, ax) for ax in (3, 4, 5)) <= nsteps * TOL_SWEEP
    assert abs(orc.total(got) - orc.total(ref)) <= 1e-13 * orc.total(ref)
    assert np.array_equal(f.cpu().numpy(), got)                        # the device copy is the same state
    absf = np.abs(ref)
    n_a, j_a, P_a = orc.moments(absf, grid, box)
    v = [np.abs(w.v_centres(d)).max() for d in range(3)]
    assert moments_err(nh.numpy(), n_r, n_a) <= 1e-12
    for a in range(3):
        assert moments_err(jh.numpy()[a], j_r[a], v[a] * n_a) <= 1e-12
    for k, (a, b) in enumerate([(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]):
        assert moments_err(Ph.numpy()[k], P_r[k], v[a] * v[b] * n_a) <= 1e-12


@pytest.mark.parametrize("nsteps", [1, 3])
def test_run_host_pipeline_2d_outflow_slab_axis(orc, nsteps):
    from paper_2305_01487_b200 import inputs
    _run(orc, inputs.harris2d(32, 16, 16, name="runhost2d"), nsteps)


def test_run_host_pipeline_2d_periodic_slab_axis(orc):
    from paper_2305_01487_b200 import inputs
    _run(orc, inputs.harris2d(32, 16, 16, bc_y=inputs.PERIODIC, name="runhost2d_periodic"), 2)


def test_run_host_pipeline_3d(orc):
    from paper_2305_01487_b200 import inputs
    _run(orc, inputs.harris3d(16, 8, name="runhost3d"), 2)


def test_run_host_ragged_slabs(orc):
    """ny = 22 over 5 slabs: slabs of 4 and 5 rows."""
    from paper_2305_01487_b200 import inputs
    _run(orc, inputs.harris2d(32, 22, 16, name="runhost2d_ragged"), 1)


def test_run_host_whole_cell_shift_on_a_lower_periodic_axis(orc):
    """|s| >= 1 along periodic x (the parent context has a scratch buffer, so mphv_step accepts it) on a grid above
    the pipeline's size threshold: the slabs have no scratch of their own, so this call must take the plain path
    (it used to run the whole-cell shift of a slab through a NULL scratch pointer)."""
    from paper_2305_01487_b200 import inputs
    w = inputs.harris2d(256, 12, 16, name="runhost2d_shift")
    _, E, B, dt = inputs.make_all(w)
    scale = 2.5
    assert np.abs(w.v_centres(0)).max() * dt * scale / w.dx(0) >= 1.0, "the test needs a whole-cell shift along x"
    assert np.abs(w.v_centres(1)).max() * dt * scale / w.dx(1) < 1.0
    _run(orc, w, 2, dt_scale=scale, with_scratch=True)
