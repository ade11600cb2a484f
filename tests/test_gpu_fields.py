"""GPU parity of the field solver and of the coupled multi-species step (include/mphv.h "closing the loop",
readings R19..R22) against the CPU oracle (oracle/mphv_fields_oracle.c, oracle/fields.py), through the C ABI.
Fields: |delta| <= 1e-12 x the largest field value (the kernels multiply by 1/dx and use FMA where the oracle
divides and rounds every product). f: the metric of parity_util. Run with ``-m gpu`` on a B200."""
import numpy as np
import pytest

from parity_util import TOL_SWEEP, rel_err

pytestmark = pytest.mark.gpu
PER, OUT = 0, 1
TOL_FIELD = 1e-12


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "these tests need a GPU"
    return t


@pytest.fixture(scope="module")
def mphv():
    from paper_2305_01487_b200 import mphv as m
    m.lib()
    return m


def _rand(shape, seed):
    return np.random.default_rng(seed).standard_normal(shape)


def _close(got, ref, scale=None):
    scale = np.abs(ref).max() if scale is None else scale
    return float(np.abs(got - ref).max()) <= TOL_FIELD * scale


GRIDS = [((16, 1, 1), (PER, PER, PER)), ((12, 10, 1), (PER, OUT, PER)), ((8, 6, 10), (PER, OUT, PER)),
         ((5, 7, 9), (OUT, OUT, OUT)), ((48, 48, 32), (PER, OUT, PER))]          # the last one: > 65536 cells (per-phase launches)


@pytest.mark.parametrize("nx,bc", GRIDS)
def test_field_kernels_match_the_oracle(torch, mphv, orc, nx, bc):
    fld = orc.fields
    dx = (0.3, 0.45, 0.2)
    g = fld.FieldGrid(nx, bc, dx, c2=2.89, inv_eps0=1.7)
    E, B, J = _rand(g.shape, 1), _rand(g.shape, 2), _rand(g.shape, 3)
    mx = mphv.Maxwell(nx, bc, dx, c2=2.89, inv_eps0=1.7)
    Ed, Bd, Jd = (torch.from_numpy(a).cuda() for a in (E, B, J))
    mx.bind(Ed, Bd)
    dt = 0.05
    # single phases
    mx.faraday(dt); fld.faraday(g, E, B, dt)
    assert _close(Bd.cpu().numpy(), B, max(np.abs(B).max(), dt * np.abs(E).max() / min(dx)))
    mx.ampere(Jd, dt); fld.ampere(g, E, B, J, dt)
    assert _close(Ed.cpu().numpy(), E, max(np.abs(E).max(), dt * 2.89 * np.abs(B).max() / min(dx)))
    mx.ampere(None, dt); fld.ampere(g, E, B, None, dt)
    assert _close(Ed.cpu().numpy(), E, max(np.abs(E).max(), dt * 2.89 * np.abs(B).max() / min(dx)))
    # the whole Maxwell step, several times
    for _ in range(5):
        mx.step(Jd, dt); fld.maxwell_step(g, E, B, J, dt)
    scale = max(np.abs(E).max(), np.abs(B).max()) * (1 + 5 * dt * 2.89 / min(dx))
    assert _close(Ed.cpu().numpy(), E, scale) and _close(Bd.cpu().numpy(), B, scale)
    # centring and charge current
    Ec, Bc = mx.centre()
    Ec_r, Bc_r = fld.to_centres(g, E, B)
    assert _close(Ec.cpu().numpy(), Ec_r) and _close(Bc.cpu().numpy(), Bc_r)
    js = [_rand(g.shape, 10 + s) for s in range(3)]
    q = [-1.0, 1.0, 2.5]
    Jsum = mx.current(q, [torch.from_numpy(j).cuda() for j in js])
    assert _close(Jsum.cpu().numpy(), fld.charge_current(g, q, js))


def test_divB_stays_zero_on_the_gpu(torch, mphv, orc):
    fld = orc.fields
    nx, bc, dx = (16, 12, 8), (PER, PER, PER), (0.3, 0.45, 0.2)
    g = fld.FieldGrid(nx, bc, dx, c2=1.0)
    E, B = _rand(g.shape, 5), np.zeros(g.shape)
    mx = mphv.Maxwell(nx, bc, dx)
    Ed, Bd = torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()
    mx.bind(Ed, Bd)
    for _ in range(20):
        mx.step(None, 0.05)
    Bn = Bd.cpu().numpy()
    assert np.abs(Bn).max() > 0.1
    assert np.abs(fld.div_B(g, Bn)).max() <= 1e-12 * np.abs(Bn).max() / min(dx)


def _two_species(orc, nx, ny, nvi, nve, mass_ratio):
    from paper_2305_01487_b200 import inputs
    wi = inputs.harris2d(nx, ny, nvi, name="ions")
    we = inputs.electrons_of(wi, mass_ratio=mass_ratio, temp_ratio=0.25, nv=nve, vmax=5.0 * np.sqrt(mass_ratio * 0.25))
    E, B = inputs.yee_fields(wi)
    fi, fe = inputs.make_f0(wi), inputs.make_f0(we)
    # a time step inside every sweep's |s| < 1: both species, fields up to twice their initial size
    dt = 0.5 * min(inputs.cfl_dt(wi, 2 * E, 2 * B), inputs.cfl_dt(we, 2 * E, 2 * B))
    return wi, we, fi, fe, E, B, dt


@pytest.mark.parametrize("concurrent", [False, True])
def test_coupled_two_species_step_matches_the_oracle(torch, mphv, orc, concurrent):
    """Ions + electrons (m_i/m_e = 16) + Maxwell on a small 2D3V Harris sheet: 3 coupled steps R22, every cell of
    both distribution functions, E, B and the species' moments against the oracle's coupled_step."""
    fld = orc.fields
    wi, we, fi, fe, E, B, dt = _two_species(orc, 16, 8, 16, 20, 16.0)
    c2, inv_eps0 = 100.0, 1.0
    g = fld.FieldGrid(wi.nx, wi.bc, tuple(wi.dx(d) if wi.nx[d] > 1 else 1.0 for d in range(3)), c2, inv_eps0)
    sims, fdev = [], []
    for w, f0 in ((wi, fi), (we, fe)):
        s = mphv.Vlasov.from_workload(w)
        fd = torch.from_numpy(f0).cuda()
        s.bind_f(fd)
        sims.append(s); fdev.append(fd)
    mx = mphv.Maxwell.from_workload(wi, c2, inv_eps0)
    Ed, Bd = torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()
    mx.bind(Ed, Bd)
    q = [1.0, -1.0]
    pl = mphv.Plasma(mx, sims, q)
    pl.set_concurrent(concurrent)
    species = [fld.Species(f0.copy(), orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi), qq, w.q_over_m)
               for (w, f0), qq in zip(((wi, fi), (we, fe)), q)]
    Er, Br = E.copy(), B.copy()
    j_now, nsteps = None, 3
    for k in range(nsteps):
        moms = fld.coupled_step(g, species, Er, Br, dt, j_now)
        j_now = [m[1] for m in moms]
    pl.step(dt, 2)
    pl.step(dt, nsteps - 2)                       # a second call continues from the kept moments
    pl.sync()
    for s, sp in enumerate(species):
        got = fdev[s].cpu().numpy()
        err = max(rel_err(got, sp.f, ax) for ax in (3, 4, 5))
        assert err <= nsteps * TOL_SWEEP, (s, err)
        n, j, P = pl.moments(s)
        assert np.abs(n.cpu().numpy() - moms[s][0]).max() <= 1e-12 * np.abs(moms[s][0]).max()
        jscale = np.abs(moms[s][2][[0, 3, 5]]).max() ** 0.5 * np.abs(moms[s][0]).max() ** 0.5
        assert np.abs(j.cpu().numpy() - moms[s][1]).max() <= 1e-12 * jscale
    fscale = max(np.abs(Er).max(), np.abs(Br).max()) * max(1.0, c2 * dt / min(g.dx[:2]))
    assert np.abs(Ed.cpu().numpy() - Er).max() <= nsteps * 1e-12 * fscale
    assert np.abs(Bd.cpu().numpy() - Br).max() <= nsteps * 1e-12 * fscale
    Ec, Bc = pl.centred_fields()
    assert Ec.shape == tuple(g.shape) and bool(torch.isfinite(Ec).all()) and bool(torch.isfinite(Bc).all())


def test_concurrent_and_serial_runs_agree_bitwise(torch, mphv, orc):
    wi, we, fi, fe, E, B, dt = _two_species(orc, 16, 8, 16, 20, 16.0)
    out = []
    for concurrent in (False, True):
        sims, fdev = [], []
        for w, f0 in ((wi, fi), (we, fe)):
            s = mphv.Vlasov.from_workload(w)
            fd = torch.from_numpy(f0).cuda()
            s.bind_f(fd)
            sims.append(s); fdev.append(fd)
        mx = mphv.Maxwell.from_workload(wi, 100.0, 1.0)
        Ed, Bd = torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()
        mx.bind(Ed, Bd)
        pl = mphv.Plasma(mx, sims, [1.0, -1.0])
        pl.set_concurrent(concurrent)
        pl.step(dt, 4)
        pl.sync()
        out.append([t.cpu().numpy() for t in (*fdev, Ed, Bd)])
        pl.close()
    for a, b in zip(*out):
        assert np.array_equal(a, b)


def test_deferred_range_check_reports_at_the_next_query(torch, mphv, orc):
    from paper_2305_01487_b200 import inputs
    w = inputs.harris2d(8, 8, 16)
    f0, E, B, dt = inputs.make_all(w)
    sim = mphv.Vlasov.from_workload(w)
    f = torch.from_numpy(f0).cuda()
    sim.bind_f(f)
    Ed, Bd = torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()
    sim.set_fields_deferred(Ed, Bd)
    sim.step(dt)
    sim.deferred_status()                                          # in range: no error
    ref = f0.copy()
    orc.step(ref, orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi), w.q_over_m, E, B, dt)
    assert max(rel_err(f.cpu().numpy(), ref, ax) for ax in (3, 4, 5)) <= TOL_SWEEP
    big = torch.from_numpy(1e3 * E).cuda()
    sim.set_fields_deferred(big, Bd)
    sim.step(dt)                                                   # enqueues; the check runs on the device
    with pytest.raises(mphv.MphvError) as ei:
        sim.deferred_status()
    assert ei.value.code == mphv.ERR_RANGE
    sim.deferred_status()                                          # the flag was cleared by the query
    sim.step(dt)                                                   # flag raised again, context still deferred ...
    fh = torch.from_numpy(f0.copy()).pin_memory()
    with pytest.raises(mphv.MphvError) as ei:                      # ... and mphv_run_host reports it when it ends
        sim.run_host(fh, 1, dt)
    assert ei.value.code == mphv.ERR_RANGE
    sim.set_fields(big, Bd)                                        # back to the immediate check
    with pytest.raises(mphv.MphvError) as ei:
        sim.step(dt)
    assert ei.value.code == mphv.ERR_RANGE


def test_landau_damping_on_the_gpu(torch, mphv):
    """Physics through the whole CUDA chain (sweeps -> fused moments -> current -> Ampere -> centring -> deferred
    set_fields -> sweeps), no oracle involved: the k = 0.5 Langmuir mode of a Maxwellian electron plasma decays
    at gamma = -0.1533 and oscillates at w = 1.4156 (roots of the kinetic dispersion relation)."""
    k, alpha = 0.5, 0.01
    nx, nv, vmax = 64, 128, 6.0
    L = 2 * np.pi / k
    dx = L / nx
    x = (np.arange(nx) + 0.5) * dx
    v = -vmax + (np.arange(nv) + 0.5) * (2 * vmax / nv)
    f0 = ((1 + alpha * np.cos(k * x))[:, None] * np.exp(-0.5 * v ** 2)[None, :] / np.sqrt(2 * np.pi)).reshape(1, 1, nx, 1, 1, nv).copy()
    sim = mphv.Vlasov((nx, 1, 1), (nv, 1, 1), (PER, PER, PER), (0.0, 0.0, 0.0), (L, 1.0, 1.0), (-vmax, 0.0, 0.0), (vmax, 1.0, 1.0), q_over_m=-1.0)
    f = torch.from_numpy(f0).cuda()
    sim.bind_f(f)
    n0 = sim.moments()[0].reshape(nx).cpu().numpy()
    rho = n0.mean() - n0
    Ex = np.cumsum(rho) * dx
    Ex -= Ex.mean()
    E = np.zeros((3, 1, 1, nx)); E[0, 0, 0] = Ex
    mx = mphv.Maxwell((nx, 1, 1), (PER, PER, PER), (dx, 1.0, 1.0))
    Ed, Bd = torch.from_numpy(E).cuda(), torch.zeros((3, 1, 1, nx), dtype=torch.float64, device="cuda")
    mx.bind(Ed, Bd)
    pl = mphv.Plasma(mx, [sim], [-1.0])
    dt = 0.5 * dx / vmax
    every = 4
    nrec = int(round(30.0 / (every * dt)))
    phase = torch.from_numpy(np.exp(-1j * k * (np.arange(nx) + 1.0) * dx)).cuda()
    amp = []
    for _ in range(nrec):
        pl.step(dt, every)
        pl.sync()
        amp.append(2.0 * abs(complex((Ed[0, 0, 0] * phase).mean().item())))
    amp = np.array(amp)
    times = every * dt * (1 + np.arange(nrec))
    pk = [i for i in range(1, nrec - 1) if amp[i] > amp[i - 1] and amp[i] >= amp[i + 1] and times[i] > 2.0]
    assert len(pk) >= 10
    tp, ap = [], []
    for i in pk:
        y0, y1, y2 = np.log(amp[i - 1]), np.log(amp[i]), np.log(amp[i + 1])
        d = 0.5 * (y0 - y2) / (y0 - 2 * y1 + y2)
        tp.append(times[i] + d * every * dt)
        ap.append(y1 - 0.25 * (y0 - y2) * d)
    gamma = np.polyfit(np.array(tp), np.array(ap), 1)[0]
    omega = np.pi / np.mean(np.diff(tp))
    assert abs(omega - 1.4156) < 0.005 * 1.4156, omega
    assert abs(gamma + 0.1533) < 0.03 * 0.1533, gamma


def test_light_wave_in_a_plasma_on_the_gpu(torch, mphv):
    """GPU twin of the oracle pin F8 (no oracle involved): a transverse wave E_y = A cos kx in a cold-ish electron
    plasma, 1D2V, through mphv_plasma_step: w^2 = w_p^2 + c^2 K^2, K = (2/dx) sin(k dx/2), neither growing nor damped.
    Faraday's law, the curl B term, the transverse current j_y and the 2V velocity sweeps (fallback kernels) in the loop."""
    k, c, A, sg = 1.0, 1.0, 0.01, 0.05
    nx, nv, vmax = 32, 24, 0.3
    L = 2 * np.pi / k
    dx = L / nx
    v = -vmax + (np.arange(nv) + 0.5) * (2 * vmax / nv)
    gauss = np.exp(-0.5 * (v / sg) ** 2) / (np.sqrt(2 * np.pi) * sg)
    f0 = np.ascontiguousarray(np.broadcast_to((gauss[:, None] * gauss[None, :])[None, None, None, None], (1, 1, nx, 1, nv, nv))).copy()
    sim = mphv.Vlasov((nx, 1, 1), (nv, nv, 1), (PER, PER, PER), (0.0, 0.0, 0.0), (L, 1.0, 1.0), (-vmax, -vmax, 0.0), (vmax, vmax, 1.0), q_over_m=-1.0)
    f = torch.from_numpy(f0).cuda()
    sim.bind_f(f)
    wp2 = float(sim.moments()[0].mean())
    x = (np.arange(nx) + 0.5) * dx
    E = np.zeros((3, 1, 1, nx)); E[1, 0, 0] = A * np.cos(k * x)
    mx = mphv.Maxwell((nx, 1, 1), (PER, PER, PER), (dx, 1.0, 1.0), c2=c * c)
    Ed, Bd = torch.from_numpy(E).cuda(), torch.zeros((3, 1, 1, nx), dtype=torch.float64, device="cuda")
    mx.bind(Ed, Bd)
    pl = mphv.Plasma(mx, [sim], [-1.0])
    dt, steps = 0.05, 400
    mode = torch.from_numpy(np.cos(k * x)).cuda()
    amp = []
    for _ in range(steps):
        pl.step(dt, 1)
        amp.append(2.0 * float((Ed[1, 0, 0] * mode).mean()))
    pl.sync()
    amp = np.array(amp)
    t = dt * (1 + np.arange(steps))
    assert np.abs(amp).max() < 1.02 * A and np.abs(amp[-80:]).max() > 0.9 * A
    zc = [t[i] - amp[i] * dt / (amp[i + 1] - amp[i]) for i in range(steps - 1) if amp[i] * amp[i + 1] < 0]
    assert len(zc) >= 8
    omega = np.pi / np.mean(np.diff(zc))
    K = 2.0 / dx * np.sin(0.5 * k * dx)
    want = np.sqrt(wp2 + c * c * K * K)
    assert abs(omega - want) < 0.005 * want, (omega, want)
    assert float(Ed[0].abs().max()) < 1e-3 * A


def test_three_species_on_different_velocity_grids(torch, mphv, orc):
    """Ions, electrons and a light positive third species, each on its own velocity grid (16^3, 20^3, 12^3), coupled
    through Maxwell: 2 steps of R22 against the oracle (every cell of every f, the fields)."""
    from paper_2305_01487_b200 import inputs
    fld = orc.fields
    wi, we, fi, fe, E, B, dt = _two_species(orc, 16, 8, 16, 20, 16.0)
    wp = inputs.variant(inputs.electrons_of(wi, mass_ratio=4.0, temp_ratio=0.5, nv=12, vmax=7.0), q_over_m=4.0, seed_offset=900)
    fp = 0.1 * inputs.make_f0(wp)
    dt = min(dt, 0.5 * inputs.cfl_dt(wp, 2 * E, 2 * B))
    c2 = 64.0
    g = fld.FieldGrid(wi.nx, wi.bc, tuple(wi.dx(d) if wi.nx[d] > 1 else 1.0 for d in range(3)), c2, 1.0)
    ws, f0s, q = (wi, we, wp), (fi, fe, fp), [1.0, -1.0, 1.0]
    sims, fdev = [], []
    for w, f0 in zip(ws, f0s):
        s = mphv.Vlasov.from_workload(w)
        fd = torch.from_numpy(f0).cuda()
        s.bind_f(fd)
        sims.append(s); fdev.append(fd)
    mx = mphv.Maxwell.from_workload(wi, c2, 1.0)
    Ed, Bd = torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()
    mx.bind(Ed, Bd)
    pl = mphv.Plasma(mx, sims, q)
    species = [fld.Species(f0.copy(), orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi), qq, w.q_over_m)
               for w, f0, qq in zip(ws, f0s, q)]
    Er, Br = E.copy(), B.copy()
    j_now = None
    for _ in range(2):
        moms = fld.coupled_step(g, species, Er, Br, dt, j_now)
        j_now = [m[1] for m in moms]
    pl.step(dt, 2)
    pl.sync()
    for s, sp in enumerate(species):
        assert max(rel_err(fdev[s].cpu().numpy(), sp.f, ax) for ax in (3, 4, 5)) <= 2 * TOL_SWEEP, s
    fscale = max(np.abs(Er).max(), np.abs(Br).max()) * max(1.0, c2 * dt / min(g.dx[:2]))
    assert np.abs(Ed.cpu().numpy() - Er).max() <= 2e-12 * fscale and np.abs(Bd.cpu().numpy() - Br).max() <= 2e-12 * fscale


def _small_plasma(torch, mphv, orc, c2=64.0):
    fld = orc.fields
    wi, we, fi, fe, E, B, dt = _two_species(orc, 16, 8, 16, 20, 16.0)
    sims, fdev = [], []
    for w, f0 in ((wi, fi), (we, fe)):
        s = mphv.Vlasov.from_workload(w)
        fd = torch.from_numpy(f0).cuda()
        s.bind_f(fd)
        sims.append(s); fdev.append(fd)
    mx = mphv.Maxwell.from_workload(wi, c2, 1.0)
    Ed, Bd = torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()
    mx.bind(Ed, Bd)
    return sims, fdev, mx, Ed, Bd, dt, (wi, we, fi, fe, E, B)


def test_destroying_the_plasma_unbinds_its_field_buffers_from_the_species(torch, mphv, orc):
    """After mphv_plasma_destroy a species must not read the freed centred-field buffers: its next step fails with
    MPHV_ERR_STATE until fields are bound again; fields the caller bound in between are kept."""
    sims, fdev, mx, Ed, Bd, dt, (wi, we, fi, fe, E, B) = _small_plasma(torch, mphv, orc)
    pl = mphv.Plasma(mx, sims, [1.0, -1.0])
    pl.step(dt, 1)
    pl.sync()
    own = (torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
    sims[1].set_fields(*own)                       # the caller's own fields on the electrons: must survive
    pl.close()
    with pytest.raises(mphv.MphvError) as ei:
        sims[0].step(dt)
    assert ei.value.code == mphv.ERR_STATE
    sims[1].step(dt)                               # still bound, not deferred
    sims[0].set_fields(*own)
    sims[0].step(dt)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(fdev[0]).all()) and bool(torch.isfinite(fdev[1]).all())


def test_invalidate_moments_after_f_was_changed_between_calls(torch, mphv, orc):
    """A species' f replaced between two mphv_plasma_step calls: with mphv_plasma_invalidate_moments the second call
    equals the oracle's coupled step started from the new f (current recomputed), bitwise equal to a fresh plasma
    object on the same state; without it the stale current of the old f goes into the opening Maxwell half step."""
    fld = orc.fields
    c2 = 64.0
    runs = {}
    for mode in ("invalidate", "fresh", "stale"):
        sims, fdev, mx, Ed, Bd, dt, (wi, we, fi, fe, E, B) = _small_plasma(torch, mphv, orc, c2)
        pl = mphv.Plasma(mx, sims, [1.0, -1.0])
        pl.step(dt, 1)
        pl.sync()
        if mode == "invalidate":                   # the state the reference run below starts from
            f_mid = [fd.cpu().numpy().copy() for fd in fdev]
            E_mid, B_mid = Ed.cpu().numpy().copy(), Bd.cpu().numpy().copy()
        fdev[1].mul_(0.5)                          # e.g. a model-border operation that changed the electrons
        torch.cuda.synchronize()
        if mode == "invalidate":
            pl.invalidate_moments()
        elif mode == "fresh":
            pl.close()
            pl = mphv.Plasma(mx, sims, [1.0, -1.0])
        pl.step(dt, 1)
        pl.sync()
        runs[mode] = [fd.cpu().numpy().copy() for fd in fdev] + [Ed.cpu().numpy().copy(), Bd.cpu().numpy().copy()]
        pl.close()
    for a, b in zip(runs["invalidate"], runs["fresh"]):
        assert np.array_equal(a, b)
    assert not np.array_equal(runs["invalidate"][2], runs["stale"][2]), "the stale current must have been visible in E"
    g = fld.FieldGrid(wi.nx, wi.bc, tuple(wi.dx(d) if wi.nx[d] > 1 else 1.0 for d in range(3)), c2, 1.0)
    f_mid[1] *= 0.5
    species = [fld.Species(f0, orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi), qq, w.q_over_m)
               for w, f0, qq in zip((wi, we), f_mid, (1.0, -1.0))]
    fld.coupled_step(g, species, E_mid, B_mid, dt, None)
    for s, sp in enumerate(species):
        assert max(rel_err(runs["invalidate"][s], sp.f, ax) for ax in (3, 4, 5)) <= 2 * TOL_SWEEP, s
    fscale = max(np.abs(E_mid).max(), np.abs(B_mid).max()) * max(1.0, c2 * dt / min(g.dx[:2]))
    assert np.abs(runs["invalidate"][2] - E_mid).max() <= 2e-12 * fscale
    assert np.abs(runs["invalidate"][3] - B_mid).max() <= 2e-12 * fscale
