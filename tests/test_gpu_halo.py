"""GPU parity of the block-decomposed path: mphv_pack_halo + mphv_sweep_x_halo +
mphv_stage_v on the blocks of a decomposed grid against the oracle's step on the WHOLE grid.
One GPU is enough: the blocks live side by side on it and the test routes the packed layers between
them exactly as halo.HaloExchange does between ranks (that exchange itself is covered over gloo in
test_halo_cpu.py)."""
import numpy as np
import pytest

from parity_util import TOL_SWEEP, rel_err

pytestmark = pytest.mark.gpu


def run_blocks(torch, mphv, halo, w, dims, f0, E, B, dt, nsteps=2, fused_x_stage=False):
    dec = halo.Decomp(w.nx, w.bc, dims)
    blocks = []
    for r in range(dec.world):
        sl = dec.local_slices(r)
        wl = dec.local_workload(w, r)
        sim = mphv.Vlasov.from_workload(wl)
        f = torch.from_numpy(f0[sl].copy()).cuda()
        sim.bind_f(f)
        sim.set_fields(torch.from_numpy(np.ascontiguousarray(E[(slice(None),) + sl])).cuda(),
                       torch.from_numpy(np.ascontiguousarray(B[(slice(None),) + sl])).cuda())
        blocks.append(dict(sim=sim, f=f, sl=sl, mom=sim.alloc_moments()))
    for _ in range(nsteps):
        if fused_x_stage:                       # x-only decomposition: mphv_stage_x_halo (S_x + S_y in one pass)
            assert dims[1] == 1 and dims[2] == 1
            packed = []
            for b in blocks:
                cnt = b["sim"].halo_count(0)
                lo, hi = (torch.empty(cnt, dtype=torch.float64, device="cuda") for _ in range(2))
                b["sim"].pack_halo(0, 0, lo)
                b["sim"].pack_halo(0, 1, hi)
                packed.append((lo, hi))
            for r, b in enumerate(blocks):
                nlo, nhi = dec.neighbour(r, 0, 0), dec.neighbour(r, 0, 1)
                n0 = b["sim"].launches
                b["sim"].stage_x_halo(dt, None if nlo is None else packed[nlo][1], None if nhi is None else packed[nhi][0])
                assert b["sim"].launches - n0 == (2 if w.nx[2] > 1 else 1), "fused S_x + S_y kernel with halo ghosts"
        for d in range(3):
            if w.nx[d] == 1 or fused_x_stage:
                continue
            if not dec.needs_exchange(d):
                for b in blocks:
                    b["sim"].sweep_x(d, dt)
                continue
            packed = []
            for b in blocks:
                cnt = b["sim"].halo_count(d)
                lo, hi = (torch.empty(cnt, dtype=torch.float64, device="cuda") for _ in range(2))
                b["sim"].pack_halo(d, 0, lo)
                b["sim"].pack_halo(d, 1, hi)
                packed.append((lo, hi))
            for r, b in enumerate(blocks):
                nlo, nhi = dec.neighbour(r, d, 0), dec.neighbour(r, d, 1)
                b["sim"].sweep_x_halo(d, dt, None if nlo is None else packed[nlo][1],
                                      None if nhi is None else packed[nhi][0])
        for b in blocks:
            b["sim"].stage_v(dt, b["mom"])
    torch.cuda.synchronize()
    got = np.empty_like(f0)
    n = np.empty(w.space_shape)
    for b in blocks:
        got[b["sl"]] = b["f"].cpu().numpy()
        n[b["sl"]] = b["mom"][0].cpu().numpy()
    return got, n


@pytest.mark.parametrize("kind,dims", [("2d", (1, 2, 1)), ("2d", (2, 1, 1)), ("2d", (3, 2, 1)),
                                       ("3d", (1, 1, 2)), ("3d", (2, 1, 2)), ("2dper", (1, 3, 1))])
def test_decomposed_blocks_match_the_global_oracle_step(orc, kind, dims):
    import torch
    from paper_2305_01487_b200 import halo, inputs, mphv
    if kind == "2d":
        w = inputs.harris2d(14, 10, 8)          # ragged: 14 = 5 + 5 + 4
    elif kind == "2dper":
        w = inputs.harris2d(8, 13, 8, bc_y=0)   # periodic y over three ranks: wrap-around neighbours
    else:
        w = inputs.harris3d(8, 4)
    f0, E, B, dt = inputs.make_all(w)
    dt *= 1.7
    got, n_g = run_blocks(torch, mphv, halo, w, dims, f0, E, B, dt)
    ref = f0.copy()
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    for _ in range(2):
        orc.step(ref, grid, box, w.q_over_m, E, B, dt)
    assert rel_err(got, ref, 3) <= 2 * TOL_SWEEP
    n_r, _, _ = orc.moments(ref, grid, box)
    assert np.max(np.abs(n_g - n_r) / np.abs(n_r)) <= 1e-12


@pytest.mark.parametrize("kind,nblocks,bcx", [("2d", 2, 0), ("2d", 3, 0), ("2d", 2, 1), ("3d", 2, 0), ("2dper", 2, 0)])
def test_x_decomposed_blocks_fused_x_stage_match_the_global_oracle_step(orc, kind, nblocks, bcx):
    """mphv_stage_x_halo on blocks side by side along x (periodic and outflow x: the end blocks of an
    outflow axis have no neighbour on one side) against the oracle's step on the whole grid."""
    import torch
    from paper_2305_01487_b200 import halo, inputs, mphv
    if kind == "2d":
        w = inputs.harris2d(8 * nblocks, 10, 8)
    elif kind == "2dper":
        w = inputs.harris2d(16, 9, 8, bc_y=0)
    else:
        w = inputs.harris3d(16, 4)
    if bcx:
        w = inputs.variant(w, bc=(1, w.bc[1], w.bc[2]))
    f0, E, B, dt = inputs.make_all(w)
    dt *= 1.7
    got, n_g = run_blocks(torch, mphv, halo, w, (nblocks, 1, 1), f0, E, B, dt, fused_x_stage=True)
    ref = f0.copy()
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    for _ in range(2):
        orc.step(ref, grid, box, w.q_over_m, E, B, dt)
    assert rel_err(got, ref, 3) <= 2 * TOL_SWEEP
    n_r, _, _ = orc.moments(ref, grid, box)
    assert np.max(np.abs(n_g - n_r) / np.abs(n_r)) <= 1e-12


def test_distributed_vlasov_single_rank_fused_x_stage(orc):
    """halo.DistributedVlasov, one rank, halo forced along x only: pack x2 -> self exchange -> mphv_stage_x_halo."""
    import torch
    from paper_2305_01487_b200 import halo, inputs
    w = inputs.harris2d(12, 10, 8)
    f0, E, B, dt = inputs.make_all(w)
    dv = halo.DistributedVlasov(w, halo.Decomp(w.nx, w.bc, (1, 1, 1)), 0, "cuda:0", force_halo=(0,))
    f = torch.from_numpy(f0).cuda()
    dv.bind_f(f)
    dv.set_fields(torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
    mom = dv.alloc_moments()
    for _ in range(2):
        dv.step_moments(dt, mom)
    torch.cuda.synchronize()
    ref = f0.copy()
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    for _ in range(2):
        orc.step(ref, grid, box, w.q_over_m, E, B, dt)
    assert rel_err(f.cpu().numpy(), ref, 3) <= 2 * TOL_SWEEP
    assert dv.sim.launches == 1 + 2 * (2 + 1 + 1), "amax; per step: pack x2, fused X stage, fused V stage"


def test_distributed_vlasov_single_rank_through_the_halo_kernels(orc):
    """halo.DistributedVlasov with one rank and force_halo: every spatial sweep goes pack -> (self)
    exchange -> halo kernel; periodic x wraps onto the block itself, outflow y has no neighbour."""
    import torch
    from paper_2305_01487_b200 import halo, inputs, mphv  # noqa: F401
    w = inputs.harris2d(12, 10, 8)
    f0, E, B, dt = inputs.make_all(w)
    dv = halo.DistributedVlasov(w, halo.Decomp(w.nx, w.bc, (1, 1, 1)), 0, "cuda:0", force_halo=True)
    f = torch.from_numpy(f0).cuda()
    dv.bind_f(f)
    dv.set_fields(torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
    mom = dv.alloc_moments()
    for _ in range(2):
        dv.step_moments(dt, mom)
    torch.cuda.synchronize()
    ref = f0.copy()
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    for _ in range(2):
        orc.step(ref, grid, box, w.q_over_m, E, B, dt)
    assert rel_err(f.cpu().numpy(), ref, 3) <= 2 * TOL_SWEEP
    assert dv.sim.launches >= 2 * (2 * 3 + 1), "pack x2 + halo sweep per spatial axis, V stage (one kernel at the default fusion level)"


def test_halo_api_errors():
    import torch
    from paper_2305_01487_b200 import inputs, mphv
    w = inputs.harris2d(8, 8, 8)
    sim = mphv.Vlasov.from_workload(w)
    assert sim.halo_count(0) == 2 * 8 * 8 ** 3 and sim.halo_count(2) == 0
    f = torch.ones(w.shape, dtype=torch.float64, device="cuda")
    sim.bind_f(f)
    buf = torch.zeros(sim.halo_count(0), dtype=torch.float64, device="cuda")
    for call, code in [(lambda: mphv.mphv_pack_halo(sim.ctx, 2, 0, buf.data_ptr()), mphv.ERR_ARG),
                       (lambda: mphv.mphv_pack_halo(sim.ctx, 0, 2, buf.data_ptr()), mphv.ERR_ARG),
                       (lambda: mphv.mphv_pack_halo(sim.ctx, 0, 0, None), mphv.ERR_ARG),
                       (lambda: mphv.mphv_sweep_x_halo(sim.ctx, 0, 0.01, buf.data_ptr(), None), mphv.ERR_ARG),   # periodic
                       (lambda: mphv.mphv_sweep_x_halo(sim.ctx, 0, 10.0, buf.data_ptr(), buf.data_ptr()), mphv.ERR_RANGE),
                       (lambda: mphv.mphv_stage_v(sim.ctx, 0.01), mphv.ERR_STATE)]:                                 # no fields
        with pytest.raises(mphv.MphvError) as ei:
            call()
        assert ei.value.code == code
    torch.cuda.synchronize()
    assert bool((f == 1.0).all())
