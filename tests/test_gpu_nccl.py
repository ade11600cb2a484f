"""The multi-GPU path over NCCL: two ranks, one GPU each, DistributedVlasov (pack -> send/recv ->
halo sweep, V stage) against the oracle's step on the whole grid. NCCL ignores tags and matches sends and receives
between a pair of ranks in issue order, so the periodic two-rank case (each rank is the other's lower AND upper
neighbour) exercises exactly what the gloo tests on CPU cannot. Skips cleanly on a box with fewer than two GPUs
(one rank per GPU is the only sound way to run it: see the profiling guide on ranks that wait on one another)."""
import os
import socket

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, dims, nsteps, q):
    import torch
    import torch.distributed as dist
    from paper_2305_01487_b200 import halo, inputs
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    torch.cuda.set_device(rank)
    dev = torch.device("cuda", rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    try:
        w = inputs.harris2d(32, 16, 16)
        dec = halo.Decomp(w.nx, w.bc, dims)
        f0, E, B, dt = inputs.make_all(w)
        sl = dec.local_slices(rank)
        El, Bl = (np.ascontiguousarray(a[(slice(None),) + sl]) for a in (E, B))
        dv = halo.DistributedVlasov(w, dec, rank, dev)
        f = torch.from_numpy(np.ascontiguousarray(f0[sl])).to(dev)
        dv.bind_f(f)
        dv.set_fields(torch.from_numpy(El).to(dev), torch.from_numpy(Bl).to(dev))
        mom = dv.alloc_moments()
        for _ in range(nsteps):
            dv.step_moments(dt, mom)
        torch.cuda.synchronize()
        parts = [None] * world
        dist.all_gather_object(parts, (sl, f.cpu().numpy(), mom[0].cpu().numpy()))
        if rank == 0:
            q.put(("ok", parts))
    except Exception as e:  # noqa: BLE001
        q.put(("error", rank, repr(e)))
        raise
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("dims", [(2, 1, 1), (1, 2, 1)])
def test_two_nccl_ranks_reproduce_the_global_step(orc, dims):
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (one NCCL rank per GPU)")
    import torch.multiprocessing as mp
    from paper_2305_01487_b200 import inputs
    from parity_util import TOL_SWEEP, rel_err
    nsteps = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, dims, nsteps, q)) for r in range(2)]
    for p in procs:
        p.start()
    try:
        res = q.get(timeout=300)
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.kill()
    assert res[0] == "ok", res
    w = inputs.harris2d(32, 16, 16)
    f0, E, B, dt = inputs.make_all(w)
    grid, box = orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi)
    ref = f0.copy()
    for _ in range(nsteps):
        orc.step(ref, grid, box, w.q_over_m, E, B, dt)
    n_ref = orc.moments(ref, grid, box)[0]
    got, n_got = np.full_like(ref, np.nan), np.full_like(n_ref, np.nan)
    for sl, blk, n in res[1]:
        got[sl] = blk
        n_got[sl] = n
    assert np.isfinite(got).all()
    assert max(rel_err(got, ref, ax) for ax in (3, 4, 5)) <= nsteps * TOL_SWEEP
    assert np.abs(n_got - n_ref).max() <= 1e-12 * np.abs(n_ref).max()
