"""Host logic of the multi-GPU path (paper_2305_01487_b200/halo.py), on CPU.

The decomposition bookkeeping is checked directly; the neighbour exchange runs for real between
world_size 2 and 4 processes over gloo. The sweeps themselves are the oracle's here (the CUDA kernels
need a GPU): each rank attaches the received ghost layers to its block, sweeps the extended block and
keeps the interior -- which must reproduce the oracle's step on the whole grid (to the last bits:
the arithmetic is the same, only a block's cell width may round differently)."""
import os
import socket

import numpy as np
import pytest

from paper_2305_01487_b200 import halo, inputs


def test_decomp_bookkeeping():
    d = halo.Decomp(nx=(18, 9, 1), bc=(0, 1, 0), dims=(4, 2, 1))
    assert d.world == 8
    cover = np.zeros((1, 9, 18), dtype=int)
    for r in range(d.world):
        assert d.rank_of(d.coords(r)) == r
        cover[d.local_slices(r)] += 1
        assert min(n for n, g in zip(d.local_nx(r), d.nx) if g > 1) >= 4
    assert (cover == 1).all(), "blocks tile the grid exactly once"
    assert [d.extent(0, c) for c in range(4)] == [5, 5, 4, 4] and [d.offset(0, c) for c in range(4)] == [0, 5, 10, 14]
    # periodic x wraps, outflow y ends have no neighbour
    r = d.rank_of((0, 0, 0))
    assert d.neighbour(r, 0, 0) == d.rank_of((3, 0, 0)) and d.neighbour(r, 0, 1) == d.rank_of((1, 0, 0))
    assert d.neighbour(r, 1, 0) is None and d.neighbour(r, 1, 1) == d.rank_of((0, 1, 0))
    assert d.neighbour(d.rank_of((2, 1, 0)), 1, 1) is None
    assert not d.needs_exchange(2)
    with pytest.raises(ValueError):
        halo.Decomp(nx=(6, 8, 1), bc=(0, 1, 0), dims=(2, 1, 1))        # 3-cell blocks


def test_choose_dims_prefers_x_only_then_the_slowest_axis():
    # x only wherever the fused X stage can take it: blocks of whole 4-cell groups, at least 8 cells
    assert halo.choose_dims((128, 64, 1), 2) == (2, 1, 1)
    assert halo.choose_dims((128, 64, 1), 8) == (8, 1, 1)
    assert halo.choose_dims((32, 32, 32), 4) == (4, 1, 1)
    assert halo.choose_dims((64, 8, 1), 8) == (8, 1, 1)
    assert halo.choose_dims((64, 1, 1), 4) == (4, 1, 1)
    for n in (1, 2, 4, 8):                                  # bench.py --gpus n: config 3 repeated n times along x
        assert halo.choose_dims((128 * n, 64, 1), n) == (n, 1, 1)
    # otherwise the slowest active axis first
    assert halo.choose_dims((12, 10, 1), 2) == (1, 2, 1)     # 6-cell blocks along x are not whole groups
    assert halo.choose_dims((32, 32, 32), 8) == (1, 1, 8)    # 4-cell blocks along x are too short
    assert halo.choose_dims((24, 64, 1), 4) == (1, 4, 1)
    assert halo.choose_dims((12, 8, 1), 4) == (2, 2, 1)
    with pytest.raises(ValueError):
        halo.choose_dims((4, 4, 1), 8)


def test_local_workload_blocks_reassemble_the_global_inputs():
    w = inputs.harris2d(12, 10, 4)
    d = halo.Decomp(w.nx, w.bc, (2, 2, 1))
    for r in range(d.world):
        wl = d.local_workload(w, r)
        sl = d.local_slices(r)
        assert np.allclose(wl.x_centres(0), w.x_centres(0)[sl[2]], rtol=0, atol=1e-13)
        assert np.allclose(wl.x_centres(1), w.x_centres(1)[sl[1]], rtol=0, atol=1e-13)
        assert wl.nv == w.nv and abs(wl.dx(0) - w.dx(0)) < 1e-15


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _sweep_block_with_ghosts(orc, blk, w_blk, d, dt, lo, hi):
    """Oracle sweep of a block along spatial dim d with ghost layers lo / hi (None = outflow end):
    sweep the extended block, keep the interior (the extended block's own boundary rule only touches
    its two outermost layers' fluxes, which lie outside the interior's stencil)."""
    ax = halo.F_AXIS[d]
    first = np.take(blk, [0, 0], axis=ax)
    last = np.take(blk, [-1, -1], axis=ax)
    ext = np.ascontiguousarray(np.concatenate([first if lo is None else lo, blk, last if hi is None else hi], axis=ax))
    nx = list(w_blk.nx)
    nx[d] += 4
    grid = orc.Grid(tuple(nx), w_blk.nv, (1, 1, 1))
    xhi = list(w_blk.xhi)
    xhi[d] = w_blk.xlo[d] + nx[d] * w_blk.dx(d)
    box = orc.Box(w_blk.xlo, tuple(xhi), w_blk.vlo, w_blk.vhi)
    orc.sweep_x(ext, grid, box, d, dt)
    n = blk.shape[ax]
    return np.ascontiguousarray(np.take(ext, np.arange(2, 2 + n), axis=ax))


def _worker(rank, world, port, dims, kind, q):
    import torch
    import torch.distributed as dist
    import oracle as orc
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = inputs.harris2d(12, 10, 6) if kind == "2d" else inputs.harris2d(64, 8, 4) if kind == "2dx8" else inputs.harris3d(8, 4)
        dec = halo.Decomp(w.nx, w.bc, dims)
        f0, E, B, dt = inputs.make_all(w)
        dt *= 1.7
        sl = dec.local_slices(rank)
        wl = dec.local_workload(w, rank)
        blk = f0[sl].copy()                      # (a leading block of f0 is already contiguous: copy, do not alias)
        El, Bl = (np.ascontiguousarray(a[(slice(None),) + sl]) for a in (E, B))
        xchg = halo.HaloExchange(dec, rank)
        for d in range(3):
            if w.nx[d] == 1:
                continue
            ax = halo.F_AXIS[d]
            if not dec.needs_exchange(d):
                orc.sweep_x(blk, orc.Grid(wl.nx, wl.nv, wl.bc), orc.Box(wl.xlo, wl.xhi, wl.vlo, wl.vhi), d, dt)
                continue
            n = blk.shape[ax]
            send_lo = torch.from_numpy(np.ascontiguousarray(np.take(blk, [0, 1], axis=ax)))
            send_hi = torch.from_numpy(np.ascontiguousarray(np.take(blk, [n - 2, n - 1], axis=ax)))
            recv_lo, recv_hi = torch.full_like(send_lo, np.nan), torch.full_like(send_hi, np.nan)
            has_lo, has_hi = xchg.exchange(d, send_lo, send_hi, recv_lo, recv_hi)
            blk = _sweep_block_with_ghosts(orc, blk, wl, d, dt, recv_lo.numpy() if has_lo else None,
                                           recv_hi.numpy() if has_hi else None)
        grid, box = orc.Grid(wl.nx, wl.nv, wl.bc), orc.Box(wl.xlo, wl.xhi, wl.vlo, wl.vhi)
        for d in range(3):
            orc.sweep_v(blk, grid, box, wl.q_over_m, El, Bl, d, dt)
        parts = [None] * world
        dist.all_gather_object(parts, (sl, blk))
        if rank == 0:
            ref = f0.copy()
            orc.step(ref, orc.Grid(w.nx, w.nv, w.bc), orc.Box(w.xlo, w.xhi, w.vlo, w.vhi), w.q_over_m, E, B, dt)
            got = np.full_like(ref, np.nan)
            for s, b in parts:
                got[s] = b
            q.put(("ok", bool(np.isfinite(got).all()), float(np.nanmax(np.abs(got - ref)) / np.max(np.abs(ref)))))
    except Exception as e:  # noqa: BLE001
        q.put(("error", rank, repr(e)))
        raise
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,dims,kind", [(2, (1, 2, 1), "2d"), (2, (2, 1, 1), "2d"), (4, (2, 2, 1), "2d"),
                                             (2, (1, 1, 2), "3d")])
def test_exchange_over_gloo_reproduces_the_global_step(orc, world, dims, kind):
    """world_size 2 and 4 over gloo: periodic wrap between two ranks (each is the other's lower AND
    upper neighbour), outflow ends, a 2 x 2 process grid, a 3-D grid."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, dims, kind, q)) for r in range(world)]
    for p in procs:
        p.start()
    try:
        res = q.get(timeout=240)
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.kill()
    assert res[0] == "ok", res
    # not bitwise: a block's cell width (xhi - xlo) / n can differ from the global one in the last bit,
    # so its Courant numbers may be one ulp off
    assert res[1] and res[2] <= 1e-15, f"blocks differ from the global oracle step (max diff / max|f| = {res[2]:.3e})"


def test_eight_blocks_along_x_as_bench_gpus_8_decomposes(orc):
    """world_size 8 over gloo on a 64 x 8 grid with the decomposition choose_dims picks (x only, 8-cell blocks): the
    bookkeeping of `bench.py --gpus 8` (block offsets, periodic wrap across 8 ranks, both ghost slabs of every block)."""
    import torch.multiprocessing as mp
    dims = halo.choose_dims((64, 8, 1), 8)
    assert dims == (8, 1, 1)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 8, port, dims, "2dx8", q)) for r in range(8)]
    for p in procs:
        p.start()
    try:
        res = q.get(timeout=400)
    finally:
        for p in procs:
            p.join(timeout=90)
            if p.is_alive():
                p.kill()
    assert res[0] == "ok", res
    assert res[1] and res[2] <= 1e-15, f"blocks differ from the global oracle step (max diff / max|f| = {res[2]:.3e})"
