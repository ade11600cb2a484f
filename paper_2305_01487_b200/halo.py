"""Spatial block decomposition of the Vlasov grid over several GPUs.

The paper parallelises by domain decomposition with boundary cells exchanged between neighbouring
blocks (sec. 3; "two boundary cells", L187). Here: one process per GPU, ranks form a
process grid ``dims = (px, py, pz)`` over the spatial grid; velocity space is never split, so the V
stage and the moments need no communication. A spatial sweep along a decomposed axis needs the two
boundary layers of each neighbour first: ``mphv_pack_halo`` (kernel) -> neighbour exchange
(``torch.distributed`` point-to-point: NCCL over NVLink on GPUs, gloo in the CPU tests) ->
``mphv_sweep_x_halo`` (kernel reading its ghost cells from the received slabs). No collective is on
the data path; the only reduction is the one-off minimum of the time step.

This module holds host logic only (who talks to whom, buffers, call order). All arithmetic of the
method runs in the CUDA kernels behind the C ABI; there is no CPU fallback.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Optional, Sequence, Tuple

PERIODIC, OUTFLOW = 0, 1
# position of spatial dimension d (x, y, z) among the axes of f [nz][ny][nx][nvz][nvy][nvx]
F_AXIS = {0: 2, 1: 1, 2: 0}


@dataclass(frozen=True)
class Decomp:
    """Process grid over the global spatial grid. rank = (cz * py + cy) * px + cx."""
    nx: Tuple[int, int, int]            # global spatial extents
    bc: Tuple[int, int, int]
    dims: Tuple[int, int, int]          # ranks per spatial dimension

    def __post_init__(self):
        for d in range(3):
            if self.dims[d] < 1:
                raise ValueError("dims must be >= 1")
            if self.dims[d] > 1 and self.nx[d] // self.dims[d] < 4:
                raise ValueError(f"dimension {d}: blocks need at least 4 cells (two boundary cells per side)")

    @property
    def world(self) -> int:
        return self.dims[0] * self.dims[1] * self.dims[2]

    def coords(self, rank: int) -> Tuple[int, int, int]:
        px, py, _ = self.dims
        return (rank % px, (rank // px) % py, rank // (px * py))

    def rank_of(self, c: Sequence[int]) -> int:
        px, py, _ = self.dims
        return (c[2] * py + c[1]) * px + c[0]

    def extent(self, d: int, c: int) -> int:
        base, rem = divmod(self.nx[d], self.dims[d])
        return base + (1 if c < rem else 0)

    def offset(self, d: int, c: int) -> int:
        base, rem = divmod(self.nx[d], self.dims[d])
        return c * base + min(c, rem)

    def local_nx(self, rank: int) -> Tuple[int, int, int]:
        c = self.coords(rank)
        return tuple(self.extent(d, c[d]) for d in range(3))

    def local_slices(self, rank: int):
        """Slices of this rank's block in a global [nz][ny][nx]... array (axes z, y, x)."""
        c = self.coords(rank)
        s = [slice(self.offset(d, c[d]), self.offset(d, c[d]) + self.extent(d, c[d])) for d in range(3)]
        return (s[2], s[1], s[0])

    def neighbour(self, rank: int, d: int, side: int) -> Optional[int]:
        """Rank owning the block below (side 0) / above (side 1) along d; None at a global outflow end.
        On a periodic axis the neighbour wraps around (and is the rank itself when dims[d] == 1)."""
        c = list(self.coords(rank))
        c[d] += 1 if side else -1
        if c[d] < 0 or c[d] >= self.dims[d]:
            if self.bc[d] != PERIODIC:
                return None
            c[d] %= self.dims[d]
        return self.rank_of(c)

    def needs_exchange(self, d: int) -> bool:
        return self.nx[d] > 1 and self.dims[d] > 1

    def local_workload(self, w, rank: int):
        """The block of workload w (a paper_2305_01487_b200.inputs.Workload) this rank owns."""
        c = self.coords(rank)
        nx, xlo, xhi = list(w.nx), list(w.xlo), list(w.xhi)
        for d in range(3):
            if w.nx[d] > 1:
                dx = (w.xhi[d] - w.xlo[d]) / w.nx[d]
                nx[d] = self.extent(d, c[d])
                xlo[d] = w.xlo[d] + self.offset(d, c[d]) * dx
                xhi[d] = xlo[d] + nx[d] * dx
        return replace(w, name=f"{w.name}_block{rank}of{self.world}", nx=tuple(nx), xlo=tuple(xlo), xhi=tuple(xhi))


def choose_dims(nx: Sequence[int], world: int) -> Tuple[int, int, int]:
    """Process grid for `world` ranks. Preferred: blocks along x ONLY when every block keeps a whole number of
    4-cell groups and at least 8 cells (nx[0] % (4 world) == 0, nx[0] / world >= 8): that is the decomposition
    whose X stage runs as one fused pass per step (mphv_stage_x_halo: one exchange, then S_x with ghost cells and
    S_y in one kernel), and the one bench.py times. Otherwise the ranks go over the slowest active spatial axis
    first (its halo slabs are contiguous in f), then the next one, keeping at least 4 cells per block; those
    decompositions take the per-sweep path (pack, exchange, mphv_sweep_x_halo per decomposed axis)."""
    if world > 1 and nx[0] > 1 and nx[0] % (4 * world) == 0 and nx[0] // world >= 8:
        return (world, 1, 1)
    dims = [1, 1, 1]
    left = world
    for d in (2, 1, 0):
        if nx[d] <= 1 or left == 1:
            continue
        p = left
        while p > 1 and (left % p or nx[d] // p < 4):
            p -= 1
        dims[d] = p
        left //= p
    if left != 1:
        raise ValueError(f"cannot place {world} ranks on a {tuple(nx)} grid with >= 4 cells per block")
    return tuple(dims)


class HaloExchange:
    """Neighbour exchange of packed boundary layers along one decomposed axis.

    ``exchange(d, send_lo, send_hi, recv_lo, recv_hi)``: send_lo / send_hi are this block's two
    lowest / highest layers (as packed by mphv_pack_halo); after the call recv_lo holds the lower
    neighbour's highest layers and recv_hi the upper neighbour's lowest layers. Returns
    (has_lo, has_hi): False where the block sits at a global outflow end (nothing received).
    Works on any torch tensors the process group's backend can move (CUDA + NCCL, CPU + gloo)."""

    TAG_UP, TAG_DOWN = 11, 12          # message travelling towards higher / lower block index

    def __init__(self, decomp: Decomp, rank: int, group=None):
        self.decomp, self.rank, self.group = decomp, rank, group

    def exchange(self, d: int, send_lo, send_hi, recv_lo, recv_hi):
        import torch.distributed as dist
        lo, hi = self.decomp.neighbour(self.rank, d, 0), self.decomp.neighbour(self.rank, d, 1)
        ops = []
        if lo == self.rank and hi == self.rank:        # periodic axis owned by one rank: wrap locally
            recv_lo.copy_(send_hi)
            recv_hi.copy_(send_lo)
            return True, True
        # fixed issue order on every rank (NCCL matches sends and receives between a pair of ranks in
        # issue order; gloo matches by tag): sends up, down; receives from below, from above
        if hi is not None:
            ops.append(dist.P2POp(dist.isend, send_hi, hi, group=self.group, tag=self.TAG_UP))
        if lo is not None:
            ops.append(dist.P2POp(dist.isend, send_lo, lo, group=self.group, tag=self.TAG_DOWN))
        if lo is not None:
            ops.append(dist.P2POp(dist.irecv, recv_lo, lo, group=self.group, tag=self.TAG_UP))
        if hi is not None:
            ops.append(dist.P2POp(dist.irecv, recv_hi, hi, group=self.group, tag=self.TAG_DOWN))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        return lo is not None, hi is not None


class DistributedVlasov:
    """One block of a decomposed grid on this rank's GPU: the mphv context of the block plus the halo
    buffers and the exchange. step / step_moments give, block by block, the result of the single-GPU
    mphv_step on the whole grid (same kernels; ghost cells from the neighbours)."""

    def __init__(self, w_global, decomp: Decomp, rank: int, device, group=None, force_halo=False):
        """force_halo: True routes EVERY active spatial sweep through pack -> exchange -> halo kernel, also
        along axes a single rank owns (periodic: the block is its own neighbour; outflow: no neighbour);
        a tuple of axes does so for those axes only."""
        import torch
        from . import mphv
        self.torch = torch
        self.decomp, self.rank = decomp, rank
        self.w = decomp.local_workload(w_global, rank)
        self.sim = mphv.Vlasov.from_workload(self.w, device=device)
        # The kernels must run on the stream the process group's point-to-point calls are ordered against: NCCL
        # work is enqueued behind the CURRENT torch stream, so the context follows it (checked again every step).
        self._stream = None
        self._follow_current_stream()
        self.xchg = HaloExchange(decomp, rank, group)
        self.buf = {}
        forced = (0, 1, 2) if force_halo is True else tuple(force_halo or ())
        self.use_halo = [self.w.nx[d] > 1 and (d in forced or decomp.needs_exchange(d)) for d in range(3)]
        for d in range(3):
            if self.use_halo[d]:
                cnt = self.sim.halo_count(d)
                self.buf[d] = [torch.empty(cnt, dtype=torch.float64, device=self.sim.device) for _ in range(4)]

    def _follow_current_stream(self):
        torch = self.torch
        if self.sim.device.type != "cuda":
            return
        cur = torch.cuda.current_stream(self.sim.device).cuda_stream
        if cur != self._stream:
            from . import mphv
            mphv.mphv_set_stream(self.sim.ctx, cur or None)
            self._stream = cur

    def bind_f(self, f, scratch=None):
        self.sim.bind_f(f, scratch)

    def set_fields(self, E, B):
        self._follow_current_stream()
        self.sim.set_fields(E, B)

    def sweep_x(self, d: int, dt: float):
        self._follow_current_stream()
        if not self.use_halo[d]:
            self.sim.sweep_x(d, dt)
            return
        send_lo, send_hi, recv_lo, recv_hi = self.buf[d]
        self.sim.pack_halo(d, 0, send_lo)
        self.sim.pack_halo(d, 1, send_hi)
        has_lo, has_hi = self.xchg.exchange(d, send_lo, send_hi, recv_lo, recv_hi)
        self.sim.sweep_x_halo(d, dt, recv_lo if has_lo else None, recv_hi if has_hi else None)

    def step(self, dt: float):
        self.step_moments(dt, None)

    def step_moments(self, dt: float, out=None):
        self._follow_current_stream()
        if self.use_halo[0] and not self.use_halo[1] and not self.use_halo[2]:
            # decomposed along x only: one exchange, then the whole X stage (S_x and S_y in one pass)
            send_lo, send_hi, recv_lo, recv_hi = self.buf[0]
            self.sim.pack_halo(0, 0, send_lo)
            self.sim.pack_halo(0, 1, send_hi)
            has_lo, has_hi = self.xchg.exchange(0, send_lo, send_hi, recv_lo, recv_hi)
            self.sim.stage_x_halo(dt, recv_lo if has_lo else None, recv_hi if has_hi else None)
        else:
            for d in range(3):
                if self.w.nx[d] > 1:
                    self.sweep_x(d, dt)
        return self.sim.stage_v(dt, out)

    def alloc_moments(self):
        return self.sim.alloc_moments()
