"""Seeded synthetic inputs for the mphv hot path (numpy only).

This module serves BOTH the CPU oracle (tests, bench cpu_baseline) and the CUDA
path. It holds none of the method's arithmetic: no flux, limiter, sweep or moment
code, and it imports neither ``oracle`` nor the CUDA binding. It only builds the
arrays f0, E, B in the boundary layout and picks a time step.

The five workloads are BASELINE.json's ``configs`` (index 0..4); the recipe is
SURVEY.md sec. 8(d) and is restated in DESIGN.md ("Input recipe"). They stand in
for the paper's Harris-sheet reconnection runs (sec. 5.1,
L261 sec. 6: n = n0 sech^2(y/lambda) + n_b, B_x = B0 tanh(y/lambda) + dB, ion
velocity grids 16^3..36^3 over +-4..5 v_A); the paper's MMS-derived initial data
are not available and not needed.

Layouts (C order, fastest last, interior cells only):
  f    [nz][ny][nx][nvz][nvy][nvx]
  E, B [3][nz][ny][nx]   component-major, cell-centred
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Tuple

import numpy as np

BASE_SEED = 230501487  # + workload index

PERIODIC, OUTFLOW = 0, 1


@dataclass(frozen=True)
class Workload:
    name: str
    index: int
    kind: str                       # "landau1d" | "harris2d" | "harris3d"
    nx: Tuple[int, int, int]
    nv: Tuple[int, int, int]
    bc: Tuple[int, int, int]
    xlo: Tuple[float, float, float]
    xhi: Tuple[float, float, float]
    vlo: Tuple[float, float, float]
    vhi: Tuple[float, float, float]
    q_over_m: float = 1.0
    steps: int = 10
    moments_every_step: bool = False
    cfl: float = 0.5
    background: float = 0.2         # n_b of the Harris sheets
    guide_bz: float = 0.0
    seed_offset: int = 0            # extra offset for test variants
    sigma: float = 1.0              # thermal spread (standard deviation) of the Maxwellians
    drift: float = 0.5              # |u_z| of the current-carrying sheet population

    @property
    def shape(self):
        return (self.nx[2], self.nx[1], self.nx[0], self.nv[2], self.nv[1], self.nv[0])

    @property
    def space_shape(self):
        return (self.nx[2], self.nx[1], self.nx[0])

    @property
    def n_cells(self) -> int:
        return int(np.prod(self.shape, dtype=np.int64))

    @property
    def n_space(self) -> int:
        return int(np.prod(self.space_shape, dtype=np.int64))

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index + self.seed_offset

    def n_sweeps(self) -> int:
        return sum(1 for n in self.nx if n > 1) + sum(1 for n in self.nv if n > 1)

    def x_centres(self, d: int) -> np.ndarray:
        n = self.nx[d]
        if n == 1:
            return np.array([0.5 * (self.xlo[d] + self.xhi[d])])
        dx = (self.xhi[d] - self.xlo[d]) / n
        return self.xlo[d] + (np.arange(n) + 0.5) * dx

    def v_centres(self, d: int) -> np.ndarray:
        n = self.nv[d]
        if n == 1:
            return np.zeros(1)      # inactive velocity dimension: v == 0
        dv = (self.vhi[d] - self.vlo[d]) / n
        return self.vlo[d] + (np.arange(n) + 0.5) * dv

    def dx(self, d: int) -> float:
        return (self.xhi[d] - self.xlo[d]) / self.nx[d]

    def dv(self, d: int) -> float:
        return 1.0 if self.nv[d] == 1 else (self.vhi[d] - self.vlo[d]) / self.nv[d]


def harris2d(nx: int, ny: int, nv: int, vmax: float = 5.0, background: float = 0.2,
             guide_bz: float = 0.0, steps: int = 10, moments_every_step: bool = False,
             index: int = 1, name: str | None = None, bc_y: int = OUTFLOW,
             seed_offset: int = 0) -> Workload:
    return Workload(
        name=name or f"harris2d_{nx}x{ny}x{nv}^3", index=index, kind="harris2d",
        nx=(nx, ny, 1), nv=(nv, nv, nv), bc=(PERIODIC, bc_y, PERIODIC),
        xlo=(0.0, -6.4, 0.0), xhi=(25.6, 6.4, 1.0),
        vlo=(-vmax,) * 3, vhi=(vmax,) * 3,
        steps=steps, moments_every_step=moments_every_step,
        background=background, guide_bz=guide_bz, seed_offset=seed_offset)


def harris3d(n: int, nv: int, vmax: float = 5.0, steps: int = 5, index: int = 4,
             name: str | None = None, seed_offset: int = 0) -> Workload:
    return Workload(
        name=name or f"harris3d_{n}^3x{nv}^3", index=index, kind="harris3d",
        nx=(n, n, n), nv=(nv, nv, nv), bc=(PERIODIC, OUTFLOW, PERIODIC),
        xlo=(0.0, -6.4, 0.0), xhi=(12.8, 6.4, 12.8),
        vlo=(-vmax,) * 3, vhi=(vmax,) * 3,
        steps=steps, moments_every_step=True, background=0.2, seed_offset=seed_offset)


def landau1d(nx: int = 64, nv: int = 128, steps: int = 20) -> Workload:
    return Workload(
        name=f"landau1d_{nx}x{nv}", index=0, kind="landau1d",
        nx=(nx, 1, 1), nv=(nv, 1, 1), bc=(PERIODIC, PERIODIC, PERIODIC),
        xlo=(0.0, 0.0, 0.0), xhi=(4.0 * np.pi, 1.0, 1.0),
        vlo=(-6.0, 0.0, 0.0), vhi=(6.0, 1.0, 1.0), steps=steps)


def config(i: int) -> Workload:
    """BASELINE.json ``configs[i]``."""
    if i == 0:
        return landau1d()
    if i == 1:
        return harris2d(32, 32, 32, index=1, name="c1_harris2d_32x32x32^3")
    if i == 2:
        return harris2d(64, 64, 32, guide_bz=0.1, moments_every_step=True, index=2,
                        name="c2_harris2d_64x64x32^3")
    if i == 3:
        return harris2d(128, 64, 40, vmax=6.0, background=0.1, index=3,
                        name="c3_harris2d_128x64x40^3")
    if i == 4:
        return harris3d(32, 32, name="c4_harris3d_32^3x32^3")
    raise ValueError("config index must be 0..4")


# --------------------------------------------------------------------------- fields

def _smooth_noise(w: Workload, rng: np.random.Generator) -> np.ndarray:
    """Seeded sum of <= 4x4(x4) low Fourier modes on the spatial grid, max-abs 1.

    Periodic in every periodic direction (integer mode numbers over the box).
    Returned shape: space_shape = (nz, ny, nx).
    """
    x, y, z = (w.x_centres(d) for d in range(3))
    L = [w.xhi[d] - w.xlo[d] for d in range(3)]
    px = 2.0 * np.pi * (x - w.xlo[0]) / L[0]
    py = 2.0 * np.pi * (y - w.xlo[1]) / L[1]
    pz = 2.0 * np.pi * (z - w.xlo[2]) / L[2]
    out = np.zeros(w.space_shape)
    mz_range = range(4) if w.nx[2] > 1 else range(1)
    my_range = range(4) if w.nx[1] > 1 else range(1)
    for mz in mz_range:
        for my in my_range:
            for mx in range(4):
                amp = rng.normal()
                ph = rng.uniform(0.0, 2.0 * np.pi)
                if mx == 0 and my == 0 and mz == 0:
                    continue
                out += amp * np.cos(mz * pz[:, None, None] + my * py[None, :, None]
                                    + mx * px[None, None, :] + ph)
    m = np.max(np.abs(out))
    return out / m if m > 0 else out


def make_fields(w: Workload):
    """E, B as float64 arrays of shape (3, nz, ny, nx)."""
    rng = np.random.default_rng(w.seed)
    E = np.zeros((3,) + w.space_shape)
    B = np.zeros((3,) + w.space_shape)
    if w.kind == "landau1d":
        x = w.x_centres(0)
        E[0, 0, 0, :] = 0.01 * np.sin(0.5 * x)
        return E, B
    y = w.x_centres(1)
    if w.kind == "harris2d":
        prof = np.tanh(y / 0.5)
    else:  # double sheet at y0 = -3.2 and +3.2
        prof = np.tanh((y + 3.2) / 0.5) - np.tanh((y - 3.2) / 0.5) - 1.0
    B[0] = prof[None, :, None] + 1e-2 * _smooth_noise(w, rng)
    B[2] = w.guide_bz
    for a in range(3):
        E[a] = 1e-2 * _smooth_noise(w, rng)
    return np.ascontiguousarray(E), np.ascontiguousarray(B)


def cfl_dt(w: Workload, E: np.ndarray, B: np.ndarray) -> float:
    """dt = cfl * min over all active sweeps of (cell width / max |speed|).

    Spatial sweeps: max |v_d| is the outermost cell centre. Velocity sweeps: the
    bound |E_d| + vmax_e |B_f| + vmax_f |B_e| (triangle inequality over the other
    two velocity components; it is attained on a symmetric velocity grid), maxed
    over spatial cells. Computed once here and handed to both sides.
    """
    lim = []
    vmax = [float(np.max(np.abs(w.v_centres(d)))) for d in range(3)]
    for d in range(3):
        if w.nx[d] > 1 and vmax[d] > 0:
            lim.append(w.dx(d) / vmax[d])
    for d in range(3):
        if w.nv[d] > 1:
            e, f_ = (d + 1) % 3, (d + 2) % 3
            a = np.abs(E[d]) + vmax[e] * np.abs(B[f_]) + vmax[f_] * np.abs(B[e])
            amax = abs(w.q_over_m) * float(np.max(a))
            if amax > 0:
                lim.append(w.dv(d) / amax)
    return float(w.cfl * min(lim))


# --------------------------------------------------------------------------- f0

def _gauss(v: np.ndarray, u: float = 0.0, sigma: float = 1.0) -> np.ndarray:
    if sigma == 1.0:
        return np.exp(-0.5 * (v - u) ** 2) / np.sqrt(2.0 * np.pi)
    return np.exp(-0.5 * ((v - u) / sigma) ** 2) / (np.sqrt(2.0 * np.pi) * sigma)


def make_f0(w: Workload, noise: float = 1e-6, density_ripple: float = 1e-3) -> np.ndarray:
    """Initial distribution, shape w.shape, float64, strictly positive.

    landau1d: (1 + 0.01 cos 0.5x) exp(-v^2/2)/sqrt(2 pi) x (1 + noise U(-1,1)).
    harris:   [sech^2((y-y0)/0.5) M(v; u_z = +-0.5) + n_b M(v; 0)]
              x (1 + density_ripple eta(x,y,z)) x (1 + noise U(-1,1)),
              M = product of unit-variance Gaussians at cell centres.
    The ripple (not in BASELINE.json) makes f vary along x from step 0 so that the
    x sweep is exercised by the parity tests; the per-cell noise makes every cell
    distinct so that an index error cannot cancel.
    """
    rng = np.random.default_rng(w.seed + 7919)
    nz, ny, nx, nvz, nvy, nvx = w.shape
    if w.kind == "landau1d":
        x = w.x_centres(0)
        v = w.v_centres(0)
        f = (1.0 + 0.01 * np.cos(0.5 * x))[:, None] * _gauss(v)[None, :]
        f = f * (1.0 + noise * rng.uniform(-1.0, 1.0, size=f.shape))
        return np.ascontiguousarray(f.reshape(w.shape))

    y = w.x_centres(1)
    sg = w.sigma
    gx, gy = _gauss(w.v_centres(0), 0.0, sg), _gauss(w.v_centres(1), 0.0, sg)
    vz = w.v_centres(2)
    ripple = 1.0 + density_ripple * _smooth_noise(w, rng)            # (nz, ny, nx)
    if w.kind == "harris2d":
        sheets = [(1.0 / np.cosh(y / 0.5) ** 2, w.drift)]
    else:
        sheets = [(1.0 / np.cosh((y + 3.2) / 0.5) ** 2, w.drift),
                  (1.0 / np.cosh((y - 3.2) / 0.5) ** 2, -w.drift)]
    # z-profile in velocity per spatial row: sum_sheets n_s(y) G(vz - u_s) + n_b G(vz)
    zprof = w.background * _gauss(vz, 0.0, sg)[None, :] + sum(
        n_s[:, None] * _gauss(vz, u, sg)[None, :] for n_s, u in sheets)  # (ny, nvz)
    plane = gy[:, None] * gx[None, :]                                # (nvy, nvx)
    f = np.empty(w.shape)
    for iz in range(nz):
        for iy in range(ny):
            cube = zprof[iy][:, None, None] * plane[None, :, :]      # (nvz, nvy, nvx)
            row = ripple[iz, iy][:, None, None, None] * cube[None]   # (nx, nvz, nvy, nvx)
            if noise:
                row = row * (1.0 + noise * rng.uniform(-1.0, 1.0, size=row.shape))
            f[iz, iy] = row
    return f


def make_all(w: Workload):
    """(f0, E, B, dt) for a workload."""
    E, B = make_fields(w)
    return make_f0(w), E, B, cfl_dt(w, E, B)


def variant(w: Workload, **kw) -> Workload:
    return replace(w, **kw)


def electrons_of(w: Workload, mass_ratio: float = 100.0, temp_ratio: float = 0.2, nv: int = 36,
                 vmax: float = 20.0) -> Workload:
    """The electron species that goes with the (ion) Harris workload w in a two-species run: same spatial
    grid and density profile (a neutral plasma), q/m = -mass_ratio, velocity grid nv^3 on [-vmax, vmax]^3 (the
    paper's electron grids: 36^3 on +-20 v_A at m_i/m_e = 100), thermal spread
    sqrt(mass_ratio * temp_ratio) (T_e / T_i = temp_ratio), sheet drift -temp_ratio * drift (the Harris
    equilibrium splits the current as the temperatures), its own seed."""
    return replace(w, name=w.name + f"_electrons_{nv}^3", nv=(nv, nv, nv), vlo=(-vmax,) * 3, vhi=(vmax,) * 3,
                   q_over_m=-mass_ratio, sigma=float(np.sqrt(mass_ratio * temp_ratio)),
                   drift=-temp_ratio * w.drift, seed_offset=w.seed_offset + 500)


def yee_fields(w: Workload):
    """Seeded STAGGERED E, B (shape (3, nz, ny, nx) each, the lattice R19 of DESIGN.md) for coupled runs: the
    Harris profile B_x = tanh(y / 0.5) (double sheet for harris3d) sampled at the positions of B_x on the lattice
    plus the 1e-2 smooth perturbation, guide field, E = 1e-2 smooth noise; zero fields for landau1d."""
    rng = np.random.default_rng(w.seed + 104729)
    E = np.zeros((3,) + w.space_shape)
    B = np.zeros((3,) + w.space_shape)
    if w.kind == "landau1d":
        return E, B
    y_edge = w.x_centres(1) + 0.5 * w.dx(1)                       # B_x sits at (i, j + 1/2, k + 1/2)
    if w.kind == "harris2d":
        prof = np.tanh(y_edge / 0.5)
    else:
        prof = np.tanh((y_edge + 3.2) / 0.5) - np.tanh((y_edge - 3.2) / 0.5) - 1.0
    B[0] = prof[None, :, None] + 1e-2 * _smooth_noise(w, rng)
    B[2] = w.guide_bz
    for a in range(3):
        E[a] = 1e-2 * _smooth_noise(w, rng)
    return np.ascontiguousarray(E), np.ascontiguousarray(B)
