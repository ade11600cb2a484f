"""ctypes binding of oracle/mphv_oracle.c (builds it with gcc on first use).

TEST INFRASTRUCTURE. Argument marshalling only; all arithmetic is in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import shutil
import subprocess
from dataclasses import dataclass, field
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "mphv_oracle.c"
_SRCS = [_SRC, _HERE / "mphv_fields_oracle.c"]
_SO = _HERE / "libmphv_oracle.so"

BC_PERIODIC, BC_OUTFLOW, BC_WALL = 0, 1, 2
OK, ERR_ARG, ERR_RANGE = 0, 1, 3


class _CGrid(C.Structure):
    _fields_ = [("nx", C.c_int32 * 3), ("nv", C.c_int32 * 3), ("bc", C.c_int32 * 3)]


class _CBox(C.Structure):
    _fields_ = [("xlo", C.c_double * 3), ("xhi", C.c_double * 3),
                ("vlo", C.c_double * 3), ("vhi", C.c_double * 3)]


@dataclass
class Grid:
    nx: tuple
    nv: tuple
    bc: tuple = (0, 0, 0)

    def c(self) -> _CGrid:
        return _CGrid((C.c_int32 * 3)(*self.nx), (C.c_int32 * 3)(*self.nv), (C.c_int32 * 3)(*self.bc))

    @property
    def n_space(self) -> int:
        return int(np.prod(self.nx))

    @property
    def shape(self) -> tuple:
        return (self.nx[2], self.nx[1], self.nx[0], self.nv[2], self.nv[1], self.nv[0])


@dataclass
class Box:
    xlo: tuple = (0.0, 0.0, 0.0)
    xhi: tuple = (1.0, 1.0, 1.0)
    vlo: tuple = (-1.0, -1.0, -1.0)
    vhi: tuple = (1.0, 1.0, 1.0)

    def c(self) -> _CBox:
        d3 = C.c_double * 3
        return _CBox(d3(*self.xlo), d3(*self.xhi), d3(*self.vlo), d3(*self.vhi))


def build(force: bool = False) -> Path:
    """Compile the oracle: -O2, OpenMP over independent pencils, no FMA contraction."""
    if not force and _SO.exists() and all(_SO.stat().st_mtime >= p.stat().st_mtime for p in _SRCS):
        return _SO
    cands = [c for c in ("/usr/bin/gcc", shutil.which("gcc"), shutil.which("cc")) if c]
    flags = ["-O2", "-std=c99", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra"]
    errs = []
    for cc in cands:
        for omp in (["-fopenmp"], []):
            tmp = _SO.with_suffix(f".{os.getpid()}.tmp")
            r = subprocess.run([cc, *flags, *omp, "-o", str(tmp), *map(str, _SRCS), "-lm"],
                               capture_output=True, text=True)
            if r.returncode == 0:
                os.replace(tmp, _SO)
                return _SO
            errs.append(f"{cc} {' '.join(omp)}: {r.stderr.strip()[-400:]}")
    raise RuntimeError("could not build the oracle:\n" + "\n".join(errs))


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        dp = C.POINTER(C.c_double)
        L.orc_sweep_pencil.argtypes = [dp, dp, C.c_int, C.c_double, C.c_int, dp, dp]
        L.orc_sweep_pencil.restype = C.c_int
        L.orc_sweep_x.argtypes = [dp, C.POINTER(_CGrid), C.POINTER(_CBox), C.c_int, C.c_double, dp]
        L.orc_sweep_x.restype = C.c_int
        L.orc_sweep_v.argtypes = [dp, C.POINTER(_CGrid), C.POINTER(_CBox), C.c_double, dp, dp, C.c_int, C.c_double]
        L.orc_sweep_v.restype = C.c_int
        L.orc_step.argtypes = [dp, C.POINTER(_CGrid), C.POINTER(_CBox), C.c_double, dp, dp, C.c_double, dp]
        L.orc_step.restype = C.c_int
        L.orc_moments.argtypes = [dp, C.POINTER(_CGrid), C.POINTER(_CBox), dp, dp, dp]
        L.orc_moments.restype = C.c_int
        L.orc_sum.argtypes = [dp, C.c_size_t]
        L.orc_sum.restype = C.c_double
        L.orc_f_count.argtypes = [C.POINTER(_CGrid)]
        L.orc_f_count.restype = C.c_size_t
        d3, d9 = C.c_double * 3, C.c_double * 9
        L.orc_boris_map.argtypes = [C.c_double, d3, d3, C.c_double, d9, d3]
        L.orc_boris_map.restype = None
        L.orc_backsub_foot.argtypes = [d9, d3, C.c_int, d3]
        L.orc_backsub_foot.restype = C.c_double
        L.orc_sweep_pencil_faces.argtypes = [dp, dp, C.c_int, dp]
        L.orc_sweep_pencil_faces.restype = C.c_int
        L.orc_sweep_v_backsub.argtypes = L.orc_sweep_v.argtypes
        L.orc_sweep_v_backsub.restype = C.c_int
        L.orc_step_backsub.argtypes = L.orc_step.argtypes
        L.orc_step_backsub.restype = C.c_int
        L.orc_maxwellian.argtypes = [C.POINTER(_CGrid), C.POINTER(_CBox), C.c_size_t, dp, dp, dp, dp]
        L.orc_maxwellian.restype = C.c_int
        L.orc_exchange_maxwellian.argtypes = [dp, C.POINTER(_CGrid), C.POINTER(_CBox), C.c_int, C.c_int, dp, dp, dp]
        L.orc_exchange_maxwellian.restype = C.c_int
        L.orc_match_moments.argtypes = [dp, C.POINTER(_CGrid), C.POINTER(_CBox), dp, dp, dp]
        L.orc_match_moments.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        L.orc_set_num_threads.restype = None
        L.orc_num_threads.argtypes = []
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _check_f(f: np.ndarray, grid: Grid):
    if f.dtype != np.float64 or not f.flags["C_CONTIGUOUS"] or f.size != int(np.prod(grid.shape)):
        raise ValueError("f must be C-contiguous float64 with prod(grid.shape) entries")


def sweep_pencil(pencil, s: float, bc: int, return_flux: bool = False):
    """1-D PFC-3 remap of one pencil; returns the new pencil (status raised as ValueError)."""
    a = np.ascontiguousarray(pencil, dtype=np.float64)
    out = np.empty_like(a)
    lo, hi = C.c_double(0.0), C.c_double(0.0)
    st = lib().orc_sweep_pencil(_p(a), _p(out), a.size, float(s), int(bc), C.byref(lo), C.byref(hi))
    if st != OK:
        raise ValueError(f"orc_sweep_pencil status {st}")
    return (out, lo.value, hi.value) if return_flux else out


def sweep_x(f: np.ndarray, grid: Grid, box: Box, dim: int, dt: float) -> float:
    """In-place spatial sweep; returns the net outflow through the axis ends."""
    _check_f(f, grid)
    net = C.c_double(0.0)
    g, b = grid.c(), box.c()
    st = lib().orc_sweep_x(_p(f), C.byref(g), C.byref(b), dim, float(dt), C.byref(net))
    if st != OK:
        raise ValueError(f"orc_sweep_x status {st}")
    return net.value


def sweep_v(f: np.ndarray, grid: Grid, box: Box, q_over_m: float, E: np.ndarray, B: np.ndarray,
            dim: int, dt: float) -> None:
    _check_f(f, grid)
    assert E.size == 3 * grid.n_space and B.size == 3 * grid.n_space
    g, b = grid.c(), box.c()
    st = lib().orc_sweep_v(_p(f), C.byref(g), C.byref(b), float(q_over_m), _p(E), _p(B), dim, float(dt))
    if st != OK:
        raise ValueError(f"orc_sweep_v status {st}")


def step(f: np.ndarray, grid: Grid, box: Box, q_over_m: float, E: np.ndarray, B: np.ndarray,
         dt: float) -> float:
    """One full split step in place; returns the net spatial outflow."""
    _check_f(f, grid)
    assert E.size == 3 * grid.n_space and B.size == 3 * grid.n_space
    net = C.c_double(0.0)
    g, b = grid.c(), box.c()
    st = lib().orc_step(_p(f), C.byref(g), C.byref(b), float(q_over_m), _p(E), _p(B), float(dt), C.byref(net))
    if st != OK:
        raise ValueError(f"orc_step status {st}")
    return net.value


def boris_map(q_over_m: float, E, B, dt: float):
    """Boris map of one spatial cell, v_new = R v_old + c: returns (R 3x3, c 3)."""
    d3, d9 = C.c_double * 3, C.c_double * 9
    R, c = d9(), d3()
    lib().orc_boris_map(float(q_over_m), d3(*map(float, E)), d3(*map(float, B)), float(dt), R, c)
    return np.array(R[:]).reshape(3, 3), np.array(c[:])


def backsub_foot(R, c, dim: int, v) -> float:
    """Foot coordinate of backsubstituted sweep `dim` at the point v (see mphv_oracle.c)."""
    d3, d9 = C.c_double * 3, C.c_double * 9
    Rf = [float(x) for x in np.asarray(R).reshape(9)]
    return float(lib().orc_backsub_foot(d9(*Rf), d3(*map(float, c)), int(dim), d3(*map(float, v))))


def sweep_pencil_faces(pencil, s_face):
    """Closed-box 1-D PFC-3 remap with one Courant number per face (n + 1 of them)."""
    a = np.ascontiguousarray(pencil, dtype=np.float64)
    sf = np.ascontiguousarray(s_face, dtype=np.float64)
    assert sf.size == a.size + 1
    out = np.empty_like(a)
    st = lib().orc_sweep_pencil_faces(_p(a), _p(out), a.size, _p(sf))
    if st != OK:
        raise ValueError(f"orc_sweep_pencil_faces status {st}")
    return out


def sweep_v_backsub(f: np.ndarray, grid: Grid, box: Box, q_over_m: float, E: np.ndarray, B: np.ndarray,
                    dim: int, dt: float) -> None:
    _check_f(f, grid)
    assert E.size == 3 * grid.n_space and B.size == 3 * grid.n_space
    g, b = grid.c(), box.c()
    st = lib().orc_sweep_v_backsub(_p(f), C.byref(g), C.byref(b), float(q_over_m), _p(E), _p(B), dim, float(dt))
    if st != OK:
        raise ValueError(f"orc_sweep_v_backsub status {st}")


def step_backsub(f: np.ndarray, grid: Grid, box: Box, q_over_m: float, E: np.ndarray, B: np.ndarray,
                 dt: float) -> float:
    """One full split step with the backsubstituted V stage, in place; returns the net spatial outflow."""
    _check_f(f, grid)
    assert E.size == 3 * grid.n_space and B.size == 3 * grid.n_space
    net = C.c_double(0.0)
    g, b = grid.c(), box.c()
    st = lib().orc_step_backsub(_p(f), C.byref(g), C.byref(b), float(q_over_m), _p(E), _p(B), float(dt), C.byref(net))
    if st != OK:
        raise ValueError(f"orc_step_backsub status {st}")
    return net.value


def moments(f: np.ndarray, grid: Grid, box: Box):
    _check_f(f, grid)
    sp = (grid.nx[2], grid.nx[1], grid.nx[0])
    n = np.empty(sp)
    j = np.empty((3,) + sp)
    P = np.empty((6,) + sp)
    g, b = grid.c(), box.c()
    st = lib().orc_moments(_p(f), C.byref(g), C.byref(b), _p(n), _p(j), _p(P))
    if st != OK:
        raise ValueError(f"orc_moments status {st}")
    return n, j, P


def maxwellian(grid: Grid, box: Box, n, j, P) -> np.ndarray:
    """Ten-moment Maxwellian cubes of `count` cells: n [count], j [3][count], P [6][count] -> [count][nvz][nvy][nvx]."""
    n = np.ascontiguousarray(n, dtype=np.float64).reshape(-1)
    count = n.size
    j = np.ascontiguousarray(j, dtype=np.float64).reshape(3, count)
    P = np.ascontiguousarray(P, dtype=np.float64).reshape(6, count)
    out = np.empty((count, grid.nv[2], grid.nv[1], grid.nv[0]))
    g, b = grid.c(), box.c()
    st = lib().orc_maxwellian(C.byref(g), C.byref(b), count, _p(n), _p(j), _p(P), _p(out))
    if st != OK:
        raise ValueError(f"orc_maxwellian status {st}")
    return out


def exchange_maxwellian(f: np.ndarray, grid: Grid, box: Box, dim: int, side: int, n_fl, j_fl, P_fl) -> None:
    """Exchange of Maxwellians in the two boundary layers at one end of spatial axis dim, in place."""
    _check_f(f, grid)
    plane = grid.n_space // grid.nx[dim]
    n_fl = np.ascontiguousarray(n_fl, dtype=np.float64); assert n_fl.size == 2 * plane
    j_fl = np.ascontiguousarray(j_fl, dtype=np.float64); assert j_fl.size == 6 * plane
    P_fl = np.ascontiguousarray(P_fl, dtype=np.float64); assert P_fl.size == 12 * plane
    g, b = grid.c(), box.c()
    st = lib().orc_exchange_maxwellian(_p(f), C.byref(g), C.byref(b), int(dim), int(side), _p(n_fl), _p(j_fl), _p(P_fl))
    if st != OK:
        raise ValueError(f"orc_exchange_maxwellian status {st}")


def match_moments(f: np.ndarray, grid: Grid, box: Box, n_t, j_t, P_t) -> None:
    """f <- M[n_t, j_t, P_t] + (f - M[moments of f]) in every spatial cell, in place."""
    _check_f(f, grid)
    n_t = np.ascontiguousarray(n_t, dtype=np.float64); assert n_t.size == grid.n_space
    j_t = np.ascontiguousarray(j_t, dtype=np.float64); assert j_t.size == 3 * grid.n_space
    P_t = np.ascontiguousarray(P_t, dtype=np.float64); assert P_t.size == 6 * grid.n_space
    g, b = grid.c(), box.c()
    st = lib().orc_match_moments(_p(f), C.byref(g), C.byref(b), _p(n_t), _p(j_t), _p(P_t))
    if st != OK:
        raise ValueError(f"orc_match_moments status {st}")


def total(f: np.ndarray) -> float:
    a = np.ascontiguousarray(f, dtype=np.float64)
    return lib().orc_sum(_p(a), a.size)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    """OpenMP threads of later oracle calls (tiny grids run much faster on one thread)."""
    lib().orc_set_num_threads(int(n))
