"""ctypes binding of oracle/mphv_fields_oracle.c (FDTD Maxwell update, staggered <-> centred
interpolation, charge current) and the coupled Vlasov-Maxwell step R22 composed from oracle calls.

TEST INFRASTRUCTURE. The arithmetic of the field update is in the C file; `coupled_step` below only
calls oracle functions in the order DESIGN.md R22 states.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import binding as _b

BC_PERIODIC, BC_OUTFLOW = 0, 1


class _CFGrid(C.Structure):
    _fields_ = [("nx", C.c_int32 * 3), ("bc", C.c_int32 * 3), ("dx", C.c_double * 3),
                ("c2", C.c_double), ("inv_eps0", C.c_double)]


@dataclass
class FieldGrid:
    """Spatial lattice of the field solver: extents, boundary rule per axis (R21), cell widths, c^2, 1/eps0."""
    nx: tuple
    bc: tuple
    dx: tuple
    c2: float = 1.0
    inv_eps0: float = 1.0

    def c(self) -> _CFGrid:
        return _CFGrid((C.c_int32 * 3)(*self.nx), (C.c_int32 * 3)(*self.bc), (C.c_double * 3)(*self.dx),
                       float(self.c2), float(self.inv_eps0))

    @property
    def n_space(self) -> int:
        return int(np.prod(self.nx))

    @property
    def shape(self) -> tuple:
        return (3, self.nx[2], self.nx[1], self.nx[0])

    @classmethod
    def of(cls, grid: "_b.Grid", box: "_b.Box", c2: float = 1.0, inv_eps0: float = 1.0) -> "FieldGrid":
        dx = tuple((box.xhi[d] - box.xlo[d]) / grid.nx[d] if grid.nx[d] > 1 else 1.0 for d in range(3))
        return cls(tuple(grid.nx), tuple(grid.bc), dx, c2, inv_eps0)


_ready = False


def _lib():
    global _ready
    L = _b.lib()
    if not _ready:
        dp, gp = C.POINTER(C.c_double), C.POINTER(_CFGrid)
        L.orc_faraday.argtypes = [gp, dp, dp, C.c_double]
        L.orc_ampere.argtypes = [gp, dp, dp, dp, C.c_double]
        L.orc_maxwell_step.argtypes = [gp, dp, dp, dp, C.c_double]
        L.orc_fields_to_centres.argtypes = [gp, dp, dp, dp, dp]
        L.orc_charge_current.argtypes = [C.c_size_t, C.c_int, dp, dp, dp]
        L.orc_div_E.argtypes = [gp, dp, dp]
        L.orc_div_B.argtypes = [gp, dp, dp]
        for name in ("orc_faraday", "orc_ampere", "orc_maxwell_step", "orc_fields_to_centres",
                     "orc_charge_current", "orc_div_E", "orc_div_B"):
            getattr(L, name).restype = C.c_int
        _ready = True
    return L


def _chk(st, what):
    if st != 0:
        raise ValueError(f"{what} status {st}")


def _fld(a, g: FieldGrid):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"] and a.size == 3 * g.n_space
    return a.ctypes.data_as(C.POINTER(C.c_double))


def faraday(g: FieldGrid, E, B, dt: float) -> None:
    """B <- B - dt curl E, in place (eq. (9); lattice R19)."""
    cg = g.c()
    _chk(_lib().orc_faraday(C.byref(cg), _fld(E, g), _fld(B, g), float(dt)), "orc_faraday")


def ampere(g: FieldGrid, E, B, J, dt: float) -> None:
    """E <- E + dt (c^2 curl B - J / eps0), in place; J cell-centred charge current or None (vacuum)."""
    cg = g.c()
    Jp = _fld(J, g) if J is not None else None
    _chk(_lib().orc_ampere(C.byref(cg), _fld(E, g), _fld(B, g), Jp, float(dt)), "orc_ampere")


def maxwell_step(g: FieldGrid, E, B, J, dt: float) -> None:
    """B(dt/2) E(dt; J) B(dt/2), in place."""
    cg = g.c()
    Jp = _fld(J, g) if J is not None else None
    _chk(_lib().orc_maxwell_step(C.byref(cg), _fld(E, g), _fld(B, g), Jp, float(dt)), "orc_maxwell_step")


def to_centres(g: FieldGrid, E, B):
    """(E_c, B_c): the staggered fields interpolated to the cell centres (R20)."""
    Ec, Bc = np.empty(g.shape), np.empty(g.shape)
    cg = g.c()
    _chk(_lib().orc_fields_to_centres(C.byref(cg), _fld(E, g), _fld(B, g), _fld(Ec, g), _fld(Bc, g)),
         "orc_fields_to_centres")
    return Ec, Bc


def charge_current(g: FieldGrid, q, j_list) -> np.ndarray:
    """J = sum_s q_s j_s (eq. (9)); j_list: one [3][nz][ny][nx] number-flux array per species."""
    qa = np.ascontiguousarray(q, dtype=np.float64)
    ja = np.ascontiguousarray(np.stack([np.asarray(j, dtype=np.float64).reshape(g.shape) for j in j_list]))
    J = np.empty(g.shape)
    dp = C.POINTER(C.c_double)
    _chk(_lib().orc_charge_current(g.n_space, len(j_list), qa.ctypes.data_as(dp), ja.ctypes.data_as(dp), _fld(J, g)),
         "orc_charge_current")
    return J


def div_E(g: FieldGrid, E) -> np.ndarray:
    out = np.empty(g.shape[1:])
    cg = g.c()
    _chk(_lib().orc_div_E(C.byref(cg), _fld(E, g), out.ctypes.data_as(C.POINTER(C.c_double))), "orc_div_E")
    return out


def div_B(g: FieldGrid, B) -> np.ndarray:
    out = np.empty(g.shape[1:])
    cg = g.c()
    _chk(_lib().orc_div_B(C.byref(cg), _fld(B, g), out.ctypes.data_as(C.POINTER(C.c_double))), "orc_div_B")
    return out


@dataclass
class Species:
    """One kinetic species of a coupled run: its f (modified in place), phase-space grid and box, charge q
    (enters the current) and q/m (enters the Lorentz force)."""
    f: np.ndarray
    grid: "_b.Grid"
    box: "_b.Box"
    q: float
    q_over_m: float


def coupled_step(g: FieldGrid, species, E, B, dt: float, j_now=None, backsub: bool = False):
    """One step of the coupled scheme R22, in place on every species' f and on the staggered E, B:
        J  = sum_s q_s j_s[f_s];  Maxwell(dt/2; J);  E_c, B_c = centred fields;
        every species: f_s <- step(dt) with E_c, B_c frozen;  J' = sum_s q_s j_s[f_s];  Maxwell(dt/2; J').
    j_now: the species' number fluxes of the present f (as returned by the previous call), else they are
    computed here. Returns the list of the species' moments (n, j, P) of the new f."""
    if j_now is None:
        j_now = [_b.moments(s.f, s.grid, s.box)[1] for s in species]
    q = [s.q for s in species]
    maxwell_step(g, E, B, charge_current(g, q, j_now), 0.5 * dt)
    Ec, Bc = to_centres(g, E, B)
    moms = []
    for s in species:
        if backsub:
            _b.step_backsub(s.f, s.grid, s.box, s.q_over_m, Ec, Bc, dt)
        else:
            _b.step(s.f, s.grid, s.box, s.q_over_m, Ec, Bc, dt)
        moms.append(_b.moments(s.f, s.grid, s.box))
    maxwell_step(g, E, B, charge_current(g, q, [m[1] for m in moms]), 0.5 * dt)
    return moms
