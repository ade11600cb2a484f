"""Thin ctypes binding of the C-ABI library ``libmphv.so`` (include/mphv.h).

Argument marshalling only: every step of the path (sweeps, moments, reductions) runs in
the CUDA kernels of ``csrc/``. PyTorch is used for device memory and streams. There is no
CPU fallback: if the library is missing it is built with nvcc, and if no sm_100 GPU is
present ``mphv_create`` fails and :class:`MphvError` is raised.

The module-level functions carry the C names (``mphv_create`` ... ``mphv_moments``) and take
raw device pointers (ints) like the C calls do; :class:`Vlasov` wraps them for torch tensors.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional, Sequence

_PKG = Path(__file__).resolve().parent
_SO = _PKG / "libmphv.so"

BC_PERIODIC, BC_OUTFLOW = 0, 1
OK, ERR_ARG, ERR_STATE, ERR_RANGE, ERR_CUDA, ERR_ARCH = 0, 1, 2, 3, 4, 5

# every symbol include/mphv.h declares (tests check the library exports each of them)
SYMBOLS = (
    "mphv_create", "mphv_destroy", "mphv_set_stream", "mphv_f_count", "mphv_space_count",
    "mphv_bind_f", "mphv_set_fields", "mphv_sweep_x", "mphv_sweep_v", "mphv_step",
    "mphv_moments", "mphv_step_moments", "mphv_run_host", "mphv_step_fields_host", "mphv_sum_f", "mphv_sum_noalloc", "mphv_launch_count",
    "mphv_set_fusion", "mphv_set_vmode", "mphv_maxwellian", "mphv_exchange_maxwellian", "mphv_match_moments", "mphv_strerror", "mphv_last_error",
    "mphv_set_timing", "mphv_timing_slots", "mphv_get_timing", "mphv_get_timing_moved",
    "mphv_stage_x", "mphv_stage_x_halo", "mphv_stage_v", "mphv_halo_count", "mphv_pack_halo", "mphv_sweep_x_halo",
    "mphv_set_fields_deferred", "mphv_deferred_status",
    "mphv_maxwell_create", "mphv_maxwell_destroy", "mphv_maxwell_set_stream", "mphv_maxwell_bind", "mphv_maxwell_faraday",
    "mphv_maxwell_ampere", "mphv_maxwell_step", "mphv_maxwell_centre", "mphv_maxwell_current", "mphv_maxwell_last_error",
    "mphv_plasma_create", "mphv_plasma_destroy", "mphv_plasma_set_concurrent", "mphv_plasma_step", "mphv_plasma_sync", "mphv_plasma_invalidate_moments",
    "mphv_plasma_moments", "mphv_plasma_centred_fields", "mphv_plasma_last_error", "mphv_set_vstage_generation",
)


class MphvError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"[{code}] {text}")
        self.code = code


class mphv_grid(C.Structure):
    _fields_ = [("nx", C.c_int32 * 3), ("nv", C.c_int32 * 3), ("bc", C.c_int32 * 3)]


class mphv_box(C.Structure):
    _fields_ = [("xlo", C.c_double * 3), ("xhi", C.c_double * 3),
                ("vlo", C.c_double * 3), ("vhi", C.c_double * 3)]


class mphv_field_grid(C.Structure):
    _fields_ = [("nx", C.c_int32 * 3), ("bc", C.c_int32 * 3), ("dx", C.c_double * 3),
                ("c2", C.c_double), ("inv_eps0", C.c_double)]


_lib = None


def lib() -> C.CDLL:
    """Load (building first if needed) the CUDA library. Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    so = _build.build()                      # no-op when up to date; raises if nvcc fails
    L = C.CDLL(str(so))
    vp, dbl, i32 = C.c_void_p, C.c_double, C.c_int
    sig = {
        "mphv_create": (vp, [C.POINTER(mphv_grid), C.POINTER(mphv_box), dbl]),
        "mphv_destroy": (i32, [vp]),
        "mphv_set_stream": (i32, [vp, vp]),
        "mphv_f_count": (C.c_size_t, [vp]),
        "mphv_space_count": (C.c_size_t, [vp]),
        "mphv_bind_f": (i32, [vp, vp, vp]),
        "mphv_set_fields": (i32, [vp, vp, vp]),
        "mphv_sweep_x": (i32, [vp, i32, dbl]),
        "mphv_sweep_v": (i32, [vp, i32, dbl]),
        "mphv_step": (i32, [vp, dbl]),
        "mphv_moments": (i32, [vp, vp, vp, vp]),
        "mphv_step_moments": (i32, [vp, dbl, vp, vp, vp]),
        "mphv_run_host": (i32, [vp, vp, i32, dbl, vp, vp, vp]),
        "mphv_step_fields_host": (i32, [vp, vp, vp, dbl, vp, vp, vp]),
        "mphv_sum_f": (i32, [vp, vp]),
        "mphv_sum_noalloc": (i32, [vp, C.c_size_t, vp, vp, C.c_char_p, C.c_size_t]),
        "mphv_launch_count": (C.c_uint64, [vp]),
        "mphv_set_fusion": (i32, [vp, i32]),
        "mphv_set_vmode": (i32, [vp, i32]),
        "mphv_maxwellian": (i32, [vp, C.c_size_t, vp, vp, vp, vp]),
        "mphv_exchange_maxwellian": (i32, [vp, i32, i32, vp, vp, vp]),
        "mphv_match_moments": (i32, [vp, vp, vp, vp]),
        "mphv_set_timing": (i32, [vp, i32]),
        "mphv_timing_slots": (i32, []),
        "mphv_get_timing": (i32, [vp, i32, C.c_char_p, C.c_size_t, C.POINTER(dbl),
                                  C.POINTER(C.c_uint64), C.POINTER(dbl)]),
        "mphv_get_timing_moved": (i32, [vp, i32, C.POINTER(dbl)]),
        "mphv_stage_x": (i32, [vp, dbl]),
        "mphv_stage_x_halo": (i32, [vp, dbl, vp, vp]),
        "mphv_stage_v": (i32, [vp, dbl, vp, vp, vp]),
        "mphv_halo_count": (C.c_size_t, [vp, i32]),
        "mphv_pack_halo": (i32, [vp, i32, i32, vp]),
        "mphv_sweep_x_halo": (i32, [vp, i32, dbl, vp, vp]),
        "mphv_strerror": (C.c_char_p, [i32]),
        "mphv_last_error": (C.c_char_p, [vp]),
        "mphv_set_fields_deferred": (i32, [vp, vp, vp]),
        "mphv_deferred_status": (i32, [vp]),
        "mphv_maxwell_create": (vp, [C.POINTER(mphv_field_grid)]),
        "mphv_maxwell_destroy": (i32, [vp]),
        "mphv_maxwell_set_stream": (i32, [vp, vp]),
        "mphv_maxwell_bind": (i32, [vp, vp, vp]),
        "mphv_maxwell_faraday": (i32, [vp, dbl]),
        "mphv_maxwell_ampere": (i32, [vp, vp, dbl]),
        "mphv_maxwell_step": (i32, [vp, vp, dbl]),
        "mphv_maxwell_centre": (i32, [vp, vp, vp]),
        "mphv_maxwell_current": (i32, [vp, i32, C.POINTER(dbl), C.POINTER(vp), vp]),
        "mphv_maxwell_last_error": (C.c_char_p, [vp]),
        "mphv_plasma_create": (vp, [vp, i32, C.POINTER(vp), C.POINTER(dbl)]),
        "mphv_plasma_destroy": (i32, [vp]),
        "mphv_plasma_set_concurrent": (i32, [vp, i32]),
        "mphv_plasma_step": (i32, [vp, dbl, i32]),
        "mphv_plasma_sync": (i32, [vp]),
        "mphv_plasma_invalidate_moments": (i32, [vp]),
        "mphv_plasma_moments": (i32, [vp, i32, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]),
        "mphv_plasma_centred_fields": (i32, [vp, C.POINTER(vp), C.POINTER(vp)]),
        "mphv_plasma_last_error": (C.c_char_p, [vp]),
        "mphv_set_vstage_generation": (i32, [vp, i32]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def loaded_library_path() -> str:
    lib()
    return str(_SO)


# ------------------------------------------------------------------ C-named functions
def mphv_strerror(code: int) -> str:
    return lib().mphv_strerror(int(code)).decode()


def mphv_last_error(ctx=None) -> str:
    return lib().mphv_last_error(ctx).decode()


def _check(ctx, st: int):
    if st != OK:
        raise MphvError(st, f"{mphv_strerror(st)}: {mphv_last_error(ctx)}")


def mphv_create(nx: Sequence[int], nv: Sequence[int], bc: Sequence[int],
                xlo: Sequence[float], xhi: Sequence[float],
                vlo: Sequence[float], vhi: Sequence[float], q_over_m: float):
    g = mphv_grid((C.c_int32 * 3)(*nx), (C.c_int32 * 3)(*nv), (C.c_int32 * 3)(*bc))
    d3 = C.c_double * 3
    b = mphv_box(d3(*xlo), d3(*xhi), d3(*vlo), d3(*vhi))
    ctx = lib().mphv_create(C.byref(g), C.byref(b), float(q_over_m))
    if not ctx:
        raise MphvError(ERR_ARG, "mphv_create failed: " + mphv_last_error(None))
    return ctx


def mphv_destroy(ctx):
    _check(None, lib().mphv_destroy(ctx))


def mphv_set_stream(ctx, cuda_stream: int):
    _check(ctx, lib().mphv_set_stream(ctx, cuda_stream))


def mphv_f_count(ctx) -> int:
    return int(lib().mphv_f_count(ctx))


def mphv_space_count(ctx) -> int:
    return int(lib().mphv_space_count(ctx))


def mphv_bind_f(ctx, f_dev: int, scratch_dev: Optional[int] = None):
    _check(ctx, lib().mphv_bind_f(ctx, f_dev, scratch_dev))


def mphv_set_fields(ctx, E_dev: int, B_dev: int):
    _check(ctx, lib().mphv_set_fields(ctx, E_dev, B_dev))


def mphv_sweep_x(ctx, dim: int, dt: float):
    _check(ctx, lib().mphv_sweep_x(ctx, int(dim), float(dt)))


def mphv_sweep_v(ctx, dim: int, dt: float):
    _check(ctx, lib().mphv_sweep_v(ctx, int(dim), float(dt)))


def mphv_step(ctx, dt: float):
    _check(ctx, lib().mphv_step(ctx, float(dt)))


def mphv_moments(ctx, n_dev: int, j_dev: int, P_dev: int):
    _check(ctx, lib().mphv_moments(ctx, n_dev, j_dev, P_dev))


def mphv_step_moments(ctx, dt: float, n_dev: int, j_dev: int, P_dev: int):
    _check(ctx, lib().mphv_step_moments(ctx, float(dt), n_dev, j_dev, P_dev))


def mphv_stage_x(ctx, dt: float):
    _check(ctx, lib().mphv_stage_x(ctx, float(dt)))


def mphv_stage_x_halo(ctx, dt: float, lo_dev, hi_dev):
    _check(ctx, lib().mphv_stage_x_halo(ctx, float(dt), lo_dev, hi_dev))


def mphv_stage_v(ctx, dt: float, n_dev=None, j_dev=None, P_dev=None):
    _check(ctx, lib().mphv_stage_v(ctx, float(dt), n_dev, j_dev, P_dev))


def mphv_halo_count(ctx, dim: int) -> int:
    return int(lib().mphv_halo_count(ctx, int(dim)))


def mphv_pack_halo(ctx, dim: int, side: int, buf_dev: int):
    _check(ctx, lib().mphv_pack_halo(ctx, int(dim), int(side), buf_dev))


def mphv_sweep_x_halo(ctx, dim: int, dt: float, lo_dev=None, hi_dev=None):
    _check(ctx, lib().mphv_sweep_x_halo(ctx, int(dim), float(dt), lo_dev, hi_dev))


def mphv_run_host(ctx, f_host: int, nsteps: int, dt: float, n_host=None, j_host=None, P_host=None):
    _check(ctx, lib().mphv_run_host(ctx, f_host, int(nsteps), float(dt), n_host, j_host, P_host))


def mphv_step_fields_host(ctx, E_host: int, B_host: int, dt: float, n_host: int, j_host: int, P_host: int):
    _check(ctx, lib().mphv_step_fields_host(ctx, E_host, B_host, float(dt), n_host, j_host, P_host))


def mphv_sum_f(ctx, sum_dev: int):
    _check(ctx, lib().mphv_sum_f(ctx, sum_dev))


SUM_NOALLOC_CHUNK = 65536
SUM_NOALLOC_MAX_COUNT = 1 << 30


def mphv_sum_noalloc(x_dev: int, count: int, sum_dev: int, stream: int | None = None):
    """Total of ``count`` doubles at ``x_dev`` into the device double at ``sum_dev``, for callers that
    cannot allocate device memory (their own memory manager holds all of HBM, or they are inside a time
    loop where cudaMalloc would stall the device): no context, scratch in a static device array of the
    library. Limits and rules (first call per device during set-up, calls on one device must not overlap
    on the GPU, ``count`` <= ``SUM_NOALLOC_MAX_COUNT``) in include/mphv.h."""
    err = C.create_string_buffer(512)
    st = lib().mphv_sum_noalloc(x_dev, int(count), sum_dev, stream, err, len(err))
    if st != OK:
        raise MphvError(st, f"{mphv_strerror(st)}: {err.value.decode(errors='replace')}")


def mphv_launch_count(ctx) -> int:
    return int(lib().mphv_launch_count(ctx))


V_PLAIN, V_BACKSUB = 0, 1


def mphv_maxwellian(ctx, count: int, n_dev, j_dev, P_dev, f_out_dev):
    _check(ctx, lib().mphv_maxwellian(ctx, int(count), n_dev, j_dev, P_dev, f_out_dev))


def mphv_match_moments(ctx, n_t_dev, j_t_dev, P_t_dev):
    _check(ctx, lib().mphv_match_moments(ctx, n_t_dev, j_t_dev, P_t_dev))


def mphv_exchange_maxwellian(ctx, dim: int, side: int, n_fl_dev, j_fl_dev, P_fl_dev):
    _check(ctx, lib().mphv_exchange_maxwellian(ctx, int(dim), int(side), n_fl_dev, j_fl_dev, P_fl_dev))


def mphv_set_vmode(ctx, mode):
    _check(ctx, lib().mphv_set_vmode(ctx, int(mode)))


def mphv_set_fusion(ctx, level):
    """level: 0 / 1 / 2 as in include/mphv.h; True means the default (1), False means 0."""
    if isinstance(level, bool):
        level = 1 if level else 0
    _check(ctx, lib().mphv_set_fusion(ctx, int(level)))


def mphv_set_timing(ctx, enabled: bool):
    _check(ctx, lib().mphv_set_timing(ctx, 1 if enabled else 0))


def mphv_timing_slots() -> int:
    return int(lib().mphv_timing_slots())


def mphv_get_timing(ctx, slot: int):
    """(name, total_ms, launches, algorithmic bytes per launch) of one timing slot."""
    name = C.create_string_buffer(64)
    ms, n, b = C.c_double(0.0), C.c_uint64(0), C.c_double(0.0)
    _check(ctx, lib().mphv_get_timing(ctx, int(slot), name, 64, C.byref(ms), C.byref(n), C.byref(b)))
    return name.value.decode(), ms.value, int(n.value), b.value


def mphv_get_timing_moved(ctx, slot: int) -> float:
    """Bytes one launch of the slot must move through HBM (one read + one write of f per pass)."""
    b = C.c_double(0.0)
    _check(ctx, lib().mphv_get_timing_moved(ctx, int(slot), C.byref(b)))
    return b.value


# ---- fields and coupled step (include/mphv.h "closing the loop")
def _check_m(m, st: int):
    if st != OK:
        raise MphvError(st, f"{mphv_strerror(st)}: {mphv_maxwell_last_error(m)}")


def _check_p(p, st: int):
    if st != OK:
        raise MphvError(st, f"{mphv_strerror(st)}: {mphv_plasma_last_error(p)}")


def mphv_set_fields_deferred(ctx, E_dev: int, B_dev: int):
    _check(ctx, lib().mphv_set_fields_deferred(ctx, E_dev, B_dev))


def mphv_deferred_status(ctx):
    _check(ctx, lib().mphv_deferred_status(ctx))


def mphv_maxwell_create(nx, bc, dx, c2: float = 1.0, inv_eps0: float = 1.0):
    g = mphv_field_grid((C.c_int32 * 3)(*nx), (C.c_int32 * 3)(*bc), (C.c_double * 3)(*dx), float(c2), float(inv_eps0))
    m = lib().mphv_maxwell_create(C.byref(g))
    if not m:
        raise MphvError(ERR_ARG, "mphv_maxwell_create failed: " + mphv_last_error(None))
    return m


def mphv_maxwell_destroy(m):
    _check_m(None, lib().mphv_maxwell_destroy(m))


def mphv_maxwell_set_stream(m, cuda_stream: int):
    _check_m(m, lib().mphv_maxwell_set_stream(m, cuda_stream))


def mphv_maxwell_bind(m, E_dev: int, B_dev: int):
    _check_m(m, lib().mphv_maxwell_bind(m, E_dev, B_dev))


def mphv_maxwell_faraday(m, dt: float):
    _check_m(m, lib().mphv_maxwell_faraday(m, float(dt)))


def mphv_maxwell_ampere(m, J_dev, dt: float):
    _check_m(m, lib().mphv_maxwell_ampere(m, J_dev, float(dt)))


def mphv_maxwell_step(m, J_dev, dt: float):
    _check_m(m, lib().mphv_maxwell_step(m, J_dev, float(dt)))


def mphv_maxwell_centre(m, Ec_dev: int, Bc_dev: int):
    _check_m(m, lib().mphv_maxwell_centre(m, Ec_dev, Bc_dev))


def mphv_maxwell_current(m, q: Sequence[float], j_dev_ptrs: Sequence[int], J_dev: int):
    n = len(q)
    qa = (C.c_double * n)(*map(float, q))
    ja = (C.c_void_p * n)(*j_dev_ptrs)
    _check_m(m, lib().mphv_maxwell_current(m, n, qa, ja, J_dev))


def mphv_maxwell_last_error(m=None) -> str:
    return lib().mphv_maxwell_last_error(m).decode()


def mphv_plasma_create(m, species_ctx: Sequence, q: Sequence[float]):
    n = len(species_ctx)
    sa = (C.c_void_p * n)(*species_ctx)
    qa = (C.c_double * n)(*map(float, q))
    p = lib().mphv_plasma_create(m, n, sa, qa)
    if not p:
        raise MphvError(ERR_ARG, "mphv_plasma_create failed: " + mphv_last_error(None))
    return p


def mphv_plasma_destroy(p):
    _check_p(None, lib().mphv_plasma_destroy(p))


def mphv_plasma_set_concurrent(p, concurrent: bool):
    _check_p(p, lib().mphv_plasma_set_concurrent(p, 1 if concurrent else 0))


def mphv_plasma_step(p, dt: float, nsteps: int = 1):
    _check_p(p, lib().mphv_plasma_step(p, float(dt), int(nsteps)))


def mphv_plasma_sync(p):
    _check_p(p, lib().mphv_plasma_sync(p))


def mphv_plasma_invalidate_moments(p):
    _check_p(p, lib().mphv_plasma_invalidate_moments(p))


def mphv_plasma_moments(p, s: int):
    """Device pointers (n, j, P) of the latest moments of species s."""
    n, j, P = C.c_void_p(), C.c_void_p(), C.c_void_p()
    _check_p(p, lib().mphv_plasma_moments(p, int(s), C.byref(n), C.byref(j), C.byref(P)))
    return n.value, j.value, P.value


def mphv_plasma_centred_fields(p):
    Ec, Bc = C.c_void_p(), C.c_void_p()
    _check_p(p, lib().mphv_plasma_centred_fields(p, C.byref(Ec), C.byref(Bc)))
    return Ec.value, Bc.value


def mphv_plasma_last_error(p=None) -> str:
    return lib().mphv_plasma_last_error(p).decode()


def mphv_set_vstage_generation(ctx, generation: int):
    _check(ctx, lib().mphv_set_vstage_generation(ctx, int(generation)))


# ------------------------------------------------------------------ torch convenience

class Vlasov:
    """One species on one GPU. Holds the context and references to the bound tensors."""

    def __init__(self, nx, nv, bc, xlo, xhi, vlo, vhi, q_over_m=1.0, device="cuda:0", stream=None):
        import torch
        self.torch = torch
        self.device = torch.device(device)
        self.nx, self.nv = tuple(nx), tuple(nv)
        self.shape = (nx[2], nx[1], nx[0], nv[2], nv[1], nv[0])
        self.space_shape = (nx[2], nx[1], nx[0])
        with torch.cuda.device(self.device):
            self.ctx = mphv_create(nx, nv, bc, xlo, xhi, vlo, vhi, q_over_m)
            if stream is not None:
                mphv_set_stream(self.ctx, stream.cuda_stream)
        self.stream = stream
        self.f = self.scratch = self.E = self.B = None
        self._sum = None

    @classmethod
    def from_workload(cls, w, **kw):
        return cls(w.nx, w.nv, w.bc, w.xlo, w.xhi, w.vlo, w.vhi, w.q_over_m, **kw)

    def _dev(self, t, count):
        torch = self.torch
        if t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != count or t.device != self.device:
            raise ValueError(f"need a contiguous float64 tensor of {count} elements on {self.device}")
        return t.data_ptr()

    def _host(self, t, count):
        torch = self.torch
        if t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != count or t.device.type != "cpu":
            raise ValueError(f"need a contiguous float64 CPU tensor of {count} elements")
        return t.data_ptr()

    def close(self):
        if self.ctx:
            mphv_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def bind_f(self, f, scratch=None):
        n = mphv_f_count(self.ctx)
        mphv_bind_f(self.ctx, self._dev(f, n), None if scratch is None else self._dev(scratch, n))
        self.f, self.scratch = f, scratch

    def set_fields(self, E, B):
        ns = mphv_space_count(self.ctx)
        mphv_set_fields(self.ctx, self._dev(E, 3 * ns), self._dev(B, 3 * ns))
        self.E, self.B = E, B

    def set_fields_deferred(self, E, B):
        ns = mphv_space_count(self.ctx)
        mphv_set_fields_deferred(self.ctx, self._dev(E, 3 * ns), self._dev(B, 3 * ns))
        self.E, self.B = E, B

    def deferred_status(self):
        mphv_deferred_status(self.ctx)

    def sweep_x(self, dim, dt):
        mphv_sweep_x(self.ctx, dim, dt)

    def sweep_v(self, dim, dt):
        mphv_sweep_v(self.ctx, dim, dt)

    def step(self, dt):
        mphv_step(self.ctx, dt)

    def alloc_moments(self):
        torch = self.torch
        sp = self.space_shape
        return (torch.empty(sp, dtype=torch.float64, device=self.device),
                torch.empty((3,) + sp, dtype=torch.float64, device=self.device),
                torch.empty((6,) + sp, dtype=torch.float64, device=self.device))

    def _mom_ptrs(self, n, j, P):
        """Device pointers of a moment triple after the dtype / contiguity / size / device check."""
        ns = mphv_space_count(self.ctx)
        return self._dev(n, ns), self._dev(j, 3 * ns), self._dev(P, 6 * ns)

    def moments(self, out=None):
        n, j, P = out if out is not None else self.alloc_moments()
        mphv_moments(self.ctx, *self._mom_ptrs(n, j, P))
        return n, j, P

    def step_moments(self, dt, out=None):
        n, j, P = out if out is not None else self.alloc_moments()
        mphv_step_moments(self.ctx, dt, *self._mom_ptrs(n, j, P))
        return n, j, P

    def stage_x(self, dt):
        mphv_stage_x(self.ctx, dt)

    def stage_x_halo(self, dt, lo=None, hi=None):
        cnt = self.halo_count(0)
        mphv_stage_x_halo(self.ctx, dt, None if lo is None else self._dev(lo, cnt),
                          None if hi is None else self._dev(hi, cnt))

    def stage_v(self, dt, out=None):
        """The V stage alone; with out = (n, j, P) tensors the moments of the result are written too."""
        if out is None:
            mphv_stage_v(self.ctx, dt)
            return None
        mphv_stage_v(self.ctx, dt, *self._mom_ptrs(*out))
        return out

    def halo_count(self, dim) -> int:
        return mphv_halo_count(self.ctx, dim)

    def pack_halo(self, dim, side, buf):
        mphv_pack_halo(self.ctx, dim, side, self._dev(buf, self.halo_count(dim)))

    def sweep_x_halo(self, dim, dt, lo=None, hi=None):
        cnt = self.halo_count(dim)
        mphv_sweep_x_halo(self.ctx, dim, dt, None if lo is None else self._dev(lo, cnt),
                          None if hi is None else self._dev(hi, cnt))

    def sum_f(self) -> float:
        torch = self.torch
        if self._sum is None:
            self._sum = torch.empty(1, dtype=torch.float64, device=self.device)
        mphv_sum_f(self.ctx, self._sum.data_ptr())
        return float(self._sum.item())

    def run_host(self, f_host, nsteps, dt, n_host=None, j_host=None, P_host=None):
        """f_host etc.: CPU float64 tensors (pinned for speed); updated in place."""
        ns = mphv_space_count(self.ctx)
        mphv_run_host(self.ctx, self._host(f_host, mphv_f_count(self.ctx)), nsteps, dt,
                      None if n_host is None else self._host(n_host, ns),
                      None if j_host is None else self._host(j_host, 3 * ns),
                      None if P_host is None else self._host(P_host, 6 * ns))

    def step_fields_host(self, E_host, B_host, dt, n_host, j_host, P_host):
        """Coupled step with f resident: host fields in, host moments out (CPU float64 tensors, pinned for speed)."""
        ns = mphv_space_count(self.ctx)
        mphv_step_fields_host(self.ctx, self._host(E_host, 3 * ns), self._host(B_host, 3 * ns), dt,
                              self._host(n_host, ns), self._host(j_host, 3 * ns), self._host(P_host, 6 * ns))

    @property
    def launches(self) -> int:
        return mphv_launch_count(self.ctx)

    def maxwellian(self, n, j, P, out=None):
        """Ten-moment Maxwellian cubes of n.numel() cells (device tensors n [count], j [3][count], P [6][count])."""
        torch = self.torch
        count = n.numel()
        nvel = self.nv[0] * self.nv[1] * self.nv[2]
        if out is None:
            out = torch.empty((count, self.nv[2], self.nv[1], self.nv[0]), dtype=torch.float64, device=self.device)
        mphv_maxwellian(self.ctx, count, self._dev(n, count), self._dev(j, 3 * count), self._dev(P, 6 * count),
                        self._dev(out, count * nvel))
        return out

    def match_moments(self, n_t, j_t, P_t):
        mphv_match_moments(self.ctx, *self._mom_ptrs(n_t, j_t, P_t))

    def exchange_maxwellian(self, dim, side, n_fl, j_fl, P_fl):
        """n_fl [2][plane], j_fl [3][2][plane], P_fl [6][2][plane]: fluid moments of the two boundary layers."""
        cnt = 2 * (mphv_space_count(self.ctx) // self.nx[dim])
        mphv_exchange_maxwellian(self.ctx, dim, side, self._dev(n_fl, cnt), self._dev(j_fl, 3 * cnt), self._dev(P_fl, 6 * cnt))

    def set_vmode(self, mode):
        mphv_set_vmode(self.ctx, mode)

    def set_vstage_generation(self, generation: int):
        mphv_set_vstage_generation(self.ctx, generation)

    def set_fusion(self, level):
        mphv_set_fusion(self.ctx, level)

    def set_timing(self, enabled: bool):
        mphv_set_timing(self.ctx, enabled)

    def timings(self):
        """{kernel name: dict(ms=total, launches=count, alg_bytes=per launch)} for slots that ran."""
        out = {}
        for s in range(mphv_timing_slots()):
            name, ms, n, b = mphv_get_timing(self.ctx, s)
            if n:
                out[name] = dict(ms=ms, launches=n, alg_bytes=b, moved_bytes=mphv_get_timing_moved(self.ctx, s))
        return out


def _from_ptr(torch, ptr: int, shape, device, keep):
    """A float64 torch view of library-owned device memory (no copy); `keep` is held so the owner outlives it."""
    n = 1
    for e in shape:
        n *= int(e)

    class _Mem:
        __cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (int(ptr), False), "version": 2}
    t = torch.as_tensor(_Mem(), device=device).view(*shape)
    t._mphv_owner = keep
    return t


class Maxwell:
    """FDTD field solver on the Vlasov cells (readings R19..R21): staggered E, B as [3][nz][ny][nx] tensors."""

    def __init__(self, nx, bc, dx, c2=1.0, inv_eps0=1.0, device="cuda:0"):
        import torch
        self.torch, self.device = torch, torch.device(device)
        self.nx = tuple(nx)
        self.ns = int(nx[0]) * int(nx[1]) * int(nx[2])
        self.shape = (3, nx[2], nx[1], nx[0])
        with torch.cuda.device(self.device):
            self.m = mphv_maxwell_create(nx, bc, dx, c2, inv_eps0)
        self.E = self.B = None

    @classmethod
    def from_workload(cls, w, c2=1.0, inv_eps0=1.0, **kw):
        return cls(w.nx, w.bc, tuple(w.dx(d) if w.nx[d] > 1 else 1.0 for d in range(3)), c2, inv_eps0, **kw)

    def _dev(self, t, count=None):
        torch = self.torch
        count = 3 * self.ns if count is None else count
        if t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != count or t.device != self.device:
            raise ValueError(f"need a contiguous float64 tensor of {count} elements on {self.device}")
        return t.data_ptr()

    def close(self):
        if self.m:
            mphv_maxwell_destroy(self.m)
            self.m = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def bind(self, E, B):
        mphv_maxwell_bind(self.m, self._dev(E), self._dev(B))
        self.E, self.B = E, B

    def faraday(self, dt):
        mphv_maxwell_faraday(self.m, dt)

    def ampere(self, J, dt):
        mphv_maxwell_ampere(self.m, None if J is None else self._dev(J), dt)

    def step(self, J, dt):
        mphv_maxwell_step(self.m, None if J is None else self._dev(J), dt)

    def centre(self, out=None):
        torch = self.torch
        Ec, Bc = out if out is not None else (torch.empty(self.shape, dtype=torch.float64, device=self.device),
                                              torch.empty(self.shape, dtype=torch.float64, device=self.device))
        mphv_maxwell_centre(self.m, self._dev(Ec), self._dev(Bc))
        return Ec, Bc

    def current(self, q, j_list, out=None):
        torch = self.torch
        J = out if out is not None else torch.empty(self.shape, dtype=torch.float64, device=self.device)
        mphv_maxwell_current(self.m, q, [self._dev(j) for j in j_list], self._dev(J))
        return J


class Plasma:
    """Kinetic species coupled through Maxwell's equations (mphv_plasma_*): the coupled step R22."""

    def __init__(self, maxwell: Maxwell, species: Sequence[Vlasov], q: Sequence[float]):
        self.maxwell, self.species = maxwell, list(species)
        self.torch, self.device = maxwell.torch, maxwell.device
        with self.torch.cuda.device(self.device):
            self.p = mphv_plasma_create(maxwell.m, [s.ctx for s in species], q)

    def close(self):
        if self.p:
            mphv_plasma_destroy(self.p)
            self.p = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_concurrent(self, concurrent: bool):
        mphv_plasma_set_concurrent(self.p, concurrent)

    def step(self, dt, nsteps=1):
        mphv_plasma_step(self.p, dt, nsteps)

    def sync(self):
        mphv_plasma_sync(self.p)

    def invalidate_moments(self):
        """Call after changing a species' f by anything but step(): the next step() recomputes the moments."""
        mphv_plasma_invalidate_moments(self.p)

    def moments(self, s: int):
        """(n, j, P) of species s as torch views of the plasma object's device buffers (call sync() first)."""
        n, j, P = mphv_plasma_moments(self.p, s)
        sp = self.maxwell.shape[1:]
        return (_from_ptr(self.torch, n, sp, self.device, self), _from_ptr(self.torch, j, (3,) + sp, self.device, self),
                _from_ptr(self.torch, P, (6,) + sp, self.device, self))

    def centred_fields(self):
        Ec, Bc = mphv_plasma_centred_fields(self.p)
        return (_from_ptr(self.torch, Ec, self.maxwell.shape, self.device, self),
                _from_ptr(self.torch, Bc, self.maxwell.shape, self.device, self))
