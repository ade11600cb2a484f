"""Parity metric of SURVEY.md sec. 8(c) / DESIGN.md: per cell, |gpu - oracle| divided by the
largest |oracle| value in the 5-point neighbourhood along a given axis (values of f span
e^-50, the scheme's rounding error scales with the stencil's magnitude, not with |f_i|)."""
import numpy as np

TOL_SWEEP = 1e-12      # BASELINE.json north_star: max relative error 1e-12 per step
TOL_MASS = 1e-13


def local_scale(ref: np.ndarray, axis: int, periodic: bool = False) -> np.ndarray:
    a = np.abs(ref)
    out = a.copy()
    n = a.shape[axis]
    for sh in (-2, -1, 1, 2):
        if periodic:
            out = np.maximum(out, np.roll(a, sh, axis=axis))
        else:
            idx = np.clip(np.arange(n) + sh, 0, n - 1)
            out = np.maximum(out, np.take(a, idx, axis=axis))
    return out


def rel_err(gpu: np.ndarray, ref: np.ndarray, axis: int) -> float:
    scale = np.maximum(local_scale(ref, axis), 1e-300)
    return float(np.max(np.abs(gpu - ref) / scale))


def moments_err(gpu, ref, absref) -> float:
    """|delta| / (sum |v_a v_b| f dV), the absolute-sum scale (j and off-diagonal P cancel)."""
    return float(np.max(np.abs(gpu - ref) / np.maximum(absref, 1e-300)))


MOMENT_PAIRS = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]          # order of the six components of P


def moment_scales(ref: np.ndarray, w, chunk: int = 512):
    """The per-component scales of SURVEY 8(c): (n, j[3], P[6]) of sum |v_a v_b| |f| dV per spatial cell, for ANY size
    of f. By separability the weights |vx|^p |vy|^q |vz|^r are applied axis by axis (three small matrix products per
    block of spatial cells), so no temporary of the size of f is made. w: the workload (v_centres, dv)."""
    nz, ny, nx, nvz, nvy, nvx = ref.shape
    ns = nz * ny * nx
    f = ref.reshape(ns, nvz, nvy, nvx)
    pw = [np.stack([np.ones_like(v), np.abs(v), v * v], axis=1) for v in (w.v_centres(0), w.v_centres(1), w.v_centres(2))]
    dV = w.dv(0) * w.dv(1) * w.dv(2)
    T = np.empty((ns, 3, 3, 3))                                         # [cell, power of vz, of vy, of vx]
    for c0 in range(0, ns, chunk):
        a = np.abs(f[c0:c0 + chunk])
        a = a @ pw[0]                                                   # (c, nvz, nvy, 3x)
        a = np.einsum("czyx,yq->czqx", a, pw[1])                        # (c, nvz, 3y, 3x)
        T[c0:c0 + chunk] = np.einsum("czqx,zr->crqx", a, pw[2])         # (c, 3z, 3y, 3x)
    T *= dV
    sp = (nz, ny, nx)

    def pick(px, py, pz):
        return T[:, pz, py, px].reshape(sp)
    n_s = pick(0, 0, 0)
    j_s = np.stack([pick(1, 0, 0), pick(0, 1, 0), pick(0, 0, 1)])
    P_s = np.stack([pick(*[(a == d) + (b == d) for d in range(3)]) for a, b in MOMENT_PAIRS])
    return n_s, j_s, P_s


def moments_worst(got, ref_moments, scales) -> float:
    """max over the ten components and all spatial cells of |gpu - oracle| / (its own absolute-sum scale)."""
    worst = 0.0
    for g, r, s in zip(got, ref_moments, scales):
        g = g.cpu().numpy() if hasattr(g, "cpu") else np.asarray(g)
        worst = max(worst, float(np.max(np.abs(g.reshape(r.shape) - r) / np.maximum(s.reshape(r.shape), 1e-300))))
    return worst
