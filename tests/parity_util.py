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
