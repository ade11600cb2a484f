"""The CUDA path against the PHYSICS directly (not through the oracle): the closed forms the oracle itself is
pinned to (BASELINE.json north_star: free streaming against f0(x - v t, v); gyration in a uniform B), run through
the C ABI on the GPU. A mistake shared by oracle and kernels (both written from the same readings) would still
have to get past these."""
from math import pi, sqrt

import numpy as np
import pytest

from test_gpu_parity import torch_cuda, mphv  # noqa: F401
from test_oracle_backsub import _plane_to_cube, _rotated_gaussian_avg

pytestmark = pytest.mark.gpu


def test_free_streaming_on_gpu_against_the_analytic_solution(torch_cuda, mphv):
    torch = torch_cuda
    nx, nv, steps = 64, 128, 20
    L = 4 * pi
    sim = mphv.Vlasov((nx, 1, 1), (nv, 1, 1), (0, 0, 0), (0, 0, 0), (L, 1, 1), (-6.0, 0, 0), (6.0, 1, 1), 1.0)
    dx, dv = L / nx, 12.0 / nv
    v = -6.0 + (np.arange(nv) + 0.5) * dv
    edges = np.arange(nx + 1) * dx
    gv = np.exp(-0.5 * v ** 2) / sqrt(2 * pi)

    def exact(t):       # x-cell average of (1 + 0.01 cos(0.5 (x - v t))) g(v), v at the cell centre
        lo, hi = edges[:-1, None] - v[None, :] * t, edges[1:, None] - v[None, :] * t
        return (1.0 + 0.01 * (np.sin(0.5 * hi) - np.sin(0.5 * lo)) / (0.5 * dx)) * gv[None, :]

    f = torch.from_numpy(np.ascontiguousarray(exact(0.0).reshape(1, 1, nx, 1, 1, nv))).cuda()
    sim.bind_f(f)
    dt = 0.5 * dx / np.max(np.abs(v))
    m0 = float(f.sum())
    for _ in range(steps):
        sim.sweep_x(0, dt)
    torch.cuda.synchronize()
    got = f.cpu().numpy().reshape(nx, nv)
    assert np.max(np.abs(got - exact(steps * dt))) <= 1e-7          # third-order scheme on a smooth wave
    assert abs(float(f.sum()) - m0) <= 1e-13 * m0 and got.min() >= 0.0


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("fusion", [0, 3])
def test_quarter_gyration_on_gpu_backsubstitution(torch_cuda, mphv, fusion, axis):
    """B = B0 e_axis, E = 0: after N backsubstituted V stages with N theta = pi/2 an off-centre Gaussian is the
    rotated Gaussian up to interpolation error (no splitting error), mass and positivity kept. Every axis in
    turn, as in B5 of tests/test_oracle_backsub.py."""
    torch = torch_cuda
    n, N, vmax, sig, centre = 64, 56, 6.0, 1.0, (1.5, 0.0)
    nv = [n, n, n]
    nv[axis] = 4
    sim = mphv.Vlasov((4, 1, 1), tuple(nv), (0, 0, 0), (0, 0, 0), (1, 1, 1), (-vmax,) * 3, (vmax,) * 3, 1.0)
    sim.set_fusion(fusion)
    sim.set_vmode(mphv.V_BACKSUB)
    b = 2 * np.tan((pi / 2) / N / 2)                                 # Boris angle per step = (pi/2)/N exactly
    E, B = np.zeros((3, 1, 1, 4)), np.zeros((3, 1, 1, 4))
    B[axis] = b
    f0 = _plane_to_cube(_rotated_gaussian_avg(n, vmax, centre, sig, 0.0), n, axis)
    f = torch.from_numpy(np.ascontiguousarray(np.broadcast_to(f0, (1, 1, 4) + f0.shape)).copy()).cuda()
    sim.bind_f(f)
    sim.set_fields(torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda())
    for _ in range(N):
        sim.stage_v(1.0)
    torch.cuda.synchronize()
    got = f.cpu().numpy()
    exact = _plane_to_cube(_rotated_gaussian_avg(n, vmax, centre, sig, pi / 2), n, axis)
    assert got.min() >= 0.0
    assert abs(got.sum() - 4 * f0.sum()) <= 1e-12 * 4 * f0.sum()
    assert np.max(np.abs(got[0, 0, 2] - exact)) / exact.max() <= 6e-3
