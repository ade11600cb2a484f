"""The test-side moment scales (parity_util.moment_scales) against the formula of SURVEY 8(c) written out directly."""
import numpy as np

from parity_util import MOMENT_PAIRS, moment_scales, moments_worst


def test_moment_scales_equal_the_direct_absolute_sums():
    from paper_2305_01487_b200 import inputs
    w = inputs.Workload(name="scales", index=1, kind="harris3d", nx=(5, 4, 6), nv=(8, 6, 4), bc=(0, 1, 0),
                        xlo=(0.0, -6.4, 0.0), xhi=(25.6, 6.4, 12.8), vlo=(-5.0, -4.0, -3.0), vhi=(5.0, 4.5, 3.5), steps=1)
    rng = np.random.default_rng(7)
    f = rng.standard_normal(w.shape)                                   # signed on purpose: the scale uses |f|
    vx, vy, vz = (w.v_centres(d) for d in range(3))
    V = [vx[None, None, None, None, None, :], vy[None, None, None, None, :, None], vz[None, None, None, :, None, None]]
    dV = w.dv(0) * w.dv(1) * w.dv(2)
    fa = np.abs(f)
    n_s, j_s, P_s = moment_scales(f, w, chunk=7)                       # ragged last block
    assert np.allclose(n_s, fa.sum(axis=(3, 4, 5)) * dV, rtol=1e-13, atol=0)
    for a in range(3):
        assert np.allclose(j_s[a], (fa * np.abs(V[a])).sum(axis=(3, 4, 5)) * dV, rtol=1e-13, atol=0)
    for k, (a, b) in enumerate(MOMENT_PAIRS):
        assert np.allclose(P_s[k], (fa * np.abs(V[a] * V[b])).sum(axis=(3, 4, 5)) * dV, rtol=1e-13, atol=0)
    ref = (n_s.copy(), j_s.copy(), P_s.copy())
    got = (n_s.copy(), j_s.copy(), P_s.copy())
    got[2][4].flat[3] += 5e-12 * P_s[4].flat[3]                        # one component of one cell off by 5e-12 of its scale
    assert abs(moments_worst(got, ref, (n_s, j_s, P_s)) - 5e-12) < 1e-15
