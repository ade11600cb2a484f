"""mphv_sum_noalloc against the existing mass sum (mphv_sum_f), on the GPU.

mphv_sum_noalloc is the one entry point for callers that cannot allocate device memory: host codes
whose own memory manager already holds all of HBM (a cudaMalloc inside the library would fail there)
and callers inside a time loop, where cudaMalloc / cudaFree would synchronise the device. Its partial
sums live in a static device array of the library instead of a context's workspace (include/mphv.h).

What is checked: its result equals that of the context path mphv_sum_f on the same f within the mass
tolerance the other GPU tests use (1e-13 relative; the two differ only in summation order), and both
equal the exactly rounded host sum. Two calls are made in a row on the shared static array -- a grid
spanning several chunks with a ragged tail first, then a grid smaller than one chunk, so that the second
call runs over what the first one left behind -- and then the first again, which must give the same
bits as before.

This file is named to be collected LAST: it is the newest entry point, and under `pytest -x` a failure
here must not hide the other tests. It passes alone in a fresh process (its first call does the
per-device set-up) and after every other test.
"""
import math

import numpy as np
import pytest

from parity_util import TOL_MASS

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need a GPU"
    return torch


@pytest.fixture(scope="module")
def mphv():
    from paper_2305_01487_b200 import mphv as m
    m.lib()
    return m


def harris(nx, nv, seed_offset):
    from paper_2305_01487_b200 import inputs
    return inputs.Workload(
        name="noalloc", index=1, kind="harris2d", nx=tuple(nx), nv=tuple(nv), bc=(0, 1, 0),
        xlo=(0.0, -6.4, 0.0), xhi=(25.6, 6.4, 12.8), vlo=(-5.0,) * 3, vhi=(5.0,) * 3,
        steps=2, seed_offset=seed_offset)


class Case:
    """One f on the device, bound to a context (the existing path) and summed on the host."""

    def __init__(self, torch, mphv, w):
        from paper_2305_01487_b200 import inputs
        f0, E, B, dt = inputs.make_all(w)
        self.torch, self.mphv = torch, mphv
        self.f = torch.from_numpy(f0).cuda()
        self.E, self.B = torch.from_numpy(E).cuda(), torch.from_numpy(B).cuda()
        self.sim = mphv.Vlasov.from_workload(w)
        self.sim.bind_f(self.f)
        self.sim.set_fields(self.E, self.B)
        self.sim.step(dt)                                    # a realistic f: one full split step of the method
        torch.cuda.synchronize()
        self.exact = math.fsum(self.f.cpu().numpy().ravel().tolist())
        self.out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")

    def existing(self) -> float:
        return self.sim.sum_f()

    def noalloc(self) -> float:
        self.out.fill_(float("nan"))
        self.mphv.mphv_sum_noalloc(self.f.data_ptr(), self.f.numel(), self.out.data_ptr(),
                                   self.torch.cuda.current_stream().cuda_stream)
        self.torch.cuda.synchronize()
        return float(self.out.item())


def test_two_calls_in_a_row_match_the_context_sum(torch_cuda, mphv):
    big = Case(torch_cuda, mphv, harris((16, 12, 1), (16, 12, 12), 31))     # 442 368 doubles: 6 chunks + 49 152
    small = Case(torch_cuda, mphv, harris((8, 8, 1), (8, 8, 8), 32))        # 32 768 doubles: half a chunk
    assert big.f.numel() > 6 * mphv.SUM_NOALLOC_CHUNK and big.f.numel() % mphv.SUM_NOALLOC_CHUNK != 0
    assert small.f.numel() < mphv.SUM_NOALLOC_CHUNK
    first = big.noalloc()                                    # call 1 (does the per-device set-up when run alone)
    second = small.noalloc()                                 # call 2, over call 1's leftovers in the static array
    for got, case in ((first, big), (second, small)):
        ref = case.existing()
        assert ref > 0.0
        assert abs(got - ref) <= TOL_MASS * abs(ref), "static-scratch sum vs mphv_sum_f"
        assert abs(got - case.exact) <= TOL_MASS * abs(case.exact), "static-scratch sum vs the exactly rounded sum"
        assert abs(ref - case.exact) <= TOL_MASS * abs(case.exact)
    assert big.noalloc() == first, "fixed chunks, fixed order: the same bits whatever ran in between"
    assert small.noalloc() == second


def test_signed_data_whole_chunks_and_empty_input(torch_cuda, mphv):
    torch = torch_cuda
    rng = np.random.default_rng(20230501)
    x_host = rng.standard_normal(3 * mphv.SUM_NOALLOC_CHUNK) * np.exp(rng.uniform(-30.0, 3.0, 3 * mphv.SUM_NOALLOC_CHUNK))
    x = torch.from_numpy(x_host).cuda()
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    scale = math.fsum(np.abs(x_host).tolist())
    for count in (x.numel(), 2 * mphv.SUM_NOALLOC_CHUNK + 1, mphv.SUM_NOALLOC_CHUNK, 1):
        mphv.mphv_sum_noalloc(x.data_ptr(), count, out.data_ptr(), stream)
        torch.cuda.synchronize()
        assert abs(float(out.item()) - math.fsum(x_host[:count].tolist())) <= TOL_MASS * scale
    mphv.mphv_sum_noalloc(x.data_ptr(), 0, out.data_ptr(), stream)
    torch.cuda.synchronize()
    assert float(out.item()) == 0.0


def test_sizes_beyond_the_static_array_are_refused(torch_cuda, mphv):
    torch = torch_cuda
    x = torch.ones(16, dtype=torch.float64, device="cuda")
    out = torch.full((1,), -7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(mphv.MphvError) as ei:               # refused before anything is launched or read
        mphv.mphv_sum_noalloc(x.data_ptr(), mphv.SUM_NOALLOC_MAX_COUNT + 1, out.data_ptr(), None)
    assert ei.value.code == mphv.ERR_RANGE and "MPHV_SUM_NOALLOC_MAX_COUNT" in str(ei.value)
    with pytest.raises(mphv.MphvError) as ei:
        mphv.mphv_sum_noalloc(x.data_ptr(), 16, None, None)
    assert ei.value.code == mphv.ERR_ARG
    torch.cuda.synchronize()
    assert float(out.item()) == -7.0
    mphv.mphv_sum_noalloc(x.data_ptr(), 16, out.data_ptr(), None)
    torch.cuda.synchronize()
    assert float(out.item()) == 16.0
