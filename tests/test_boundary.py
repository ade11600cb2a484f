"""CPU-side checks of the C-ABI boundary: the CUDA library builds with nvcc for sm_100a,
loads without a GPU, and exports every symbol include/mphv.h declares. No compute calls."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = ROOT / "include" / "mphv.h"


def declared_symbols():
    text = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(mphv_[a-z_0-9]+)\s*\(", text)))


@pytest.fixture(scope="module")
def mphv():
    from paper_2305_01487_b200 import mphv as m
    m.lib()
    return m


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("mphv_create", "mphv_set_fields", "mphv_sweep_x", "mphv_sweep_v", "mphv_step", "mphv_moments"):
        assert name in syms


def test_library_exports_every_declared_symbol(mphv):
    L = C.CDLL(mphv.loaded_library_path())
    syms = declared_symbols()
    assert len(syms) >= 15
    for name in syms:
        assert hasattr(L, name), f"{name} declared in mphv.h but not exported"
    assert sorted(mphv.SYMBOLS) == syms, "binding's SYMBOLS list and header disagree"


def test_binding_has_same_names(mphv):
    for name in declared_symbols():
        assert callable(getattr(mphv, name)), f"python binding lacks {name}"


def test_strerror_and_null_handling_without_gpu(mphv):
    assert mphv.mphv_strerror(0) == "MPHV_OK"
    assert "RANGE" in mphv.mphv_strerror(mphv.ERR_RANGE)
    L = mphv.lib()
    assert L.mphv_f_count(None) == 0
    assert L.mphv_destroy(None) == mphv.ERR_ARG
    assert L.mphv_step(None, 0.1) == mphv.ERR_ARG
    assert L.mphv_create(None, None, 1.0) is None
    assert "NULL" in mphv.mphv_last_error(None)


def test_create_validates_arguments_before_touching_cuda(mphv):
    ok = dict(nx=(8, 1, 1), nv=(8, 1, 1), bc=(0, 0, 0), xlo=(0, 0, 0), xhi=(1, 1, 1),
              vlo=(-1, 0, 0), vhi=(1, 1, 1), q_over_m=1.0)
    for bad in (dict(nx=(0, 1, 1)), dict(nx=(3, 1, 1)), dict(nv=(2, 1, 1)), dict(bc=(2, 0, 0)),
                dict(xhi=(0, 1, 1)), dict(vhi=(-1, 1, 1)), dict(q_over_m=float("nan"))):
        with pytest.raises(mphv.MphvError):
            mphv.mphv_create(**{**ok, **bad})


def test_no_cpu_fallback_create_fails_loudly_without_sm100(mphv):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(mphv.MphvError) as ei:
        mphv.mphv_create((8, 1, 1), (8, 1, 1), (0, 0, 0), (0, 0, 0), (1, 1, 1), (-1, 0, 0), (1, 1, 1), 1.0)
    assert "CUDA" in str(ei.value) or "device" in str(ei.value)


def test_product_never_imports_the_oracle():
    pkg = ROOT / "paper_2305_01487_b200"
    for p in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + [HEADER]:
        txt = p.read_text()
        assert "import oracle" not in txt and "from oracle" not in txt and "mphv_oracle" not in txt, p
    orc = (ROOT / "oracle" / "mphv_oracle.c").read_text() + (ROOT / "oracle" / "binding.py").read_text()
    assert "mphv.h" not in orc and "paper_2305_01487_b200" not in orc.replace("paper_2305_01487_b200/csrc", "")
