"""C-ABI library: loads, exports every symbol include/lb.h declares, and checks its arguments
without a GPU (no compute calls here)."""
import ctypes as C
import os
import re

import pytest

from paper_2112_08264_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2112_08264_b200.build import build_lib
    build_lib()
    return B.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "lb.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lbs?_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    names = declared_symbols()
    assert len(names) >= 14
    assert sorted(B.SYMBOLS) == names
    for n in names:
        assert hasattr(L, n), n


def test_enums_match_header():
    src = open(os.path.join(ROOT, "include", "lb.h")).read()
    for name in ("LB_OK", "LB_EINVAL", "LB_ENOMEM", "LB_ECUDA", "LB_ESTATE", "LB_F64", "LB_F32",
                 "LB_KERNEL_AUTO", "LB_KERNEL_TWOPASS", "LB_KERNEL_ONEPASS", "LB_KERNEL_TMA", "LB_KERNEL_HALO", "LB_KERNEL_NODE",
                 "LB_OPT_ZC", "LB_OPT_DIAG", "LB_OPT_BALANCE", "LB_MODEL_SHAN_CHEN", "LB_MODEL_COLOUR_GRADIENT"):
        m = re.search(name + r"\s*=\s*(-?\d+)", src)
        assert m and int(m.group(1)) == getattr(B, name), name


@pytest.mark.parametrize("args", [
    (0, 4, 4, 1.0, 1.0, 1.2), (4, -1, 4, 1.0, 1.0, 1.2), (4, 4, 0, 1.0, 1.0, 1.2),
    (4, 4, 4, 0.5, 1.0, 1.2), (4, 4, 4, 1.0, 0.3, 1.2), (4, 4, 4, float("nan"), 1.0, 1.2),
    (4, 4, 4, 1.0, float("inf"), 1.2), (4, 4, 4, 1.0, 1.0, float("nan")), (4, 4, 4, 1.0, 1.0, float("inf")),
    (2048, 2048, 1024, 1.0, 1.0, 1.2),
])
def test_create_rejects_bad_arguments(L, args):
    assert L.lb_create(*args) is None
    assert B.lb_last_error() != ""
    with pytest.raises(B.LBError):
        B.lb_create(*args)


def test_create_rejects_bad_dtype(L):
    assert L.lb_create_ex(4, 4, 4, 1.0, 1.0, 1.2, 7, None) is None


def test_null_context_calls_fail_cleanly(L):
    L.lb_destroy(None)                                   # no-op
    assert L.lb_step(None, 1) == B.LB_EINVAL
    assert L.lb_sync(None) == B.LB_EINVAL
    assert L.lb_set_kernel(None, 0) == B.LB_EINVAL
    assert L.lb_get_populations(None, None) == B.LB_EINVAL
    assert L.lb_launch_count(None) == 0
    assert b"sm_100a" in L.lb_version()


def test_no_gpu_means_loud_failure_not_fallback(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(B.LBError) as ei:
        B.lb_create(8, 8, 8, 1.0, 1.0, 1.2)
    assert "CUDA" in str(ei.value) or "cuda" in str(ei.value)


def _code_lines(path):
    """import / #include lines only (docstrings may name the other side to disown it)."""
    out = []
    for line in open(path):
        t = line.strip()
        if t.startswith(("import ", "from ", "#include")) or "CDLL(" in t or "dlopen" in t:
            out.append(t)
    return "\n".join(out)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2112_08264_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = _code_lines(os.path.join(dirpath, fn))
                assert "oracle" not in txt and "ora" not in txt.replace("import", ""), fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp")):
            txt = _code_lines(os.path.join(ROOT, "oracle", fn))
            assert "paper_2112_08264_b200" not in txt and "csrc" not in txt and "lb.h" not in txt, fn
