"""Host-side checks of the boundary (no GPU): the C-ABI library builds for sm_100a, loads, and
exports every symbol include/foremoe.h declares; host-detectable argument errors are reported
without touching CUDA."""
import ctypes as C
import os
import re

import pytest

from paper_2606_11867_b200 import binding as fm
from paper_2606_11867_b200 import build as fbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    return fbuild.build()


def test_header_symbols_exported(libpath):
    hdr = open(os.path.join(ROOT, "include", "foremoe.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\bint\s+(foremoe_\w+)\s*\(", hdr)))
    assert declared == sorted(fm.EXPORTS)
    lib = C.CDLL(libpath)
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.foremoe_version() >= 100


def test_workspace_bytes_and_invalid_shapes(libpath):
    s = fm.Shape(L=48, E=128, K=8, P=8, Nb=16, Nr=2, T=524288, n_mb=32, H=2048)
    n = fm.workspace_bytes(s)
    assert 0 < n < (1 << 30)
    import dataclasses
    for bad in (dict(K=0), dict(K=33), dict(E=127), dict(Nb=15), dict(H=7), dict(n_mb=0),
                dict(act_dtype=2), dict(T=(1 << 31) // 8), dict(placement_mb_stride=5)):
        with pytest.raises(fm.ForeMoEError) as ei:
            fm.workspace_bytes(dataclasses.replace(s, **bad))
        assert ei.value.code == fm.ERR_INVALID_ARG
    # per-micro-step placement stride is accepted
    fm.workspace_bytes(dataclasses.replace(s, placement_mb_stride=s.L * s.S))


def test_null_pointers_rejected_before_any_cuda_call(libpath):
    s = fm.Shape(L=1, E=8, K=2, P=4, Nb=2, Nr=1, T=16, n_mb=1, H=8, act_dtype=fm.ACT_FP32)
    lib = fm.lib()
    cs = s.c()
    assert lib.foremoe_load_hist(C.byref(cs), None, None, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_assign(C.byref(cs), *([None] * 11), 0, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_dispatch(C.byref(cs), 0, 0, 1, None, None, None, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_combine(C.byref(cs), 0, 0, 1, None, None, None, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_step_host(C.byref(cs), *([None] * 10), 0, None, None) == fm.ERR_INVALID_ARG


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    monkeypatch.setattr(fm, "_lib", None)
    monkeypatch.setattr(fm, "LIB_PATH", str(tmp_path / "missing.so"))
    with pytest.raises(ImportError):
        fm.lib()
