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


def test_exported_symbols_are_exactly_the_declared_ones(libpath):
    """Nothing is exported that include/foremoe.h does not declare (nm -D), debug setters included."""
    import subprocess
    hdr = open(os.path.join(ROOT, "include", "foremoe.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(?:int|void)\s+(foremoe_\w+)\s*\(", hdr))
    out = subprocess.run(["nm", "-D", "--defined-only", libpath], capture_output=True, text=True, check=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln and ln.split()[-1].startswith("foremoe_")}
    assert exported == declared, (exported ^ declared)
    # the boundary keeps no tunable global state: sweep knobs exist only in the
    # separate -DFOREMOE_TUNING build, never in the product library or its header
    assert not [n for n in exported if "debug" in n or "tuning" in n]


@pytest.mark.parametrize("lang,std", [("c", "c99"), ("c", "c11"), ("c++", "c++14")])
def test_header_is_plain_c(tmp_path, lang, std):
    """The boundary is a C ABI: the header compiles on its own as C and as C++ (no torch, no CUDA types)."""
    import subprocess
    src = tmp_path / ("t." + ("c" if lang == "c" else "cpp"))
    src.write_text('#include "foremoe.h"\nint main(void) { foremoe_shape_t s; (void)s; return sizeof(s) == 48 ? 0 : 1; }\n')
    exe = tmp_path / "t"
    subprocess.run(["gcc" if lang == "c" else "g++", "-std=" + std, "-Wall", "-Wextra", "-Werror", "-pedantic",
                    "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    assert subprocess.run([str(exe)]).returncode == 0          # 12 x int32: the ctypes mirror has the same size
    assert C.sizeof(fm._CShape) == 48


def test_workspace_bytes_and_invalid_shapes(libpath):
    s = fm.Shape(L=48, E=128, K=8, P=8, Nb=16, Nr=2, T=524288, n_mb=32, H=2048)
    n = fm.workspace_bytes(s)
    assert 0 < n < (1 << 30)
    import dataclasses
    for bad in (dict(K=0), dict(K=33), dict(E=127), dict(Nb=15), dict(H=7), dict(n_mb=0),
                dict(act_dtype=2), dict(T=(1 << 31) // 8), dict(placement_mb_stride=5), dict(flags=2)):
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
    assert lib.foremoe_plan(C.byref(cs), *([None] * 12), 0, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_dispatch(C.byref(cs), 0, 0, 1, None, None, None, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_combine(C.byref(cs), 0, 0, 1, None, None, None, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_step_host(C.byref(cs), *([None] * 10), 0, None, None) == fm.ERR_INVALID_ARG
    # the widened entry points check their arguments on the host as well
    assert lib.foremoe_combine_bwd(C.byref(cs), 0, 0, 1, *([None] * 9)) == fm.ERR_INVALID_ARG
    assert lib.foremoe_dispatch_bwd(C.byref(cs), 0, 0, 1, *([None] * 6)) == fm.ERR_INVALID_ARG
    assert lib.foremoe_base_placement(C.byref(cs), None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_base_placement_machines(C.byref(cs), 2, 1, 1, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_microstep_placement(C.byref(cs), 1, None, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_replication(C.byref(cs), 1, None, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_swap_relocation(C.byref(cs), 1, 2, 8, 1, 0, None, None, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_source_ids(C.byref(cs), 2, None, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_local_placement(C.byref(cs), 2, None, None, None, None) == fm.ERR_INVALID_ARG
    assert lib.foremoe_traffic(C.byref(cs), 2, None, None, None) == fm.ERR_INVALID_ARG
    for M in (0, 3):                                  # M must divide P = 4
        one = (C.c_int32 * 64)()
        assert lib.foremoe_traffic(C.byref(cs), M, one, one, None) == fm.ERR_INVALID_ARG


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    monkeypatch.setattr(fm, "_lib", None)
    monkeypatch.setattr(fm, "LIB_PATH", str(tmp_path / "missing.so"))
    with pytest.raises(ImportError):
        fm.lib()


def test_launch_fact_memo_keeps_several_shapes_per_kernel(tmp_path):
    """The per-device memo of launch facts holds four shapes per kernel instantiation at once (keys that
    are all multiples of 32 must not share one way): tests/memo_check.cu, host code only."""
    import subprocess
    exe = tmp_path / "memo_check"
    subprocess.run([fbuild.NVCC, "-std=c++17", "-O1", os.path.join(ROOT, "tests", "memo_check.cu"), "-o", str(exe)],
                   check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0 and "memo ok" in out.stdout, out.stdout + out.stderr
