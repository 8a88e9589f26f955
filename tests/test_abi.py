"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol include/fvnl.h declares; the
host-side argument checks that need no device; the product package holds no route into the oracle."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "fvnl.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fvnl_[a-z_]+)\s*\(", src)))


def test_header_declares_the_boundary():
    names = declared_functions()
    for must in ("fvnl_create", "fvnl_set_state", "fvnl_step", "fvnl_get_state", "fvnl_set_bc", "fvnl_destroy",
                 "fvnl_workspace_bytes", "fvnl_set_clock", "fvnl_get_info", "fvnl_strerror"):
        assert must in names


def test_library_builds_loads_and_exports_every_symbol():
    from paper_1311_3004_b200 import build
    path = build.build()
    lib = ctypes.CDLL(path)
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in include/fvnl.h but not exported"


def test_python_binding_has_the_same_names():
    import paper_1311_3004_b200 as P
    for name in declared_functions():
        assert callable(getattr(P, name)), name


def test_host_side_checks_without_a_device():
    import torch
    import paper_1311_3004_b200 as P
    assert P.fvnl_workspace_bytes(3, 8) == 0
    assert P.fvnl_workspace_bytes(8, 8, 16) == 0
    assert 0 < P.fvnl_workspace_bytes(1024, 1024, 32) < P.fvnl_workspace_bytes(1024, 1024, 64) * 0.52
    n = P.fvnl_workspace_bytes(1024, 1024)
    # clock + two states + the analytic ghost cells of the edges (9 doubles per edge cell, two buffers), nothing else
    assert n >= 6 * 1024 * 1024 * 8 and n < 6 * 1024 * 1024 * 8 + 4096 + 2 * (9 * 8 * (4 * 1024 + 12) + 256)
    assert P.fvnl_strerror(0) == "ok"
    assert "argument" in P.fvnl_strerror(P.EARG)
    med = P.fvnl_medium(1500.0, 1000.0, 3.5, 4.3e-6)
    rc, h = P.fvnl_create(2, 2, 1.0, 1.0, med)
    assert rc == P.EARG
    if not torch.cuda.is_available():
        rc, h = P.fvnl_create(16, 16, 1.0, 1.0, med)
        assert rc == P.ECUDA                                  # no CPU fallback: no device -> error
        with pytest.raises(RuntimeError):
            P.Solver(16, 16, 1.0, 1.0, 1500.0, 1000.0, 3.5, 0.0)


def test_product_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_1311_3004_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), f"{f} mentions the oracle"


def test_option_and_kind_constants_match_the_header():
    """The enums of include/fvnl.h and the constants of the Python binding are the same numbers."""
    import paper_1311_3004_b200 as P
    src = open(os.path.join(ROOT, "include", "fvnl.h")).read()
    found = {}
    for body in re.findall(r"enum\s*\{(.*?)\}", src, flags=re.S):
        for name, val in re.findall(r"(FVNL_[A-Z0-9_]+)\s*=\s*(-?\d+)", body):
            found[name] = int(val)
    for name in ("FVNL_OPT_KERNEL", "FVNL_OPT_ROWS_PER_BLOCK", "FVNL_OPT_KERNEL_TIMING", "FVNL_OPT_VARIANT",
                 "FVNL_OPT_SMALL_GRID", "FVNL_KERNEL_DEFAULT", "FVNL_KERNEL_UNFUSED"):
        assert name in found, name
        assert getattr(P, name[len("FVNL_"):]) == found[name], name
