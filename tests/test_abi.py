"""Boundary checks that need no GPU: the C-ABI library builds for sm_100a, loads, and exports
every symbol include/echo.h declares; host-side argument validation returns error codes."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2604_09603_b200 import build, echo
    build.build_library()
    return echo.load_library()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "echo.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(echo_[a-z_]+)\s*\(", src)))


def test_header_symbols_exported(lib):
    names = declared_symbols()
    assert {"echo_gate_select", "echo_verify_attn", "echo_accept", "echo_create"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in echo.h but not exported by libecho.so"


def test_binding_lists_same_symbols():
    from paper_2604_09603_b200 import echo
    assert sorted(echo.EXPORTS) == declared_symbols()


def test_strerror_and_workspace(lib):
    assert lib.echo_strerror(0) == b"ok"
    assert b"workspace" in lib.echo_strerror(-3)
    lib.echo_workspace_bytes.restype = C.c_size_t
    assert lib.echo_workspace_bytes(128, 10240, 2048, 64, 0) >= 16 * 2048 * 64 * 129 * 4   # max_splits <= 0: the limit, 16
    assert lib.echo_workspace_bytes(128, 10240, 2048, 64, 2) >= 2 * 2048 * 64 * 129 * 4
    one = lib.echo_workspace_bytes(128, 10240, 2048, 64, 1)                               # unsplit: no partials at all
    assert 10240 * 8 <= one < 4 * 1024 * 1024
    assert lib.echo_workspace_bytes(256, 0, 4096, 0, 1) >= (4096 + 256) * 8               # echo_accept_stochastic statistics
    assert lib.echo_workspace_bytes(-1, 0, 0, 0, 1) == 0
    assert lib.echo_attn_splits(None, 4, 2) == -1


def test_null_arguments_rejected(lib):
    assert lib.echo_gate_select(None, None, None, None, None) == -1
    assert lib.echo_verify_attn(None, None, None, 0, 8, 1, None, None, None, C.c_float(1.0), None) == -1
    assert lib.echo_accept(None, None, None, 0, None, None, None) == -1
    assert lib.echo_gate_keys(None, None, None, None, None, None) == -1
    assert lib.echo_gate_select_keys(None, None, None, None, None, 0, None, None) == -1
    assert lib.echo_accept_stochastic(None, None, None, 0, None, None, None) == -1
    assert lib.echo_calibrate(None, None, C.c_double(0.5), None, None) == -1
    assert lib.echo_draft_expand(None, None, None, None, None, None) == -1
    assert lib.echo_argmax_shard(None, None, None, 8, 8, 0, None, None) == -1
    assert lib.echo_argmax_merge(None, None, None, 1, None, None) == -1
    assert lib.echo_destroy(None) == -1
    assert lib.echo_set_option(None, 1, 1) == -1


def test_create_fails_loudly_without_b200(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    rc = lib.echo_create(C.byref(h), 0, 1 << 20)
    assert rc < 0 and not h.value


def test_no_cpu_fallback_in_binding():
    import torch
    from paper_2604_09603_b200 import echo
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        echo.EchoContext()


def test_product_does_not_import_oracle():
    """the product path never routes through the oracle (bench.py / smoke() may, explicitly)."""
    pkg = os.path.join(ROOT, "paper_2604_09603_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle\b|oracle/|import_module\(.oracle", re.M)
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dp, f)).read()), f
