"""echo_gate_select_noalloc (include/echo.h): the selection step for callers that cannot allocate -- no context, no
workspace, its scratch a fixed array inside libecho.so.  Checked against the existing path (echo_gate_select) bit for
bit, on two calls in a row whose sizes differ (the second call finds the first one's keys in the shared scratch).
Collected last on purpose (pytest -x: a failure here hides nothing)."""
import numpy as np
import pytest

from paper_2604_09603_b200 import workloads as W
from gpu_util import dev, get_ctx, run_gate_select, assert_selection_equal

pytestmark = pytest.mark.gpu


def _noalloc(echo, ctx, wl, status, schedule=0):
    g = wl.gate
    cap = wl.capacity()
    sel = ctx.alloc_selection(wl.R, wl.N, cap)       # the caller's outputs (allocated by the caller, ahead of the call)
    args = (dev(wl.cand_offsets), dev(wl.parent), dev(wl.logq))
    return sel, args, lambda: echo.gate_select_noalloc(*args, g.depth_mask, g.log_tau, g.w_max, g.budget, sel, status,
                                                       static_k=g.static_k, schedule=schedule,
                                                       max_cand=max(1, wl.max_cand))


@pytest.mark.parametrize("schedule", [0, 1])
def test_noalloc_matches_gate_select_twice_in_a_row(schedule):
    import torch
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    big, small = W.make_config(2), W.make_config(1, R=5)
    assert small.N < big.N <= echo.NOALLOC_MAX_CAND
    want = {}
    for name, wl in (("big", big), ("small", small)):
        for path in (1, 0):                          # the existing path: three kernels, and its default form
            ctx.set_option(echo.OPT_GATE_PATH, path)
            want[name, path] = run_gate_select(ctx, wl, schedule=schedule).to_host()
        assert_selection_equal(want[name, 1], want[name, 0])
    runs = [(name, wl) + _noalloc(echo, ctx, wl, status, schedule) for name, wl in (("big", big), ("small", small), ("big", big))]
    runs[0][4]()                                     # first call on this device: looks up the scratch address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _, _, _, _, call in runs[1:]:                # two calls in a row on one stream, nothing in between
        call()
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "device memory was allocated inside the calls"
    for name, wl, sel, _, _ in runs:
        assert_selection_equal(sel.to_host(), want[name, 0])
    assert int(status.item()) == 0


def test_noalloc_static_trees_and_status_flags():
    import torch
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    wl = W.make_config(2, static=True, gated=False, R=9)
    sel, _, call = _noalloc(echo, ctx, wl, status)
    call()
    assert_selection_equal(sel.to_host(), run_gate_select(ctx, wl).to_host())
    assert int(status.item()) == 0
    offs = np.asarray([0, 3], np.int32)
    parent = np.asarray([-1, 2, 0], np.int32)        # parent[1] = 2 >= 1
    logq = np.asarray([0.0, 0.5, -1.0], np.float32)  # logq > 0
    s2 = ctx.alloc_selection(1, 3, 4)
    echo.gate_select_noalloc(dev(offs), dev(parent), dev(logq), 0, np.zeros(32, np.float32), 0, 3, s2, status)
    f = int(status.item())
    assert f & echo.DEV_BAD_PARENT and f & echo.DEV_BAD_LOGQ


def test_noalloc_rejects_sizes_beyond_its_scratch():
    import torch
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    lib = echo.load_library()
    assert b"ECHO_NOALLOC_MAX_CAND" in lib.echo_strerror(echo.ERR_TOO_LARGE)
    n = echo.NOALLOC_MAX_CAND + 1
    R = (n + 127) // 128
    offs = np.minimum(np.arange(R + 1, dtype=np.int64) * 128, n).astype(np.int32)
    parent = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    logq = torch.zeros(n, dtype=torch.float32, device="cuda")
    sel = ctx.alloc_selection(R, n, 8)
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    with pytest.raises(echo.EchoError) as e:
        echo.gate_select_noalloc(dev(offs), parent, logq, 0, np.zeros(32, np.float32), 0, 8, sel, status)
    assert e.value.code == echo.ERR_TOO_LARGE
    assert lib.echo_gate_select_noalloc(None, None, None, None, None) == echo.ERR_INVALID_ARG
    # exactly at the limit it runs
    sel = ctx.alloc_selection(R, n - 1, 8)
    offs[-1] = n - 1
    echo.gate_select_noalloc(dev(offs), parent[:n - 1], logq[:n - 1], 0, np.zeros(32, np.float32), 0, 8, sel, status)
    got = sel.to_host()
    # equal scores: (request, node) order
    assert got["n_selected"] == 8 and got["sel_req"].tolist() == [0] * 8 and got["sel_node"].tolist() == list(range(8))
    assert int(status.item()) == 0
