"""Test-side marshalling between seeded workloads, the CUDA binding and the oracle (no arithmetic)."""
import numpy as np

from helpers import torch_bf16_to_bits


def dev(a, device="cuda"):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).to(device)


_CTX = {}
GATE = {"path": 0, "cluster": 0}  # ECHO_OPT_GATE_PATH / ECHO_OPT_GATE_CLUSTER that get_ctx() applies (test fixtures set it)


def get_ctx():
    from paper_2604_09603_b200 import echo
    if "ctx" not in _CTX:
        _CTX["ctx"] = echo.EchoContext(0, 1 << 30)
    ctx = _CTX["ctx"]
    ctx.set_option(echo.OPT_FORCE_SPLITS, 0)
    ctx.set_option(echo.OPT_ATTN_PATH, 0)
    ctx.set_option(echo.OPT_NUM_CTAS, 0)
    ctx.set_option(echo.OPT_ATTN_SAFE, 0)
    ctx.set_option(echo.OPT_ATTN_PLAN, 0)
    ctx.set_option(echo.OPT_GATE_PATH, GATE["path"])
    ctx.set_option(echo.OPT_GATE_CLUSTER, GATE["cluster"])
    return ctx


def run_gate_select(ctx, wl, gate=None, capacity=None, schedule=0):
    g = gate or wl.gate
    return ctx.gate_select(dev(wl.cand_offsets), dev(wl.parent), dev(wl.logq), g.depth_mask, g.log_tau, g.w_max,
                           g.budget, g.static_k, capacity=capacity, max_cand=max(1, wl.max_cand), schedule=schedule)


def make_kv(wl, k, v):
    from paper_2604_09603_b200 import echo
    return echo.PagedKV(k, v, dev(wl.page_table), dev(wl.prefix_len))


def assert_selection_equal(got, want):
    assert got["n_selected"] == want["n_selected"]
    n = want["n_selected"]
    for key in ("sel_offsets", "cut_depth", "cand_depth"):
        np.testing.assert_array_equal(got[key][:len(want[key])], want[key], err_msg=key)
    np.testing.assert_array_equal(got["path_score"][:len(want["path_score"])].view(np.uint32),
                                  want["path_score"].view(np.uint32), err_msg="path_score bits")
    for key in ("sel_node", "sel_req", "parent_local", "sel_depth"):
        np.testing.assert_array_equal(got[key][:n], want[key][:n], err_msg=key)
    np.testing.assert_array_equal(got["anc_mask"][:n].reshape(-1, 4), want["anc_mask"][:n], err_msg="anc_mask")


def pools_bits(k, v):
    return torch_bf16_to_bits(k), torch_bf16_to_bits(v)
