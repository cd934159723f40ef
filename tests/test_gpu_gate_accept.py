"""-m gpu parity: echo_gate_select and echo_accept (CUDA, through the C ABI) against the CPU oracle.
Bar: bit-exact selection indices, masks, path-score bits, accepted lengths and slot maps."""
import json
import os

import numpy as np
import pytest

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W
from helpers import oracle_gate_select, packed_tokens, torch_bf16_to_bits
import gpu_util
from gpu_util import dev, get_ctx, run_gate_select, make_kv, assert_selection_equal

pytestmark = pytest.mark.gpu
GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "w1.json")))


@pytest.fixture(autouse=True, params=["auto", "chain", "cluster2", "cluster1"])
def gate_path(request):
    """Every test of this file runs echo_gate_select as the one-cluster kernel with its default cluster size, as the
    three-kernel chain, and as a cluster of two CTAs / one CTA (several requests per thread group; the chain again
    where a CTA would get more than 32 requests)."""
    gpu_util.GATE.update({"auto": dict(path=0, cluster=0), "chain": dict(path=1, cluster=0),
                          "cluster2": dict(path=0, cluster=2), "cluster1": dict(path=0, cluster=1)}[request.param])
    yield request.param
    gpu_util.GATE.update(path=0, cluster=0)


def _w1_workload():
    offs = np.asarray(GOLD["cand_offsets"], np.int32)
    parent = np.asarray(GOLD["parent"], np.int32)
    logq = np.asarray(GOLD["logq"], np.float32)
    return offs, parent, logq


@pytest.mark.parametrize("B", list(range(0, 11)))
def test_w1_selection_all_budgets(B):
    ctx = get_ctx()
    offs, parent, logq = _w1_workload()
    sel = ctx.gate_select(dev(offs), dev(parent), dev(logq), 0, np.zeros(32, np.float32), 0, B, capacity=16)
    want = orc.gate_select(offs, parent, logq, 0, np.zeros(32, np.float32), 0, B)
    assert_selection_equal(sel.to_host(), want)
    if B in (6, 7):
        g = GOLD[f"B{B}"]
        assert np.diff(sel.to_host()["sel_offsets"]).tolist() == g["K"]


def test_w1_gated_priority():
    ctx = get_ctx()
    offs, parent, logq = _w1_workload()
    g = GOLD["gated"]
    lt = np.zeros(32, np.float32)
    lt[g["depth"]] = np.float32(np.log(np.float64(g["tau"])))
    for B in (8, 9):
        sel = ctx.gate_select(dev(offs), dev(parent), dev(logq), 1 << g["depth"], lt, g["w_max"], B, capacity=16)
        want = orc.gate_select(offs, parent, logq, 1 << g["depth"], lt, g["w_max"], B)
        got = sel.to_host()
        assert_selection_equal(got, want)
        assert got["cut_depth"].tolist() == g["cut_depth"]


CASES = [(0, True, False, None), (0, False, False, None), (1, True, False, None), (1, False, False, None),
         (2, True, False, None), (2, False, True, None), (3, True, False, None), (4, True, False, None),
         (2, True, False, 7), (3, False, False, 3)]


@pytest.mark.parametrize("cfg,gated,static,R", CASES)
def test_gate_select_configs(cfg, gated, static, R):
    ctx = get_ctx()
    wl = W.make_config(cfg, gated=gated, static=static, R=R)
    sel = run_gate_select(ctx, wl)
    want = oracle_gate_select(orc, wl)
    assert_selection_equal(sel.to_host(), want)
    assert ctx.device_status() == 0


@pytest.mark.parametrize("budget", [0, 1, 5, 95, 96, 500])
def test_gate_select_budget_edges(budget):
    ctx = get_ctx()
    wl = W.make_config(0, gated=True)
    g = wl.gate.replace(budget=budget)
    sel = run_gate_select(ctx, wl, g, capacity=max(1, min(budget, wl.N)))
    assert_selection_equal(sel.to_host(), oracle_gate_select(orc, wl, g))


def test_gate_select_ties_and_special_values():
    """equal scores across requests and -inf confidences: order (score desc, request, node)."""
    ctx = get_ctx()
    R, C = 6, 9
    offs = np.arange(R + 1, dtype=np.int32) * C
    parent = np.tile(np.asarray([-1, 0, 0, 1, 1, 2, 2, 3, 3], np.int32), R)
    logq = np.tile(np.asarray([0, -1, -1, -0.5, -0.5, -0.5, -np.inf, -2, -2], np.float32), R)
    for B in (1, 5, 6, 7, 13, 20, 30, 54):
        sel = ctx.gate_select(dev(offs), dev(parent), dev(logq), 0, np.zeros(32, np.float32), 0, B, capacity=64)
        want = orc.gate_select(offs, parent, logq, 0, np.zeros(32, np.float32), 0, B)
        assert_selection_equal(sel.to_host(), want)


def test_gate_select_strict_threshold_and_absent_level():
    ctx = get_ctx()
    offs = np.asarray([0, 3, 6], np.int32)
    parent = np.asarray([-1, 0, 1, -1, 0, 1], np.int32)
    logq = np.asarray([-0.5, -0.25, -0.25, -0.5, -0.5, -0.25], np.float32)
    lt = np.zeros(32, np.float32)
    lt[1] = np.float32(-0.75)   # request 0: m = -0.75 == tau -> fail (strict); request 1: -1.0 fails
    lt[7] = np.float32(0.0)     # absent level: skipped
    mask = (1 << 1) | (1 << 7)
    sel = ctx.gate_select(dev(offs), dev(parent), dev(logq), mask, lt, 1, 6, capacity=8)
    want = orc.gate_select(offs, parent, logq, mask, lt, 1, 6)
    got = sel.to_host()
    assert_selection_equal(got, want)
    assert got["cut_depth"].tolist() == [1, 1]


def test_device_status_flags_bad_inputs():
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    offs = np.asarray([0, 3], np.int32)
    parent = np.asarray([-1, 2, 0], np.int32)       # parent[1] = 2 >= 1
    logq = np.asarray([0.0, 0.5, -1.0], np.float32)  # logq > 0
    ctx.gate_select(dev(offs), dev(parent), dev(logq), 0, np.zeros(32, np.float32), 0, 3, capacity=4)
    f = ctx.device_status()
    assert f & echo.DEV_BAD_PARENT and f & echo.DEV_BAD_LOGQ
    assert ctx.device_status() == 0


def test_gate_select_empty_batch_and_requests_without_candidates():
    """R = 0 selects nothing and writes sel_offsets[0] = n_selected = 0; requests without candidates (equal
    offsets) sit between requests that have some, first and last included."""
    import torch
    ctx = get_ctx()
    z32 = lambda n: torch.zeros(n, dtype=torch.int32, device="cuda")
    sel = ctx.gate_select(z32(1), z32(0), torch.zeros(0, device="cuda"), 0, np.zeros(32, np.float32), 0, 8, capacity=8)
    torch.cuda.synchronize()
    assert int(sel.n_selected.item()) == 0 and int(sel.sel_offsets[0].item()) == 0
    assert ctx.device_status() == 0
    wl = W.make_config(0, gated=True)
    sizes = np.diff(wl.cand_offsets)
    keep = np.ones(wl.R, bool)
    keep[[0, wl.R // 2, wl.R - 1]] = False
    offs = np.concatenate([[0], np.cumsum(np.where(keep, sizes, 0))]).astype(np.int32)
    rows = np.concatenate([np.arange(wl.cand_offsets[i], wl.cand_offsets[i + 1]) for i in range(wl.R) if keep[i]])
    parent, logq = wl.parent[rows], wl.logq[rows]
    g = wl.gate
    for budget in (5, g.budget):
        sel = ctx.gate_select(dev(offs), dev(parent), dev(logq), g.depth_mask, g.log_tau, g.w_max, budget,
                              capacity=max(1, budget))
        want = orc.gate_select(offs, parent, logq, g.depth_mask, g.log_tau, g.w_max, budget)
        assert_selection_equal(sel.to_host(), want)
    assert ctx.device_status() == 0


def test_device_status_flags_overflows():
    """a request with more than 128 candidates (declared as 128) and a chain deeper than 31: flagged, never a trap,
    and the well-formed request next to them is still selected from"""
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    n_big = 140
    offs = np.asarray([0, n_big, n_big + 40, n_big + 43], np.int32)
    parent = np.concatenate([np.full(n_big, -1), np.arange(-1, 39), [-1, 0, 0]]).astype(np.int32)   # roots; one chain; a tree
    logq = np.full(len(parent), -0.1, np.float32)
    sel = ctx.gate_select(dev(offs), dev(parent), dev(logq), 0, np.zeros(32, np.float32), 0, 16, capacity=16, max_cand=128)
    got = sel.to_host()
    f = ctx.device_status()
    assert f & echo.DEV_CAND_OVERFLOW and f & echo.DEV_DEPTH_OVERFLOW
    assert got["n_selected"] <= 16 and got["sel_offsets"][-1] == got["n_selected"]
    assert ctx.device_status() == 0


def test_error_codes_on_gpu():
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    wl = W.make_config(0)
    with pytest.raises(echo.EchoError) as e:
        run_gate_select(ctx, wl, wl.gate.replace(budget=32), capacity=8)     # capacity < budget
    assert e.value.code == echo.ERR_INVALID_ARG
    with pytest.raises(echo.EchoError) as e:
        run_gate_select(ctx, wl, wl.gate.replace(budget=-1), capacity=8)
    assert e.value.code == echo.ERR_INVALID_ARG


# ------------------------------------------------------------------------------ acceptance
def _accept_case(wl, gate=None, num_layers=2, logits=False):
    import torch
    ctx = get_ctx()
    sel = run_gate_select(ctx, wl, gate)
    hs = sel.to_host()
    want_sel = oracle_gate_select(orc, wl, gate)
    assert_selection_equal(hs, want_sel)
    draft, target, glob = packed_tokens(wl, want_sel)
    cap = sel.capacity
    n = want_sel["n_selected"]
    dpad = np.zeros(max(1, cap), np.int32); dpad[:n] = draft
    tpad = np.zeros(max(1, cap), np.int32); tpad[:n] = target
    _, k, v = W.draw_qkv(wl, 1, device="cuda", num_layers=num_layers)
    kb, vb = torch_bf16_to_bits(k).copy(), torch_bf16_to_bits(v).copy()
    kv = make_kv(wl, k, v)
    if logits:
        lg = W.draw_logits(wl, glob, device="cuda")
        if lg.shape[0] < cap:
            lg = torch.cat([lg, torch.zeros(cap - lg.shape[0], lg.shape[1], dtype=lg.dtype, device="cuda")])
        acc = ctx.accept(sel, kv, dev(dpad), dev(wl.prev_token), target_logits=lg, vocab=wl.vocab)
        tt = orc.argmax_bf16(torch_bf16_to_bits(lg[:n]), wl.vocab)
        np.testing.assert_array_equal(acc.target_token[:n].cpu().numpy(), tt)
        target = tt
    else:
        acc = ctx.accept(sel, kv, dev(dpad), dev(wl.prev_token), target_token=dev(tpad))
    want = orc.accept(want_sel, draft, wl.prev_token, target, wl.R)
    wc = orc.compact_kv(want_sel, want, kb, vb, wl.page_table, wl.prefix_len, wl.R)
    got = acc.to_host()
    for key in ("accept_len", "last_node", "bonus_token", "accept_idx"):
        np.testing.assert_array_equal(got[key][:wl.R], want[key], err_msg=key)
    for key in ("slot_src", "slot_dst", "new_len"):
        np.testing.assert_array_equal(got[key][:wl.R], wc[key], err_msg=key)
    np.testing.assert_array_equal(torch_bf16_to_bits(k), kb, err_msg="compacted K pool")
    np.testing.assert_array_equal(torch_bf16_to_bits(v), vb, err_msg="compacted V pool")
    return got


@pytest.mark.parametrize("cfg,gated,static,R", [(0, True, False, None), (0, False, False, None),
                                                 (1, True, False, None), (2, True, False, 16),
                                                 (2, False, True, 8), (3, True, False, 16), (4, True, False, 24)])
def test_accept_configs(cfg, gated, static, R):
    wl = W.make_config(cfg, gated=gated, static=static, R=R)
    got = _accept_case(wl)
    assert got["accept_len"].max() <= 32


def test_accept_w1():
    ctx = get_ctx()
    offs, parent, logq = _w1_workload()
    a = GOLD["accept"]
    sel = ctx.gate_select(dev(offs), dev(parent), dev(logq), 0, np.zeros(32, np.float32), 0, a["budget"], capacity=8)
    draft = np.zeros(8, np.int32); draft[:4] = a["draft_token"]; draft[4:7] = [1, 2, 3]
    target = np.zeros(8, np.int32); target[:4] = a["target_token"]
    import torch
    from paper_2604_09603_b200 import echo
    pt = np.asarray([a["page_table"], [0, 1]], np.int32)
    k = torch.zeros(1, 8, 1, 16, 128, dtype=torch.bfloat16, device="cuda")
    kv = echo.PagedKV(k, k.clone(), dev(pt), dev(np.asarray([a["prefix_len"], 3], np.int32)))
    acc = ctx.accept(sel, kv, dev(draft), dev(np.asarray([a["prev_token"], 999], np.int32)), target_token=dev(target))
    got = acc.to_host()
    assert got["accept_len"].tolist() == [a["accept_len"], 0]
    assert got["bonus_token"].tolist() == [a["bonus_token"], -1]
    assert got["slot_src"][0, :3].tolist() == a["slot_src"]
    assert got["slot_dst"][0, :3].tolist() == a["slot_dst"]
    assert got["new_len"].tolist() == [a["new_len"], 3]
    assert (got["accept_idx"][1] == -1).all() and got["last_node"].tolist() == [3, -1]


def test_accept_logits_argmax_small():
    wl = W.make_config(4, R=6)
    _accept_case(wl, logits=True, num_layers=1)


def test_argmax_ties_lowest_index():
    import torch
    ctx = get_ctx()
    wl = W.make_config(0, gated=False)
    sel = run_gate_select(ctx, wl)
    n = int(sel.n_selected.item())
    V, ld = 1000, 1008
    g = torch.Generator(device="cuda"); g.manual_seed(5)
    lg = torch.randn(sel.capacity, ld, generator=g, device="cuda").to(torch.bfloat16)
    lg[0, :] = 1.0                       # all equal -> 0
    lg[1, 700] = 9.0; lg[1, 300] = 9.0   # duplicate max -> lower index
    lg[2, 999] = 50.0                    # last valid column
    lg[3, 1003] = 99.0                   # beyond vocab: ignored
    lg[4, 5] = -0.0; lg[4, :5] = -1.0; lg[4, 6:] = -1.0; lg[4, 900] = 0.0   # -0 == +0 -> index 5
    _, k, v = W.draw_qkv(wl, 1, device="cuda")
    acc = ctx.accept(sel, make_kv(wl, k, v), dev(np.zeros(sel.capacity, np.int32)), dev(wl.prev_token),
                     target_logits=lg, vocab=V, compact=False)
    got = acc.target_token[:n].cpu().numpy()
    want = orc.argmax_bf16(torch_bf16_to_bits(lg[:n]), V)
    np.testing.assert_array_equal(got, want)
    assert got[0] == 0 and got[1] == 300 and got[2] == 999 and got[3] < 1000 and got[4] == 5


# ---------------------------------------------------------------- NEXT-1: Algorithm 1 as printed (schedule = ALG1)
A1 = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "alg1.json")))


@pytest.mark.parametrize("B", list(range(0, 11)))
def test_alg1_hand_example_all_budgets(B):
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    offs = np.asarray(GOLD["cand_offsets"], np.int32)
    parent = np.asarray(GOLD["parent"], np.int32)
    logq = np.asarray(GOLD["logq"], np.float32)
    lt = np.zeros(32, np.float32)
    sel = ctx.gate_select(dev(offs), dev(parent), dev(logq), 0, lt, 0, B, capacity=16, schedule=echo.SCHED_ALG1)
    got = sel.to_host()
    want = orc.gate_select(offs, parent, logq, 0, lt, 0, B, schedule=1)
    assert_selection_equal(got, want)
    order = sorted(tuple(x) for x in A1["grant_order"][:B])
    assert sorted(zip(got["sel_req"].tolist(), got["sel_node"].tolist())) == order


@pytest.mark.parametrize("cfg,gated,R", [(0, True, None), (0, False, None), (1, True, None), (2, True, None),
                                         (3, True, None), (4, True, None), (2, False, 7)])
def test_alg1_configs(cfg, gated, R):
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    wl = W.make_config(cfg, gated=gated, R=R)
    sel = run_gate_select(ctx, wl, schedule=echo.SCHED_ALG1)
    want = oracle_gate_select(orc, wl, schedule=1)
    assert_selection_equal(sel.to_host(), want)
    assert ctx.device_status() == 0


@pytest.mark.parametrize("budget", [0, 1, 7, 40, 95, 96, 500])
def test_alg1_budget_edges_and_widening(budget):
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    wl = W.make_config(0, gated=True)
    g = wl.gate.replace(budget=budget)
    sel = run_gate_select(ctx, wl, g, capacity=max(budget, 1), schedule=echo.SCHED_ALG1)
    assert_selection_equal(sel.to_host(), oracle_gate_select(orc, wl, g, schedule=1))


# ---------------------------------------------------------------- one budget shared by several ranks
def _slice_oracle(want, r0, r1):
    """the packed arrays of requests [r0, r1) of a selection over the merged batch, rebased to a rank-local view"""
    offs = want["sel_offsets"]
    a, b = int(offs[r0]), int(offs[r1])
    return dict(n_selected=b - a, sel_offsets=(offs[r0:r1 + 1] - offs[r0]).astype(np.int32),
                sel_node=want["sel_node"][a:b], sel_req=(want["sel_req"][a:b] - r0).astype(np.int32),
                parent_local=want["parent_local"][a:b], sel_depth=want["sel_depth"][a:b],
                anc_mask=want["anc_mask"][a:b], path_score=None, cand_depth=None, cut_depth=want["cut_depth"][r0:r1])


@pytest.mark.parametrize("cfgs,schedule", [((2, 2), 0), ((1, 3, 0), 0), ((2, 2), 1), ((0, 4, 1), 1)])
def test_global_budget_across_ranks_equals_merged_batch(cfgs, schedule):
    """Ranks with their own requests share ONE budget: keys of all ranks, one threshold, each rank packs its own.
    The ranks run one after the other on this GPU and torch.cat stands in for the all-gather (they share nothing
    else); the oracle selects on the merged batch."""
    import torch
    ctx = get_ctx()
    wls = [W.make_config(c, R=5 + 3 * i, seed=777 + i) for i, c in enumerate(cfgs)]
    g0 = wls[0].gate
    budget = sum(w.N for w in wls) // 3
    offs = np.concatenate([[0]] + [w.cand_offsets[1:] + sum(x.N for x in wls[:i]) for i, w in enumerate(wls)]).astype(np.int32)
    parent = np.concatenate([w.parent for w in wls])
    logq = np.concatenate([w.logq for w in wls])
    want = orc.gate_select(offs, parent, logq, g0.depth_mask, g0.log_tau, g0.w_max, budget, 0, schedule=schedule)
    sels, keys, dts = [], [], []
    for i, w in enumerate(wls):
        dt = (dev(w.cand_offsets), dev(w.parent), dev(w.logq))
        sel = ctx.alloc_selection(w.R, w.N, min(budget, w.N))
        k = ctx.gate_keys(*dt, g0.depth_mask, g0.log_tau, g0.w_max, budget, sel, schedule=schedule,
                          cand_index_base=sum(x.N for x in wls[:i]), request_base=sum(x.R for x in wls[:i]),
                          max_cand=max(1, w.max_cand))
        sels.append(sel); keys.append(k.clone()); dts.append(dt)   # one context plays all ranks: its key buffer is reused
    n_max = max(k.numel() for k in keys)
    gathered = torch.cat([torch.cat([k, torch.full((n_max - k.numel(),), -1, dtype=torch.int64, device=k.device)]) for k in keys])
    total = 0
    for i, w in enumerate(wls):
        ctx.gate_select_keys(*dts[i], g0.depth_mask, g0.log_tau, g0.w_max, budget, keys[i], gathered, sels[i],
                             schedule=schedule, max_cand=max(1, w.max_cand))
        got = sels[i].to_host()
        r0 = sum(x.R for x in wls[:i])
        exp = _slice_oracle(want, r0, r0 + w.R)
        assert got["n_selected"] == exp["n_selected"]
        for key in ("sel_offsets", "sel_node", "sel_req", "parent_local", "sel_depth", "anc_mask", "cut_depth"):
            np.testing.assert_array_equal(np.asarray(got[key])[:len(exp[key])], exp[key], err_msg=f"rank {i} {key}")
        total += got["n_selected"]
    assert total == want["n_selected"] <= budget
    assert ctx.device_status() == 0
