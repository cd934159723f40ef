"""Pins for the CPU oracle (-m "not gpu"): the oracle against what the paper and the
mathematics fix -- worked example W1 (tests/golden/w1.json), closed forms, special cases
that reduce to textbook routines, brute force on tiny inputs, invariants."""
import itertools
import json
import os

import numpy as np
import pytest

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W
from helpers import f32_to_bf16_bits, bf16_bits_to_f32, oracle_gate_select, packed_tokens

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "w1.json")))
INT32_MAX = 2**31 - 1


def _w1(budget, depth_mask=0, log_tau=None, w_max=0):
    lt = np.zeros(32, np.float32) if log_tau is None else log_tau
    return orc.gate_select(np.asarray(GOLD["cand_offsets"], np.int32), np.asarray(GOLD["parent"], np.int32),
                           np.asarray(GOLD["logq"], np.float32), depth_mask, lt, w_max, budget)


def _per_req(sel, key):
    o = sel["sel_offsets"]
    return [list(map(int, sel[key][o[i]:o[i + 1]])) for i in range(len(o) - 1)]


# ------------------------------------------------------------------ W1 (S1-S5)
def test_w1_scores_depths():
    s = _w1(9)
    assert s["path_score"].tolist() == GOLD["S"]
    assert s["cand_depth"].tolist() == GOLD["depth"]


@pytest.mark.parametrize("B", [6, 7])
def test_w1_selection(B):
    g = GOLD[f"B{B}"]
    s = _w1(B)
    assert np.diff(s["sel_offsets"]).tolist() == g["K"]
    assert _per_req(s, "sel_node") == g["nodes"]
    assert _per_req(s, "parent_local") == g["parent_local"]
    o = s["sel_offsets"]
    assert [[int(s["anc_mask"][k, 0]) for k in range(o[i], o[i + 1])] for i in range(2)] == g["masks"]
    assert not s["anc_mask"][:, 1:].any()


def test_w1_total_order_prefixes():
    order = [tuple(x) for x in GOLD["total_order"]]
    for B in range(10):
        s = _w1(B)
        got = sorted(zip(s["sel_req"].tolist(), s["sel_node"].tolist()))
        assert got == sorted(order[:B])


def test_w1_gated():
    g = GOLD["gated"]
    lt = np.zeros(32, np.float32)
    lt[g["depth"]] = np.float32(np.log(np.float64(g["tau"])))
    assert abs(float(lt[2]) - g["log_tau"]) < 1e-7
    s9 = _w1(9, 1 << g["depth"], lt, g["w_max"])
    assert s9["cut_depth"].tolist() == g["cut_depth"]
    assert s9["n_selected"] == 9
    assert [int(m) for m in s9["anc_mask"][5:, 0]] == g["B9_req1_masks"]
    s8 = _w1(8, 1 << g["depth"], lt, g["w_max"])
    got = set(zip(s8["sel_req"].tolist(), s8["sel_node"].tolist()))
    assert tuple(g["B8_dropped"]) not in got and (0, 4) in got and len(got) == 8
    # w_max = 0 disables Phase 2: node (1,2) never selected even with ample budget (G-8)
    s = _w1(9, 1 << g["depth"], lt, 0)
    assert s["n_selected"] == 8


def test_w1_accept_and_compaction():
    a = GOLD["accept"]
    s = _w1(a["budget"])
    draft = np.zeros(s["n_selected"], np.int32); tgt = np.zeros_like(draft)
    draft[:4] = a["draft_token"]; tgt[:4] = a["target_token"]
    draft[4:] = [1, 2, 3]; tgt[4:] = [7, 7, 7]
    prev = np.asarray([a["prev_token"], 999], np.int32)
    acc = orc.accept(s, draft, prev, tgt, 2)
    assert acc["accept_len"].tolist() == [a["accept_len"], 0]
    assert acc["accept_idx"][0, :3].tolist() == a["path_local"]
    assert acc["last_node"].tolist() == [a["best"], -1]
    assert acc["bonus_token"].tolist() == [a["bonus_token"], -1]
    rng = np.random.default_rng(0)
    kp = rng.integers(0, 2**16, size=(2, 8, 2, 16, 128), dtype=np.uint16)
    vp = rng.integers(0, 2**16, size=(2, 8, 2, 16, 128), dtype=np.uint16)
    k0, v0 = kp.copy(), vp.copy()
    table = np.asarray([a["page_table"], [0, 1]], np.int32)
    c = orc.compact_kv(s, acc, kp, vp, table, np.asarray([a["prefix_len"], 3], np.int32), 2)
    assert c["slot_src"][0, :3].tolist() == a["slot_src"] and c["slot_dst"][0, :3].tolist() == a["slot_dst"]
    assert (c["slot_src"][0, 3:] == -1).all() and (c["slot_src"][1] == -1).all()
    assert c["new_len"].tolist() == [a["new_len"], 3]
    # row 39 -> 38 moved, everything else untouched
    assert (kp[:, 2, :, 6, :] == k0[:, 2, :, 7, :]).all() and (vp[:, 2, :, 6, :] == v0[:, 2, :, 7, :]).all()
    kp[:, 2, :, 6, :] = k0[:, 2, :, 6, :]; vp[:, 2, :, 6, :] = v0[:, 2, :, 6, :]
    assert (kp == k0).all() and (vp == v0).all()


# ------------------------------------------------------------------ S1 / S2 closed forms
def test_chain_scores_exact_and_monotone():
    n = 20
    logq = np.asarray([-(2.0 ** -k) for k in range(n)], np.float32)
    S, d = orc.path_scores(np.asarray([0, n], np.int32), W.tree_chain(n), logq)
    exact = np.cumsum(logq.astype(np.float64))        # all partial sums fit in 24 bits
    assert (S.astype(np.float64) == exact).all()
    assert d.tolist() == list(range(n))
    wl = W.make_config(2, R=8)
    S, d = orc.path_scores(wl.cand_offsets, wl.parent, wl.logq)
    for i in range(wl.R):
        b = wl.cand_offsets[i]
        for j in range(wl.cand_offsets[i + 1] - b):
            p = wl.parent[b + j]
            if p >= 0:
                assert S[b + j] <= S[b + p] and d[b + j] == d[b + p] + 1   # I1
    assert not np.signbit(S[S == 0]).any()            # no -0 (G-13)


def test_fp32_order_matters_reference():
    # S is the fp32 sequential sum, not the rounded fp64 sum: pick values where they differ
    logq = np.asarray([-1.0, -2.0 ** -24, -2.0 ** -24, -2.0 ** -24], np.float32)
    S, _ = orc.path_scores(np.asarray([0, 4], np.int32), W.tree_chain(4), logq)
    assert S[3] == np.float32(-1.0)                   # each tiny add rounds back to -1 (ties-to-even)
    assert np.float32(np.sum(logq.astype(np.float64))) != S[3]


def test_gate_special_cases():
    wl = W.make_config(0)
    S, d = orc.path_scores(wl.cand_offsets, wl.parent, wl.logq)
    lt = np.zeros(32, np.float32)
    assert (orc.gate_cut_depth(wl.cand_offsets, S, d, 0, lt) == INT32_MAX).all()       # gates off
    lt[0] = np.inf
    assert (orc.gate_cut_depth(wl.cand_offsets, S, d, 1, lt) == 0).all()               # tau = +inf at root
    # strictness: threshold exactly equal to the level max fails (G-4)
    b, e = wl.cand_offsets[0], wl.cand_offsets[1]
    m2 = max(S[j] for j in range(b, e) if d[j] == 2)
    lt = np.zeros(32, np.float32); lt[2] = m2
    assert orc.gate_cut_depth(wl.cand_offsets, S, d, 1 << 2, lt)[0] == 2
    lt[2] = np.nextafter(np.float32(m2), np.float32(-np.inf))
    assert orc.gate_cut_depth(wl.cand_offsets, S, d, 1 << 2, lt)[0] == INT32_MAX
    # absent level is skipped (G-5)
    lt = np.zeros(32, np.float32); lt[20] = np.inf
    assert (orc.gate_cut_depth(wl.cand_offsets, S, d, 1 << 20, lt) == INT32_MAX).all()


# ------------------------------------------------------------------ S3-S5 brute force + invariants
def _beats(a, b):
    """explicit pairwise comparator of the total order (tier asc, S desc, request asc, node asc)."""
    if a[0] != b[0]:
        return a[0] < b[0]
    if a[1] != b[1]:
        return a[1] > b[1]
    if a[2] != b[2]:
        return a[2] < b[2]
    return a[3] < b[3]


def _brute_select(wl, gate):
    """rank-by-counting formulation: node selected iff fewer than B eligible nodes beat it."""
    S, d = orc.path_scores(wl.cand_offsets, wl.parent, wl.logq)
    cut = orc.gate_cut_depth(wl.cand_offsets, S, d, gate.depth_mask, gate.log_tau)
    elig = []
    for i in range(wl.R):
        b, e = wl.cand_offsets[i], wl.cand_offsets[i + 1]
        for j in range(e - b):
            if d[b + j] < cut[i]:
                elig.append((0, float(S[b + j]), i, j))
            elif d[b + j] == cut[i]:
                better = sum(1 for k in range(e - b) if d[b + k] == cut[i] and k != j and
                             (S[b + k] > S[b + j] or (S[b + k] == S[b + j] and k < j)))
                if better < gate.w_max:
                    elig.append((1, float(S[b + j]), i, j))
    out = []
    for a in elig:
        if sum(1 for b_ in elig if _beats(b_, a)) < gate.budget:
            out.append((a[2], a[3]))
    return sorted(out), len(elig)


@pytest.mark.parametrize("gated", [False, True])
@pytest.mark.parametrize("budget", [0, 1, 17, 32, 95, 96, 500])
def test_select_bruteforce_cfg0(gated, budget):
    wl = W.make_config(0, gated=gated)
    g = wl.gate.replace(budget=budget)
    s = oracle_gate_select(orc, wl, g)
    want, n_elig = _brute_select(wl, g)
    assert sorted(zip(s["sel_req"].tolist(), s["sel_node"].tolist())) == want
    assert s["n_selected"] == min(budget, n_elig)                                     # I3


@pytest.mark.parametrize("cfg,R", [(1, 6), (2, 5), (3, 5), (4, 12)])
def test_select_invariants(cfg, R):
    wl = W.make_config(cfg, R=R)
    s = oracle_gate_select(orc, wl)
    want, n_elig = _brute_select(wl, wl.gate)
    assert sorted(zip(s["sel_req"].tolist(), s["sel_node"].tolist())) == want
    o = s["sel_offsets"]
    for i in range(wl.R):                                                             # I2 ancestor closure
        nodes = s["sel_node"][o[i]:o[i + 1]].tolist()
        assert nodes == sorted(nodes)
        for l, j in enumerate(nodes):
            p = wl.parent[wl.cand_offsets[i] + j]
            pl = s["parent_local"][o[i] + l]
            assert (p < 0 and pl == -1) or nodes[pl] == p
            m = sum(int(s["anc_mask"][o[i] + l, w]) << (32 * w) for w in range(4))
            assert bin(m).count("1") == s["sel_depth"][o[i] + l] + 1 and (m >> l) & 1 and m < (2 << l)
    # I5: gates off and B >= N => everything selected
    g = W.Gate(budget=wl.N + 5)
    s = oracle_gate_select(orc, wl, g)
    assert s["n_selected"] == wl.N and (np.diff(s["sel_offsets"]) == np.diff(wl.cand_offsets)).all()


def test_static_and_roots_only():
    wl = W.make_config(2, R=4, static=True)
    s = oracle_gate_select(orc, wl)
    assert np.diff(s["sel_offsets"]).tolist() == [60] * 4
    S = s["path_score"]
    for i in range(4):
        b = wl.cand_offsets[i]
        chosen = set(s["sel_node"][s["sel_offsets"][i]:s["sel_offsets"][i + 1]].tolist())
        worst_in = min(S[b + j] for j in chosen)
        assert all(S[b + j] <= worst_in for j in range(80) if j not in chosen)
    # I7: one certain root per request, B = R => exactly the roots
    wl = W.make_config(0, gated=False)
    s = oracle_gate_select(orc, wl, W.Gate(budget=wl.R))
    assert s["sel_node"].tolist() == [0] * wl.R
    # I8 tie-break: two identical requests, odd budget -> request 0 gets the extra node
    offs = np.asarray([0, 3, 6], np.int32); par = np.asarray([-1, 0, 0, -1, 0, 0], np.int32)
    lq = np.asarray([0, -1, -1, 0, -1, -1], np.float32)
    s = orc.gate_select(offs, par, lq, 0, np.zeros(32, np.float32), 0, 3)
    assert sorted(zip(s["sel_req"].tolist(), s["sel_node"].tolist())) == [(0, 0), (0, 1), (1, 0)]
    # -inf (confidence 0) is legal and sorts last
    lq = np.asarray([0, -np.inf, -1, 0, -1, -1], np.float32)
    s = orc.gate_select(offs, par, lq, 0, np.zeros(32, np.float32), 0, 5)
    assert (0, 1) not in set(zip(s["sel_req"].tolist(), s["sel_node"].tolist()))
