"""Pins of the Algorithm-1-literal scheduler of the oracle (NEXT-1): the hand-run example of
tests/golden/alg1.json, invariants that hold for any input, the ample-budget case where it must agree with the
(separately pinned) global top-B selection, and an order-based brute force on small random forests."""
import json
import os

import numpy as np
import pytest

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
W1 = json.load(open(os.path.join(HERE, "golden", "w1.json")))
A1 = json.load(open(os.path.join(HERE, "golden", "alg1.json")))
OFFS = np.asarray(W1["cand_offsets"], np.int32)
PARENT = np.asarray(W1["parent"], np.int32)
LOGQ = np.asarray(W1["logq"], np.float32)


def _by_req(sel, R):
    out = [[] for _ in range(R)]
    for i, j in sel:
        out[i].append(j)
    return out


def test_alg1_hand_example_every_budget():
    S, depth = orc.path_scores(OFFS, PARENT, LOGQ)
    lt = np.zeros(32, np.float32)
    order = [tuple(x) for x in A1["grant_order"]]
    for B in range(0, 11):
        sel, cut = orc.select_alg1(OFFS, S, depth, 0, lt, B, 0)
        assert sel == sorted(order[:B]) and cut == {}
    assert _by_req(orc.select_alg1(OFFS, S, depth, 0, lt, 3, 0)[0], 2) == A1["B3"]["nodes"]
    out = orc.gate_select(OFFS, PARENT, LOGQ, 0, lt, 0, 6, schedule=1)
    assert _by_req(list(zip(out["sel_req"].tolist(), out["sel_node"].tolist())), 2) == A1["B6"]["nodes"]
    assert out["parent_local"].tolist() == sum(A1["B6"]["parent_local"], [])
    assert out["masks"] == sum(A1["B6"]["masks"], [])


def test_alg1_hand_example_gated():
    S, depth = orc.path_scores(OFFS, PARENT, LOGQ)
    g = A1["gated"]
    lt = np.zeros(32, np.float32)
    lt[g["depth"]] = np.float32(np.log(np.float64(g["tau"])))
    sel8, cut8 = orc.select_alg1(OFFS, S, depth, 1 << g["depth"], lt, 8, g["w_max"])
    assert _by_req(sel8, 2) == g["B8"]["nodes"] and cut8 == {}
    sel9, cut9 = orc.select_alg1(OFFS, S, depth, 1 << g["depth"], lt, 9, g["w_max"])
    assert _by_req(sel9, 2) == g["B9"]["nodes"] and cut9 == {1: 2}
    # w_max = 0: the truncated request is never widened, whatever the budget
    sel, _ = orc.select_alg1(OFFS, S, depth, 1 << g["depth"], lt, 100, 0)
    assert (1, 2) not in sel and len(sel) == 8


def _eligible(wl, S, depth, cut, w_max):
    el = set()
    for i in range(wl.R):
        b, e = int(wl.cand_offsets[i]), int(wl.cand_offsets[i + 1])
        for j in range(e - b):
            if depth[b + j] < cut[i]:
                el.add((i, j))
        lvl = sorted([j for j in range(e - b) if depth[b + j] == cut[i]], key=lambda j: (-float(S[b + j]), j))
        el |= {(i, j) for j in lvl[:w_max]}
    return el


@pytest.mark.parametrize("cfg,R", [(0, None), (1, 6), (2, 9), (3, 5), (4, 12)])
def test_alg1_invariants_and_ample_budget(cfg, R):
    wl = W.make_config(cfg, R=R)
    g = wl.gate
    S, depth = orc.path_scores(wl.cand_offsets, wl.parent, wl.logq)
    cut = orc.gate_cut_depth(wl.cand_offsets, S, depth, g.depth_mask, g.log_tau)
    el = _eligible(wl, S, depth, cut, g.w_max)
    for B in (0, 1, wl.R, len(el) // 2, len(el) - 1, len(el), wl.N + 5):
        sel, _ = orc.select_alg1(wl.cand_offsets, S, depth, g.depth_mask, g.log_tau, B, g.w_max)
        s = set(sel)
        assert len(sel) == len(s) == min(B, len(el)) and s <= el          # Eq. 4 and eligibility
        for (i, j) in sel:                                                  # ancestor closure (I2)
            p = int(wl.parent[wl.cand_offsets[i] + j])
            assert p < 0 or (i, p) in s
        dep = lambda i, j: int(depth[wl.cand_offsets[i] + j])
        for (i, j) in el - s:                                               # priority rule
            if dep(i, j) < cut[i]:  # a depth-extension node was left out: nothing deeper and no widening was granted
                assert all(dep(a, b_) < cut[a] and dep(a, b_) <= dep(i, j) for (a, b_) in s)
        if B >= len(el):                                                    # ample budget: same set as global top-B
            assert sel == orc.select(wl.cand_offsets, S, depth, cut, B, g.w_max)


@pytest.mark.parametrize("seed", range(6))
def test_alg1_equals_order_bruteforce(seed):
    """Alg. 1's grants, read as a sequence, are the eligible nodes sorted by (phase, depth, request, rank in level):
    brute force with Python's sorted() on random small forests and random gates."""
    rng = np.random.default_rng(seed)
    R = int(rng.integers(1, 6))
    sizes = rng.integers(1, 12, R)
    offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)
    parent = np.concatenate([[-1 if (j == 0 or rng.random() < 0.2) else int(rng.integers(0, j)) for j in range(n)]
                             for n in sizes]).astype(np.int32)
    logq = np.log(rng.uniform(0.05, 1.0, offs[-1])).astype(np.float32)
    S, depth = orc.path_scores(offs, parent, logq)
    mask = int(rng.integers(0, 16))
    lt = np.log(rng.uniform(0.05, 0.9, 32)).astype(np.float32)
    w_max = int(rng.integers(0, 4))
    cut = orc.gate_cut_depth(offs, S, depth, mask, lt)
    keyed = []
    for i in range(R):
        b, e = int(offs[i]), int(offs[i + 1])
        for d in set(int(x) for x in depth[b:e]):
            lvl = sorted([j for j in range(e - b) if depth[b + j] == d], key=lambda j: (-float(S[b + j]), j))
            for rank, j in enumerate(lvl):
                if d < cut[i]:
                    keyed.append((0, d, i, rank, j))
                elif d == cut[i] and rank < w_max:
                    keyed.append((1, d, i, rank, j))
    keyed.sort()
    for B in range(0, len(keyed) + 2):
        sel, _ = orc.select_alg1(offs, S, depth, mask, lt, B, w_max)
        assert sel == sorted((i, j) for (_, _, i, _, j) in keyed[:B])
