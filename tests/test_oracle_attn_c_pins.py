"""Pins for the plain-C attention oracle oracle/echo_oracle_attn.c (-m "not gpu"): the numpy oracle (pinned in
test_oracle_attn_pins.py by closed forms and a separately written dense softmax) on every row of cfg0 and on samples of
the other shapes; closed forms computed here from gathers of the test's own (Q = 0, a dominant key, a dominant key
outside the visible set); the result does not depend on the number of threads."""
import numpy as np
import pytest

from helpers import bf16_bits_to_f32, f32_to_bf16_bits, oracle_gate_select, torch_bf16_to_bits
from oracle import attn_c, echo_oracle as orc
from paper_2604_09603_b200 import workloads as W

SM_SCALE = 1.0 / np.sqrt(128.0)


def _case(cfg, R=None, gated=True, seed_rows=0, n_rows=None):
    wl = W.make_config(cfg, R=R, gated=gated) if R else W.make_config(cfg, gated=gated)
    sel = oracle_gate_select(orc, wl)
    q, k, v = W.draw_qkv(wl, max(1, sel["n_selected"]), device="cpu")
    qb, kb, vb = torch_bf16_to_bits(q), torch_bf16_to_bits(k), torch_bf16_to_bits(v)
    rows = None
    if n_rows:
        rng = np.random.default_rng(seed_rows)
        rows = sorted({(int(rng.integers(0, sel["n_selected"])), int(rng.integers(0, wl.Hq))) for _ in range(n_rows)})
    return wl, sel, qb, kb, vb, rows


def _visible(wl, sel, k):
    """token positions node k sees, from the selection's parent links (not from its masks)"""
    i = int(sel["sel_req"][k])
    off = int(sel["sel_offsets"][i])
    P = int(wl.prefix_len[i])
    pos, l = list(range(P)), k - off
    chain = []
    while l >= 0:
        chain.append(P + l)
        l = int(sel["parent_local"][off + l])
    return i, pos + sorted(chain)


def _row(wl, pool_bits, i, kvh, t):
    return bf16_bits_to_f32(pool_bits[0, wl.page_table[i][t // 16], kvh, t % 16, :]).astype(np.float64)


@pytest.mark.parametrize("gated", [False, True])
def test_c_oracle_equals_numpy_oracle_cfg0_every_row(gated):
    wl, sel, qb, kb, vb, _ = _case(0, gated=gated)
    O, L = orc.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE)
    O2, L2 = attn_c.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE)
    assert O2.shape == O.shape and L2.shape == L.shape
    assert np.abs(O - O2).max() <= 1e-13 and np.abs(L - L2).max() <= 1e-12


@pytest.mark.parametrize("cfg,R", [(1, 4), (2, 3), (3, 2), (4, 3)])
def test_c_oracle_equals_numpy_oracle_sampled_rows(cfg, R):
    """the other head groupings (G = 4, 8, 16), long prefixes, chains and wide trees"""
    wl, sel, qb, kb, vb, rows = _case(cfg, R=R, seed_rows=cfg, n_rows=48)
    want = orc.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=rows)
    O2, L2 = attn_c.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=rows)
    for j, r in enumerate(rows):
        assert np.abs(want[r][0] - O2[j]).max() <= 1e-13 and abs(want[r][1] - L2[j]) <= 1e-12


def test_c_oracle_q_zero_closed_form():
    """Q = 0: every visible key weighs the same => out = mean of the visible V rows, lse = ln |visible set|"""
    wl, sel, qb, kb, vb, _ = _case(0)
    O2, L2 = attn_c.verify_attn(sel, np.zeros_like(qb), kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE)
    G = wl.Hq // wl.Hkv
    for k in range(sel["n_selected"]):
        i, pos = _visible(wl, sel, k)
        for h in (0, wl.Hq - 1):
            mean_v = np.mean([_row(wl, vb, i, h // G, t) for t in pos], axis=0)
            assert np.abs(O2[k, h] - mean_v).max() <= 1e-13
            assert abs(L2[k, h] - np.log(len(pos))) <= 1e-12


def test_c_oracle_dominant_key_inside_and_outside_the_visible_set():
    """one key 2^12 times the query direction: if the node sees it, out = that key's V row and lse = its logit; planted
    at a tree position the node does NOT see (a sibling's), it changes nothing"""
    wl, sel, qb, kb, vb, _ = _case(0, gated=False)
    G = wl.Hq // wl.Hkv
    base_O, base_L = attn_c.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE)
    n = sel["n_selected"]
    checked_in = checked_out = 0
    for k in range(n):
        i, pos = _visible(wl, sel, k)
        off, P = int(sel["sel_offsets"][i]), int(wl.prefix_len[i])
        K_i = int(sel["sel_offsets"][i + 1]) - off
        hidden = [P + l for l in range(K_i) if P + l not in pos]
        h = (3 * k) % wl.Hq
        kvh = h // G
        qv = bf16_bits_to_f32(qb[k, h]).astype(np.float64)
        for t, seen in ((pos[len(pos) // 2], True), (pos[-1], True)) + (((hidden[0], False),) if hidden else ()):
            kb2 = kb.copy()
            kb2[0, wl.page_table[i][t // 16], kvh, t % 16, :] = f32_to_bf16_bits((qv * 4096.0).astype(np.float32))
            O2, L2 = attn_c.verify_attn(sel, qb, kb2, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=[(k, h)])
            if seen:
                s_t = float(np.float32(SM_SCALE)) * float(np.dot(bf16_bits_to_f32(kb2[0, wl.page_table[i][t // 16], kvh, t % 16]).astype(np.float64), qv))
                assert np.abs(O2[0] - _row(wl, vb, i, kvh, t)).max() <= 1e-9     # every other weight is < e^-1000
                assert abs(L2[0] - s_t) <= 1e-9 * max(1.0, abs(s_t))
                checked_in += 1
            else:
                assert np.array_equal(O2[0], base_O[k, h]) and L2[0] == base_L[k, h]
                checked_out += 1
    assert checked_in >= 2 * n and checked_out >= 4


def test_c_oracle_thread_count_invariance_and_argument_checks():
    wl, sel, qb, kb, vb, rows = _case(1, R=3, n_rows=40)
    a = attn_c.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=rows, threads=1)
    for t in (2, 3, 8, 64):
        b = attn_c.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=rows, threads=t)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    e = attn_c.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=[])
    assert e[0].shape == (0, 128) and e[1].shape == (0,)
    with pytest.raises(AssertionError):
        attn_c.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=[(10**6, 0)])
    assert attn_c.host_threads() >= 1
