"""Pins for the oracle's attention / argmax / acceptance (-m "not gpu")."""
import itertools

import numpy as np
import pytest

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W
from helpers import f32_to_bf16_bits, bf16_bits_to_f32, oracle_gate_select, packed_tokens

SCALE = 1.0 / np.sqrt(128.0)


def _pools(wl, rng, layers=1):
    shape = (layers, wl.num_pages, wl.Hkv, 16, 128)
    return (f32_to_bf16_bits(rng.standard_normal(shape)), f32_to_bf16_bits(rng.standard_normal(shape)))


def _dense_kv(wl, i, pool, kvh, n, layer=0):
    """contiguous [n][128] float64 rows of request i's sequence, read through the page table."""
    return np.stack([bf16_bits_to_f32(pool[layer, wl.page_table[i, t // 16], kvh, t % 16]).astype(np.float64)
                     for t in range(n)])


def _ancestors_by_walk(parent_local, l):
    s = set()
    while l >= 0:
        s.add(l); l = int(parent_local[l])
    return s


def test_bruteforce_dense_masked_softmax_cfg0():
    """(iv): dense [rows x positions] score matrix, mask rebuilt by walking parent_local."""
    wl = W.make_config(0)
    sel = oracle_gate_select(orc, wl)
    rng = np.random.default_rng(1)
    kp, vp = _pools(wl, rng)
    q = f32_to_bf16_bits(rng.standard_normal((sel["n_selected"], wl.Hq, 128)))
    O, L = orc.verify_attn(sel, q, kp, vp, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SCALE)
    o = sel["sel_offsets"]
    for i in range(wl.R):
        K_i, P = int(o[i + 1] - o[i]), int(wl.prefix_len[i])
        if K_i == 0:
            continue
        pl = sel["parent_local"][o[i]:o[i + 1]]
        mask = np.zeros((K_i, P + K_i), bool)
        mask[:, :P] = True
        for l in range(K_i):
            for a in _ancestors_by_walk(pl, l):
                mask[l, P + a] = True
        for h in range(wl.Hq):
            Kd = _dense_kv(wl, i, kp, h // wl.G, P + K_i); Vd = _dense_kv(wl, i, vp, h // wl.G, P + K_i)
            Q = bf16_bits_to_f32(q[o[i]:o[i + 1], h]).astype(np.float64)
            s = np.where(mask, np.float64(np.float32(SCALE)) * (Q @ Kd.T), -np.inf)
            p = np.exp(s - s.max(1, keepdims=True))
            want = (p / p.sum(1, keepdims=True)) @ Vd
            np.testing.assert_allclose(O[o[i]:o[i + 1], h], want, rtol=1e-12, atol=1e-13)
            np.testing.assert_allclose(L[o[i]:o[i + 1], h], np.log(np.exp(s).sum(1)), rtol=1e-12)


def _chain_workload(P, n, Hq=4, Hkv=2, seed=5):
    rng = np.random.default_rng(seed)
    t = W.tree_chain(n)
    c = np.full(n, 0.5)
    return W._assemble("chain", seed, rng, Hq, Hkv, 1000, W.Gate(budget=n), [t], [c], [P]), rng


def test_chain_equals_causal_attention():
    """(ii): chain tree == causal attention of the last K tokens of a length P+K sequence."""
    P, n = 37, 9
    wl, rng = _chain_workload(P, n)
    sel = oracle_gate_select(orc, wl)
    assert sel["n_selected"] == n
    kp, vp = _pools(wl, rng)
    q = f32_to_bf16_bits(rng.standard_normal((n, wl.Hq, 128)))
    O, L = orc.verify_attn(sel, q, kp, vp, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SCALE)
    T = P + n
    causal = np.tril(np.ones((T, T), bool))[P:]            # rows of the last n tokens
    for h in range(wl.Hq):
        Kd = _dense_kv(wl, 0, kp, h // wl.G, T); Vd = _dense_kv(wl, 0, vp, h // wl.G, T)
        Q = bf16_bits_to_f32(q[:, h]).astype(np.float64)
        s = np.where(causal, np.float64(np.float32(SCALE)) * (Q @ Kd.T), -np.inf)
        p = np.exp(s - s.max(1, keepdims=True)); p /= p.sum(1, keepdims=True)
        np.testing.assert_allclose(O[:, h], p @ Vd, rtol=1e-12, atol=1e-13)


def test_single_node_equals_decode_attention():
    """(iii): one node == decode attention over P+1 keys."""
    wl, rng = _chain_workload(50, 1)
    sel = oracle_gate_select(orc, wl)
    kp, vp = _pools(wl, rng)
    q = f32_to_bf16_bits(rng.standard_normal((1, wl.Hq, 128)))
    O, L = orc.verify_attn(sel, q, kp, vp, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SCALE)
    for h in range(wl.Hq):
        Kd = _dense_kv(wl, 0, kp, h // wl.G, 51); Vd = _dense_kv(wl, 0, vp, h // wl.G, 51)
        s = np.float64(np.float32(SCALE)) * (Kd @ bf16_bits_to_f32(q[0, h]).astype(np.float64))
        w = np.exp(s - np.log(np.exp(s).sum()))
        np.testing.assert_allclose(O[0, h], w @ Vd, rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(L[0, h], np.log(np.exp(s).sum()), rtol=1e-13)


def test_q_zero_closed_form_and_invariances():
    """(i) Q=0 => mean of visible V rows, lse = ln(P + depth + 1); (v) page permutation
    invariance (bit-identical); (vii) sibling isolation; (viii) one-hot key."""
    wl = W.make_config(0, gated=False)
    sel = oracle_gate_select(orc, wl)
    rng = np.random.default_rng(2)
    kp, vp = _pools(wl, rng)
    n = sel["n_selected"]
    q0 = np.zeros((n, wl.Hq, 128), np.uint16)
    O, L = orc.verify_attn(sel, q0, kp, vp, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SCALE)
    o = sel["sel_offsets"]
    for k in range(n):
        i = int(sel["sel_req"][k]); P = int(wl.prefix_len[i])
        anc = _ancestors_by_walk(sel["parent_local"][o[i]:o[i + 1]], k - o[i])
        pos = list(range(P)) + [P + a for a in sorted(anc)]
        assert len(pos) == P + int(sel["sel_depth"][k]) + 1
        for h in (0, wl.Hq - 1):
            Vd = _dense_kv(wl, i, vp, h // wl.G, P + int(o[i + 1] - o[i]))
            np.testing.assert_allclose(O[k, h], Vd[pos].mean(0), rtol=1e-12, atol=1e-14)
            assert abs(L[k, h] - np.log(len(pos))) < 1e-12
    # (v) permute physical pages
    q = f32_to_bf16_bits(rng.standard_normal((n, wl.Hq, 128)))
    O1, L1 = orc.verify_attn(sel, q, kp, vp, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SCALE)
    perm = rng.permutation(wl.num_pages)
    inv = np.empty_like(perm); inv[perm] = np.arange(wl.num_pages)
    table2 = np.where(wl.page_table >= 0, inv[np.maximum(wl.page_table, 0)], -1)
    O2, L2 = orc.verify_attn(sel, q, kp[:, perm], vp[:, perm], table2, wl.prefix_len, wl.Hq, wl.Hkv, SCALE)
    assert (O1 == O2).all() and (L1 == L2).all()
    # (vii) perturb K/V of a non-ancestor tree node of request 3: rows not descending from it unchanged
    i = 3; b = int(o[i]); K_i = int(o[i + 1] - o[i]); P = int(wl.prefix_len[i])
    pl = sel["parent_local"][b:b + K_i]
    victim = K_i - 1
    pos = P + victim
    kp2, vp2 = kp.copy(), vp.copy()
    kp2[0, wl.page_table[i, pos // 16], :, pos % 16] ^= 0x0040
    vp2[0, wl.page_table[i, pos // 16], :, pos % 16] ^= 0x0040
    O3, L3 = orc.verify_attn(sel, q, kp2, vp2, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SCALE)
    for l in range(K_i):
        same = (O3[b + l] == O1[b + l]).all() and (L3[b + l] == L1[b + l]).all()
        assert same == (victim not in _ancestors_by_walk(pl, l))
    assert (O3[:b] == O1[:b]).all()
    # (viii) one-hot: q = 16 * k_t for one prefix key => O ~ v_t
    k = b; t = 5; h = 0
    krow = bf16_bits_to_f32(kp[0, wl.page_table[i, 0], 0, t])
    qh = q.copy(); qh[k, h] = f32_to_bf16_bits(krow * 16.0)
    Oh, _ = orc.verify_attn(sel, qh, kp, vp, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SCALE, rows=[(k, h)])[(k, h)]
    np.testing.assert_allclose(Oh, bf16_bits_to_f32(vp[0, wl.page_table[i, 0], 0, t]), atol=1e-6)


def test_rows_subset_matches_full():
    wl = W.make_config(0)
    sel = oracle_gate_select(orc, wl)
    rng = np.random.default_rng(3)
    kp, vp = _pools(wl, rng)
    q = f32_to_bf16_bits(rng.standard_normal((sel["n_selected"], wl.Hq, 128)))
    O, L = orc.verify_attn(sel, q, kp, vp, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SCALE)
    sub = orc.verify_attn(sel, q, kp, vp, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SCALE, rows=[(3, 1), (20, 7)])
    for (k, h), (o_, l_) in sub.items():
        assert (o_ == O[k, h]).all() and l_ == L[k, h]


# ------------------------------------------------------------------ S8
def test_argmax_pins():
    rng = np.random.default_rng(4)
    V, ld = 1000, 1024
    x = f32_to_bf16_bits(rng.standard_normal((6, ld)))
    x[:, V:] = f32_to_bf16_bits(np.float32(100.0))          # padding columns beyond vocab are ignored
    x[0, 700] = x[0, 30] = f32_to_bf16_bits(np.float32(9.0))  # duplicate max: lower index wins
    x[1, :] = f32_to_bf16_bits(np.float32(-1.5))             # all equal => 0
    x[2, V - 1] = f32_to_bf16_bits(np.float32(50.0))
    x[3, 10] = 0x0000; x[3, 5] = 0x8000                      # +0 and -0 compare equal
    x[3, :V] = np.where(bf16_bits_to_f32(x[3, :V]) > 0, 0x8000, x[3, :V]).astype(np.uint16)
    got = orc.argmax_bf16(x, V)
    for r in range(6):                                        # explicit strict-'>' first-max scan
        best, bi = -np.inf, -1
        row = bf16_bits_to_f32(x[r])
        for v in range(V):
            if row[v] > best or bi < 0:
                best, bi = row[v], v
        assert got[r] == bi
    assert got[0] == 30 and got[1] == 0 and got[2] == V - 1


def _partitions(V):
    """vocabulary partitions: equal shards of 1, 2, 3, 8 ranks, a lopsided one, and one with empty shards"""
    eq = lambda W_: [(V * r // W_, V * (r + 1) // W_) for r in range(W_)]
    return [eq(1), eq(2), eq(3), eq(8), [(0, 1), (1, V - 1), (V - 1, V)], [(0, 8), (8, 8), (8, V)]]


def test_sharded_argmax_is_the_argmax():
    """SURVEY 8(e), vocabulary-sharded S8: per-shard (maximum, first index) pairs merged by (greater value, then lower
    index) give the first maximum of the whole row -- for every partition, with the maximum duplicated across shard
    boundaries, -0 / +0 in different shards, all-equal and all -inf rows."""
    rng = np.random.default_rng(11)
    V, ld = 1000, 1024
    bits = lambda v: f32_to_bf16_bits(np.float32(v))
    x = f32_to_bf16_bits(rng.standard_normal((8, ld)))
    x[:, V:] = bits(100.0)                                   # padding beyond the vocabulary
    x[0, 900] = x[0, 499] = x[0, 500] = bits(9.0)            # the same maximum in several shards: lowest index
    x[1, :] = bits(-1.5)                                     # all equal => 0
    x[2, :V] = 0xFF80                                        # all -inf => 0
    x[3, :V] = bits(-2.0); x[3, 700] = 0x8000; x[3, 20] = 0x0000; x[3, 10] = 0x8000   # -0 at 10 wins over +0 at 20
    x[4, V - 1] = bits(50.0)                                 # last column
    x[5, :V] = 0xFF80; x[5, 640] = bits(-3.0)                # one finite logit among -inf
    want = orc.argmax_bf16(x, V)
    assert want[0] == 499 and want[1] == 0 and want[2] == 0 and want[3] == 10 and want[4] == V - 1 and want[5] == 640
    for part in _partitions(V):
        vals, idxs = [], []
        for v0, v1 in part:
            if v1 > v0:
                a, b = orc.argmax_shard_pairs(x, v0, v1)
                assert ((b >= v0) & (b < v1)).all()
                assert (bf16_bits_to_f32(x[np.arange(8), b]) == a).all()          # the value is the logit at the index
                assert (bf16_bits_to_f32(x[:, v0:v1]).max(axis=1) == a).all()     # and the shard's maximum
                assert not np.signbit(a[a == 0]).any()                            # -0 reported as +0
                vals.append(a); idxs.append(b)
        np.testing.assert_array_equal(orc.merge_argmax_pairs(vals, idxs), want, err_msg=str(part))
    # a wrong tie rule shows: taking the LAST shard on equal values would give 900 / V-1 style answers
    a0, b0 = orc.argmax_shard_pairs(x, 0, 500)
    a1, b1 = orc.argmax_shard_pairs(x, 500, V)
    assert b0[0] == 499 and b1[0] == 500 and a0[0] == a1[0]


# ------------------------------------------------------------------ S9 / S10
def _all_paths(parent_local):
    n = len(parent_local)
    paths = []
    for l in range(n):
        p, cur = [], l
        while cur >= 0:
            p.append(cur); cur = int(parent_local[cur])
        paths.append(p[::-1])
    return paths


@pytest.mark.parametrize("cfg,R,gated", [(0, None, False), (0, None, True), (1, 6, True), (3, 4, True), (4, 10, True)])
def test_accept_exhaustive_paths(cfg, R, gated):
    wl = W.make_config(cfg, gated=gated, R=R)
    sel = oracle_gate_select(orc, wl)
    draft, tgt, _ = packed_tokens(wl, sel)
    acc = orc.accept(sel, draft, wl.prev_token, tgt, wl.R)
    o = sel["sel_offsets"]
    total = 0
    for i in range(wl.R):
        b, K_i = int(o[i]), int(o[i + 1] - o[i])
        best = []
        for path in _all_paths(sel["parent_local"][b:b + K_i]):      # every root-to-node path
            ok = draft[b + path[0]] == wl.prev_token[i]
            for a, c in zip(path[:-1], path[1:]):
                ok = ok and draft[b + c] == tgt[b + a]
            if ok and len(path) > len(best):                         # first (lowest end index) of max length
                best = path
        assert acc["accept_len"][i] == len(best)
        assert acc["accept_idx"][i, :len(best)].tolist() == [b + a for a in best]
        assert (acc["accept_idx"][i, len(best):] == -1).all()
        if best:
            assert acc["last_node"][i] == b + best[-1] and acc["bonus_token"][i] == tgt[b + best[-1]]
        else:
            assert acc["last_node"][i] == -1 and acc["bonus_token"][i] == -1
        total += len(best)
    if cfg in (1, 3):
        assert total > 0


def test_accept_chain_and_compaction_invariants():
    n, P = 12, 41
    wl, rng = _chain_workload(P, n)
    sel = oracle_gate_select(orc, wl)
    draft = np.arange(100, 100 + n, dtype=np.int32)
    tgt = np.arange(101, 101 + n, dtype=np.int32)
    acc = orc.accept(sel, draft, np.asarray([100], np.int32), tgt, 1)
    assert acc["accept_len"][0] == n and acc["bonus_token"][0] == 100 + n
    kp, vp = _pools(wl, rng, layers=2)
    k0, v0 = kp.copy(), vp.copy()
    c = orc.compact_kv(sel, acc, kp, vp, wl.page_table, wl.prefix_len, 1)
    assert (c["slot_src"][0, :n] == c["slot_dst"][0, :n]).all() and (kp == k0).all() and (vp == v0).all()
    assert orc.accept(sel, draft, np.asarray([7], np.int32), tgt, 1)["accept_len"][0] == 0      # root mismatch
    tgt2 = tgt.copy(); tgt2[4] = 0
    assert orc.accept(sel, draft, np.asarray([100], np.int32), tgt2, 1)["accept_len"][0] == 5
    # general tree: invariants of the slot maps
    wl = W.make_config(1, R=6)
    sel = oracle_gate_select(orc, wl)
    d, t, _ = packed_tokens(wl, sel)
    acc = orc.accept(sel, d, wl.prev_token, t, wl.R)
    rng = np.random.default_rng(9)
    kp, vp = _pools(wl, rng, layers=2)
    k0, v0 = kp.copy(), vp.copy()
    c = orc.compact_kv(sel, acc, kp, vp, wl.page_table, wl.prefix_len, wl.R)
    touched = np.zeros((wl.num_pages * 16,), bool)
    for i in range(wl.R):
        L, P = int(acc["accept_len"][i]), int(wl.prefix_len[i])
        assert c["new_len"][i] == P + L
        dst_pos = [P + t_ for t_ in range(L)]
        assert c["slot_dst"][i, :L].tolist() == [int(wl.page_table[i, p // 16]) * 16 + p % 16 for p in dst_pos]
        src_pos = [P + int(acc["accept_idx"][i, t_] - sel["sel_offsets"][i]) for t_ in range(L)]
        assert all(a < b for a, b in zip(src_pos, src_pos[1:])) and all(s >= d_ for s, d_ in zip(src_pos, dst_pos))
        for t_ in range(L):
            s, d_ = int(c["slot_src"][i, t_]), int(c["slot_dst"][i, t_])
            assert (kp[:, d_ // 16, :, d_ % 16] == k0[:, s // 16, :, s % 16]).all()
            assert (vp[:, d_ // 16, :, d_ % 16] == v0[:, s // 16, :, s % 16]).all()
            touched[d_] = True
    flat_k = kp.transpose(1, 3, 0, 2, 4).reshape(wl.num_pages * 16, -1)
    flat_k0 = k0.transpose(1, 3, 0, 2, 4).reshape(wl.num_pages * 16, -1)
    assert (flat_k[~touched] == flat_k0[~touched]).all()
