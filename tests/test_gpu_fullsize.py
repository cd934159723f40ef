"""-m gpu parity at BASELINE.json's full sizes and on the branches only large inputs reach:
cfg1 (R=32) attention on every row (cfg2 / cfg3 on every row: test_zx_attn_every_row.py);
cfg2 / cfg2-static / cfg3 / cfg4 (R=256) attention on a STRATIFIED row sample
(first and last row of every 128-row tile, last valid row, deepest and root nodes, for the requests with extreme K_i
and P_i and 16 random ones, topped up with uniform rows); cfg4 acceptance from the full 4096 x 151 936 logits, greedy
and at temperature 1; k_select's uncached branch (N > 16 384 keys) and k_plan's multi-pass loop (R > 256)."""
import numpy as np
import pytest

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W
from helpers import oracle_gate_select, packed_tokens, torch_bf16_to_bits, bf16_bits_to_f32
from gpu_util import dev, get_ctx, run_gate_select, make_kv, assert_selection_equal

pytestmark = pytest.mark.gpu
TOL_O, TOL_LSE = 1e-2, 1e-3
SM_SCALE = 1.0 / np.sqrt(128.0)
TILE_M = 128


def stratified_rows(wl, sel, target, seed):
    """(packed node, query head) pairs that cover what a uniform sample misses: per chosen request and KV head the
    first and the last valid row of EVERY row tile of the kernel (rows are ordered (node, head in group), 128 per tile),
    the rows of the deepest node and of a root; chosen requests = largest / smallest K_i > 0, longest / shortest P_i,
    16 random ones; then uniform rows up to `target`."""
    rng = np.random.default_rng(seed)
    offs = sel["sel_offsets"].astype(np.int64)
    K = np.diff(offs)
    P = wl.prefix_len.astype(np.int64)
    act = np.flatnonzero(K > 0)
    G = wl.Hq // wl.Hkv
    chosen = {int(act[np.argmax(K[act])]), int(act[np.argmin(K[act])]), int(act[np.argmax(P[act])]),
              int(act[np.argmin(P[act])])}
    chosen |= set(int(x) for x in rng.choice(act, size=min(16, len(act)), replace=False))
    rows = set()
    for i in sorted(chosen):
        n_rows = int(K[i]) * G
        depth = sel["sel_depth"][offs[i]:offs[i + 1]]
        special = [int(np.argmax(depth)), int(np.argmin(depth))]
        for kvh in range(wl.Hkv):
            for rt in range((n_rows + TILE_M - 1) // TILE_M):
                for r in (rt * TILE_M, min(n_rows, (rt + 1) * TILE_M) - 1):
                    rows.add((int(offs[i]) + r // G, kvh * G + r % G))
            for l in special:
                rows.add((int(offs[i]) + l, kvh * G + int(rng.integers(0, G))))
    n = int(sel["n_selected"])
    rows |= {(0, 0), (n - 1, wl.Hq - 1)}
    while len(rows) < target:
        rows.add((int(rng.integers(0, n)), int(rng.integers(0, wl.Hq))))
    return sorted(rows)


def _attn_case(wl, gate=None):
    ctx = get_ctx()
    sel = run_gate_select(ctx, wl, gate)
    want_sel = oracle_gate_select(orc, wl, gate)
    assert_selection_equal(sel.to_host(), want_sel)
    q, k, v = W.draw_qkv(wl, max(1, sel.capacity), device="cuda")
    out, lse = ctx.verify_attn(sel, make_kv(wl, k, v), q, SM_SCALE)
    assert ctx.device_status() == 0
    return want_sel, q, k, v, out, lse


def _check_rows(wl, want_sel, q, k, v, out, lse, rows):
    qb, kb, vb = torch_bf16_to_bits(q), torch_bf16_to_bits(k), torch_bf16_to_bits(v)
    o_gpu = bf16_bits_to_f32(torch_bf16_to_bits(out))
    l_gpu = lse.cpu().numpy()
    res = orc.verify_attn(want_sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=rows)
    eo = max(np.abs(o_gpu[k_, h].astype(np.float64) - res[(k_, h)][0]).max() for (k_, h) in rows)
    el = max(abs(float(l_gpu[k_, h]) - res[(k_, h)][1]) for (k_, h) in rows)
    assert eo <= TOL_O, f"max|dO| = {eo}"
    assert el <= TOL_LSE, f"max|dlse| = {el}"


def test_attn_cfg1_full_batch_every_row():
    """cfg1 at its full size (R = 32, B = 1024, 32 / 8 heads): all 32 768 (node, head) rows against the oracle."""
    wl = W.make_config(1)
    want_sel, q, k, v, out, lse = _attn_case(wl)
    n = want_sel["n_selected"]
    assert n == wl.gate.budget
    qb, kb, vb = torch_bf16_to_bits(q), torch_bf16_to_bits(k), torch_bf16_to_bits(v)
    O, L = orc.verify_attn(want_sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE)
    o_gpu = bf16_bits_to_f32(torch_bf16_to_bits(out))[:n].astype(np.float64)
    assert np.isfinite(o_gpu).all()
    assert np.abs(o_gpu - O).max() <= TOL_O
    assert np.abs(lse.cpu().numpy()[:n].astype(np.float64) - L).max() <= TOL_LSE


@pytest.mark.parametrize("cfg,static,target", [(2, False, 2000), (2, True, 2000), (3, False, 2000), (4, False, 640)])
def test_attn_full_size_stratified_rows(cfg, static, target):
    wl = W.make_config(cfg, static=static, gated=not static)
    want_sel, q, k, v, out, lse = _attn_case(wl)
    n = want_sel["n_selected"]
    assert n == (wl.R * 60 if static else wl.gate.budget)
    rows = stratified_rows(wl, want_sel, target, seed=200 + cfg)
    assert len(rows) >= target
    _check_rows(wl, want_sel, q, k, v, out, lse, rows)
    o_gpu = bf16_bits_to_f32(torch_bf16_to_bits(out))[:n]
    assert np.isfinite(o_gpu).all() and np.isfinite(lse.cpu().numpy()[:n]).all()


def test_attn_many_requests_planner_multi_pass():
    """R = 300 > PLAN_THREADS (256): k_plan's request loop takes a second pass (cfg1 shape, 4 heads per group)."""
    wl = W.make_config(1, R=300)
    want_sel, q, k, v, out, lse = _attn_case(wl)
    rows = stratified_rows(wl, want_sel, 600, seed=301)
    rows += [(int(want_sel["sel_offsets"][i]), 0) for i in range(256, 300) if want_sel["sel_offsets"][i + 1] > want_sel["sel_offsets"][i]]
    _check_rows(wl, want_sel, q, k, v, out, lse, sorted(set(rows)))


@pytest.mark.parametrize("gate_path", [1, 2])
@pytest.mark.parametrize("schedule", [0, 1])
def test_gate_select_more_keys_than_the_register_cache(schedule, gate_path):
    """N = 16 800 > 16 384: as three kernels, k_select reads the keys from global memory in every radix pass (the branch
    the merged key population of 8 request-sharded ranks takes); as one cluster, 16 CTAs take 14 requests each in two
    rounds."""
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    ctx.set_option(echo.OPT_GATE_PATH, gate_path)
    wl = W.make_config(2, R=210)
    assert wl.N > 16384
    sel = run_gate_select(ctx, wl, schedule=schedule)
    assert_selection_equal(sel.to_host(), oracle_gate_select(orc, wl, schedule=schedule))
    assert ctx.device_status() == 0


def test_gate_select_more_requests_than_a_cluster_takes():
    """R = 520 > 16 CTAs x 32 requests: echo_gate_select falls back to the three-kernel chain by itself, and refuses
    when the cluster kernel is forced."""
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    wl = W.make_config(1, R=520)
    sel = run_gate_select(ctx, wl)
    assert_selection_equal(sel.to_host(), oracle_gate_select(orc, wl))
    ctx.set_option(echo.OPT_GATE_PATH, 2)
    with pytest.raises(echo.EchoError) as e:
        run_gate_select(ctx, wl)
    assert e.value.code == echo.ERR_UNSUPPORTED
    ctx.set_option(echo.OPT_GATE_PATH, 0)


def test_global_budget_eight_ranks_key_population():
    """8 ranks x 32 requests x 80 candidates = 20 480 keys through echo_gate_keys / echo_gate_select_keys: one
    threshold over the gathered population (uncached radix select), every rank's packed arrays equal the oracle's
    selection on the merged batch."""
    import torch
    ctx = get_ctx()
    wls = [W.make_config(2, R=32, seed=900 + i) for i in range(8)]
    g0 = wls[0].gate
    budget = 8 * g0.budget
    n_before = np.concatenate([[0], np.cumsum([w.N for w in wls])]).astype(np.int64)
    r_before = np.concatenate([[0], np.cumsum([w.R for w in wls])]).astype(np.int64)
    offs = np.concatenate([[0]] + [w.cand_offsets[1:] + n_before[i] for i, w in enumerate(wls)]).astype(np.int32)
    want = orc.gate_select(offs, np.concatenate([w.parent for w in wls]), np.concatenate([w.logq for w in wls]),
                           g0.depth_mask, g0.log_tau, g0.w_max, budget, 0)
    sels, keys, dts = [], [], []
    for i, w in enumerate(wls):
        dt = (dev(w.cand_offsets), dev(w.parent), dev(w.logq))
        sel = ctx.alloc_selection(w.R, w.N, min(budget, w.N))
        k = ctx.gate_keys(*dt, g0.depth_mask, g0.log_tau, g0.w_max, budget, sel, cand_index_base=int(n_before[i]),
                          request_base=int(r_before[i]), max_cand=w.max_cand)
        sels.append(sel); keys.append(k.clone()); dts.append(dt)
    gathered = torch.cat(keys)
    assert gathered.numel() > 16384
    total = 0
    for i, w in enumerate(wls):
        ctx.gate_select_keys(*dts[i], g0.depth_mask, g0.log_tau, g0.w_max, budget, keys[i], gathered, sels[i],
                             max_cand=w.max_cand)
        got = sels[i].to_host()
        a, b = int(want["sel_offsets"][r_before[i]]), int(want["sel_offsets"][r_before[i + 1]])
        assert got["n_selected"] == b - a
        np.testing.assert_array_equal(got["sel_offsets"], want["sel_offsets"][r_before[i]:r_before[i + 1] + 1] - a)
        for key in ("sel_node", "parent_local", "sel_depth"):
            np.testing.assert_array_equal(got[key], want[key][a:b], err_msg=f"rank {i} {key}")
        np.testing.assert_array_equal(got["sel_req"], want["sel_req"][a:b] - r_before[i])
        np.testing.assert_array_equal(got["anc_mask"].reshape(-1, 4), want["anc_mask"][a:b])
        total += got["n_selected"]
    assert total == want["n_selected"] == budget
    assert ctx.device_status() == 0


def test_accept_cfg4_full_size_from_logits():
    """cfg4 at R = 256: fused argmax over the full [4096][151 936] bf16 logits, acceptance walk, slot maps and the
    compacted pools, all bit-exact."""
    from test_gpu_gate_accept import _accept_case
    wl = W.make_config(4)
    got = _accept_case(wl, logits=True, num_layers=1)
    assert got["accept_len"].max() <= 32 and got["accept_len"].sum() > 0


def test_stochastic_cfg4_full_size():
    """echo_accept_stochastic at cfg4's full size (R = 256, 4096 + 256 rows of 151 936 logits)."""
    from test_gpu_stochastic import _case
    want = _case(4, None, 1.0, seed=404)
    assert len(want["bonus_cdf"]) == 256
