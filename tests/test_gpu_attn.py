"""-m gpu parity: echo_verify_attn (CUDA, through the C ABI) against the fp64 oracle.
Bar (BASELINE.json north_star): max|O - O_oracle| <= 1e-2 on the bf16 output, max|lse - lse_oracle| <= 1e-3."""
import numpy as np
import pytest

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W
from helpers import oracle_gate_select, torch_bf16_to_bits, bf16_bits_to_f32
from gpu_util import dev, get_ctx, run_gate_select, make_kv, assert_selection_equal

pytestmark = pytest.mark.gpu
TOL_O, TOL_LSE = 1e-2, 1e-3
SM_SCALE = 1.0 / np.sqrt(128.0)


def _setup(wl, gate=None, poison=False, q_zero=False):
    ctx = get_ctx()
    sel = run_gate_select(ctx, wl, gate)
    want_sel = oracle_gate_select(orc, wl, gate)
    assert_selection_equal(sel.to_host(), want_sel)   # the attention below runs on the GPU's own selection
    cap = max(1, sel.capacity)
    q, k, v = W.draw_qkv(wl, cap, device="cuda")
    if q_zero:
        q.zero_()
    if poison:
        K = np.diff(want_sel["sel_offsets"])
        W.poison_unused_slots(wl, k, v, used_extra=K)
    return ctx, sel, want_sel, q, k, v


def _compare(wl, want_sel, q, k, v, out, lse, rows=None):
    n = want_sel["n_selected"]
    qb, kb, vb = torch_bf16_to_bits(q), torch_bf16_to_bits(k), torch_bf16_to_bits(v)
    o_gpu = bf16_bits_to_f32(torch_bf16_to_bits(out)).astype(np.float64)
    l_gpu = lse.cpu().numpy().astype(np.float64)
    if rows is None:
        O, L = orc.verify_attn(want_sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE)
        eo = np.abs(o_gpu[:n] - O).max() if n else 0.0
        el = np.abs(l_gpu[:n] - L).max() if n else 0.0
    else:
        res = orc.verify_attn(want_sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=rows)
        eo = max(np.abs(o_gpu[k_, h] - res[(k_, h)][0]).max() for (k_, h) in rows)
        el = max(abs(l_gpu[k_, h] - res[(k_, h)][1]) for (k_, h) in rows)
    assert np.isfinite(o_gpu[:n]).all() and np.isfinite(l_gpu[:n]).all()
    assert eo <= TOL_O, f"max|dO| = {eo}"
    assert el <= TOL_LSE, f"max|dlse| = {el}"
    return eo, el


PATHS = [1, 2]


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("splits", [0, 1, 2, 3, 7])
@pytest.mark.parametrize("gated", [True, False])
def test_attn_cfg0_full(path, splits, gated):
    from paper_2604_09603_b200 import echo
    wl = W.make_config(0, gated=gated)
    ctx, sel, want_sel, q, k, v = _setup(wl, poison=True)
    ctx.set_option(echo.OPT_ATTN_PATH, path)
    ctx.set_option(echo.OPT_FORCE_SPLITS, splits)
    out, lse = ctx.verify_attn(sel, make_kv(wl, k, v), q, SM_SCALE)
    _compare(wl, want_sel, q, k, v, out, lse)
    assert ctx.device_status() == 0


@pytest.mark.parametrize("path", PATHS)
def test_attn_q_zero_closed_form(path):
    """Q = 0: O = mean of the visible V rows, lse = ln(P_i + depth + 1) (closed form, SURVEY 8(c) pin (i))."""
    from paper_2604_09603_b200 import echo
    wl = W.make_config(0, gated=False)
    ctx, sel, want_sel, q, k, v = _setup(wl, q_zero=True, poison=True)
    ctx.set_option(echo.OPT_ATTN_PATH, path)
    out, lse = ctx.verify_attn(sel, make_kv(wl, k, v), q, SM_SCALE)
    n = want_sel["n_selected"]
    expect = np.log(wl.prefix_len[want_sel["sel_req"]].astype(np.float64) + want_sel["sel_depth"] + 1.0)
    got = lse.cpu().numpy()[:n]
    assert np.abs(got - expect[:, None]).max() <= TOL_LSE
    _compare(wl, want_sel, q, k, v, out, lse)


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("cfg,R,static", [(1, 3, False), (2, 3, False), (2, 2, True), (3, 2, False), (4, 4, False)])
def test_attn_scaled_configs_sampled(path, cfg, R, static):
    """cfg1-4 shapes at reduced batch: several KV tiles, ragged tails, G = 4 / 8 / 16; sampled rows."""
    from paper_2604_09603_b200 import echo
    wl = W.make_config(cfg, R=R, static=static, gated=not static)
    ctx, sel, want_sel, q, k, v = _setup(wl, poison=True)
    ctx.set_option(echo.OPT_ATTN_PATH, path)
    out, lse = ctx.verify_attn(sel, make_kv(wl, k, v), q, SM_SCALE)
    n = want_sel["n_selected"]
    rng = np.random.default_rng(cfg)
    rows = [(int(rng.integers(0, n)), int(rng.integers(0, wl.Hq))) for _ in range(96)]
    rows += [(0, 0), (n - 1, wl.Hq - 1)]
    _compare(wl, want_sel, q, k, v, out, lse, rows=rows)
    assert ctx.device_status() == 0


@pytest.mark.parametrize("path", PATHS)
def test_attn_edge_prefix_zero_and_empty_request(path):
    """P_i = 0 (tree only), a request that gets no budget (K_i = 0), P_i a multiple of the tile."""
    from paper_2604_09603_b200 import echo
    wl = W.make_config(0, gated=False, R=6)
    wl.prefix_len[:] = np.asarray([0, 128, 1, 256, 15, 16], np.int32)
    wl.page_table, wl.num_pages = W.paged_layout(np.random.default_rng(11), wl.prefix_len, np.diff(wl.cand_offsets))
    wl.logq[wl.cand_offsets[2]:wl.cand_offsets[3]] = np.float32(-50.0)   # request 2 loses every slot
    g = wl.gate.replace(budget=40)
    ctx, sel, want_sel, q, k, v = _setup(wl, g, poison=True)
    assert np.diff(want_sel["sel_offsets"])[2] == 0
    ctx.set_option(echo.OPT_ATTN_PATH, path)
    for splits in (1, 2):
        ctx.set_option(echo.OPT_FORCE_SPLITS, splits)
        out, lse = ctx.verify_attn(sel, make_kv(wl, k, v), q, SM_SCALE)
        _compare(wl, want_sel, q, k, v, out, lse)


@pytest.mark.parametrize("path", PATHS)
def test_attn_sibling_isolation(path):
    """perturbing K/V of a non-ancestor tree node leaves a row unchanged bit for bit."""
    import torch
    from paper_2604_09603_b200 import echo
    wl = W.make_config(0, gated=False)
    ctx, sel, want_sel, q, k, v = _setup(wl)
    ctx.set_option(echo.OPT_ATTN_PATH, path)
    ctx.set_option(echo.OPT_FORCE_SPLITS, 1)
    kv = make_kv(wl, k, v)
    out0, lse0 = ctx.verify_attn(sel, kv, q, SM_SCALE)
    out0, lse0 = out0.clone(), lse0.clone()
    offs = want_sel["sel_offsets"]
    i = 3
    Ki = int(offs[i + 1] - offs[i])
    masks = want_sel["masks"][offs[i]:offs[i + 1]]
    victim = Ki - 1                                    # last packed node of request 3: nobody's ancestor but itself
    pos = int(wl.prefix_len[i]) + victim
    pg, sl = int(wl.page_table[i, pos // 16]), pos % 16
    k[0, pg, :, sl, :] = 3.0
    v[0, pg, :, sl, :] = -7.0
    out1, lse1 = ctx.verify_attn(sel, kv, q, SM_SCALE)
    keep = [int(offs[i]) + l for l in range(Ki) if not (masks[l] >> victim) & 1]
    assert len(keep) == Ki - 1
    assert torch.equal(out0[keep], out1[keep]) and torch.equal(lse0[keep], lse1[keep])
    assert not torch.equal(out0[int(offs[i]) + victim], out1[int(offs[i]) + victim])


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("regime", ["all_low", "low_then_normal", "late_spike"])
def test_attn_extreme_scores(path, regime):
    """Scores far from the reference the tcgen05 kernel starts every item with (0): a first tile whose weights all
    underflow (two-pass fallback takes the reference from the data), a later tile that overflows it (O rescaled in
    TMEM), and one dominant key deep in the prefix.  Oracle: plain fp64 softmax, no running maximum."""
    import torch
    from paper_2604_09603_b200 import echo
    wl = W.make_config(1, R=3, gated=True)
    ctx, sel, want_sel, q, k, v = _setup(wl, poison=False)
    ctx.set_option(echo.OPT_ATTN_PATH, path)
    K = np.diff(want_sel["sel_offsets"])

    def set_k0(i, positions, value):
        pos = np.asarray(positions)
        pg = torch.from_numpy(wl.page_table[i, pos // 16].astype(np.int64)).cuda()
        sl = torch.from_numpy((pos % 16).astype(np.int64)).cuda()
        k[0, pg, :, sl, 0] = value

    q[:, :, 0] = 40.0                      # score = (40 k_0 + N(0, 127)) / sqrt(128)
    for i in range(wl.R):
        total = int(wl.prefix_len[i] + K[i])
        if regime == "all_low":            # every score near -141 (log2 domain -204)
            set_k0(i, np.arange(total), -40.0)
        elif regime == "low_then_normal":  # first KV tile near -141, the rest N(0, 3.5^2)
            set_k0(i, np.arange(min(128, total)), -40.0)
        else:                              # one key at +106 in the third tile
            set_k0(i, [300], 30.0)
    out, lse = ctx.verify_attn(sel, make_kv(wl, k, v), q, SM_SCALE)
    n = want_sel["n_selected"]
    rng = np.random.default_rng(5)
    rows = [(int(rng.integers(0, n)), int(rng.integers(0, wl.Hq))) for _ in range(48)] + [(0, 0), (n - 1, wl.Hq - 1)]
    _compare(wl, want_sel, q, k, v, out, lse, rows=rows)
    assert ctx.device_status() == 0


@pytest.mark.parametrize("cfg,R,splits", [(0, None, 1), (0, None, 3), (1, 3, 0), (2, 3, 1)])
def test_attn_safe_form_on_regular_scores(cfg, R, splits):
    """ECHO_OPT_ATTN_SAFE: every item takes the tcgen05 kernel's safe form (running row maximum, O rescaled in TMEM,
    one warpgroup) -- the form an item is redone in when its row sums leave the fast form's window -- on ordinary
    scores, where the oracle and the fast form are known to agree."""
    from paper_2604_09603_b200 import echo
    wl = W.make_config(cfg, R=R, gated=True)
    ctx, sel, want_sel, q, k, v = _setup(wl, poison=True)
    ctx.set_option(echo.OPT_ATTN_PATH, 2)
    ctx.set_option(echo.OPT_ATTN_SAFE, 1)
    ctx.set_option(echo.OPT_FORCE_SPLITS, splits)
    out, lse = ctx.verify_attn(sel, make_kv(wl, k, v), q, SM_SCALE)
    n = want_sel["n_selected"]
    if cfg == 0:
        _compare(wl, want_sel, q, k, v, out, lse)
    else:
        rng = np.random.default_rng(31 + cfg)
        rows = [(int(rng.integers(0, n)), int(rng.integers(0, wl.Hq))) for _ in range(96)] + [(0, 0), (n - 1, wl.Hq - 1)]
        _compare(wl, want_sel, q, k, v, out, lse, rows=rows)
    assert ctx.device_status() == 0


@pytest.mark.parametrize("cfg,static", [(2, False), (2, True), (3, False)])
def test_attn_full_size_bench_configuration(cfg, static):
    """BASELINE.json's full sizes (BS=128) in the launch configuration bench.py times (default path, default
    splits): 130 sampled (node, head) rows -- first and last row of the batch, the rest uniform -- against the
    oracle, which computes each row on its own."""
    from paper_2604_09603_b200 import echo
    wl = W.make_config(cfg, static=static, gated=not static)
    ctx, sel, want_sel, q, k, v = _setup(wl)
    ctx.set_option(echo.OPT_ATTN_PATH, 0)
    ctx.set_option(echo.OPT_FORCE_SPLITS, 0)
    out, lse = ctx.verify_attn(sel, make_kv(wl, k, v), q, SM_SCALE)
    n = want_sel["n_selected"]
    assert n == (wl.R * 60 if static else wl.gate.budget)
    rng = np.random.default_rng(100 + cfg)
    rows = [(int(rng.integers(0, n)), int(rng.integers(0, wl.Hq))) for _ in range(128)] + [(0, 0), (n - 1, wl.Hq - 1)]
    _compare(wl, want_sel, q, k, v, out, lse, rows=rows)
    assert ctx.device_status() == 0


def test_step_is_cuda_graph_capturable():
    """The three calls never synchronise or read device results on the host (include/echo.h): one verify step is
    captured into a CUDA graph (the paper serves under CUDA graphs) and replayed on new Q; results equal the
    eager run bit for bit."""
    import torch
    wl = W.make_config(1, R=4, gated=True)
    ctx, sel, want_sel, q, k, v = _setup(wl)
    from paper_2604_09603_b200 import echo
    ctx.set_option(echo.OPT_ATTN_PATH, 0)
    ctx.set_option(echo.OPT_FORCE_SPLITS, 0)
    kv = make_kv(wl, k, v)
    g = wl.gate
    cap = sel.capacity
    d_off, d_par, d_lq = dev(wl.cand_offsets), dev(wl.parent), dev(wl.logq)
    out = torch.zeros_like(q)
    lse = torch.zeros(cap, wl.Hq, dtype=torch.float32, device="cuda")

    def step():
        ctx.gate_select(d_off, d_par, d_lq, g.depth_mask, g.log_tau, g.w_max, g.budget, g.static_k, capacity=cap,
                        max_cand=wl.max_cand, out=sel)
        ctx.verify_attn(sel, kv, q, SM_SCALE, out=out, lse=lse)

    step()
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        step()  # warm-up on the capture stream
        side.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            step()
    torch.cuda.synchronize()
    q.copy_(torch.randn_like(q))
    out.zero_(); lse.zero_()
    graph.replay()
    torch.cuda.synchronize()
    out_g, lse_g = out.clone(), lse.clone()
    out.zero_(); lse.zero_()
    step()
    torch.cuda.synchronize()
    assert torch.equal(out_g, out) and torch.equal(lse_g, lse)
    _compare(wl, want_sel, q, k, v, out_g, lse_g)


@pytest.mark.parametrize("path", PATHS)
def test_attn_second_layer_of_a_two_layer_pool(path):
    """pools [2 layers][pages][Hkv][16][128]: attention over layer 1 reads layer 1's pages only (4-D tensor map
    coordinate = ((layer * pages + page) * Hkv + head) * 2)."""
    from paper_2604_09603_b200 import echo
    wl = W.make_config(1, R=3, gated=True)
    ctx = get_ctx()
    sel = run_gate_select(ctx, wl)
    want_sel = oracle_gate_select(orc, wl)
    q, k, v = W.draw_qkv(wl, max(1, sel.capacity), device="cuda", num_layers=2)
    ctx.set_option(echo.OPT_ATTN_PATH, path)
    ctx.set_option(echo.OPT_FORCE_SPLITS, 0)
    kv = make_kv(wl, k, v)
    n = want_sel["n_selected"]
    rng = np.random.default_rng(9)
    rows = [(int(rng.integers(0, n)), int(rng.integers(0, wl.Hq))) for _ in range(40)] + [(0, 0), (n - 1, wl.Hq - 1)]
    qb, kb, vb = torch_bf16_to_bits(q), torch_bf16_to_bits(k), torch_bf16_to_bits(v)
    for layer in (1, 0):
        out, lse = ctx.verify_attn(sel, kv, q, SM_SCALE, layer=layer)
        res = orc.verify_attn(want_sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, layer=layer,
                              rows=rows)
        o_gpu = bf16_bits_to_f32(torch_bf16_to_bits(out)).astype(np.float64)
        l_gpu = lse.cpu().numpy().astype(np.float64)
        assert max(np.abs(o_gpu[k_, h] - res[(k_, h)][0]).max() for (k_, h) in rows) <= TOL_O
        assert max(abs(l_gpu[k_, h] - res[(k_, h)][1]) for (k_, h) in rows) <= TOL_LSE
    assert ctx.device_status() == 0


@pytest.mark.parametrize("world", [2, 4])
def test_attn_head_sharded_equals_unsharded(world):
    """NEXT-4 / SURVEY 8(e): rank r runs the same call on its KV heads' shard of Q and the pools; the concatenation
    of the ranks' outputs is the unsharded output bit for bit (one GPU, the shards run one after the other: they
    share nothing and wait on nothing)."""
    import torch
    from paper_2604_09603_b200 import echo, sharding
    wl = W.make_config(1, R=5, gated=True)
    ctx, sel, want_sel, q, k, v = _setup(wl)
    ctx.set_option(echo.OPT_ATTN_PATH, 0)
    ctx.set_option(echo.OPT_FORCE_SPLITS, 1)
    out, lse = ctx.verify_attn(sel, make_kv(wl, k, v), q, SM_SCALE)
    outs, lses = [], []
    for r in range(world):
        qs, ks, vs = sharding.shard_attention_inputs(q, k, v, r, world)
        o_r, l_r = ctx.verify_attn(sel, make_kv(wl, ks, vs), qs, SM_SCALE)
        outs.append(o_r.clone()); lses.append(l_r.clone())
    n = want_sel["n_selected"]
    assert torch.equal(torch.cat(outs, dim=1)[:n], out[:n]) and torch.equal(torch.cat(lses, dim=1)[:n], lse[:n])


@pytest.mark.parametrize("cfg,R,splits", [(0, None, 0), (0, None, 3), (1, None, 0), (1, 300, 1), (1, 300, 2), (2, 40, 16)])
def test_attn_work_list_planned_in_kernel_or_by_k_plan(cfg, R, splits):
    """The tcgen05 kernel plans its work list itself for up to 512 (request, split) pairs, else k_plan runs in front of
    it (R x splits = 600 and 640 here; ECHO_OPT_ATTN_PLAN = 1 forces it): same items in another order, so the
    outputs are equal bit for bit -- and right (oracle on sampled rows)."""
    import torch
    from paper_2604_09603_b200 import echo
    wl = W.make_config(cfg, R=R, gated=True)
    ctx, sel, want_sel, q, k, v = _setup(wl)
    kv = make_kv(wl, k, v)
    ctx.set_option(echo.OPT_ATTN_PATH, 2)
    ctx.set_option(echo.OPT_FORCE_SPLITS, splits)
    res = []
    for plan in (0, 1):
        ctx.set_option(echo.OPT_ATTN_PLAN, plan)
        out, lse = ctx.verify_attn(sel, kv, q, SM_SCALE)
        torch.cuda.synchronize()
        res.append((out, lse))
    n = want_sel["n_selected"]
    assert torch.equal(res[0][0][:n], res[1][0][:n]) and torch.equal(res[0][1][:n], res[1][1][:n])
    assert ctx.device_status() == 0
    rng = np.random.default_rng(17)
    rows = sorted({(int(a), int(b)) for a, b in zip(rng.integers(0, n, 40), rng.integers(0, wl.Hq, 40))})
    rows += [(0, 0), (n - 1, wl.Hq - 1)]
    _compare(wl, want_sel, q, k, v, res[0][0], res[0][1], rows=sorted(set(rows)))
    ctx.set_option(echo.OPT_ATTN_PLAN, 0)
    ctx.set_option(echo.OPT_ATTN_PATH, 0)
    ctx.set_option(echo.OPT_FORCE_SPLITS, 0)
