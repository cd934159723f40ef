"""-m gpu parity: echo_accept_stochastic (CUDA, through the C ABI) against the fp64 oracle.  The decisions compare a
uniform draw with an fp32 probability, so the seeded uniforms of knife-edge decisions are redrawn until every decision
of the oracle has a margin of 2e-4 (the kernel's fp32 / ex2.approx error is ~1e-5): then paths and slot maps are exact.
The bonus token is an inverse-CDF draw over 10^4..10^5 tokens: it must be the oracle's token whenever the draw is
more than EPS = 1e-6 away from both ends of that token's CDF interval, and otherwise a token whose interval is within
EPS of the draw (DESIGN.md R:T-4: the kernel's CDF is good to ~3e-7)."""
import numpy as np
import pytest
import torch

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W
from helpers import oracle_gate_select, packed_tokens, torch_bf16_to_bits
from gpu_util import dev, get_ctx, run_gate_select, make_kv, assert_selection_equal

pytestmark = pytest.mark.gpu
MARGIN = 2e-4
EPS = 1e-6


def _logits(rng, rows, V, bump_at, ld):
    x = torch.from_numpy((rng.normal(0, 2.0, (rows, ld))).astype(np.float32))
    x[torch.arange(rows), torch.from_numpy(np.asarray(bump_at, np.int64))] += 5.0
    return x.to(torch.bfloat16).cuda()


def _case(cfg, R, temperature, seed, num_layers=1, mask_frac=0.0):
    ctx = get_ctx()
    wl = W.make_config(cfg, R=R)
    sel = run_gate_select(ctx, wl)
    want_sel = oracle_gate_select(orc, wl)
    assert_selection_equal(sel.to_host(), want_sel)
    draft, target, _ = packed_tokens(wl, want_sel)
    n, cap, V = want_sel["n_selected"], sel.capacity, wl.vocab
    ld = (V + 7) // 8 * 8
    rng = np.random.default_rng(seed)
    tl = _logits(rng, cap, V, np.concatenate([target, np.zeros(cap - n, np.int64)]), ld)
    rl = _logits(rng, wl.R, V, wl.prev_token, ld)
    if mask_frac > 0:   # banned / grammar-masked tokens: -inf logits, in aligned runs of 8 and scattered
        for t_ in (tl, rl):
            m = torch.from_numpy(rng.random((t_.shape[0], ld // 8)) < mask_frac).cuda()
            t_.view(t_.shape[0], ld // 8, 8)[m] = float("-inf")
            t_[torch.from_numpy(rng.random((t_.shape[0], ld)) < 0.05).cuda()] = float("-inf")
            t_[:, :2048] = float("-inf")          # a whole thread-chunk worth of leading tokens masked
        tl[torch.arange(cap).cuda(), torch.from_numpy(np.concatenate([target, np.zeros(cap - n, np.int64)])).cuda()] = 6.0
        rl[torch.arange(wl.R).cuda(), torch.from_numpy(wl.prev_token.astype(np.int64)).cuda()] = 6.0
    tlb, rlb = torch_bf16_to_bits(tl), torch_bf16_to_bits(rl)
    ua = rng.random(cap).astype(np.float32)
    ub = rng.random(wl.R).astype(np.float32)
    for attempt in range(50):
        want = orc.accept_stochastic(want_sel, draft, rlb, tlb, V, temperature, ua, ub, wl.R)
        close = sorted({k_ for (k_, pr) in want["decisions"] if abs(float(ua[k_]) - pr) < MARGIN})
        if not close:
            break
        ua[close] = rng.random(len(close)).astype(np.float32)   # redraw only the knife-edge uniforms
    else:
        pytest.fail("no uniforms with a safe margin")
    assert want["min_margin"] >= MARGIN
    dpad = np.zeros(cap, np.int32); dpad[:n] = draft
    _, k, v = W.draw_qkv(wl, 1, device="cuda", num_layers=num_layers)
    kb, vb = torch_bf16_to_bits(k).copy(), torch_bf16_to_bits(v).copy()
    acc = ctx.accept_stochastic(sel, make_kv(wl, k, v), dev(dpad), tl, rl, V, temperature, dev(ua), dev(ub))
    got = acc.to_host()
    for key in ("accept_len", "last_node", "accept_idx"):
        np.testing.assert_array_equal(got[key][:wl.R], want[key], err_msg=key)
    # the bonus draw (see the module docstring)
    exact = 0
    for i in range(wl.R):
        t, cdf, u = int(got["bonus_token"][i]), want["bonus_cdf"][i], want["bonus_u"][i]
        w = int(want["bonus_token"][i])
        wlo = cdf[w - 1] if w > 0 else 0.0
        if wlo + EPS < u < cdf[w] - EPS:
            assert t == w, f"request {i}: token {t}, oracle {w} with margin {min(u - wlo, cdf[w] - u):.2e}"
            exact += 1
        lo = cdf[t - 1] if t > 0 else 0.0
        assert 0 <= t < V and cdf[t] > lo, f"request {i}: token {t} has no residual mass"
        assert lo - EPS <= u <= cdf[t] + EPS, f"request {i}: token {t} [{lo}, {cdf[t]}] vs draw {u}"
    assert exact >= 1 or wl.R < 4
    wc = orc.compact_kv(want_sel, want, kb, vb, wl.page_table, wl.prefix_len, wl.R)
    for key in ("slot_src", "slot_dst", "new_len"):
        np.testing.assert_array_equal(got[key][:wl.R], wc[key], err_msg=key)
    np.testing.assert_array_equal(torch_bf16_to_bits(k), kb, err_msg="compacted K pool")
    np.testing.assert_array_equal(torch_bf16_to_bits(v), vb, err_msg="compacted V pool")
    assert ctx.device_status() == 0
    return want


@pytest.mark.parametrize("cfg,R,temperature", [(0, None, 1.0), (0, None, 0.6), (1, 6, 1.0), (2, 5, 0.8), (4, 8, 1.0)])
def test_stochastic_accept_matches_oracle(cfg, R, temperature):
    want = _case(cfg, R, temperature, seed=100 + cfg)
    assert 0 <= want["accept_len"].min() and want["accept_len"].max() <= 32


@pytest.mark.parametrize("cfg,R", [(0, None), (4, 8)])
def test_stochastic_accept_with_masked_logits(cfg, R):
    """-inf logits (banned tokens): a thread of k_softmax_stats whose every chunk is masked must contribute no mass
    and no NaN ((-inf) - (-inf)); paths, bonus tokens and slot maps still match the oracle."""
    want = _case(cfg, R, 1.0, seed=300 + cfg, mask_frac=0.5)
    assert all(np.isfinite(c).all() for c in want["bonus_cdf"])


def test_low_temperature_is_greedy_on_gpu():
    """T = 0.02 with a 5-logit lead: p is one-hot to fp32 precision, so the call reproduces echo_accept."""
    ctx = get_ctx()
    wl = W.make_config(0)
    sel = run_gate_select(ctx, wl)
    want_sel = oracle_gate_select(orc, wl)
    draft, target, _ = packed_tokens(wl, want_sel)
    n, cap, V = want_sel["n_selected"], sel.capacity, wl.vocab
    rng = np.random.default_rng(5)
    tl = _logits(rng, cap, V, np.concatenate([target, np.zeros(cap - n, np.int64)]), V)
    rl = _logits(rng, wl.R, V, wl.prev_token, V)
    tt = orc.argmax_bf16(torch_bf16_to_bits(tl[:n]), V)
    prev = orc.argmax_bf16(torch_bf16_to_bits(rl), V)
    greedy = orc.accept(want_sel, draft, prev, tt, wl.R)
    dpad = np.zeros(cap, np.int32); dpad[:n] = draft
    _, k, v = W.draw_qkv(wl, 1, device="cuda")
    ua, ub = rng.random(cap).astype(np.float32) * 0.99, rng.random(wl.R).astype(np.float32) * 0.99
    acc = ctx.accept_stochastic(sel, make_kv(wl, k, v), dev(dpad), tl, rl, V, 0.02, dev(ua), dev(ub)).to_host()
    np.testing.assert_array_equal(acc["accept_len"][:wl.R], greedy["accept_len"])
    np.testing.assert_array_equal(acc["last_node"][:wl.R], greedy["last_node"])
    has = greedy["last_node"] >= 0
    np.testing.assert_array_equal(acc["bonus_token"][:wl.R][has], greedy["bonus_token"][has])
    np.testing.assert_array_equal(acc["bonus_token"][:wl.R][~has], prev[~has])
