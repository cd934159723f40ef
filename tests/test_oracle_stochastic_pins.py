"""Pins of the stochastic tree acceptance of the oracle (NEXT-2): the T -> 0 limit is the greedy
acceptance (pinned separately), the emitted token at every position is distributed exactly as the target's p (the
speculative-sampling guarantee), and hand-computed decisions on a two-child example."""
import numpy as np
import pytest

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W
from helpers import oracle_gate_select, packed_tokens


def _f32_to_bf16_bits(x):
    u = np.asarray(x, np.float32).view(np.uint32)
    return ((u + 0x7FFF + ((u >> 16) & 1)) >> 16).astype(np.uint16)


def test_hand_example_two_children():
    # one request, root context p = softmax([ln 4, ln 2, ln 1, ln 1]) = [.5, .25, .125, .125]; children tokens 1 then 0
    sel = dict(sel_offsets=np.asarray([0, 2]), parent_local=np.asarray([-1, -1]))
    V = 4
    root = _f32_to_bf16_bits(np.log(np.asarray([[4.0, 2.0, 1.0, 1.0]])))
    tl = _f32_to_bf16_bits(np.log(np.asarray([[1.0, 1.0, 1.0, 5.0], [1.0, 1.0, 6.0, 1.0]])))
    draft = np.asarray([1, 0], np.int32)
    run = lambda ua, ub: orc.accept_stochastic(sel, draft, root, tl, V, 1.0, np.asarray(ua, np.float32), np.asarray([ub], np.float32), 1)
    r = run([0.2, 0.9], 0.0)            # child 0 (token 1, p = .25): 0.2 < .25 accepted; then node 0 has no children
    assert r["accept_len"][0] == 1 and r["last_node"][0] == 0 and r["bonus_token"][0] == 0   # u_bonus 0 -> first token
    r = run([0.3, 0.6], 0.99)           # child 0 rejected (removes token 1, m = .25); child 1 (token 0): .5/.75 = .667 > .6
    assert r["accept_len"][0] == 1 and r["last_node"][0] == 1 and r["bonus_token"][0] == 3   # last token of node 1's p
    r = run([0.3, 0.7], 0.5)            # both rejected: residual [0, 0, .5, .5] of mass .25 -> u = .5 picks token 3
    assert r["accept_len"][0] == 0 and r["last_node"][0] == -1 and r["bonus_token"][0] == 3
    r = run([0.3, 0.7], 0.49)
    assert r["bonus_token"][0] == 2


def test_emitted_token_is_distributed_as_p():
    """root with three children: over a fine grid of the uniforms, the first emitted token (an accepted child's token
    or the bonus token) has exactly the target distribution."""
    V = 6
    p = np.asarray([0.05, 0.3, 0.1, 0.25, 0.2, 0.1])
    root = _f32_to_bf16_bits(np.log(p)[None])
    p = orc.softmax_bits(root[0], V, 1.0)                      # the bf16-rounded distribution the oracle sees
    sel = dict(sel_offsets=np.asarray([0, 3]), parent_local=np.asarray([-1, -1, -1]))
    draft = np.asarray([3, 1, 4], np.int32)
    tl = _f32_to_bf16_bits(np.zeros((3, V)))
    n = 24
    g = (np.arange(n) + 0.5) / n
    counts = np.zeros(V)
    for u0 in g:
        for u1 in g:
            for u2 in g:
                # the bonus draw is averaged analytically over its uniform: residual / its mass
                r = orc.accept_stochastic(sel, draft, root, tl, V, 1.0, np.asarray([u0, u1, u2], np.float32),
                                          np.asarray([0.5], np.float32), 1)
                if r["accept_len"][0] >= 1:
                    counts[draft[r["accept_idx"][0, 0]]] += 1.0
                else:
                    res = p.copy(); res[draft] = 0.0
                    counts += res / res.sum()
    assert np.abs(counts / n ** 3 - p).max() < 1.5 / n


@pytest.mark.parametrize("cfg", [0, 1])
def test_zero_temperature_limit_is_greedy(cfg):
    """T -> 0: p is one-hot at the argmax, a child is accepted iff its token is the target's greedy token, the bonus
    token is the argmax after the last accepted node: the greedy acceptance O9 (siblings carry distinct tokens)."""
    wl = W.make_config(cfg, R=4 if cfg else None)
    sel = oracle_gate_select(orc, wl)
    draft, target, _ = packed_tokens(wl, sel)
    n, V = sel["n_selected"], wl.vocab
    rng = np.random.default_rng(cfg)
    tl = rng.normal(0, 1, (n, V)).astype(np.float32); tl[np.arange(n), target] = 30.0
    rl = rng.normal(0, 1, (wl.R, V)).astype(np.float32); rl[np.arange(wl.R), wl.prev_token] = 30.0
    greedy = orc.accept(sel, draft, wl.prev_token, target, wl.R)
    st = orc.accept_stochastic(sel, draft, _f32_to_bf16_bits(rl), _f32_to_bf16_bits(tl), V, 1e-3,
                               rng.random(n).astype(np.float32) * 0.999, rng.random(wl.R).astype(np.float32), wl.R)
    assert greedy["accept_len"].sum() > 0
    assert np.array_equal(st["accept_len"], greedy["accept_len"])
    assert np.array_equal(st["last_node"], greedy["last_node"])
    assert np.array_equal(st["accept_idx"], greedy["accept_idx"])
    has = greedy["last_node"] >= 0
    assert np.array_equal(st["bonus_token"][has], greedy["bonus_token"][has])
    assert np.array_equal(st["bonus_token"][~has], np.asarray(wl.prev_token)[~has])
