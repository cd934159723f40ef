"""-m gpu: S8 over vocabulary-sharded logits.  One GPU plays the tensor-parallel
ranks one after the other: echo_argmax_shard on each rank's columns, the ranks' keys stacked the way the all-gather
lays them out, echo_argmax_merge.  Checked bit-exactly against the oracle: the per-shard (maximum, first index) pairs,
the argmax over the unsharded row, and -- through echo_accept -- the same acceptance as the fused argmax gives.
Collected after the other GPU tests and before test_zz_no_alloc.py (which has to stay last)."""
import numpy as np
import pytest

from gpu_util import dev, get_ctx, make_kv, run_gate_select
from helpers import oracle_gate_select, packed_tokens, torch_bf16_to_bits
from oracle import echo_oracle as orc
from paper_2604_09603_b200 import sharding, workloads as W

pytestmark = pytest.mark.gpu


def _decode(keys):
    """(value as fp32, global index) held by the 64-bit keys of echo.h"""
    k = keys.cpu().numpy().view(np.uint64)
    o = (k >> np.uint64(32)).astype(np.uint32)
    bits = np.where(o & np.uint32(0x80000000), o & np.uint32(0x7FFFFFFF), ~o)
    return bits.astype(np.uint32).view(np.float32), (np.uint64(0x7FFFFFFF) - (k & np.uint64(0xFFFFFFFF))).astype(np.int64)


def _sharded_tokens(ctx, sel, lg, V, world, n, bits):
    """the ranks' shards of lg [capacity][ld] one after the other; returns the merged tokens (device int32)"""
    import torch
    cap = sel.capacity
    gathered = torch.empty(world, cap, dtype=torch.int64, device="cuda")
    for r in range(world):
        v0, v1 = sharding.vocab_shard(r, world, V)
        if v1 == v0:
            gathered[r].zero_()
            continue
        ctx.argmax_shard(sel, lg[:, v0:v1], v0, out=gathered[r])      # a column view: row pitch stays lg's
        val, idx = _decode(gathered[r])
        wv, wi = orc.argmax_shard_pairs(bits[:n], v0, v1)
        np.testing.assert_array_equal(idx[:n], wi, err_msg=f"rank {r}/{world}: first index")
        np.testing.assert_array_equal(val[:n].view(np.uint32), wv.view(np.uint32), err_msg=f"rank {r}/{world}: maximum")
        assert (gathered[r, n:] == 0).all()                            # rows behind the packed nodes: key 0
    return ctx.argmax_merge(sel, gathered, world)


@pytest.mark.parametrize("world", [1, 2, 3, 8])
def test_sharded_argmax_cfg4_rows(world):
    """cfg4's vocabulary (151 936 columns) and logits; acceptance from the merged tokens = acceptance from the logits"""
    import torch
    ctx = get_ctx()
    wl = W.make_config(4, R=6)
    sel = run_gate_select(ctx, wl, capacity=wl.gate.budget + 8)       # some rows behind the packed nodes
    want_sel = oracle_gate_select(orc, wl)
    n = want_sel["n_selected"]
    assert int(sel.n_selected.item()) == n and 0 < n < sel.capacity
    draft, _, glob = packed_tokens(wl, want_sel)
    lg = W.draw_logits(wl, glob, device="cuda")
    lg = torch.cat([lg, torch.randn(sel.capacity - n, lg.shape[1], device="cuda").to(torch.bfloat16)])
    bits = torch_bf16_to_bits(lg)
    tok = _sharded_tokens(ctx, sel, lg, wl.vocab, world, n, bits)
    want_tok = orc.argmax_bf16(bits[:n], wl.vocab)
    np.testing.assert_array_equal(tok[:n].cpu().numpy(), want_tok)
    dpad = np.zeros(sel.capacity, np.int32); dpad[:n] = draft
    _, k, v = W.draw_qkv(wl, 1, device="cuda")
    kv = make_kv(wl, k, v)
    a = ctx.accept(sel, kv, dev(dpad), dev(wl.prev_token), target_token=tok, compact=False).to_host()
    b = ctx.accept(sel, kv, dev(dpad), dev(wl.prev_token), target_logits=lg, vocab=wl.vocab, compact=False).to_host()
    want = orc.accept(want_sel, draft, wl.prev_token, want_tok, wl.R)
    for key in ("accept_len", "last_node", "bonus_token", "accept_idx"):
        np.testing.assert_array_equal(a[key][:wl.R], want[key], err_msg=key)
        np.testing.assert_array_equal(a[key][:wl.R], b[key][:wl.R], err_msg=key + " (fused argmax)")
    assert ctx.device_status() == 0


@pytest.mark.parametrize("world", [1, 2, 3, 8])
@pytest.mark.parametrize("V,ld", [(1000, 1008), (1003, 1008), (20, 24)])
def test_sharded_argmax_ties_and_edges(world, V, ld):
    """the same maximum in several shards (lowest index), -0 / +0 in different shards, all-equal and all -inf rows, a
    vocabulary that is not a multiple of 8, columns beyond it, ranks without columns (V < 8 x world)"""
    import torch
    ctx = get_ctx()
    wl = W.make_config(0, gated=False)
    sel = run_gate_select(ctx, wl, capacity=wl.gate.budget + 8)
    n = int(sel.n_selected.item())
    assert 8 <= n < sel.capacity
    g = torch.Generator(device="cuda"); g.manual_seed(5 + V)
    lg = torch.randn(sel.capacity, ld, generator=g, device="cuda").to(torch.bfloat16)
    lg[:, V:] = 100.0                                         # beyond the vocabulary: never read
    hi, mid = V - 1, V // 2
    lg[0, :] = 1.0; lg[0, V:] = 100.0                         # all equal -> 0
    lg[1, hi] = 9.0; lg[1, mid] = 9.0; lg[1, mid - 1] = 9.0   # duplicate maximum across a shard boundary
    lg[2, hi] = 50.0                                          # last column of the vocabulary
    lg[3, :V] = float("-inf")                                 # all -inf -> 0
    lg[4, :V] = -1.0; lg[4, 3] = -0.0; lg[4, hi] = 0.0        # -0 == +0 -> index 3
    lg[5, :V] = float("-inf"); lg[5, mid] = -3.0              # one finite logit
    lg[6, :V] = -2.0; lg[6, V - 2] = -1.0                     # maximum in the scalar tail when V % 8 != 0
    bits = torch_bf16_to_bits(lg)
    tok = _sharded_tokens(ctx, sel, lg, V, world, n, bits)[:n].cpu().numpy()
    want = orc.argmax_bf16(bits[:n], V)
    np.testing.assert_array_equal(tok, want)
    assert tok[0] == 0 and tok[1] == mid - 1 and tok[2] == hi and tok[3] == 0 and tok[4] == 3 and tok[5] == mid
    assert tok[6] == V - 2
    assert ctx.device_status() == 0


# keys written out by hand from include/echo.h: ordered(v) = bits | 0x80000000 for v >= 0, ~bits for v < 0 (-0 counts
# as +0), in the high word; 0x7FFFFFFF - (vocab_base + first index) in the low word
HAND_KEYS = [  # (planted logits {column: value}, fill value, expected key) for a shard of 16 columns at vocab_base 16
    ({5: 1.0}, -1.0, 0xBF800000_7FFFFFEA),            # 1.0 = 0x3F800000 at global index 21
    ({}, -2.0, 0x3FFFFFFF_7FFFFFEF),                  # all -2.0 = 0xC0000000: first index, 16
    ({}, float("-inf"), 0x007FFFFF_7FFFFFEF),         # all -inf = 0xFF800000: first index
    ({9: -0.0}, -1.0, 0x80000000_7FFFFFE6),           # -0 reported as +0 at global index 25
    ({3: 0.5, 12: 0.5}, 0.25, 0xBF000000_7FFFFFEC),   # duplicate maximum 0.5 = 0x3F000000: lower index, 19
    ({15: 3.0}, 0.0, 0xC0400000_7FFFFFE0),            # last column, global index 31; 3.0 = 0x40400000
]


def test_argmax_shard_keys_by_hand():
    import torch
    ctx = get_ctx()
    wl = W.make_config(0, gated=False)
    sel = run_gate_select(ctx, wl)
    assert int(sel.n_selected.item()) >= len(HAND_KEYS)
    lg = torch.zeros(sel.capacity, 32, dtype=torch.bfloat16, device="cuda")
    lg[:, :16] = 77.0                                              # another rank's columns: never read
    for r, (planted, fill, _) in enumerate(HAND_KEYS):
        lg[r, 16:] = fill
        for c, val in planted.items():
            lg[r, 16 + c] = val
    keys = ctx.argmax_shard(sel, lg[:, 16:], 16).cpu().numpy().view(np.uint64)
    for r, (_, _, want) in enumerate(HAND_KEYS):
        assert int(keys[r]) == want, (r, hex(int(keys[r])), hex(want))
    tok = ctx.argmax_merge(sel, torch.stack([torch.zeros_like(ctx.argmax_shard(sel, lg[:, 16:], 16)),
                                             ctx.argmax_shard(sel, lg[:, 16:], 16)]), 2).cpu().numpy()
    assert tok[:len(HAND_KEYS)].tolist() == [21, 16, 16, 25, 19, 31]    # key 0 (a rank without columns) never wins
    assert ctx.device_status() == 0


def test_sharding_helper_one_rank_equals_fused_argmax():
    """sharding.sharded_argmax with one rank (no collective) against echo_accept's own argmax"""
    import torch
    ctx = get_ctx()
    wl = W.make_config(4, R=4)
    sel = run_gate_select(ctx, wl)
    n = int(sel.n_selected.item())
    glob = (wl.cand_offsets[sel.to_host()["sel_req"][:n]] + sel.to_host()["sel_node"][:n]).astype(np.int64)
    lg = W.draw_logits(wl, glob, device="cuda")
    lg = torch.cat([lg, torch.zeros(sel.capacity - n, lg.shape[1], dtype=lg.dtype, device="cuda")])
    bufs = {}
    for _ in range(2):                                         # the buffers are reused by the second call
        tok = sharding.sharded_argmax(ctx, sel, lg, 0, 1, wl.vocab, bufs=bufs)
    np.testing.assert_array_equal(tok[:n].cpu().numpy(), orc.argmax_bf16(torch_bf16_to_bits(lg[:n]), wl.vocab))
    assert ctx.device_status() == 0


def test_argmax_shard_rejects_bad_arguments():
    import torch
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    wl = W.make_config(0, gated=False)
    sel = run_gate_select(ctx, wl)
    lg = torch.zeros(sel.capacity, 64, dtype=torch.bfloat16, device="cuda")
    for kw in (dict(vocab_base=-1), dict(vocab_base=0, vocab_shard=0), dict(vocab_base=0, vocab_shard=65),
               dict(vocab_base=2**31 - 8, vocab_shard=64)):
        with pytest.raises(echo.EchoError) as e:
            ctx.argmax_shard(sel, lg, **kw)
        assert e.value.code == echo.ERR_INVALID_ARG
    with pytest.raises(echo.EchoError) as e:
        ctx.argmax_shard(sel, lg[:, 4:], 4)                     # a shard that does not start on a 16-byte boundary
    assert e.value.code == echo.ERR_INVALID_ARG
    with pytest.raises(echo.EchoError) as e:
        ctx.argmax_merge(sel, torch.zeros(sel.capacity, dtype=torch.int64, device="cuda"), 0)
    assert e.value.code == echo.ERR_INVALID_ARG
