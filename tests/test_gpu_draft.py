"""-m gpu parity: echo_draft_expand (CUDA, through the C ABI) against the oracle, bit-exact, and the hand-over to
echo_gate_select: a tree built on the device level by level gives the selection the oracle gives for that tree."""
import numpy as np
import pytest
import torch

from oracle import echo_oracle as orc
from paper_2604_09603_b200 import workloads as W
from gpu_util import dev, get_ctx, assert_selection_equal

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("R,L,k", [(1, 1, 1), (4, 3, 8), (128, 8, 10), (37, 3, 16)])
def test_draft_expand_levels_and_gate_select(R, L, k):
    ctx = get_ctx()
    rng = np.random.default_rng(R * 100 + k)
    C = L * k
    offs = (np.arange(R + 1) * C).astype(np.int32)
    d_offs = dev(offs)
    d_parent = torch.full((R * C,), -7, dtype=torch.int32, device="cuda")
    d_logq = torch.zeros(R * C, dtype=torch.float32, device="cuda")
    d_tok = torch.zeros(R * C, dtype=torch.int32, device="cuda")
    ps_h = np.zeros((R, 1), np.float32)
    d_ps = dev(ps_h)
    parent_h, logq_h, tok_h = np.zeros((R, C), np.int32), np.zeros((R, C), np.float32), np.zeros((R, C), np.int32)
    for lvl in range(L):
        kp = 1 if lvl == 0 else k
        cl, ct = W.draw_draft_level(rng, R, kp, k)
        if lvl == 1:
            cl[:, :, 1] = cl[:, :, 0]                      # exact ties inside and across parents
        want = orc.draft_expand(lvl, k, ps_h, cl, ct)
        d_score = torch.zeros(R, k, dtype=torch.float32, device="cuda")
        ctx.draft_expand(lvl, k, d_ps, dev(cl), dev(ct), d_offs, d_parent, d_logq, d_tok, d_score)
        np.testing.assert_array_equal(d_score.cpu().numpy(), want["score"])
        sl = slice(lvl * k, (lvl + 1) * k)
        parent_h[:, sl] = -1 if lvl == 0 else (lvl - 1) * k + want["sel_parent"]
        logq_h[:, sl], tok_h[:, sl] = want["logq"], want["token"]
        ps_h, d_ps = want["score"], d_score
    np.testing.assert_array_equal(d_parent.cpu().numpy().reshape(R, C), parent_h)
    np.testing.assert_array_equal(d_logq.cpu().numpy().reshape(R, C), logq_h)
    np.testing.assert_array_equal(d_tok.cpu().numpy().reshape(R, C), tok_h)
    assert ctx.device_status() == 0
    # the device-built trees go straight into the gate (no host round trip)
    lt = np.zeros(32, np.float32)
    lt[0], lt[min(2, L - 1)] = np.float32(np.log(0.2)), np.float32(np.log(0.1))
    mask = 1 | (1 << min(2, L - 1))
    budget = max(1, R * C // 3)
    sel = ctx.gate_select(d_offs, d_parent, d_logq, mask, lt, k, budget, capacity=budget, max_cand=C)
    want_sel = orc.gate_select(offs, parent_h.reshape(-1), logq_h.reshape(-1), mask, lt, k, budget)
    assert_selection_equal(sel.to_host(), want_sel)


def test_draft_expand_edges():
    from paper_2604_09603_b200 import echo
    ctx = get_ctx()
    # a tree range too short for the level: status bit, nothing written past the range
    offs = dev(np.asarray([0, 4], np.int32))
    par = torch.full((4,), -7, dtype=torch.int32, device="cuda")
    lq = torch.zeros(4, device="cuda"); tok = torch.zeros(4, dtype=torch.int32, device="cuda")
    sc = torch.zeros(1, 4, device="cuda")
    cl, ct = W.draw_draft_level(np.random.default_rng(0), 1, 4, 4)
    ctx.draft_expand(1, 4, dev(np.zeros((1, 4), np.float32)), dev(cl), dev(ct), offs, par, lq, tok, sc)
    assert ctx.device_status() == echo.DEV_TREE_OVERFLOW and (par.cpu().numpy() == -7).all()
    with pytest.raises(Exception):
        ctx.draft_expand(0, 17, sc, sc, tok, offs, par, lq, tok, sc)       # topk > ECHO_MAX_TOPK
