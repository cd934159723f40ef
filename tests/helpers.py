"""Test-side helpers (no method arithmetic): bf16 bit conversion and oracle input marshalling."""
import numpy as np


def f32_to_bf16_bits(x):
    """round-to-nearest-even float32 -> bf16 bit patterns (uint16)."""
    u = np.asarray(x, np.float32).view(np.uint32).astype(np.uint64)
    r = ((u >> 16) & 1) + 0x7FFF
    return ((u + r) >> 16).astype(np.uint16)


def bf16_bits_to_f32(b):
    return (np.asarray(b).astype(np.uint32) << 16).view(np.float32)


def torch_bf16_to_bits(t):
    import torch
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def oracle_gate_select(orc, wl, gate=None, schedule=0):
    g = gate or wl.gate
    return orc.gate_select(wl.cand_offsets, wl.parent, wl.logq, g.depth_mask, g.log_tau, g.w_max,
                           g.budget, g.static_k, schedule=schedule)


def packed_tokens(wl, sel):
    """draft / target tokens in packed order from the per-candidate ground truth."""
    glob = wl.cand_offsets[sel["sel_req"]] + sel["sel_node"] if sel["n_selected"] else np.zeros(0, np.int64)
    glob = np.asarray(glob, np.int64)
    return wl.draft_token[glob], wl.target_after[glob], glob
