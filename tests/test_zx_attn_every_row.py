"""-m gpu: verify attention on EVERY (node, head) row of BASELINE.json's BS=128 configurations (cfg2: 131 072 rows,
cfg3: 65 536) and on every row of seeded request samples of the static-60 run and of cfg4, against the fp64 definition
computed by the plain-C oracle (oracle/echo_oracle_attn.c) on all host cores.  Collected after the other attention
tests (a failure here must not hide them under pytest -x) and before test_zz_no_alloc.py."""
import numpy as np
import pytest

from helpers import bf16_bits_to_f32, torch_bf16_to_bits
from paper_2604_09603_b200 import workloads as W
from test_gpu_fullsize import SM_SCALE, TOL_LSE, TOL_O, _attn_case

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,static,requests", [(2, False, None), (3, False, None), (2, True, 24), (4, False, 32)])
def test_attn_full_size_every_row(cfg, static, requests):
    """cfg2 and cfg3 at full size: EVERY (node, head) row -- 131 072 / 65 536 of them -- against the fp64 definition,
    computed by the plain-C oracle on all host cores ("full parity on cfg0-3"); the static-60 run (491 520
    rows) on every row of a seeded sample of 24 requests, cfg4 (R = 256, prefixes up to 32 768) on every row of a seeded
    sample of 32 requests ("else on a seeded sample of 32 requests")."""
    from oracle import attn_c
    wl = W.make_config(cfg, static=static, gated=not static)
    want_sel, q, k, v, out, lse = _attn_case(wl)
    n = want_sel["n_selected"]
    qb, kb, vb = torch_bf16_to_bits(q), torch_bf16_to_bits(k), torch_bf16_to_bits(v)
    o_gpu = bf16_bits_to_f32(torch_bf16_to_bits(out))[:n]
    l_gpu = lse.cpu().numpy()[:n]
    assert np.isfinite(o_gpu).all() and np.isfinite(l_gpu).all()
    if requests is None:
        O, L = attn_c.verify_attn(want_sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE)
        eo, el = np.abs(o_gpu - O).max(), np.abs(l_gpu - L).max()
    else:
        offs = want_sel["sel_offsets"]
        act = np.flatnonzero(np.diff(offs) > 0)
        reqs = np.sort(np.random.default_rng(400 + cfg).choice(act, size=min(requests, len(act)), replace=False))
        nodes = np.concatenate([np.arange(offs[i], offs[i + 1]) for i in reqs])
        rows = [(int(k_), h) for k_ in nodes for h in range(wl.Hq)]
        O, L = attn_c.verify_attn(want_sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=rows)
        eo = np.abs(o_gpu[nodes].reshape(-1, 128) - O).max()
        el = np.abs(l_gpu[nodes].reshape(-1) - L).max()
    assert eo <= TOL_O, f"max|dO| = {eo}"
    assert el <= TOL_LSE, f"max|dlse| = {el}"
