"""N > 1 path on CPU: two gloo processes run the host-side logic bench.py uses under torchrun:
per-rank batches are disjoint, rank 0 reproduces the single-GPU workload, the step time is the max over ranks and the
token counts are sums -- and each rank's selection (computed by the oracle here: no GPU) depends on its own batch only."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2604_09603_b200 import sharding


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import echo_oracle as orc
        wl = sharding.rank_workload(0, rank)
        g = wl.gate
        sel = orc.gate_select(wl.cand_offsets, wl.parent, wl.logq, g.depth_mask, g.log_tau, g.w_max, g.budget, g.static_k)
        n_sel = int(sel["n_selected"])
        ms = 10.0 + 5.0 * rank            # rank 1 is the slow one
        (t_max, e_max), (n_all, acc_all) = sharding.reduce_step_stats([ms, ms / 1e3], [n_sel, rank + 1], world,
                                                                       torch.device("cpu"), dist)
        gathered = [None] * world
        dist.all_gather_object(gathered, (n_sel, float(wl.logq.sum()), wl.prefix_len.tolist()))
        out[rank] = dict(t_max=t_max, e_max=e_max, n_all=n_all, acc_all=acc_all, gathered=gathered, n_sel=n_sel)
    finally:
        dist.destroy_process_group()


def test_two_rank_reduction_and_disjoint_batches():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = {k: dict(v) for k, v in out.items()}
    assert set(res) == {0, 1}
    for r in (0, 1):
        assert res[r]["t_max"] == 15.0 and res[r]["e_max"] == pytest.approx(0.015)   # max over ranks
        assert res[r]["acc_all"] == 3.0                                              # 1 + 2
        assert res[r]["n_all"] == res[0]["n_sel"] + res[1]["n_sel"]                  # sum over ranks
    g = res[0]["gathered"]
    assert g[0][1] != g[1][1]                      # different draws per rank
    assert g == res[1]["gathered"]                 # both ranks saw the same exchange
    # whole-job value = all ranks' units / slowest rank's time
    assert sharding.job_throughput(res[0]["n_all"], 4, res[0]["t_max"]) == pytest.approx(res[0]["n_all"] * 4 / 0.015)


def test_rank0_is_the_single_gpu_workload():
    from paper_2604_09603_b200 import workloads as W
    a, b = sharding.rank_workload(0, 0), W.make_config(0)
    assert np.array_equal(a.logq, b.logq) and np.array_equal(a.page_table, b.page_table)
    assert sharding.rank_seed(2, 3) == W.SEED_BASE + 2 + 3000
    t, c = sharding.reduce_step_stats([1.5], [7], 1, torch.device("cpu"))
    assert t == [1.5] and c == [7.0]


def test_head_shards_partition_the_heads():
    for Hq, Hkv, W_ in [(64, 8, 1), (64, 8, 2), (64, 8, 8), (32, 8, 4), (64, 4, 4)]:
        q_seen, kv_seen = [], []
        for r in range(W_):
            hq, hkv = sharding.head_shard(r, W_, Hq, Hkv)
            q_seen += list(range(Hq))[hq]
            kv_seen += list(range(Hkv))[hkv]
            G = Hq // Hkv
            assert [h // G for h in list(range(Hq))[hq]] == sorted(list(range(Hkv))[hkv] * G)   # groups stay whole
        assert q_seen == list(range(Hq)) and kv_seen == list(range(Hkv))
    with pytest.raises(ValueError):
        sharding.head_shard(0, 3, 64, 8)
    q = torch.arange(2 * 8 * 4).reshape(2, 8, 4)
    kp = torch.arange(1 * 3 * 2 * 16 * 4).reshape(1, 3, 2, 16, 4)
    qs, ks, vs = sharding.shard_attention_inputs(q, kp, kp + 1, 1, 2)
    assert qs.shape == (2, 4, 4) and ks.shape == (1, 3, 1, 16, 4) and qs.is_contiguous()
    assert torch.equal(qs, q[:, 4:]) and torch.equal(vs, kp[:, :, 1:] + 1)


class _FakeCtx:
    """records what sharding.global_budget_gate_select passes to the two halves of the gate (no GPU here)"""
    device = torch.device("cpu")

    def gate_keys(self, cand_offsets, parent, logq, depth_mask, log_tau, w_max, budget, sel, static_k=0, schedule=0,
                  cand_index_base=0, request_base=0, max_cand=128):
        self.bases = (cand_index_base, request_base)
        return torch.arange(parent.numel(), dtype=torch.int64) + 1000 * cand_index_base

    def gate_select_keys(self, cand_offsets, parent, logq, depth_mask, log_tau, w_max, budget, local_keys, all_keys,
                         sel, static_k=0, schedule=0, max_cand=128):
        return dict(local=local_keys.clone(), all=all_keys.clone(), bases=self.bases, budget=budget)


def _worker_global(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2604_09603_b200 import workloads as W
        N, R = (7, 2) if rank == 0 else (4, 3)                      # ranks of different sizes: padding is exercised
        offs = torch.tensor([0, 3, N] if rank == 0 else [0, 1, 2, N], dtype=torch.int32)
        gate = W.Gate(budget=5)
        res = sharding.global_budget_gate_select(_FakeCtx(), rank, world, offs, torch.zeros(N, dtype=torch.int32),
                                                 torch.zeros(N), gate, None, dist=dist)
        out[rank] = {k: (v.tolist() if hasattr(v, "tolist") else v) for k, v in res.items()}
    finally:
        dist.destroy_process_group()


def test_global_budget_exchange_under_gloo():
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker_global, args=(2, _free_port(), out), nprocs=2, join=True)
        res = {k: dict(v) for k, v in out.items()}
    assert res[0]["bases"] == (0, 0) and res[1]["bases"] == (7, 2)          # exclusive prefix sums of (N, R)
    want_all = list(range(7)) + [7000 + i for i in range(4)] + [-1] * 3     # rank 1 padded to the largest N
    assert res[0]["all"] == want_all and res[1]["all"] == want_all
    assert res[0]["local"] == list(range(7)) and res[1]["local"] == [7000 + i for i in range(4)]
    assert res[0]["budget"] == res[1]["budget"] == 5
    assert sharding.rank_bases([3, 4, 5], 2) == 7 and sharding.rank_bases([3, 4, 5], 0) == 0


def test_vocab_shards_partition_the_vocabulary():
    for V, W_ in [(151936, 1), (151936, 2), (151936, 8), (128256, 4), (1000, 3), (1003, 8), (20, 8), (5, 2)]:
        edges = [sharding.vocab_shard(r, W_, V) for r in range(W_)]
        assert edges[0][0] == 0 and edges[-1][1] == V
        for (a0, a1), (b0, b1) in zip(edges, edges[1:]):
            assert a1 == b0 and a0 <= a1                         # contiguous, in rank order
        assert all(v0 % 8 == 0 for v0, _ in edges)               # 16-byte aligned shard starts
        sizes = [v1 - v0 for v0, v1 in edges]
        if V >= 8 * W_:
            assert max(sizes) - min(sizes) <= 8 + 7              # as equal as whole 8-column blocks allow
    with pytest.raises(ValueError):
        sharding.vocab_shard(2, 2, 100)


class _FakeArgmaxCtx:
    """stands in for the two kernels of the vocabulary-sharded S8 (no GPU here): keys in the layout echo.h gives them"""

    def argmax_shard(self, sel, logits_shard, vocab_base, vocab_shard=None, out=None):
        x = logits_shard.float().numpy()
        j = x.argmax(axis=1)
        v = (x[np.arange(x.shape[0]), j] + np.float32(0)).astype(np.float32).view(np.uint32).astype(np.uint64)
        o = np.where(v >> 31, ~v & 0xFFFFFFFF, v | 0x80000000)
        key = (o << np.uint64(32)) | (np.uint64(0x7FFFFFFF) - (vocab_base + j).astype(np.uint64))
        out.copy_(torch.from_numpy(key.view(np.int64)))
        return out

    def argmax_merge(self, sel, pairs_all, world, out=None):
        k = pairs_all.numpy().view(np.uint64).reshape(world, -1)
        out.copy_(torch.from_numpy((0x7FFFFFFF - (k.max(axis=0) & np.uint64(0xFFFFFFFF)).astype(np.int64)).astype(np.int32)))
        return out


class _Sel:
    capacity = 5


def _worker_vocab(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        V = 40
        g = torch.Generator().manual_seed(3)
        full = torch.randn(_Sel.capacity, V, generator=g).to(torch.bfloat16)
        full[0, 7] = full[0, 33] = 9.0          # the same maximum on both ranks: rank 0's index wins
        full[1, 39] = 9.0                       # last column, rank 1
        v0, v1 = sharding.vocab_shard(rank, world, V)
        tok = sharding.sharded_argmax(_FakeArgmaxCtx(), _Sel(), full[:, v0:v1], rank, world, V, dist=dist)
        out[rank] = dict(tok=tok.tolist(), want=full.float().argmax(dim=1).tolist(), shard=(v0, v1))
    finally:
        dist.destroy_process_group()


def test_sharded_argmax_exchange_under_gloo():
    """the head-sharded path's one exchange: both ranks end with the argmax over the WHOLE vocabulary"""
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker_vocab, args=(2, _free_port(), out), nprocs=2, join=True)
        res = {k: dict(v) for k, v in out.items()}
    assert res[0]["shard"] == (0, 16) and res[1]["shard"] == (16, 40)
    assert res[0]["tok"] == res[1]["tok"] == res[0]["want"]
    assert res[0]["tok"][0] == 7 and res[0]["tok"][1] == 39

