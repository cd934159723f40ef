"""Host-side logic of the multi-GPU path: the verify step shards by request.

Each rank owns its own batch of requests and their KV pages (DP attention); there is no data-path collective.
What the ranks exchange is the measurement only: the step time is the MAX over ranks, the token counts are SUMs.
The functions take the process group's device so that the same code runs under NCCL (bench.py on GPUs) and under
gloo on CPU (tests/test_sharding_gloo.py).
"""
from __future__ import annotations

from . import workloads as W


def rank_seed(config_id: int, rank: int) -> int:
    """Seed of rank `rank`'s batch: disjoint per rank, rank 0 reproduces the single-GPU workload."""
    return W.SEED_BASE + config_id + 1000 * rank


def rank_workload(config_id: int, rank: int, **kw):
    return W.make_config(config_id, seed=rank_seed(config_id, rank), **kw)


def reduce_step_stats(times_ms, counts, world: int, device, dist=None):
    """times_ms: per-rank durations (any number) -> max over ranks; counts: per-rank totals -> sum over ranks.
    Returns (list of floats, list of floats).  With world == 1 no collective runs."""
    import torch
    t = torch.tensor([float(x) for x in times_ms], dtype=torch.float64, device=device)
    c = torch.tensor([float(x) for x in counts], dtype=torch.float64, device=device)
    if world > 1:
        if dist is None:
            import torch.distributed as dist  # noqa: PLC0415
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.cpu()], [float(x) for x in c.cpu()]


def job_throughput(total_units: float, steps: int, max_ms: float) -> float:
    """Whole-job units per second: units all ranks processed per step x steps / slowest rank's time."""
    return total_units * steps / (max_ms * 1e-3)


def head_shard(rank: int, world: int, Hq: int, Hkv: int):
    """Head-sharded (tensor-parallel style) split of the verify attention: rank r owns the KV
    heads [r Hkv/W, (r+1) Hkv/W) of every page and the query heads of those groups.  Attention is independent per
    KV head, so S6-S7 need no collective; S1-S5 and S9 are replicated (kilobytes); S10 compacts each rank's heads.
    Returns (slice over query heads, slice over KV heads)."""
    if world < 1 or not (0 <= rank < world) or Hkv % world or Hq % Hkv:
        raise ValueError(f"cannot shard Hq={Hq} Hkv={Hkv} over {world} ranks")
    per = Hkv // world
    G = Hq // Hkv
    return slice(rank * per * G, (rank + 1) * per * G), slice(rank * per, (rank + 1) * per)


def shard_attention_inputs(q, k_pool, v_pool, rank: int, world: int):
    """q [cap][Hq][128], pools [layers][pages][Hkv][16][128] (torch tensors) -> this rank's contiguous shards."""
    hq, hkv = head_shard(rank, world, q.shape[1], k_pool.shape[2])
    return q[:, hq].contiguous(), k_pool[:, :, hkv].contiguous(), v_pool[:, :, hkv].contiguous()
