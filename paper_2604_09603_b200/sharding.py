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


def vocab_shard(rank: int, world: int, vocab: int, align: int = 8):
    """Columns [v0, v1) of the target logits that rank `rank` of a tensor-parallel group holds (with the
    KV heads sharded, the logits are sharded over the vocabulary): contiguous, in rank order, every boundary but the
    last a multiple of `align` columns (16-byte rows for the streaming loads), sizes as equal as that allows.  A rank
    may hold no columns when vocab < world * align."""
    if world < 1 or not (0 <= rank < world) or vocab < 1 or align < 1:
        raise ValueError(f"cannot shard a vocabulary of {vocab} over {world} ranks")
    blocks = (vocab + align - 1) // align
    b0 = blocks * rank // world
    b1 = blocks * (rank + 1) // world
    return min(vocab, b0 * align), min(vocab, b1 * align)


def sharded_argmax(ctx, sel, logits_shard, rank: int, world: int, vocab: int, dist=None, bufs=None):
    """S8 when the ranks hold vocabulary shards of the logits: every rank reduces its columns to one 64-bit (max, first
    index) key per packed node (echo_argmax_shard), the ranks all-gather the keys (capacity x 8 B each -- the one
    exchange of the head-sharded path), and every rank takes the greatest key per row (echo_argmax_merge).  Returns the
    int32 target tokens for ctx.accept(target_token=...).  `logits_shard` = [capacity][v1 - v0] of vocab_shard(rank,
    world, vocab); `bufs` keeps the key buffers between steps.  No host synchronisation."""
    import torch
    if dist is None and world > 1:
        import torch.distributed as dist  # noqa: PLC0415
    v0, v1 = vocab_shard(rank, world, vocab)
    bufs = bufs if bufs is not None else {}
    cap = max(1, sel.capacity)
    if "pairs" not in bufs or bufs["pairs"].numel() != cap or bufs["gathered"].numel() != world * cap:
        bufs["pairs"] = torch.zeros(cap, dtype=torch.int64, device=logits_shard.device)
        bufs["gathered"] = torch.zeros(world * cap, dtype=torch.int64, device=logits_shard.device)
        bufs["token"] = torch.zeros(cap, dtype=torch.int32, device=logits_shard.device)
    if v1 > v0:
        ctx.argmax_shard(sel, logits_shard, v0, v1 - v0, out=bufs["pairs"])
    else:
        bufs["pairs"].zero_()  # a rank without columns: the smallest key, never the maximum
    if world > 1:
        dist.all_gather_into_tensor(bufs["gathered"], bufs["pairs"])
    else:
        bufs["gathered"].copy_(bufs["pairs"])
    return ctx.argmax_merge(sel, bufs["gathered"], world, out=bufs["token"])


def rank_bases(sizes, rank: int):
    """Exclusive prefix sum of per-rank sizes (candidates or requests): the base this rank's keys carry."""
    return int(sum(int(x) for x in sizes[:rank]))


def exchange_sizes(N: int, R: int, world: int, dist=None):
    """[(N_r, R_r)] of every rank, exchanged once at set-up (host integers: batch shapes are known on the host)."""
    if world == 1:
        return [(int(N), int(R))]
    if dist is None:
        import torch.distributed as dist  # noqa: PLC0415
    out = [None] * world
    dist.all_gather_object(out, (int(N), int(R)))
    return [tuple(x) for x in out]


def global_budget_gate_select(ctx, rank: int, world: int, cand_offsets, parent, logq, gate, sel, max_cand=128,
                              schedule=0, dist=None, all_sizes=None, bufs=None):
    """Request-sharded ranks that share ONE verification budget (the paper's batch-wide K_max, Eq. 4, over the whole
    data-parallel group): the only exchange of the path.  Every rank computes its keys, the ranks
    all-gather them (N x 8 B, padded with "not eligible" to the largest N), and each selects against all keys and
    packs its own requests.  `gate.budget` is the global budget.  `all_sizes` = exchange_sizes(...) (taken here if not
    given); `bufs` = a dict the call keeps its padded / gathered key buffers in between steps.  No host
    synchronisation: sizes are host integers, everything else stays on the stream."""
    import torch
    if dist is None and world > 1:
        import torch.distributed as dist  # noqa: PLC0415
    R, N = cand_offsets.numel() - 1, parent.numel()
    if all_sizes is None:
        all_sizes = exchange_sizes(N, R, world, dist)
    Ns = [n for n, _ in all_sizes]
    Rs = [r for _, r in all_sizes]
    keys = ctx.gate_keys(cand_offsets, parent, logq, gate.depth_mask, gate.log_tau, gate.w_max, gate.budget, sel,
                         static_k=gate.static_k, schedule=schedule, cand_index_base=rank_bases(Ns, rank),
                         request_base=rank_bases(Rs, rank), max_cand=max_cand)
    n_max = max(1, max(Ns))
    bufs = bufs if bufs is not None else {}
    if "padded" not in bufs or bufs["padded"].numel() != n_max or bufs["gathered"].numel() != world * n_max:
        bufs["padded"] = torch.full((n_max,), -1, dtype=torch.int64, device=keys.device)
        bufs["gathered"] = torch.empty(world * n_max, dtype=torch.int64, device=keys.device)
    padded, gathered = bufs["padded"], bufs["gathered"]
    padded[:N].copy_(keys)
    if world > 1:
        dist.all_gather_into_tensor(gathered, padded)
    else:
        gathered.copy_(padded)
    return ctx.gate_select_keys(cand_offsets, parent, logq, gate.depth_mask, gate.log_tau, gate.w_max, gate.budget,
                                keys, gathered, sel, static_k=gate.static_k, schedule=schedule, max_cand=max_cand)
