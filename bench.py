"""bench.py -- one "step" = one pass of the whole super-tree verify step (echo_gate_select ->
echo_verify_attn (one layer) -> echo_accept) over one synthetic batch.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

Prints ONE JSON line (rank 0).  metric = verified draft tokens/s (BASELINE.json); `roofline` is
the verify-attention kernel against the measured HBM peak; `cpu_baseline` is the CPU oracle timed
on a bounded sample; `e2e` repeats the step with host buffers (pinned H2D of the step inputs,
D2H of the results inside the timed region; the paged KV cache is resident serving state).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
SM_SCALE = 1.0 / np.sqrt(128.0)
WORKLOADS = {1: "cfg1 LLaMA-3.1-8B shape BS=32 B=1024", 2: "cfg2 LLaMA-3.3-70B shape BS=128 B=2048",
             3: "cfg3 Qwen3-235B shape BS=128 B=1024", 4: "cfg4 stress BS=256 B=4096 logits argmax",
             0: "cfg0 tiny"}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def tensor_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        if "bf16_tflops" in d:
            return float(d["bf16_tflops"]), "measured (MEASURED_PEAKS.json bf16_tflops, burst)"
    return 2250.0, "fallback (B200_PROFILING.md nominal dense bf16)"


class ClockSampler(threading.Thread):
    """samples SM clock, power and throttle reasons during the timed region: NVML every 2 ms when pynvml is there
    (the default run lasts ~15 ms), else nvidia-smi every 100 ms"""

    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, idx=0):
        super().__init__(daemon=True)
        self.idx, self.stop_flag, self.rows, self.power = idx, False, [], []

    def _run_nvml(self):
        import pynvml
        pynvml.nvmlInit()
        h = pynvml.nvmlDeviceGetHandleByIndex(self.idx)
        mx = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
        bits = [pynvml.nvmlClocksThrottleReasonHwSlowdown, pynvml.nvmlClocksThrottleReasonHwThermalSlowdown,
                pynvml.nvmlClocksThrottleReasonSwThermalSlowdown, pynvml.nvmlClocksThrottleReasonSwPowerCap]
        while not self.stop_flag:
            r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
            self.rows.append([str(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)), str(mx)] +
                             ["Active" if r & b else "Not Active" for b in bits])
            self.power.append(pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0)
            time.sleep(0.002)

    def run(self):
        try:
            self._run_nvml()
            return
        except Exception:
            pass
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self.stop_flag:
            try:
                o = subprocess.run(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                                   capture_output=True, text=True, timeout=5).stdout.strip()
                if o:
                    self.rows.append([x.strip() for x in o.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(int(r[0]) for r in self.rows if r[0].isdigit())
        reasons = [n for i, n in enumerate(self.NAMES) if any(len(r) > 2 + i and r[2 + i] == "Active" for r in self.rows)]
        out = {"sm_mhz": sm[len(sm) // 2] if sm else None,
               "sm_max_mhz": int(self.rows[0][1]) if self.rows[0][1].isdigit() else None, "reasons": reasons,
               "samples": len(self.rows)}
        if self.power:
            out["power_w_max"] = max(self.power)
        return out


def algorithmic_bytes(wl, sel_h):
    """K and V of every visible page once per KV head + Q read + O write + LSE."""
    K = np.diff(sel_h["sel_offsets"]).astype(np.int64)
    P = wl.prefix_len.astype(np.int64)
    act = K > 0
    kvb = (2 * wl.Hkv * 128 * 2 * (P + K))[act].sum()
    qo = (2 * K * wl.Hq * 128 * 2 + 4 * K * wl.Hq).sum()
    depth = sel_h["sel_depth"].astype(np.int64)
    flops = (4 * 128 * wl.Hq * (P[sel_h["sel_req"]] + depth + 1)).sum()
    return int(kvb + qo), int(flops)


def oracle_sample(wl, n_attn_nodes=6, qkv=None):
    """The CPU oracle as it stands on a bounded sample: gating + acceptance on the whole batch,
    attention (all Hq heads) for `n_attn_nodes` packed nodes.  Returns (tokens/s, description, cores)."""
    from oracle import echo_oracle as orc           # cpu_baseline / reference arm only
    g = wl.gate
    t0 = time.perf_counter()
    sel = orc.gate_select(wl.cand_offsets, wl.parent, wl.logq, g.depth_mask, g.log_tau, g.w_max, g.budget, g.static_k)
    t_gate = time.perf_counter() - t0
    n = sel["n_selected"]
    glob = wl.cand_offsets[sel["sel_req"]] + sel["sel_node"]
    t0 = time.perf_counter()
    orc.accept(sel, wl.draft_token[glob], wl.prev_token, wl.target_after[glob], wl.R)
    t_acc = time.perf_counter() - t0
    rng = np.random.default_rng(1)
    nodes = sorted(set(int(x) for x in rng.integers(0, max(1, n), size=n_attn_nodes)))
    if qkv is None:
        # same distribution as the GPU arm (bf16 N(0,1)), drawn on the host for the sampled requests only
        # timing depends on shapes only: finite bf16 bit patterns (|x| in [2^-7, 2)) with random signs
        def bits(shape):
            return (rng.integers(0x3C00, 0x4000, size=shape, dtype=np.uint16) |
                    (rng.integers(0, 2, size=shape, dtype=np.uint16) << 15))
        qb = bits((max(1, n), wl.Hq, 128))
        pool = bits((1, wl.num_pages, wl.Hkv, 16, 128))
        kb = vb = pool
    else:
        qb, kb, vb = qkv
    rows = [(k, h) for k in nodes for h in range(wl.Hq)]
    t0 = time.perf_counter()
    orc.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=rows)
    t_attn = time.perf_counter() - t0
    t_total = t_attn + (t_gate + t_acc) * len(nodes) / max(1, n)
    desc = (f"{wl.name}: attention of {len(nodes)} packed nodes x {wl.Hq} heads ({t_attn:.2f}s) + the nodes' share of "
            f"gating ({t_gate:.2f}s) and acceptance ({t_acc:.2f}s) over all {n} nodes")
    return len(nodes) / t_total, desc, 1


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle (kind 'oracle') on the same config / metric, rank 0 only."""
    if rank != 0:
        return
    from paper_2604_09603_b200 import workloads as W
    wl = W.make_config(args.config)
    vals = []
    for _ in range(args.warmup):
        oracle_sample(wl, n_attn_nodes=1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        v, desc, cores = oracle_sample(wl, n_attn_nodes=args.ref_nodes)
        vals.append(v)
    dt = time.perf_counter() - t0
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": "verified draft tokens/s", "value": value, "unit": "tokens/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config]},
            "cpu_baseline": {"value": value, "unit": "tokens/s", "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_gpu(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2604_09603_b200 import build, echo, sharding, workloads as W

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    build.build_library()
    heads = args.shard == "heads" and world > 1
    # requests: every rank its own batch (weak scaling); heads: every rank the KV heads [r Hkv/W, (r+1) Hkv/W) of
    # the same batch (strong scaling, no collective either: attention is independent per KV head)
    wl = sharding.rank_workload(args.config, 0 if heads else rank, static=args.static, gated=not args.static)
    if args.gating != "sparse" and not args.static:
        wl.gate = wl.gate.ablation(args.gating)
    g = wl.gate
    schedule = {"topb": echo.SCHED_TOPB, "alg1": echo.SCHED_ALG1}[args.schedule]
    cap = wl.capacity()
    ctx = echo.EchoContext(local_rank, 0)
    ctx.ensure_workspace(wl.R, wl.N, cap, wl.Hq, wl.Hkv)
    if args.attn_path:
        ctx.set_option(echo.OPT_ATTN_PATH, args.attn_path)
    if args.splits:
        ctx.set_option(echo.OPT_FORCE_SPLITS, args.splits)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()

    h_in = {"cand_offsets": pin(wl.cand_offsets), "parent": pin(wl.parent), "logq": pin(wl.logq),
            "prev": pin(wl.prev_token)}
    d_in = {k: v.to(dev) for k, v in h_in.items()}
    q, k, v = W.draw_qkv(wl, cap, device=str(dev))
    if heads:
        q, k, v = sharding.shard_attention_inputs(q, k, v, rank, world)
    kv = echo.PagedKV(k, v, d(wl.page_table), d(wl.prefix_len))
    sel = ctx.alloc_selection(wl.R, wl.N, cap)
    acc = ctx.alloc_accept(wl.R, cap)
    out = torch.zeros_like(q)
    lse = torch.zeros(cap, q.shape[1], dtype=torch.float32, device=dev)

    g_global, gb_bufs = g.replace(budget=g.budget * world), {}
    all_sizes = sharding.exchange_sizes(wl.N, wl.R, world, dist) if args.global_budget else None

    def gate(din, sel_=None):
        if args.global_budget and not heads:  # one budget of world x B over the ranks' requests: the one exchange of the path
            return sharding.global_budget_gate_select(ctx, rank, world, din["cand_offsets"], din["parent"], din["logq"],
                                                      g_global, sel_ or sel, max_cand=wl.max_cand, schedule=schedule,
                                                      dist=dist, all_sizes=all_sizes, bufs=gb_bufs)
        return ctx.gate_select(din["cand_offsets"], din["parent"], din["logq"], g.depth_mask, g.log_tau, g.w_max,
                               g.budget, g.static_k, capacity=cap, max_cand=wl.max_cand, out=sel_ or sel,
                               schedule=schedule)

    gate(d_in)
    sel_h = sel.to_host()
    n_sel = sel_h["n_selected"]
    glob = (wl.cand_offsets[sel_h["sel_req"]] + sel_h["sel_node"]).astype(np.int64)
    pad = lambda a: np.concatenate([a, np.zeros(cap - len(a), a.dtype)]).astype(np.int32)
    h_in["draft"] = pin(pad(wl.draft_token[glob]))
    h_in["target"] = pin(pad(wl.target_after[glob]))
    d_in["draft"], d_in["target"] = h_in["draft"].to(dev), h_in["target"].to(dev)
    logits = None
    if args.config == 4:
        logits = W.draw_logits(wl, glob, device=str(dev))
        if logits.shape[0] < cap:
            logits = torch.cat([logits, torch.zeros(cap - logits.shape[0], logits.shape[1], dtype=logits.dtype, device=dev)])
    root_logits = u_acc = u_bon = None
    if logits is not None and args.temperature > 0:  # acceptance at temperature > 0 (NEXT-2) instead of the argmax
        gen = torch.Generator(device=dev).manual_seed(W.SEED_BASE + 7)
        root_logits = torch.randn(wl.R, logits.shape[1], generator=gen, device=dev, dtype=torch.float32).to(torch.bfloat16)
        root_logits[torch.arange(wl.R, device=dev), d(wl.prev_token).long()] += 8.0
        u_acc = torch.rand(cap, generator=gen, device=dev)
        u_bon = torch.rand(wl.R, generator=gen, device=dev)
    bytes_alg, flops_alg = algorithmic_bytes(wl, sel_h)
    if heads:
        bytes_alg, flops_alg = bytes_alg // world, flops_alg // world

    ev = lambda: torch.cuda.Event(enable_timing=True)
    attn_ev = [(ev(), ev()) for _ in range(args.steps)]
    gate_ev = [(ev(), ev()) for _ in range(args.steps)]
    acc_ev = [ev() for _ in range(args.steps)]

    def step(din, i=None, qq=q, bufs=None):
        sel_, acc_, out_, lse_ = bufs or (sel, acc, out, lse)
        if i is not None:
            gate_ev[i][0].record()
        gate(din, sel_)
        if i is not None:
            gate_ev[i][1].record(); attn_ev[i][0].record()
        ctx.verify_attn(sel_, kv, qq, SM_SCALE, out=out_, lse=lse_)
        if i is not None:
            attn_ev[i][1].record()
        if logits is not None and args.temperature > 0:
            ctx.accept_stochastic(sel_, kv, din["draft"], logits, root_logits, wl.vocab, args.temperature, u_acc, u_bon,
                                  out=acc_)
        elif logits is not None:
            ctx.accept(sel_, kv, din["draft"], din["prev"], target_logits=logits, vocab=wl.vocab, out=acc_)
        else:
            ctx.accept(sel_, kv, din["draft"], din["prev"], target_token=din["target"], out=acc_)
        if i is not None:
            acc_ev[i].record()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(d_in)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    barrier()
    e0, e1 = ev(), ev()
    e0.record()
    for i in range(args.steps):
        step(d_in, i)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    sampler.stop_flag = True
    t_attn = float(np.mean([a.elapsed_time(b) for a, b in attn_ev]))
    t_gate = float(np.mean([a.elapsed_time(b) for a, b in gate_ev]))
    t_acc = float(np.mean([attn_ev[i][1].elapsed_time(acc_ev[i]) for i in range(args.steps)]))
    t_attn_min = float(np.min([a.elapsed_time(b) for a, b in attn_ev]))
    accepted = int(acc.accept_len[:wl.R].sum().item())
    # the step before the path: warm-up calibration of the gates, timed outside the step
    calib_us = None
    if rank == 0 and args.calibrate_samples > 0:
        tr = W.draw_calibration_traces(np.random.default_rng(W.SEED_BASE), args.calibrate_samples)
        d_tr = [d(a) for a in tr]
        for _ in range(3):
            ctx.calibrate(*d_tr, 0.65)
        c0, c1 = ev(), ev()
        torch.cuda.synchronize()
        c0.record()
        for _ in range(10):
            ctx.calibrate(*d_tr, 0.65)
        c1.record()
        torch.cuda.synchronize()
        calib_us = c0.elapsed_time(c1) * 100.0
    # the step on the other side of the path (NEXT-4): the candidate trees built on the device, level by level
    draft_us = None
    if rank == 0 and args.calibrate_samples > 0:
        rng = np.random.default_rng(W.SEED_BASE + 1)
        Ld, kd = 8, 10
        lv = [W.draw_draft_level(rng, wl.R, 1 if l_ == 0 else kd, kd) for l_ in range(Ld)]
        d_lv = [(d(a), d(b)) for a, b in lv]
        t_off = d((np.arange(wl.R + 1) * Ld * kd).astype(np.int32))
        t_par = torch.zeros(wl.R * Ld * kd, dtype=torch.int32, device=dev)
        t_lq = torch.zeros(wl.R * Ld * kd, dtype=torch.float32, device=dev)
        t_tok = torch.zeros_like(t_par)
        sc = [torch.zeros(wl.R, kd, dtype=torch.float32, device=dev) for _ in range(Ld + 1)]
        ps0 = torch.zeros(wl.R, 1, dtype=torch.float32, device=dev)

        def build_tree():
            for l_ in range(Ld):
                ctx.draft_expand(l_, kd, ps0 if l_ == 0 else sc[l_], d_lv[l_][0], d_lv[l_][1], t_off, t_par, t_lq, t_tok,
                                 sc[l_ + 1], max_cand=Ld * kd)
        for _ in range(3):
            build_tree()
        c0, c1 = ev(), ev()
        torch.cuda.synchronize()
        c0.record()
        for _ in range(10):
            build_tree()
        c1.record()
        torch.cuda.synchronize()
        draft_us = c0.elapsed_time(c1) * 100.0
    return dict(calib_us=calib_us, draft_us=draft_us, heads=heads, t_acc=t_acc, t_attn_min=t_attn_min, torch=torch, dist=dist, wl=wl, ctx=ctx, dev=dev, ms=ms, t_attn=t_attn, t_gate=t_gate, n_sel=n_sel,
                accepted=accepted, bytes_alg=bytes_alg, flops_alg=flops_alg, step=step, h_in=h_in, d_in=d_in, q=q,
                out=out, lse=lse, acc=acc, sel=sel, sampler=sampler, barrier=barrier, cap=cap, logits=logits)


def run_e2e(r, args):
    """Same step through the public API with HOST buffers: pinned H2D of the step's inputs (trees, logq, Q,
    tokens) and D2H of its results (out, lse, acceptance) inside the timed region, every step; the paged KV cache
    is resident serving state and is not re-uploaded.  Three streams and two sets of device
    buffers: the upload of step i+1 and the download of step i-1 overlap the kernels of step i (PCIe is full
    duplex); each step still moves all of its own bytes."""
    torch, dev, ctx, wl = r["torch"], r["dev"], r["ctx"], r["wl"]
    h_in = r["h_in"]
    h_q = r["q"].cpu().pin_memory()
    sets = []
    for n in range(2):
        d_in = {k_: t.to(dev) for k_, t in h_in.items()}
        q = torch.empty_like(r["q"])
        sel = ctx.alloc_selection(wl.R, wl.N, r["cap"])
        acc = ctx.alloc_accept(wl.R, r["cap"])
        out, lse = torch.zeros_like(r["out"]), torch.zeros_like(r["lse"])
        outs = [out, lse, acc.accept_len, acc.accept_idx, acc.bonus_token, acc.new_len, sel.n_selected]
        h_outs = [torch.empty_like(t, device="cpu").pin_memory() for t in outs]
        ev = [torch.cuda.Event() for _ in range(3)]  # upload done, kernels done, download done
        sets.append(dict(d_in=d_in, q=q, bufs=(sel, acc, out, lse), outs=outs, h_outs=h_outs, ev=ev))
    h2d = sum(t.numel() * t.element_size() for t in h_in.values()) + h_q.numel() * h_q.element_size()
    d2h = sum(t.numel() * t.element_size() for t in sets[0]["outs"])
    s_up, s_run, s_down = torch.cuda.Stream(dev), torch.cuda.Stream(dev), torch.cuda.Stream(dev)

    def one(i):
        st = sets[i % 2]
        up, run, down = st["ev"]
        with torch.cuda.stream(s_up):
            s_up.wait_event(run)          # the kernels of step i-2 have read this set's inputs
            for k_, t in h_in.items():
                st["d_in"][k_].copy_(t, non_blocking=True)
            st["q"].copy_(h_q, non_blocking=True)
            up.record(s_up)
        with torch.cuda.stream(s_run):
            s_run.wait_event(up)
            s_run.wait_event(down)        # the results of step i-2 have left this set's output buffers
            r["step"](st["d_in"], None, st["q"], st["bufs"])
            run.record(s_run)
        with torch.cuda.stream(s_down):
            s_down.wait_event(run)
            for ht, t in zip(st["h_outs"], st["outs"]):
                ht.copy_(t, non_blocking=True)
            down.record(s_down)

    for i in range(max(2, args.warmup // 2)):
        one(i)
    r["barrier"]()
    t0 = time.perf_counter()
    for i in range(args.steps):
        one(i)
    r["barrier"]()
    dt = time.perf_counter() - t0
    n_dev = int(sets[(args.steps - 1) % 2]["h_outs"][6].item())
    assert n_dev == r["n_sel"], (n_dev, r["n_sel"])  # the downloaded result is the step's
    return dt, int(h2d), int(d2h)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (default 2: BS=128)")
    ap.add_argument("--impl", default="echo", choices=["echo", "reference"])
    ap.add_argument("--attn-path", type=int, default=0)
    ap.add_argument("--splits", type=int, default=0)
    ap.add_argument("--ref-nodes", type=int, default=32, help="--impl reference: packed nodes of oracle attention per step (~0.75 s)")
    ap.add_argument("--baseline-nodes", type=int, default=512, help="cpu_baseline leg: packed nodes of oracle attention (~12 s once)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--schedule", default="topb", choices=["topb", "alg1"],
                    help="topb: global top-B (north_star); alg1: Algorithm 1 as printed (SURVEY 8(f) NEXT-1)")
    ap.add_argument("--gating", default="sparse", choices=["sparse", "dense", "fixed"],
                    help="the paper's ablation variants (PAPER.md:254-258): gate every depth / one threshold")
    ap.add_argument("--calibrate-samples", type=int, default=160000,
                    help="warm-up traces for echo_calibrate, timed outside the step (0 = skip)")
    ap.add_argument("--shard", default="requests", choices=["requests", "heads"],
                    help="N > 1: requests = each rank its own batch (weak); heads = KV-head shards of one batch (strong)")
    ap.add_argument("--global-budget", action="store_true",
                    help="request-sharded ranks share ONE budget of N x B: keys are all-gathered before the select")
    ap.add_argument("--temperature", type=float, default=0.0,
                    help="config 4: > 0 accepts by speculative sampling at this temperature instead of greedy argmax")
    ap.add_argument("--static", action="store_true", help="cfg2's static-tree comparison run: 60 fixed nodes per request, gates off")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    local_rank = int(os.environ.get("LOCAL_RANK", 0))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    r = run_gpu(args, rank, world, local_rank)
    torch, dist = r["torch"], r["dist"]
    e2e_dt, h2d, d2h = run_e2e(r, args)
    from paper_2604_09603_b200 import sharding
    (ms, e2e_dt), (n_sel_all, acc_all) = sharding.reduce_step_stats(
        [r["ms"], e2e_dt], [r["n_sel"] / (world if r["heads"] else 1), r["accepted"] / (world if r["heads"] else 1)],
        world, r["dev"], dist)
    if rank == 0:
        peak, peak_src = peaks()
        achieved = r["bytes_alg"] / (r["t_attn"] * 1e-3) / 1e9
        tpeak, tpeak_src = tensor_peak()
        # the static-60 run has ~400 FLOP per byte, above the ridge of the measured peaks: its roof is the tensor pipe
        tensor_bound = r["flops_alg"] / r["bytes_alg"] > tpeak * 1e12 / (peak * 1e9)
        tflops = r["flops_alg"] / (r["t_attn"] * 1e-3) / 1e12
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.csv")  # measured DRAM bytes per launch from the ncu --set full capture
        if os.path.exists(tp):
            for ln in open(tp).read().splitlines()[1:]:
                f = ln.split(",")
                if f and f[0] == f"cfg{args.config}":
                    traffic = int(f[1])
        wl = r["wl"]
        units = wl.R * wl.Hkv
        splits = args.splits or 1
        if not args.splits:  # the library's split policy (csrc/verify_attn.cu), to count launches
            sms = torch.cuda.get_device_properties(0).multi_processor_count
            while splits < 8 and units * splits < sms:
                splits *= 2
        launches = 3 + 2 + (1 if splits > 1 else 0) + 1 + (1 if args.config == 4 else 0)  # gate 3, plan + attn, merge, accept, argmax
        line = {"metric": "verified draft tokens/s", "value": sharding.job_throughput(n_sel_all, args.steps, ms), "unit": "tokens/s",
                "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "strong" if r["heads"] else "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": {"workload": WORKLOADS[args.config] + (" static-60 trees" if args.static else "")
                           + (" global-budget" if args.global_budget else "")
                           + (f" temperature={args.temperature}" if args.temperature > 0 and args.config == 4 else "") + ("" if args.schedule == "topb" else " schedule=alg1") + ("" if args.gating == "sparse" else f" gating={args.gating}"),
                           "requests": wl.R, "verified_nodes_per_step": r["n_sel"],
                           "accepted_per_step": r["accepted"], "l2": "inputs larger than L2 (KV pool >> 126 MB)"
                           if r["bytes_alg"] > 4e8 else "working set near L2 size: KV not flushed",
                           "attn_ms": r["t_attn"], "attn_ms_min": r["t_attn_min"], "gate_ms": r["t_gate"], "accept_ms": r["t_acc"],
                           "yield": r["accepted"] / max(1, r["n_sel"]), "attn_flops": r["flops_alg"],
                           "attn_tflops": r["flops_alg"] / (r["t_attn"] * 1e-3) / 1e12,
                           "calibrate_us": r["calib_us"], "calibrate_samples": args.calibrate_samples,
                           "draft_tree_8x10_us": r["draft_us"]},
                "accepted_tokens_per_s": acc_all * args.steps / (ms * 1e-3),
                "roofline": {"bound": "tensor" if tensor_bound else "hbm", "achieved": tflops if tensor_bound else achieved,
                             "peak": tpeak if tensor_bound else peak, "unit": "TFLOP/s" if tensor_bound else "GB/s",
                             "frac": tflops / tpeak if tensor_bound else achieved / peak,
                             "traffic": None if args.static else traffic, "peak_source": tpeak_src if tensor_bound else peak_src, "kernel": "echo_verify_attn (plan + k_verify_attn_tc"
                             + (" + k_lse_merge)" if splits > 1 else ")"), "bytes_per_launch": r["bytes_alg"], "flops_per_launch": r["flops_alg"]},
                "e2e": {"value": n_sel_all * args.steps / e2e_dt, "unit": "tokens/s", "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": d2h},
                "gpu_launches": launches * args.steps, "clocks": r["sampler"].summary()}
        if not args.no_cpu_baseline:
            try:
                v, desc, cores = oracle_sample(wl, n_attn_nodes=args.baseline_nodes)
                line["cpu_baseline"] = {"value": v, "unit": "tokens/s", "cores": cores, "kind": "oracle", "sample": desc}
            except Exception as e:  # the baseline leg must never take the GPU number down with it
                line["cpu_baseline"] = {"value": None, "unit": "tokens/s", "cores": 1, "kind": "oracle", "sample": f"failed: {e}"}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
