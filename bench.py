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
NOMINAL_GBS, NOMINAL_TFLOPS = 8000.0, 2250.0  # BASELINE.json north_star: "about 8 TB/s"; dense bf16 nominal
WORKLOADS = {1: "cfg1 LLaMA-3.1-8B shape BS=32 B=1024", 2: "cfg2 LLaMA-3.3-70B shape BS=128 B=2048",
             3: "cfg3 Qwen3-235B shape BS=128 B=1024", 4: "cfg4 stress BS=256 B=4096 logits argmax",
             0: "cfg0 tiny"}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def tensor_peak(sustained=False):
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        if sustained and "bf16_tflops_sustained" in d:
            return float(d["bf16_tflops_sustained"]), "measured (MEASURED_PEAKS.json bf16_tflops_sustained)"
        if "bf16_tflops" in d:
            return float(d["bf16_tflops"]), "measured (MEASURED_PEAKS.json bf16_tflops, burst)"
    return (1400.0, "fallback (B200_PROFILING.md, sustained)") if sustained else (1590.0, "fallback (B200_PROFILING.md, burst)")


class ClockSampler:
    """nvidia-smi in loop mode (-lms 20) for the whole measurement: SM clock, power and throttle reasons every 20 ms.
    The SM clock UNDER the kernels comes from the library's probe kernel (echo_probe_sm_clock): the verify step is
    shorter than any NVML sampling period and NVML reads the idle clock between kernels."""

    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, idx=0):
        self.idx, self.proc, self.marks = idx, None, {}

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t0 = time.time()
        except Exception:
            self.proc = None

    def mark(self, name):
        self.marks[name] = time.time()

    def stop(self):
        rows = []
        if self.proc is not None:
            time.sleep(0.05)
            self.proc.terminate()
            try:
                out, _ = self.proc.communicate(timeout=5)
            except Exception:
                self.proc.kill()
                out = ""
            rows = [[x.strip() for x in ln.split(",")] for ln in out.splitlines() if ln.count(",") >= 6]
        self.rows, self.t1 = rows, time.time()
        return rows

    def window(self, a, b):
        """rows sampled between the marks a and b (samples are evenly spaced over the run: -lms has no timestamps)"""
        if not self.rows or a not in self.marks or b not in self.marks:
            return []
        n, span = len(self.rows), max(1e-6, self.t1 - self.t0)
        i0 = int(n * (self.marks[a] - self.t0) / span)
        i1 = int(np.ceil(n * (self.marks[b] - self.t0) / span))
        return self.rows[max(0, i0):max(i0 + 1, min(n, i1))]

    def summary(self, rows, probe_mhz):
        """`clocks` object: sm_mhz = the probe kernel's median (the clock the kernels ran at), NVML's view beside it"""
        out = {"sm_mhz": float(np.median(probe_mhz)) if len(probe_mhz) else None, "sm_mhz_source":
               "echo_probe_sm_clock (clock64 / globaltimer in a kernel queued inside the measured region)",
               "sm_max_mhz": None, "reasons": [], "nvml_samples": len(rows)}
        allrows = rows or getattr(self, "rows", [])
        if allrows:
            mx = [int(float(r[1])) for r in allrows if r[1].replace(".", "").isdigit()]
            out["sm_max_mhz"] = mx[0] if mx else None
        if rows:
            sm = sorted(int(float(r[0])) for r in rows if r[0].replace(".", "").isdigit())
            out["nvml_sm_mhz"] = sm[len(sm) // 2] if sm else None
            pw = [float(r[2]) for r in rows if r[2].replace(".", "").isdigit()]
            out["power_w_max"] = max(pw) if pw else None
            out["reasons"] = [n for i, n in enumerate(self.NAMES) if any(r[3 + i] == "Active" for r in rows)]
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


def host_qkv_bits(wl, n):
    """bf16 bit patterns for the oracle legs: the CPU time depends on shapes only, so finite random patterns (|x| in
    [2^-7, 2), random signs) stand in for the device's N(0,1) draw; K and V share one pool"""
    rng = np.random.default_rng(1)

    def bits(shape):
        return (rng.integers(0x3C00, 0x4000, size=shape, dtype=np.uint16) |
                (rng.integers(0, 2, size=shape, dtype=np.uint16) << 15))
    pool = bits((1, wl.num_pages, wl.Hkv, 16, 128))
    return bits((max(1, n), wl.Hq, 128)), pool, pool


def oracle_sample(wl, n_attn_nodes=6, qkv=None, sel=None):
    """The CPU oracle as it stands on a bounded sample: gating + acceptance (numpy, one core) on the whole batch,
    attention (all Hq heads; the plain-C restatement of the definition, oracle/echo_oracle_attn.c, on every host core
    this process may use) for `n_attn_nodes` packed nodes, all of them if the batch has no more.
    Returns (tokens/s, description, threads used by the attention, which is > 98 % of the work)."""
    from oracle import attn_c, echo_oracle as orc    # cpu_baseline / reference arm only
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
    if n_attn_nodes >= n:
        nodes = list(range(n))
    else:
        nodes = sorted(set(int(x) for x in rng.choice(max(1, n), size=n_attn_nodes, replace=False)))
    qb, kb, vb = qkv if qkv is not None else host_qkv_bits(wl, n)
    rows = [(k, h) for k in nodes for h in range(wl.Hq)]
    threads = attn_c.host_threads()
    attn_c.build()
    t0 = time.perf_counter()
    attn_c.verify_attn(sel, qb, kb, vb, wl.page_table, wl.prefix_len, wl.Hq, wl.Hkv, SM_SCALE, rows=rows, threads=threads)
    t_attn = time.perf_counter() - t0
    t_total = t_attn + (t_gate + t_acc) * len(nodes) / max(1, n)
    desc = (f"{wl.name}: attention of {len(nodes)} of {n} packed nodes x {wl.Hq} heads by the plain-C fp64 oracle on "
            f"{threads} threads ({t_attn:.2f}s) + the nodes' share of gating ({t_gate:.2f}s) and acceptance ({t_acc:.2f}s; "
            f"numpy, one core) over all {n} nodes")
    return len(nodes) / t_total, desc, threads


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle (kind 'oracle') on the same config / metric, rank 0 only."""
    if rank != 0:
        return
    from paper_2604_09603_b200 import workloads as W
    wl = W.make_config(args.config)
    qkv = host_qkv_bits(wl, wl.capacity())
    vals = []
    for _ in range(args.warmup):
        oracle_sample(wl, n_attn_nodes=8, qkv=qkv)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        v, desc, cores = oracle_sample(wl, n_attn_nodes=args.ref_nodes, qkv=qkv)
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


class Case:
    """One workload resident on the device and its step (echo_gate_select -> echo_verify_attn -> echo_accept)."""

    def __init__(self, ctx, echo, sharding, W, torch, dev, cfg, rank=0, world=1, static=False, gating="sparse",
                 schedule="topb", heads=False, global_budget=False, temperature=0.0, attn_path=0, splits=0, dist=None,
                 kv_pools=1):
        self.ctx, self.torch, self.dev, self.cfg, self.static = ctx, torch, dev, cfg, static
        self.world, self.rank, self.heads, self.dist = world, rank, heads, dist
        wl = sharding.rank_workload(cfg, 0 if heads else rank, static=static, gated=not static)
        if gating != "sparse" and not static:
            wl.gate = wl.gate.ablation(gating)
        self.wl, g = wl, wl.gate
        self.schedule = {"topb": echo.SCHED_TOPB, "alg1": echo.SCHED_ALG1}[schedule]
        cap = self.cap = wl.capacity()
        ctx.ensure_workspace(wl.R, wl.N, cap, wl.Hq, wl.Hkv)
        ctx.set_option(echo.OPT_ATTN_PATH, attn_path)
        ctx.set_option(echo.OPT_FORCE_SPLITS, splits)
        d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        self.h_in = {"cand_offsets": pin(wl.cand_offsets), "parent": pin(wl.parent), "logq": pin(wl.logq),
                     "prev": pin(wl.prev_token)}
        self.d_in = {k: v.to(dev) for k, v in self.h_in.items()}
        q, k, v = W.draw_qkv(wl, cap, device=str(dev))
        if heads:
            q, k, v = sharding.shard_attention_inputs(q, k, v, rank, world)
        self.q = q
        pt, pl = d(wl.page_table), d(wl.prefix_len)
        # a working set near the L2 size (cfg1: 189 MB) is measured over >= 4 KV pools taken in turn, so that every
        # step streams its KV from HBM; the copies hold the same values
        self.kvs = [echo.PagedKV(k, v, pt, pl)] + [echo.PagedKV(k.clone(), v.clone(), pt, pl) for _ in range(kv_pools - 1)]
        self.sel = ctx.alloc_selection(wl.R, wl.N, cap)
        self.acc = ctx.alloc_accept(wl.R, cap)
        self.out = torch.zeros_like(q)
        self.lse = torch.zeros(cap, q.shape[1], dtype=torch.float32, device=dev)
        self.global_budget = global_budget and not heads
        self.g_global, self.gb_bufs = g.replace(budget=g.budget * world), {}
        self.all_sizes = sharding.exchange_sizes(wl.N, wl.R, world, dist) if self.global_budget else None
        self.sharding, self.echo = sharding, echo
        self.gate(self.d_in)
        sel_h = self.sel_h = self.sel.to_host()
        self.n_sel = sel_h["n_selected"]
        glob = (wl.cand_offsets[sel_h["sel_req"]] + sel_h["sel_node"]).astype(np.int64)
        pad = lambda a: np.concatenate([a, np.zeros(cap - len(a), a.dtype)]).astype(np.int32)
        self.h_in["draft"] = pin(pad(wl.draft_token[glob]))
        self.h_in["target"] = pin(pad(wl.target_after[glob]))
        self.d_in["draft"], self.d_in["target"] = self.h_in["draft"].to(dev), self.h_in["target"].to(dev)
        self.logits = self.root_logits = self.u_acc = self.u_bon = None
        self.temperature = temperature
        self.vocab_sharded, self.am_bufs = False, {}
        if cfg == 4:
            lg = W.draw_logits(wl, glob, device=str(dev))
            if lg.shape[0] < cap:
                lg = torch.cat([lg, torch.zeros(cap - lg.shape[0], lg.shape[1], dtype=lg.dtype, device=dev)])
            if heads and temperature <= 0:
                # head-sharded ranks hold a vocabulary shard of the logits: S8 = per-rank (max, index)
                # keys, one all-gather of capacity x 8 B, merge -- sharding.sharded_argmax
                v0, v1 = sharding.vocab_shard(rank, world, wl.vocab)
                lg = lg[:, v0:v1].contiguous()
                self.vocab_sharded = True
            self.logits = lg
            if temperature > 0:  # acceptance at temperature > 0 (NEXT-2) instead of the argmax
                gen = torch.Generator(device=dev).manual_seed(W.SEED_BASE + 7)
                rl = torch.randn(wl.R, lg.shape[1], generator=gen, device=dev, dtype=torch.float32).to(torch.bfloat16)
                rl[torch.arange(wl.R, device=dev), d(wl.prev_token).long()] += 8.0
                self.root_logits = rl
                self.u_acc = torch.rand(cap, generator=gen, device=dev)
                self.u_bon = torch.rand(wl.R, generator=gen, device=dev)
        self.bytes_alg, self.flops_alg = algorithmic_bytes(wl, sel_h)
        if heads:
            self.bytes_alg, self.flops_alg = self.bytes_alg // world, self.flops_alg // world
        self.steps_done = 0

    def gate(self, din, sel_=None):
        wl, g, ctx = self.wl, self.wl.gate, self.ctx
        if self.global_budget:  # one budget of world x B over the ranks' requests: the one exchange of the path
            return self.sharding.global_budget_gate_select(ctx, self.rank, self.world, din["cand_offsets"], din["parent"],
                                                           din["logq"], self.g_global, sel_ or self.sel,
                                                           max_cand=wl.max_cand, schedule=self.schedule, dist=self.dist,
                                                           all_sizes=self.all_sizes, bufs=self.gb_bufs)
        return ctx.gate_select(din["cand_offsets"], din["parent"], din["logq"], g.depth_mask, g.log_tau, g.w_max, g.budget,
                               g.static_k, capacity=self.cap, max_cand=wl.max_cand, out=sel_ or self.sel,
                               schedule=self.schedule)

    def step(self, din=None, ev=None, qq=None, bufs=None):
        """one pass of the hot path; ev = (gate0, gate1/attn0, attn1, acc1) CUDA events to record, or None"""
        din = din or self.d_in
        sel_, acc_, out_, lse_ = bufs or (self.sel, self.acc, self.out, self.lse)
        kv = self.kvs[self.steps_done % len(self.kvs)]
        self.steps_done += 1
        ctx, wl = self.ctx, self.wl
        if ev:
            ev[0].record()
        self.gate(din, sel_)
        if ev:
            ev[1].record()
        ctx.verify_attn(sel_, kv, self.q if qq is None else qq, SM_SCALE, out=out_, lse=lse_)
        if ev:
            ev[2].record()
        if self.logits is not None and self.temperature > 0:
            ctx.accept_stochastic(sel_, kv, din["draft"], self.logits, self.root_logits, wl.vocab, self.temperature,
                                  self.u_acc, self.u_bon, out=acc_)
        elif self.vocab_sharded:
            tok = self.sharding.sharded_argmax(ctx, sel_, self.logits, self.rank, self.world, wl.vocab, dist=self.dist,
                                               bufs=self.am_bufs)
            ctx.accept(sel_, kv, din["draft"], din["prev"], target_token=tok, out=acc_)
        elif self.logits is not None:
            ctx.accept(sel_, kv, din["draft"], din["prev"], target_logits=self.logits, vocab=wl.vocab, out=acc_)
        else:
            ctx.accept(sel_, kv, din["draft"], din["prev"], target_token=din["target"], out=acc_)
        if ev:
            ev[3].record()

    def roofline(self, attn_ms, sustained=False):
        """attention against the roof that bounds it: measured HBM copy peak, or the measured bf16 matmul peak when the
        workload's FLOP per byte is above the ridge of the two (the static-60 run)"""
        peak, peak_src = peaks()
        tpeak, tpeak_src = tensor_peak(sustained)
        tensor_bound = self.flops_alg / self.bytes_alg > tensor_peak(False)[0] * 1e12 / (peak * 1e9)
        gbs = self.bytes_alg / (attn_ms * 1e-3) / 1e9
        tfl = self.flops_alg / (attn_ms * 1e-3) / 1e12
        return {"bound": "tensor" if tensor_bound else "hbm", "achieved": tfl if tensor_bound else gbs,
                "peak": tpeak if tensor_bound else peak, "unit": "TFLOP/s" if tensor_bound else "GB/s",
                "frac": tfl / tpeak if tensor_bound else gbs / peak, "peak_source": tpeak_src if tensor_bound else peak_src,
                # the same figure against the nominal roofs north_star names (about 8 TB/s; 2.25 PFLOP/s dense bf16)
                "frac_nominal": tfl / NOMINAL_TFLOPS if tensor_bound else gbs / NOMINAL_GBS,
                "peak_nominal": NOMINAL_TFLOPS if tensor_bound else NOMINAL_GBS,
                "attn_ms": attn_ms, "bytes_per_launch": self.bytes_alg, "flops_per_launch": self.flops_alg}


def timed_steps(case, steps, warmup, barrier, probe_every=0):
    """`warmup` untimed steps, then exactly `steps` steps between two events; per-step gate / attention / acceptance
    events; SM clock probes (outside the per-call events) before, every `probe_every` steps, and after.
    Returns dict(ms, attn, gate, acc lists, probe MHz list, launches)."""
    torch, ctx = case.torch, case.ctx
    ev = lambda: torch.cuda.Event(enable_timing=True)
    evs = [(ev(), ev(), ev(), ev()) for _ in range(steps)]
    n_probe = 2 + (steps // probe_every if probe_every else 0)
    probes = torch.zeros(n_probe + 1, dtype=torch.float32, device=case.dev)
    for _ in range(warmup):
        case.step()
    barrier()
    l0 = ctx.launch_count()
    e0, e1 = ev(), ev()
    pi = 0
    ctx.probe_sm_clock(probes[pi:pi + 1]); pi += 1        # clock state going in (20 us, ahead of the timed region)
    e0.record()
    for i in range(steps):
        case.step(ev=evs[i])
        if probe_every and (i + 1) % probe_every == 0 and i + 1 < steps:
            ctx.probe_sm_clock(probes[pi:pi + 1]); pi += 1
    e1.record()
    ctx.probe_sm_clock(probes[pi:pi + 1]); pi += 1        # and coming out, with no idle gap in between
    l1 = ctx.launch_count()
    barrier()
    attn = [a[1].elapsed_time(a[2]) for a in evs]
    gate = [a[0].elapsed_time(a[1]) for a in evs]
    acc = [a[2].elapsed_time(a[3]) for a in evs]
    mhz = probes[:pi].cpu().numpy().tolist()
    # the probes inside a long leg take 20 us each: not part of any per-call time, but inside e0..e1
    ms = e0.elapsed_time(e1) - 0.02 * max(0, pi - 2)
    return dict(ms=ms, attn=attn, gate=gate, acc=acc, mhz=mhz[1:] if len(mhz) > 1 else mhz, launches=l1 - l0 - pi)


def graph_steps(case, steps, barrier):
    """The same step captured ONCE into a CUDA graph (one graph = one pass over the KV pools) and replayed: what a
    serving loop does (the paper serves under CUDA graphs), and the only timing of a small batch that the host's
    launch calls do not bound.  Returns (ms per step, steps replayed)."""
    torch = case.torch
    n = len(case.kvs)
    side = torch.cuda.Stream(device=case.dev)
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        for _ in range(n):
            case.step()
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            for _ in range(n):
                case.step()
    torch.cuda.synchronize()
    reps = max(1, steps // n)
    for _ in range(3):
        g.replay()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        g.replay()
    e1.record()
    barrier()
    return e0.elapsed_time(e1) / (reps * n), reps * n


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
    ctx = echo.EchoContext(local_rank, 0)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    mk = lambda cfg, static=False, **kw: Case(ctx, echo, sharding, W, torch, dev, cfg, rank=rank, world=world, static=static,
                                              dist=dist, **kw)
    case = mk(args.config, args.static, gating=args.gating, schedule=args.schedule, heads=heads,
              global_budget=args.global_budget, temperature=args.temperature, attn_path=args.attn_path,
              splits=args.splits, kv_pools=4 if args.config == 1 else 1)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    sampler.mark("burst0")
    t = timed_steps(case, args.steps, args.warmup, barrier)
    sampler.mark("burst1")
    r = dict(torch=torch, dist=dist, dev=dev, ctx=ctx, case=case, wl=case.wl, heads=heads, barrier=barrier, sampler=sampler,
             ms=t["ms"], t_attn=float(np.mean(t["attn"])), t_attn_min=float(np.min(t["attn"])),
             t_gate=float(np.mean(t["gate"])), t_acc=float(np.mean(t["acc"])), mhz=t["mhz"], launches=t["launches"],
             n_sel=case.n_sel, accepted=int(case.acc.accept_len[:case.wl.R].sum().item()), sustained=None, sub={},
             calib_us=None, draft_us=None, graph=None)
    if world == 1 and not args.global_budget:
        try:
            g_ms, g_n = graph_steps(case, args.steps, barrier)
            r["graph"] = {"ms_per_step": g_ms, "steps": g_n, "value": sharding.job_throughput(case.n_sel, 1, g_ms)}
        except Exception as e:  # an extra leg: never at the headline's cost
            r["graph"] = {"error": repr(e)[:200]}
    # ---- second leg: the same step back to back for >= --sustained-seconds: the regime a serving loop runs in (the
    # part reaches its power cap after ~100 ms and the SM clock drops; MEASURED_PEAKS.json keeps a sustained matmul
    # figure for the same reason)
    if args.sustained_seconds > 0:
        n = int(min(20000, max(200, args.sustained_seconds * 1e3 / max(1e-3, t["ms"] / args.steps))))
        sampler.mark("sus0")
        ts = timed_steps(case, n, 0, barrier, probe_every=max(1, n // 16))
        sampler.mark("sus1")
        tail = ts["attn"][len(ts["attn"]) // 2:]          # second half: the clocks have settled
        roof = case.roofline(float(np.mean(tail)), sustained=True)
        roof.update(steps=n, seconds=ts["ms"] * 1e-3, ms_per_step=ts["ms"] / n, sm_mhz=float(np.median(ts["mhz"][len(ts["mhz"]) // 2:])),
                    attn_ms_first_100=float(np.mean(ts["attn"][:100])),
                    value=sharding.job_throughput(case.n_sel, n, ts["ms"]))
        r["sustained"] = roof
    # ---- the other shapes north_star names, one sub-record each (rank 0's view; not part of `value`)
    if rank == 0 and args.subrecords and world == 1:
        for name, cfg, static in (("cfg1", 1, False), ("cfg3", 3, False), ("cfg2_static60", 2, True), ("cfg4", 4, False)):
            if cfg == args.config and static == args.static:
                continue
            try:
                c = mk(cfg, static, kv_pools=4 if cfg == 1 else 1)
                tt = timed_steps(c, 30 if cfg != 4 else 12, 5, barrier)
                rec = c.roofline(float(np.mean(tt["attn"])))
                rec.update(workload=WORKLOADS[cfg] + (" static-60 trees" if static else ""), steps=len(tt["attn"]),
                           ms_per_step=tt["ms"] / len(tt["attn"]), attn_ms_min=float(np.min(tt["attn"])),
                           gate_ms=float(np.mean(tt["gate"])), accept_ms=float(np.mean(tt["acc"])),
                           verified_nodes_per_step=c.n_sel, value=c.n_sel * len(tt["attn"]) / (tt["ms"] * 1e-3),
                           sm_mhz=float(np.median(tt["mhz"])), kv_pools=len(c.kvs))
                g_ms, g_n = graph_steps(c, len(tt["attn"]), barrier)
                rec.update(graph_ms_per_step=g_ms, graph_value=c.n_sel / (g_ms * 1e-3))
                r["sub"][name] = rec
                del c
                torch.cuda.empty_cache()
            except Exception as e:  # a sub-record must never take the headline number down with it
                r["sub"][name] = {"error": repr(e)[:200]}
        # back to the headline case's options (the sub-cases share the context)
        ctx.set_option(echo.OPT_ATTN_PATH, args.attn_path)
        ctx.set_option(echo.OPT_FORCE_SPLITS, args.splits)
        ctx.ensure_workspace(case.wl.R, case.wl.N, case.cap, case.wl.Hq, case.wl.Hkv)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    wl = case.wl
    # the step before the path: warm-up calibration of the gates, timed outside the step
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
        r["calib_us"] = c0.elapsed_time(c1) * 100.0
        # the step on the other side of the path (NEXT-4): the candidate trees built on the device, level by level
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
        r["draft_us"] = c0.elapsed_time(c1) * 100.0
        ctx.ensure_workspace(case.wl.R, case.wl.N, case.cap, case.wl.Hq, case.wl.Hkv)
    return r


def run_e2e(r, args):
    """Same step through the public API with HOST buffers: pinned H2D of the step's inputs (trees, logq, Q,
    tokens) and D2H of its results (out, lse, acceptance) inside the timed region, every step; the paged KV cache
    is resident serving state and is not re-uploaded.  Three streams and two sets of device
    buffers: the upload of step i+1 and the download of step i-1 overlap the kernels of step i (PCIe is full
    duplex); each step still moves all of its own bytes."""
    torch, dev, ctx, case = r["torch"], r["dev"], r["ctx"], r["case"]
    wl, h_in = case.wl, case.h_in
    h_q = case.q.cpu().pin_memory()
    sets = []
    for n in range(2):
        d_in = {k_: t.to(dev) for k_, t in h_in.items()}
        q = torch.empty_like(case.q)
        sel = ctx.alloc_selection(wl.R, wl.N, case.cap)
        acc = ctx.alloc_accept(wl.R, case.cap)
        out, lse = torch.zeros_like(case.out), torch.zeros_like(case.lse)
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
            case.step(st["d_in"], None, st["q"], st["bufs"])
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
    ap.add_argument("--steps", type=int, default=100,
                    help="timed steps of the headline leg (default: ~30 ms at cfg2, inside the burst-clock window that "
                         "MEASURED_PEAKS.json's copy figure was taken in; the sustained leg follows)")
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (default 2: BS=128)")
    ap.add_argument("--impl", default="echo", choices=["echo", "reference"])
    ap.add_argument("--attn-path", type=int, default=0)
    ap.add_argument("--splits", type=int, default=0)
    ap.add_argument("--ref-nodes", type=int, default=256,
                    help="--impl reference: packed nodes of oracle attention per step (~0.2 s on 8 cores at cfg2)")
    ap.add_argument("--baseline-nodes", type=int, default=2048,
                    help="cpu_baseline leg: packed nodes of oracle attention (cfg2: the whole batch, ~13 s on 8 cores; "
                         "cfg4's long prefixes: a quarter of this)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sustained-seconds", type=float, default=2.0,
                    help="length of the second timed leg (back-to-back steps under the power cap); 0 = skip")
    ap.add_argument("--no-subrecords", dest="subrecords", action="store_false",
                    help="skip the per-shape sub-records (cfg1, cfg3, cfg2 static-60, cfg4)")
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
        case, wl, sampler = r["case"], r["wl"], r["sampler"]
        sampler.stop()
        roof = case.roofline(r["t_attn"])
        traffic, traffic_src = None, None
        tp = os.path.join(ROOT, "profiles", "traffic.csv")  # DRAM bytes per launch from the committed ncu --set full capture
        if os.path.exists(tp) and not args.static:
            for ln in open(tp).read().splitlines()[1:]:
                f = ln.split(",")
                if f and f[0] == f"cfg{args.config}":
                    traffic, traffic_src = int(f[1]), "not measured in this run: " + ",".join(f[3:])
        splits = int(r["ctx"].lib.echo_attn_splits(r["ctx"]._h, wl.R, wl.Hkv)) if not args.splits else args.splits
        roofline = {k_: roof[k_] for k_ in ("bound", "achieved", "peak", "unit", "frac", "frac_nominal", "peak_nominal")}
        roofline.update(traffic=traffic, traffic_source=traffic_src, peak_source=roof["peak_source"],
                        kernel="echo_verify_attn (k_plan + k_verify_attn_tc" + (" + k_lse_merge)" if splits > 1 else ")"),
                        bytes_per_launch=case.bytes_alg, flops_per_launch=case.flops_alg)
        cfg_name = (WORKLOADS[args.config] + (" static-60 trees" if args.static else "")
                    + (" global-budget" if args.global_budget else "")
                    + (f" temperature={args.temperature}" if args.temperature > 0 and args.config == 4 else "")
                    + ("" if args.schedule == "topb" else " schedule=alg1") + ("" if args.gating == "sparse" else f" gating={args.gating}"))
        line = {"metric": "verified draft tokens/s", "value": sharding.job_throughput(n_sel_all, args.steps, ms), "unit": "tokens/s",
                "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "strong" if r["heads"] else "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": {"workload": cfg_name, "requests": wl.R, "verified_nodes_per_step": r["n_sel"],
                           "accepted_per_step": r["accepted"],
                           "l2": "inputs larger than L2 (KV pool >> 126 MB)" if case.bytes_alg * len(case.kvs) > 4e8
                           else "working set near L2 size: KV not flushed",
                           "kv_pools_rotated": len(case.kvs),
                           "attn_ms": r["t_attn"], "attn_ms_min": r["t_attn_min"], "gate_ms": r["t_gate"], "accept_ms": r["t_acc"],
                           "yield": r["accepted"] / max(1, r["n_sel"]), "attn_flops": case.flops_alg,
                           "attn_tflops": case.flops_alg / (r["t_attn"] * 1e-3) / 1e12,
                           "calibrate_us": r["calib_us"], "calibrate_samples": args.calibrate_samples,
                           "draft_tree_8x10_us": r["draft_us"]},
                "accepted_tokens_per_s": acc_all * args.steps / (ms * 1e-3),
                "roofline": roofline,
                "roofline_sustained": r["sustained"],
                "configs": r["sub"],
                "cuda_graph": r["graph"],
                "e2e": {"value": n_sel_all * args.steps / e2e_dt, "unit": "tokens/s", "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": d2h},
                "gpu_launches": r["launches"],
                "clocks": sampler.summary(sampler.window("burst0", "burst1"), r["mhz"])}
        if r["sustained"] is not None:
            line["clocks_sustained"] = sampler.summary(sampler.window("sus0", "sus1"), [r["sustained"]["sm_mhz"]])
        if not args.no_cpu_baseline:
            try:
                v, desc, cores = oracle_sample(wl, n_attn_nodes=args.baseline_nodes // (4 if args.config == 4 else 1))
                line["cpu_baseline"] = {"value": v, "unit": "tokens/s", "cores": cores, "kind": "oracle", "sample": desc}
            except Exception as e:  # the baseline leg must never take the GPU number down with it
                line["cpu_baseline"] = {"value": None, "unit": "tokens/s", "cores": 1, "kind": "oracle", "sample": f"failed: {e}"}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
