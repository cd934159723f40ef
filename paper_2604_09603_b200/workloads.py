"""Seeded synthetic inputs for the ECHO super-tree verify step.

This module is shared by the CUDA path's tests/bench and by the CPU oracle's
tests.  It holds NONE of the method's arithmetic: it only draws candidate
trees, draft confidences, prefix lengths, page tables, tokens and Q/K/V values
with the shapes `BASELINE.json` `configs[0..4]` name (recipe: SURVEY.md §8(d),
restated in DESIGN.md §4).  The paper's serving runs use MT-Bench / HumanEval /
GSM8K / CNN-DM / Alpaca requests; those are not available here
and only shapes / distributions are taken (tree depth 8, top-k 10, 60 total
tokens: PAPER.md:450-451; thresholds: PAPER.md:446; vocab sizes:
PAPER.md:438-442).

Everything that is structural is drawn on the host with
``numpy.random.Generator(PCG64(seed))``; bulk Q/K/V/logit values are drawn with a
``torch.Generator`` on the device they are needed on.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional

import numpy as np

PAGE_SIZE = 16
HEAD_DIM = 128
SEED_BASE = 60480
INT32_MAX = 2**31 - 1

# calibrated gate tables printed by the paper
GATES_LLAMA8B = {0: 0.2, 5: 0.35, 8: 0.5}
GATES_QWEN235B = {0: 0.15, 3: 0.3, 5: 0.5}


@dataclass
class Gate:
    """Gate parameters (Alg. 1 inputs)."""
    depth_mask: int = 0
    log_tau: np.ndarray = field(default_factory=lambda: np.zeros(32, np.float32))
    w_max: int = 0
    budget: int = 0
    static_k: int = 0

    @staticmethod
    def from_taus(taus: Dict[int, float], w_max: int, budget: int, static_k: int = 0) -> "Gate":
        g = Gate(w_max=w_max, budget=budget, static_k=static_k)
        for d, t in taus.items():
            g.depth_mask |= (1 << d)
            # logs are INPUTS, taken once on the host (SURVEY G-2)
            g.log_tau[d] = np.float32(np.log(np.float64(t))) if t > 0 else np.float32(-np.inf)
        return g

    def taus(self) -> Dict[int, float]:
        return {d: float(np.exp(np.float64(self.log_tau[d]))) for d in range(32) if (self.depth_mask >> d) & 1}

    def ablation(self, variant: str, max_depth: int = 8) -> "Gate":
        """The two simplified variants of the paper's ablation, which the paper does not
        parametrise (readings R:L-5, L-6): "dense" gates every depth below `max_depth` with the calibrated
        thresholds interpolated linearly over depth (held constant outside the calibrated range); "fixed" keeps the
        sweet-spot depths and uses one threshold, the median of the calibrated ones."""
        t = self.taus()
        if variant == "sparse" or not t:
            return self.replace()
        ds = sorted(t)
        if variant == "dense":
            new = {d: float(np.interp(d, ds, [t[x] for x in ds])) for d in range(max_depth)}
        elif variant == "fixed":
            new = {d: float(np.median([t[x] for x in ds])) for d in ds}
        else:
            raise ValueError(variant)
        return Gate.from_taus(new, self.w_max, self.budget, self.static_k)

    def replace(self, **kw) -> "Gate":
        g = Gate(self.depth_mask, self.log_tau.copy(), self.w_max, self.budget, self.static_k)
        for k, v in kw.items():
            setattr(g, k, v)
        return g


@dataclass
class Workload:
    name: str
    seed: int
    R: int
    Hq: int
    Hkv: int
    vocab: int
    gate: Gate
    cand_offsets: np.ndarray      # int32 [R+1]
    parent: np.ndarray            # int32 [N] request-local, -1 = root, parent[j] < j
    conf: np.ndarray              # float64 [N] draft confidence q(x|h)
    logq: np.ndarray              # float32 [N] = (float)log(conf)
    prefix_len: np.ndarray        # int32 [R]
    page_table: np.ndarray        # int32 [R][max_pages]
    num_pages: int
    draft_token: np.ndarray       # int32 [N] per candidate
    target_after: np.ndarray      # int32 [N] target's greedy token AFTER candidate j
    prev_token: np.ndarray        # int32 [R] target's greedy token after the committed prefix

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv

    @property
    def N(self) -> int:
        return int(self.cand_offsets[-1])

    @property
    def max_cand(self) -> int:
        return int(np.max(np.diff(self.cand_offsets))) if self.R else 0

    @property
    def max_pages(self) -> int:
        return int(self.page_table.shape[1])

    def capacity(self, gate: Optional[Gate] = None) -> int:
        g = gate or self.gate
        if g.static_k > 0:
            return max(1, self.R * g.static_k)
        return max(1, g.budget)


# --------------------------------------------------------------------------
# trees
# --------------------------------------------------------------------------
def _depths(parent: np.ndarray) -> np.ndarray:
    d = np.zeros(len(parent), np.int32)
    for j, p in enumerate(parent):
        d[j] = 0 if p < 0 else d[p] + 1
    return d


def tree_random_recursive(rng, n: int, max_depth: int) -> np.ndarray:
    """cfg0: single root, parent[j] ~ U{0..j-1}, re-drawn until depth <= max_depth."""
    parent = np.full(n, -1, np.int32)
    depth = np.zeros(n, np.int32)
    for j in range(1, n):
        while True:
            p = int(rng.integers(0, j))
            if depth[p] + 1 <= max_depth:
                break
        parent[j] = p
        depth[j] = depth[p] + 1
    return parent


def tree_levels(rng, levels: int, width: int, max_children: int) -> np.ndarray:
    """cfg1-4: `levels` x `width` nodes, level 0 = `width` roots; each node of
    level l>=1 picks a parent uniformly in level l-1 (<= max_children each)."""
    parent = np.full(levels * width, -1, np.int32)
    for l in range(1, levels):
        cnt = np.zeros(width, np.int32)
        for w in range(width):
            while True:
                p = int(rng.integers(0, width))
                if cnt[p] < max_children:
                    break
            cnt[p] += 1
            parent[l * width + w] = (l - 1) * width + p
    return parent


def tree_chain(n: int) -> np.ndarray:
    return np.arange(-1, n - 1, dtype=np.int32)


def sibling_groups(parent: np.ndarray) -> Dict[int, List[int]]:
    """children lists in node order; key -1 = the virtual parent of the roots."""
    groups: Dict[int, List[int]] = {}
    for j, p in enumerate(parent):
        groups.setdefault(int(p), []).append(j)
    return groups


# --------------------------------------------------------------------------
# confidences
# --------------------------------------------------------------------------
def conf_softmax_siblings(rng, parent: np.ndarray) -> np.ndarray:
    conf = np.zeros(len(parent), np.float64)
    for p, ch in sibling_groups(parent).items():
        z = rng.standard_normal(len(ch))
        e = np.exp(z - z.max())
        conf[ch] = e / e.sum()
    return conf


def conf_dirichlet(rng, parent: np.ndarray, alpha: float, width: int) -> np.ndarray:
    conf = np.zeros(len(parent), np.float64)
    for p, ch in sibling_groups(parent).items():
        k = max(width, len(ch))
        d = np.sort(rng.dirichlet(np.full(k, alpha)))[::-1]
        conf[ch] = d[: len(ch)]
    return conf


def conf_bimodal(rng, parent: np.ndarray, sharp_depths=(0, 5)) -> np.ndarray:
    depth = _depths(parent)
    conf = np.zeros(len(parent), np.float64)
    for j in range(len(parent)):
        if int(depth[j]) in sharp_depths:
            conf[j] = rng.beta(8, 2) if rng.random() < 0.9 else rng.beta(1, 5)
        else:
            conf[j] = rng.beta(2, 2)
    return conf


# --------------------------------------------------------------------------
# tokens / acceptance ground truth (drawn for ALL candidates before selection)
# --------------------------------------------------------------------------
def draw_tokens(rng, parent: np.ndarray, conf: np.ndarray, vocab: int):
    n = len(parent)
    draft = np.zeros(n, np.int32)
    after = rng.integers(0, vocab - 1, size=n).astype(np.int32)   # leaves keep this
    prev = vocab - 1
    for p, ch in sibling_groups(parent).items():
        toks = rng.choice(vocab - 1, size=len(ch), replace=False).astype(np.int32)
        draft[ch] = toks
        u = rng.random()
        cum = np.cumsum(conf[ch])
        m = int(np.searchsorted(cum, u, side="right"))
        tok = int(toks[m]) if m < len(ch) else vocab - 1          # reserved miss token
        if p < 0:
            prev = tok
        else:
            after[p] = tok
    return draft, after, np.int32(prev)


# --------------------------------------------------------------------------
# paged layout
# --------------------------------------------------------------------------
def paged_layout(rng, prefix_len: np.ndarray, cand: np.ndarray, spare: float = 0.10):
    need = (prefix_len.astype(np.int64) + cand + PAGE_SIZE - 1) // PAGE_SIZE
    total = int(need.sum())
    num_pages = total + max(1, int(np.ceil(total * spare)))
    perm = rng.permutation(num_pages).astype(np.int32)
    max_pages = int(need.max()) if len(need) else 1
    table = np.full((len(prefix_len), max(1, max_pages)), -1, np.int32)
    o = 0
    for i, n in enumerate(need):
        table[i, :n] = perm[o:o + n]
        o += int(n)
    return table, num_pages


def _assemble(name, seed, rng, Hq, Hkv, vocab, gate, trees, confs, prefix_len) -> Workload:
    R = len(trees)
    offs = np.zeros(R + 1, np.int32)
    offs[1:] = np.cumsum([len(t) for t in trees])
    parent = np.concatenate(trees).astype(np.int32) if R else np.zeros(0, np.int32)
    conf = np.concatenate(confs) if R else np.zeros(0)
    with np.errstate(divide="ignore"):
        logq = np.log(conf.astype(np.float64)).astype(np.float32)
    logq = np.minimum(logq, np.float32(0.0))
    drafts, afters, prevs = [], [], []
    for t, c in zip(trees, confs):
        d, a, p = draw_tokens(rng, t, c, vocab)
        drafts.append(d); afters.append(a); prevs.append(p)
    prefix_len = np.asarray(prefix_len, np.int32)
    table, num_pages = paged_layout(rng, prefix_len, np.diff(offs))
    return Workload(name, seed, R, Hq, Hkv, vocab, gate, offs, parent, conf, logq, prefix_len,
                    table, num_pages,
                    np.concatenate(drafts).astype(np.int32) if R else np.zeros(0, np.int32),
                    np.concatenate(afters).astype(np.int32) if R else np.zeros(0, np.int32),
                    np.asarray(prevs, np.int32))


def make_config(cfg: int, gated: bool = True, static: bool = False, R: Optional[int] = None,
                seed: Optional[int] = None) -> Workload:
    """BASELINE.json configs[cfg]; `R` overrides the batch size (scaled-down parity cases)."""
    seed = SEED_BASE + cfg if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    if cfg == 0:
        P = [17, 64, 100, 255]
        if R is not None:
            P = [P[i % 4] for i in range(R)]
        trees = [tree_random_recursive(rng, 24, 6) for _ in P]
        confs = []
        for t in trees:
            c = conf_softmax_siblings(rng, t)
            c[0] = 1.0
            confs.append(c)
        gate = Gate.from_taus({1: 0.5, 3: 0.25}, w_max=4, budget=32) if gated else Gate(budget=32)
        return _assemble("cfg0-tiny", seed, rng, 8, 2, 32000, gate, trees, confs, P)
    if cfg == 1:
        R = 32 if R is None else R
        P = rng.integers(512, 2049, size=R)
        trees = [tree_levels(rng, 8, 8, 8) for _ in range(R)]
        confs = [conf_dirichlet(rng, t, 0.3, 8) for t in trees]
        gate = Gate.from_taus(GATES_LLAMA8B if gated else {}, w_max=8, budget=1024 * R // 32)
        return _assemble("cfg1-llama8b", seed, rng, 32, 8, 128256, gate, trees, confs, P)
    if cfg == 2:
        R = 128 if R is None else R
        P = rng.integers(1024, 4097, size=R)
        trees = [tree_levels(rng, 8, 10, 10) for _ in range(R)]
        confs = [conf_dirichlet(rng, t, 0.3, 10) for t in trees]
        if static:
            gate = Gate(budget=60 * R, static_k=60)       # EAGLE-3 "Total Tokens = 60"
        else:
            gate = Gate.from_taus(GATES_LLAMA8B if gated else {}, w_max=10, budget=2048 * R // 128)
        return _assemble("cfg2-llama70b" + ("-static60" if static else ""), seed, rng, 64, 8, 128256,
                         gate, trees, confs, P)
    if cfg == 3:
        R = 128 if R is None else R
        P = rng.integers(2048, 8193, size=R)
        trees = [tree_levels(rng, 8, 10, 10) for _ in range(R)]
        confs = [conf_bimodal(rng, t) for t in trees]
        gate = Gate.from_taus(GATES_QWEN235B if gated else {}, w_max=10, budget=1024 * R // 128)
        return _assemble("cfg3-qwen235b", seed, rng, 64, 4, 151936, gate, trees, confs, P)
    if cfg == 4:
        R = 256 if R is None else R
        z = rng.standard_normal(R)
        P = np.minimum(32768, np.maximum(16, np.rint(np.exp(np.log(8192.0) + 1.0 * z)))).astype(np.int64)
        trees, confs = [], []
        for _ in range(R):
            if rng.random() < 0.5:
                t = tree_chain(12)
                confs.append(conf_dirichlet(rng, t, 0.3, 8)); trees.append(t)
            else:
                t = tree_levels(rng, 3, 16, 16)
                confs.append(conf_dirichlet(rng, t, 0.3, 16)); trees.append(t)
        gate = Gate.from_taus(GATES_QWEN235B if gated else {}, w_max=16, budget=4096 * R // 256)
        return _assemble("cfg4-stress", seed, rng, 64, 8, 151936, gate, trees, confs, P)
    raise ValueError(f"unknown config {cfg}")


# --------------------------------------------------------------------------
# bulk values (torch; imported lazily so the numpy-only oracle tests stay light)
# --------------------------------------------------------------------------
def draw_qkv(wl: Workload, capacity: int, device: str = "cpu", num_layers: int = 1,
             poison_unused: bool = False):
    """Q bf16 [capacity][Hq][128]; K/V pools bf16 [layers][num_pages][Hkv][16][128] ~ N(0,1)."""
    import torch
    g = torch.Generator(device=device)
    g.manual_seed(wl.seed)
    q = torch.randn(capacity, wl.Hq, HEAD_DIM, generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
    shape = (num_layers, wl.num_pages, wl.Hkv, PAGE_SIZE, HEAD_DIM)
    k = torch.empty(shape, device=device, dtype=torch.bfloat16)
    v = torch.empty(shape, device=device, dtype=torch.bfloat16)
    chunk = max(1, (1 << 26) // (wl.Hkv * PAGE_SIZE * HEAD_DIM))
    for t in (k, v):
        for l in range(num_layers):
            for s in range(0, wl.num_pages, chunk):
                e = min(wl.num_pages, s + chunk)
                t[l, s:e] = torch.randn(e - s, wl.Hkv, PAGE_SIZE, HEAD_DIM, generator=g, device=device,
                                        dtype=torch.float32).to(torch.bfloat16)
    if poison_unused:
        poison_unused_slots(wl, k, v)
    return q, k, v


def poison_unused_slots(wl: Workload, k, v, used_extra: Optional[np.ndarray] = None):
    """Fill every slot that no request may read (past P_i + C_i, spare pages) with NaN bit patterns."""
    import torch
    used = np.zeros((wl.num_pages, PAGE_SIZE), bool)
    cand = np.diff(wl.cand_offsets) if used_extra is None else used_extra
    for i in range(wl.R):
        n = int(wl.prefix_len[i]) + int(cand[i])
        for pos in range(n):
            used[wl.page_table[i, pos // PAGE_SIZE], pos % PAGE_SIZE] = True
    m = torch.from_numpy(~used).to(k.device)
    nan = torch.tensor(float("nan"), dtype=torch.bfloat16, device=k.device)
    for t in (k, v):
        t.permute(1, 3, 0, 2, 4)[m] = nan


def draw_logits(wl: Workload, sel_cand: np.ndarray, device: str = "cpu", ld: Optional[int] = None):
    """cfg4 form: bf16 N(0,1) logits [n_sel][ld>=V] with a +8 bump at the ground-truth target token
    of each selected node (`sel_cand` = global candidate index per packed node); no bump on a miss."""
    import torch
    V = wl.vocab
    ld = V if ld is None else ld
    n = len(sel_cand)
    g = torch.Generator(device=device)
    g.manual_seed(wl.seed + 7)
    logits = torch.empty(n, ld, device=device, dtype=torch.bfloat16)
    step = max(1, (1 << 26) // ld)
    for s in range(0, n, step):
        e = min(n, s + step)
        logits[s:e] = torch.randn(e - s, ld, generator=g, device=device, dtype=torch.float32).to(torch.bfloat16)
    tgt = torch.from_numpy(wl.target_after[sel_cand].astype(np.int64)).to(device)
    rows = torch.arange(n, device=device)
    hit = tgt != (V - 1)
    bumped = (logits[rows[hit], tgt[hit]].float() + 8.0).to(torch.bfloat16)
    logits[rows[hit], tgt[hit]] = bumped
    return logits


def draw_calibration_traces(rng, M: int, ties: bool = False, separation=(0.7, 0.1, 0.1, 0.3, 0.1, 0.6, 0.05, 0.0)):
    """Warm-up traces for echo_calibrate (stand-in for the paper's warm-up runs): M samples of
    (depth < 8, layer confidence in (0, 1], accepted).  Accepted samples draw Beta(2,2) shifted up by half the
    depth's `separation`, rejected ones down, so depths 0 and 5 ("root and target depth") separate
    well and the others do not.  `ties` rounds confidences to 1/64.  No method arithmetic here."""
    sep = np.asarray(separation, np.float64)
    depth = rng.integers(0, len(sep), M).astype(np.uint8)
    acc = rng.random(M) < 0.4
    conf = np.clip(rng.beta(2, 2, M) + sep[depth] * (acc - 0.5), 1e-6, 1.0)
    if ties:
        conf = np.maximum(np.round(conf * 64) / 64, 1.0 / 64)
    return depth, conf.astype(np.float32), acc.astype(np.uint8)


def draw_draft_level(rng, R: int, k_prev: int, k: int, vocab: int = 32000, alpha: float = 0.3):
    """Stand-in for the draft model's output at one level: each of the k_prev parents proposes its k most likely next
    tokens, probabilities Dirichlet(alpha) sorted descending (as a top-k would return them), tokens distinct among
    siblings.  logq = (float) log(probability) taken here on the host (SURVEY G-2).  No method arithmetic."""
    pr = -np.sort(-rng.dirichlet(np.full(k, alpha), size=(R, k_prev)), axis=-1)
    logq = np.log(np.maximum(pr, 1e-30)).astype(np.float32)
    tok = np.stack([[rng.choice(vocab, k, replace=False) for _ in range(k_prev)] for _ in range(R)]).astype(np.int32)
    return logq, tok
