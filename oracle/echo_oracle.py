"""CPU ORACLE for the ECHO super-tree verify step -- TEST INFRASTRUCTURE ONLY.

Plain, slow, obviously-correct numpy / pure-Python restatement of what the hot
path computes.  It shares no code with the CUDA path (`paper_2604_09603_b200/csrc`)
and imports nothing from the package.  Only `tests/`, `__graft_entry__.smoke()`
and `bench.py`'s cpu_baseline / `--impl reference` legs may import it.

Citations `P:<n>` are lines of /root/reference/PAPER.md; `S:<id>` are readings
of SURVEY.md §8(c), restated in DESIGN.md §3.

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): worked example W1
(tests/golden/w1.json), exactly-representable chain scores, Q=0 closed form,
chain == dense causal attention, single node == decode attention, brute-force
dense masked softmax, Python `sorted()` selection, exhaustive path enumeration.
Functions beyond the hot path and their pins: `select_alg1`
(tests/test_oracle_alg1_pins.py: hand-run example tests/golden/alg1.json,
invariants, ample budget = global top-B, order brute force), `calibrate`
(tests/test_oracle_calibrate_pins.py: closed forms, brute force over pairs,
scikit-learn roc_auc_score / roc_curve), `draft_expand`
(tests/test_oracle_draft_pins.py: hand example, brute-force top-k, Eq. 5 scores of
the built tree), `accept_stochastic` (tests/test_oracle_stochastic_pins.py: hand
example, emitted-token distribution on a grid of uniforms, T -> 0 = `accept`).
`argmax_shard_pairs` / `merge_argmax_pairs` (vocabulary-sharded S8;
tests/test_oracle_pins.py: merged over any partition they are `argmax_bf16`, with
ties, -0 / +0 and all -inf rows across the shard boundaries).
The paper prints no numeric example of this path, so parity with
"the paper's values" is unpinned; every function below is pinned by the
mathematics listed above.

`oracle/echo_oracle_attn.c` (wrapper `oracle/attn_c.py`) restates `verify_attn` as plain C loops over POSIX
threads, for every-row parity at full size and the multi-core CPU baseline; it is pinned against this file's
`verify_attn` and by closed forms of its own (tests/test_oracle_attn_c_pins.py).

Precision: path scores fp32 sequential root->leaf (north_star); attention fp64.
"""
from __future__ import annotations

import numpy as np

INT32_MAX = 2**31 - 1
PAGE = 16
D = 128


# ---------------------------------------------------------------- O1 (S1)
def path_scores(cand_offsets, parent, logq):
    """Eq. 5: S[j] = S[pa(j)] + log q[j], fp32, strictly root->leaf
    in node-index order (parent[j] < j); roots: S = 0.0f + logq (S:G-1, G-3, G-13)."""
    N = int(cand_offsets[-1])
    S = np.zeros(N, np.float32)
    depth = np.zeros(N, np.uint8)
    for i in range(len(cand_offsets) - 1):
        b = int(cand_offsets[i])
        for j in range(int(cand_offsets[i + 1]) - b):
            p = int(parent[b + j])
            if p < 0:
                depth[b + j] = 0
                S[b + j] = np.float32(0.0) + np.float32(logq[b + j])
            else:
                depth[b + j] = depth[b + p] + 1
                S[b + j] = np.float32(S[b + p]) + np.float32(logq[b + j])
    return S, depth


# ---------------------------------------------------------------- O2 (S2)
def gate_cut_depth(cand_offsets, S, depth, depth_mask, log_tau):
    """Eq. 6-7; Alg. 1 l.8.  m[i][d] = max_j S over level d;
    for gated depths ascending: pass iff m > log_tau[d] (log domain, strict; S:G-4);
    an absent level is skipped (S:G-5); first failure = cut depth, else INT32_MAX."""
    R = len(cand_offsets) - 1
    cut = np.full(R, INT32_MAX, np.int32)
    for i in range(R):
        b, e = int(cand_offsets[i]), int(cand_offsets[i + 1])
        for d in range(32):
            if not (depth_mask >> d) & 1:
                continue
            lvl = [S[j] for j in range(b, e) if depth[j] == d]
            if not lvl:
                continue
            m = max(lvl)
            if not (np.float32(m) > np.float32(log_tau[d])):
                cut[i] = d
                break
    return cut


# ---------------------------------------------------------------- O3 (S3)
def select(cand_offsets, S, depth, cut, budget, w_max, static_k=0):
    """Eq. 4; Alg. 1; priority rule P:162-167 (S:G-7..G-12, G-15).
    Returns the selected (request, node) pairs as a set-like sorted list."""
    R = len(cand_offsets) - 1
    if static_k > 0:
        out = []
        for i in range(R):
            b, e = int(cand_offsets[i]), int(cand_offsets[i + 1])
            order = sorted(range(e - b), key=lambda j: (-float(S[b + j]), j))
            out += [(i, j) for j in order[:static_k]]
        return sorted(out)
    elig = []
    for i in range(R):
        b, e = int(cand_offsets[i]), int(cand_offsets[i + 1])
        c = int(cut[i])
        for j in range(e - b):
            if depth[b + j] < c:
                elig.append((0, -float(S[b + j]), i, j))           # tier 0: depth extension
        lvl = sorted([j for j in range(e - b) if depth[b + j] == c], key=lambda j: (-float(S[b + j]), j))
        for j in lvl[:max(0, w_max)]:
            elig.append((1, -float(S[b + j]), i, j))               # tier 1: width expansion
    elig.sort()
    return sorted((i, j) for (_, _, i, j) in elig[:max(0, budget)])


# ---------------------------------------------------------------- O3' (NEXT-1): Algorithm 1 as printed
def select_alg1(cand_offsets, S, depth, depth_mask, log_tau, budget, w_max):
    """Algorithm 1, followed line by line in the paper's order (readings R:L-1..L-4):
    Phase 1 walks the depths; at each depth the active requests are visited in request order while budget is left;
    a request whose gate passes (or whose depth is not gated) appends its level -- the candidate tree already holds
    the W_topk drafted nodes of that level (S:G-9) -- and pays for it; one whose gate fails leaves active_set for
    trunc_set.  Phase 2 visits trunc_set in insertion order and widens each by up to W_max nodes of its truncation
    level.  The cap of Eq. 4 is never exceeded: a level (or a widening) that does not fit is granted best-first by
    (S desc, node asc) as far as the budget goes (R:L-1).  Paper depth d = 1 is depth 0 here (S:G-1).
    Returns (sorted list of (request, node), cut depth per request for the requests that were truncated)."""
    R = len(cand_offsets) - 1
    G = [[] for _ in range(R)]
    budget = max(0, int(budget))
    active = list(range(R))
    trunc = []
    cut = {}
    d = -1
    while budget > 0 and active:                       # l.5
        d += 1                                         # l.6
        if d >= 32:
            break
        for i in list(active):                         # l.7, request order
            if budget <= 0:
                break
            b, e = int(cand_offsets[i]), int(cand_offsets[i + 1])
            lvl = [j for j in range(e - b) if depth[b + j] == d]
            if not lvl:                                # R:L-2: the drafted tree ends here; nothing to extend or widen
                active.remove(i)
                continue
            if (depth_mask >> d) & 1:                  # l.8
                m = max(S[b + j] for j in lvl)
                is_pass = bool(np.float32(m) > np.float32(log_tau[d]))
            else:
                is_pass = True
            if is_pass:                                # l.9-11
                lvl.sort(key=lambda j: (-float(S[b + j]), j))
                grant = lvl[:budget]
                G[i] += grant
                budget -= len(grant)
            else:                                      # l.12-13
                active.remove(i)
                trunc.append(i)
                cut[i] = d
    for i in trunc:                                    # l.18-21 (garbled in the paper: R:L-4)
        if budget <= 0:
            break
        b, e = int(cand_offsets[i]), int(cand_offsets[i + 1])
        lvl = sorted([j for j in range(e - b) if depth[b + j] == cut[i]], key=lambda j: (-float(S[b + j]), j))
        w = min(budget, max(0, int(w_max)), len(lvl))
        G[i] += lvl[:w]
        budget -= w
    return sorted((i, j) for i in range(R) for j in G[i]), cut


# ---------------------------------------------------------------- O4 + O5 (S4, S5)
def pack(cand_offsets, parent, depth, selected, R):
    """Flatten & Pack, Fig. 3(3): request asc, node asc (S:P-1); CSR offsets,
    local parent remap, 128-bit ancestor-or-self masks as Python ints (S5)."""
    sel_offsets = np.zeros(R + 1, np.int32)
    sel_node, sel_req, parent_local, sel_depth, masks = [], [], [], [], []
    by_req = [[] for _ in range(R)]
    for (i, j) in selected:
        by_req[i].append(j)
    for i in range(R):
        nodes = sorted(by_req[i])
        loc = {j: l for l, j in enumerate(nodes)}
        b = int(cand_offsets[i])
        req_masks = []
        for l, j in enumerate(nodes):
            p = int(parent[b + j])
            pl = -1 if p < 0 else loc[p]          # KeyError = ancestor closure (I2) violated
            sel_node.append(j); sel_req.append(i); parent_local.append(pl)
            sel_depth.append(int(depth[b + j]))
            req_masks.append((1 << l) | (req_masks[pl] if pl >= 0 else 0))
        masks += req_masks
        sel_offsets[i + 1] = sel_offsets[i] + len(nodes)
    anc = np.zeros((len(masks), 4), np.uint32)
    for k, m in enumerate(masks):
        for w in range(4):
            anc[k, w] = (m >> (32 * w)) & 0xFFFFFFFF
    return dict(n_selected=len(sel_node), sel_offsets=sel_offsets,
                sel_node=np.asarray(sel_node, np.int32), sel_req=np.asarray(sel_req, np.int32),
                parent_local=np.asarray(parent_local, np.int32),
                sel_depth=np.asarray(sel_depth, np.uint8), anc_mask=anc, masks=masks)


def gate_select(cand_offsets, parent, logq, depth_mask, log_tau, w_max, budget, static_k=0, schedule=0):
    """S1-S5 end to end (what `echo_gate_select` must reproduce bit-exactly).  schedule 0 = global top-B
    (north_star, S:G-10); 1 = Algorithm 1 as printed (NEXT-1); `cut_depth` is the gate's verdict in both."""
    R = len(cand_offsets) - 1
    S, depth = path_scores(cand_offsets, parent, logq)
    if static_k > 0:
        cut = np.full(R, INT32_MAX, np.int32)
    else:
        cut = gate_cut_depth(cand_offsets, S, depth, depth_mask, log_tau)
    if schedule == 1 and static_k <= 0:
        sel, _ = select_alg1(cand_offsets, S, depth, depth_mask, log_tau, budget, w_max)
    else:
        sel = select(cand_offsets, S, depth, cut, budget, w_max, static_k)
    out = pack(cand_offsets, parent, depth, sel, R)
    out.update(path_score=S, cand_depth=depth, cut_depth=cut)
    return out


# ---------------------------------------------------------------- O6 + O7 (S6, S7)
def bf16_bits_to_f64(u16):
    """exact bf16 (stored as uint16 bit patterns) -> float64."""
    return (np.asarray(u16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def visible_positions(P_i, mask):
    """prefix [0,P_i) then P_i + a for every set bit a of the ancestor-or-self mask (S:A-1, A-2)."""
    return list(range(int(P_i))) + [int(P_i) + a for a in range(128) if (mask >> a) & 1]


def verify_attn(sel, q_bits, k_pool_bits, v_pool_bits, page_table, prefix_len, Hq, Hkv, sm_scale,
                layer=0, rows=None):
    """Plain dense definition softmax(sm_scale * q K^T) V over the visible set, fp64, no
    splitting, no online softmax (S:A-1..A-5).  q_bits uint16 [cap][Hq][128]; pools uint16
    [layers][pages][Hkv][16][128].  `rows` = optional list of (packed node, head) pairs to
    compute (sampled parity at full size); default all.  Returns {(k,h): (O[128], lse)} if
    rows given else (out [n][Hq][128] f64, lse [n][Hq] f64)."""
    G = Hq // Hkv
    offs = sel["sel_offsets"]
    n = int(sel["n_selected"])
    sel_req = sel["sel_req"]
    scale = float(np.float32(sm_scale))

    def one(k, heads):
        i = int(sel_req[k])
        l = k - int(offs[i])
        pos = visible_positions(prefix_len[i], sel["masks"][k] if "masks" in sel else
                                sum(int(sel["anc_mask"][k, w]) << (32 * w) for w in range(4)))
        pg = np.asarray([page_table[i][t // PAGE] for t in pos], np.int64)
        sl = np.asarray([t % PAGE for t in pos], np.int64)
        res = {}
        cache = {}
        for h in heads:
            kvh = h // G
            if kvh not in cache:
                cache[kvh] = (bf16_bits_to_f64(k_pool_bits[layer, pg, kvh, sl, :]),
                              bf16_bits_to_f64(v_pool_bits[layer, pg, kvh, sl, :]))
            Kt, Vt = cache[kvh]
            qv = bf16_bits_to_f64(q_bits[k, h, :])
            s = scale * (Kt @ qv)
            M = s.max()
            e = np.exp(s - M)
            Z = e.sum()
            res[h] = ((e @ Vt) / Z, M + np.log(Z))
        return res

    if rows is not None:
        out = {}
        by_k = {}
        for (k, h) in rows:
            by_k.setdefault(int(k), []).append(int(h))
        for k, hs in by_k.items():
            r = one(k, hs)
            for h in hs:
                out[(k, h)] = r[h]
        return out
    O = np.zeros((n, Hq, D), np.float64)
    L = np.zeros((n, Hq), np.float64)
    for k in range(n):
        r = one(k, range(Hq))
        for h in range(Hq):
            O[k, h], L[k, h] = r[h]
    return O, L


# ---------------------------------------------------------------- O8 (S8)
def argmax_bf16(logits_bits, vocab):
    """greedy target token: first maximum of each row over v < vocab (S:C-3).
    numpy.argmax returns the first occurrence; pinned against an explicit strict-'>' scan."""
    x = (np.asarray(logits_bits)[:, :vocab].astype(np.uint32) << 16).view(np.float32)
    return np.argmax(x, axis=1).astype(np.int32)


def argmax_shard_pairs(logits_bits, v0, v1):
    """S8 on one vocabulary shard (tensor-parallel ranks hold columns [v0, v1) of the logits): per row
    the shard's maximum (fp32 value of the bf16 logit, -0 taken as +0, S:C-3) and the GLOBAL index of its first
    occurrence.  Pinned (tests/test_oracle_pins.py): merged over any partition of the vocabulary it is `argmax_bf16`."""
    x = (np.asarray(logits_bits)[:, v0:v1].astype(np.uint32) << 16).view(np.float32)
    j = np.argmax(x, axis=1)
    val = x[np.arange(x.shape[0]), j] + np.float32(0.0)
    return val.astype(np.float32), (v0 + j).astype(np.int32)


def merge_argmax_pairs(values, indices):
    """values / indices [W][rows] from `argmax_shard_pairs` -> token per row: the greatest value, then the lowest
    index (the first maximum of the whole row, S:C-3)."""
    values, indices = np.asarray(values), np.asarray(indices)
    out = np.zeros(values.shape[1], np.int32)
    for r in range(values.shape[1]):
        best = 0
        for w in range(1, values.shape[0]):
            if values[w, r] > values[best, r] or (values[w, r] == values[best, r] and indices[w, r] < indices[best, r]):
                best = w
        out[r] = indices[best, r]
    return out


# ---------------------------------------------------------------- O9 (S9)
def accept(sel, draft_token, prev_token, target_token, R):
    """Greedy acceptance (S:C-1, C-2, C-4, C-5): acc[l] = parent accepted
    and draft[l] == target token after the parent (roots: == prev_token); best = accepted
    node of maximum depth, lowest local index; path = its ancestor-or-self set ascending."""
    offs = sel["sel_offsets"]
    accept_len = np.zeros(R, np.int32)
    last_node = np.full(R, -1, np.int32)
    bonus = np.full(R, -1, np.int32)
    accept_idx = np.full((R, 32), -1, np.int32)
    for i in range(R):
        b, e = int(offs[i]), int(offs[i + 1])
        acc = []
        best, best_d = -1, -1
        for l in range(e - b):
            pl = int(sel["parent_local"][b + l])
            if pl < 0:
                a = int(draft_token[b + l]) == int(prev_token[i])
            else:
                a = acc[pl] and int(draft_token[b + l]) == int(target_token[b + pl])
            acc.append(bool(a))
            if a and int(sel["sel_depth"][b + l]) > best_d:
                best, best_d = l, int(sel["sel_depth"][b + l])
        if best < 0:
            continue
        m = sum(int(sel["anc_mask"][b + best, w]) << (32 * w) for w in range(4))
        path = [a for a in range(128) if (m >> a) & 1]
        accept_len[i] = len(path)
        accept_idx[i, :len(path)] = [b + a for a in path]
        last_node[i] = b + best
        bonus[i] = int(target_token[b + best])
    return dict(accept_len=accept_len, accept_idx=accept_idx, last_node=last_node, bonus_token=bonus)


# ---------------------------------------------------------------- O10 (S10)
def compact_kv(sel, acc, k_pool_bits, v_pool_bits, page_table, prefix_len, R):
    """KV-slot compaction (S:C-6): path node t moves from position P_i + a_t to P_i + t;
    slot(i,pos) = page_table[i][pos/16]*16 + pos%16; all layers, all KV heads, K and V; every
    read happens before any write.  Pools (uint16 views) are updated IN PLACE."""
    slot_src = np.full((R, 32), -1, np.int32)
    slot_dst = np.full((R, 32), -1, np.int32)
    new_len = np.zeros(R, np.int32)
    offs = sel["sel_offsets"]
    for i in range(R):
        P = int(prefix_len[i])
        L = int(acc["accept_len"][i])
        new_len[i] = P + L
        tmp = []
        for t in range(L):
            a = int(acc["accept_idx"][i, t]) - int(offs[i])
            sp, dp = P + a, P + t
            slot_src[i, t] = int(page_table[i][sp // PAGE]) * PAGE + sp % PAGE
            slot_dst[i, t] = int(page_table[i][dp // PAGE]) * PAGE + dp % PAGE
            s = int(slot_src[i, t])
            tmp.append((k_pool_bits[:, s // PAGE, :, s % PAGE, :].copy(),
                        v_pool_bits[:, s // PAGE, :, s % PAGE, :].copy()))
        for t in range(L):
            d = int(slot_dst[i, t])
            k_pool_bits[:, d // PAGE, :, d % PAGE, :] = tmp[t][0]
            v_pool_bits[:, d // PAGE, :, d % PAGE, :] = tmp[t][1]
    return dict(slot_src=slot_src, slot_dst=slot_dst, new_len=new_len)


# ---------------------------------------------------------------- O11 (NEXT-3): warm-up calibration of the gates
def calibrate(depth, conf, accepted, delta):
    """Offline calibration, P:115 (and P:446): per depth d, the separability of the layer confidences c_{i,d} of
    accepted versus rejected samples is the AUC (Hanley & McNeil 1982: the Wilcoxon / Mann-Whitney statistic,
    AUC = (#{c_pos > c_neg} + 0.5 #{c_pos == c_neg}) / (n_pos n_neg)); sweet spots D_sig = {d : AUC_d > delta};
    tau_d "maximises the separation between the two distributions": the observed value v that maximises
    J(v) = #pos(c > v)/n_pos - #neg(c > v)/n_neg (Youden's J = the Kolmogorov-Smirnov distance of the two empirical
    CDFs; the gate is c > tau, Eq. 7), the smallest such v on ties (readings R:K-1..K-3).  Plain
    definitions on exact integers; a depth with no accepted or no rejected sample gets AUC 0.5 and tau 0 and is
    never a sweet spot.  Returns dict(auc f64[32], tau f32[32], n_pos, n_neg i64[32], depth_mask)."""
    depth = np.asarray(depth).astype(np.int64)
    conf = np.asarray(conf, np.float32)
    accepted = np.asarray(accepted).astype(bool)
    auc = np.full(32, 0.5, np.float64)
    tau = np.zeros(32, np.float32)
    n_pos = np.zeros(32, np.int64)
    n_neg = np.zeros(32, np.int64)
    mask = 0
    for d in range(32):
        m = depth == d
        pos = np.sort(conf[m & accepted])
        neg = np.sort(conf[m & ~accepted])
        n_pos[d], n_neg[d] = len(pos), len(neg)
        if len(pos) == 0 or len(neg) == 0:
            continue
        less = np.searchsorted(neg, pos, side="left").astype(np.int64)      # negatives strictly below each positive
        leq = np.searchsorted(neg, pos, side="right").astype(np.int64)
        two_u = int((2 * less + (leq - less)).sum())                         # 2 x the Mann-Whitney U
        auc[d] = float(two_u) / float(2 * len(pos) * len(neg))
        best_v, best_num = None, None
        for v in np.unique(np.concatenate([pos, neg])):                      # ascending: the first maximum is kept
            p_gt = len(pos) - int(np.searchsorted(pos, v, side="right"))
            n_gt = len(neg) - int(np.searchsorted(neg, v, side="right"))
            num = p_gt * len(neg) - n_gt * len(pos)                          # J(v) n_pos n_neg, an integer
            if best_num is None or num > best_num:
                best_v, best_num = v, num
        tau[d] = best_v
        if auc[d] > delta:
            mask |= 1 << d
    return dict(auc=auc, tau=tau, n_pos=n_pos, n_neg=n_neg, depth_mask=mask)


# ---------------------------------------------------------------- O12 (NEXT-4): draft-side level expansion
def draft_expand(level, k, parent_score, child_logq, child_token):
    """One level of the draft tree built from the draft model's top-k outputs (EAGLE-style dynamic expansion, the step
    the paper takes from its base system, "topk tokens"; readings R:D-1..D-3).  Per request:
    the k_prev nodes of the previous level (k_prev = 1 virtual root with score 0 at level 0, else k) each propose k
    children with draft log-probabilities; the cumulative score of a candidate is fl32(S_parent + logq) (Eq. 5), and
    the level keeps the k best by (score desc, parent slot asc, child rank asc), in that order.
    parent_score f32 [R][k_prev]; child_logq f32 / child_token i32 [R][k_prev][k].
    Returns dict(sel_parent i32 [R][k] (slot in the previous level, -1 at level 0), logq f32 [R][k], token i32 [R][k],
    score f32 [R][k])."""
    parent_score = np.asarray(parent_score, np.float32)
    child_logq = np.asarray(child_logq, np.float32)
    child_token = np.asarray(child_token, np.int32)
    R, k_prev, kk = child_logq.shape
    assert kk == k and (k_prev == 1 if level == 0 else k_prev == k)
    sel_parent = np.zeros((R, k), np.int32)
    logq = np.zeros((R, k), np.float32)
    token = np.zeros((R, k), np.int32)
    score = np.zeros((R, k), np.float32)
    for i in range(R):
        cands = []
        for p in range(k_prev):
            for c in range(k):
                s = np.float32(np.float32(parent_score[i, p]) + child_logq[i, p, c])
                cands.append((-float(s), p, c, s))
        cands.sort(key=lambda t: (t[0], t[1], t[2]))
        for slot, (_, p, c, s) in enumerate(cands[:k]):
            sel_parent[i, slot] = -1 if level == 0 else p
            logq[i, slot] = child_logq[i, p, c]
            token[i, slot] = child_token[i, p, c]
            score[i, slot] = s
    return dict(sel_parent=sel_parent, logq=logq, token=token, score=score)


# ---------------------------------------------------------------- O13 (NEXT-2): stochastic tree acceptance
def softmax_bits(row_bits, vocab, temperature):
    """softmax(logits / T) of one bf16 row in fp64 (plain definition)."""
    x = bf16_bits_to_f64(np.asarray(row_bits)[:vocab]) / float(np.float32(temperature))
    x = x - x.max()
    e = np.exp(x)
    return e / e.sum()


def accept_stochastic(sel, draft_token, root_logits_bits, target_logits_bits, vocab, temperature, u_accept, u_bonus, R):
    """Tree acceptance at temperature > 0 under the speculative-sampling conditions the paper cites,
    in the multi-round form tree drafters use when the draft proposes its top-k deterministically (so q = 1 on a
    proposed token; readings R:T-1..T-4).  Per request, starting from the distribution p after the last
    committed token (root_logits) with nothing removed: the children of the current node are tried in packed order;
    child c with token x is accepted iff u_accept[c] < p'(x), p' = p with the tokens rejected so far at this node
    removed and renormalised; a rejected token is removed; an accepted child becomes the current node and p becomes
    softmax(target_logits[c] / T).  When no child is accepted the bonus token is drawn from the residual p' by
    inverse CDF in vocabulary order with u_bonus[i] (smallest v whose cumulative residual mass exceeds u (1 - m)).
    Emits exactly p at every position (checked in the pins).  Returns accept_len / accept_idx / last_node /
    bonus_token like `accept`, plus for the tests: min_margin (smallest |u - p'| over the decisions) and, per request,
    the normalised residual CDF and the bonus draw (a token t is a valid draw within eps iff
    cdf[t-1] - eps <= u <= cdf[t] + eps and its residual mass is positive), and `decisions` = (packed node, p') of
    every accept / reject test in the order they were taken."""
    offs = sel["sel_offsets"]
    accept_len = np.zeros(R, np.int32)
    last_node = np.full(R, -1, np.int32)
    bonus = np.full(R, -1, np.int32)
    accept_idx = np.full((R, 32), -1, np.int32)
    margins = []  # |u - p'| of every accept / reject decision: the GPU tests redraw uniforms that sit on a knife edge
    decisions = []  # (packed node, p') of every decision, so that a test can redraw just the knife-edge uniforms
    cdfs, targets = [], []  # residual CDF and u (1 - m) of the bonus draw: neighbouring tokens are a rounding apart
    for i in range(R):
        b, e = int(offs[i]), int(offs[i + 1])
        pl = [int(x) for x in sel["parent_local"][b:e]]
        p = softmax_bits(root_logits_bits[i], vocab, temperature)
        cur, path = -1, []
        while True:
            removed, m, nxt = [], 0.0, None
            for c in [l for l in range(e - b) if pl[l] == cur]:
                x = int(draft_token[b + c])
                px = 0.0 if x in removed else float(p[x])
                pr = px / (1.0 - m) if (1.0 - m) > 0.0 else 0.0
                u = float(np.float32(u_accept[b + c]))
                margins.append(abs(u - pr))
                decisions.append((b + c, pr))
                if u < pr:
                    nxt = c
                    break
                if x not in removed:
                    removed.append(x)
                    m += float(p[x])
            if nxt is None or len(path) >= 32:
                break
            path.append(nxt)
            cur = nxt
            p = softmax_bits(target_logits_bits[b + nxt], vocab, temperature)
        r = p.copy()
        r[removed] = 0.0
        cdf = np.cumsum(r)
        target = float(np.float32(u_bonus[i])) * cdf[-1]
        v = int(np.searchsorted(cdf, target, side="right"))
        v = min(v, int(np.flatnonzero(r)[-1]))
        cdfs.append(cdf / cdf[-1])
        targets.append(target / cdf[-1])
        bonus[i] = v
        accept_len[i] = len(path)
        accept_idx[i, :len(path)] = [b + a for a in path]
        last_node[i] = b + cur if cur >= 0 else -1
    return dict(accept_len=accept_len, accept_idx=accept_idx, last_node=last_node, bonus_token=bonus,
                min_margin=min(margins) if margins else 1.0, bonus_cdf=cdfs, bonus_u=targets, decisions=decisions)
