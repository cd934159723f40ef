// echo_gate_select: S1-S5 of the super-tree verify step (include/echo.h).
//   k_score_gate  : one CTA per request -- path scores (Eq. 5), level maxima and the
//                   sparse gate (Eq. 6-7), tier assignment (Alg. 1) and a
//                   unique 64-bit selection key per candidate.
//   k_select      : one CTA -- radix select of the budget-th smallest key (Eq. 4), per-request
//                   counts and CSR offsets.
//   k_pack        : one CTA per request -- Flatten & Pack (Fig. 3(3)) with local parents and 128-bit
//                   ancestor masks.
// These steps move < 1 MB and are latency-bound: three launches, no host sync.  (Tried in
// round 2: scoring in CTAs of eight requests whose last one, by a ticket, runs the select -- and the packing too: no
// gain, 30 us against 28; packing by that one CTA is a chain of dependent loads per eight requests, 58 us.)
#include "common.cuh"

namespace {

struct GateParams {
  uint32_t depth_mask;
  float log_tau[32];
  int32_t w_max;
  int32_t static_k;
  int32_t schedule;
  int32_t cand_base;  // global index of this call's first candidate / request (> 0 only when several ranks share
  int32_t req_base;   // one budget)
};

__device__ __forceinline__ float f32_unordered(uint32_t o) {
  uint32_t u = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o;
  return __uint_as_float(u);
}

constexpr uint64_t KEY_INELIGIBLE = ~0ull;

// key order == (tier asc, S desc, request asc, node asc): tier in bit 63, inverted ordered score in
// bits 31..62, global candidate index (monotone in (request, node)) in bits 0..30.
__device__ __forceinline__ uint64_t make_key(int tier, float S, int g) {
  return ((uint64_t)tier << 63) | ((uint64_t)(~f32_ordered(S)) << 31) | (uint64_t)(uint32_t)g;
}

// ECHO_SCHED_ALG1 (Algorithm 1 as printed): the grants of Phase 1 (depth by depth,
// request order inside a depth, a level best-first) and then Phase 2 (truncated requests in the order they were
// truncated, the W_max best nodes of the truncation level) are, read as one sequence, the eligible nodes sorted by
// (phase, depth, request, rank in level); taking the first K_max of that order is the algorithm, including the
// level that only partly fits (readings R:L-1..L-4).
__device__ __forceinline__ uint64_t make_key_alg1(int phase, int depth, int request, int rank) {
  return ((uint64_t)phase << 63) | ((uint64_t)depth << 56) | ((uint64_t)(uint32_t)request << 16) | (uint64_t)rank;
}

// Shared memory of one request's scoring (one 128-thread group)
struct ScoreSmem {
  int par[ECHO_MAX_CAND];
  float lq[ECHO_MAX_CAND];
  float S[ECHO_MAX_CAND];
  int d[ECHO_MAX_CAND];
  uint32_t lvlmax[ECHO_MAX_DEPTH];
  int cut;
};

// S1-S2 and the selection keys of request i; j = candidate = thread in the request's 128-thread group.  `active` is
// false for a group without a request (it still takes part in the CTA-wide barriers).
__device__ __forceinline__ void score_gate_request(
    bool active, int i, int j, ScoreSmem& sm, const int32_t* __restrict__ cand_offsets,
    const int32_t* __restrict__ parent, const float* __restrict__ logq, const GateParams& gp,
    float* __restrict__ path_score, uint8_t* __restrict__ cand_depth, int32_t* __restrict__ cut_depth,
    uint64_t* __restrict__ keys, uint32_t* __restrict__ status) {
  int b = 0, C_all = 0;
  if (active) { b = cand_offsets[i]; C_all = cand_offsets[i + 1] - b; }
  const int C = min(C_all, ECHO_MAX_CAND);
  uint32_t bad = 0;
  if (C_all > ECHO_MAX_CAND) {  // more candidates than a request may have (R:G-14): flag, and make the excess
    bad |= ECHO_DEV_CAND_OVERFLOW;  // ineligible so that the select never reads an unwritten key
    for (int t = ECHO_MAX_CAND + j; t < C_all; t += ECHO_MAX_CAND) keys[b + t] = KEY_INELIGIBLE;
  }
  if (j < ECHO_MAX_DEPTH) sm.lvlmax[j] = 0u;
  if (j < C) {
    int p = parent[b + j];
    float lq = logq[b + j];
    if (p >= j || p < -1) { bad |= ECHO_DEV_BAD_PARENT; p = -1; }
    if (!(lq <= 0.0f)) bad |= ECHO_DEV_BAD_LOGQ;
    sm.par[j] = p;
    sm.lq[j] = lq;
  }
  __syncthreads();

  float S = 0.0f;
  int d = 0;
  if (j < C) {
    // S1: every node replays the root->leaf chain of fp32 adds in order, so the value is
    // bit-identical to the sequential recurrence (R:G-3); __fadd_rn forbids contraction.
    int chain[ECHO_MAX_DEPTH];
    int n = 0, c = j;
    while (c >= 0 && n < ECHO_MAX_DEPTH) { chain[n++] = c; c = sm.par[c]; }
    if (c >= 0) bad |= ECHO_DEV_DEPTH_OVERFLOW;
    for (int k = n - 1; k >= 0; --k) S = __fadd_rn(S, sm.lq[chain[k]]);
    d = n - 1;
    sm.S[j] = S;
    sm.d[j] = d;
    path_score[b + j] = S;
    cand_depth[b + j] = (uint8_t)d;
    atomicMax(&sm.lvlmax[d], f32_ordered(S));  // S2: m[i][d] (Eq. 6 in the log domain)
  }
  if (bad) atomicOr(status, bad);
  __syncthreads();

  if (j == 0 && active) {
    int cut = ECHO_CUT_NEVER;
    if (gp.static_k <= 0) {
      for (int dd = 0; dd < ECHO_MAX_DEPTH; ++dd) {
        if (!((gp.depth_mask >> dd) & 1u) || sm.lvlmax[dd] == 0u) continue;  // ungated or absent level (R:G-5)
        if (!(f32_unordered(sm.lvlmax[dd]) > gp.log_tau[dd])) { cut = dd; break; }  // Eq. 7, strict (R:G-4)
      }
    }
    sm.cut = cut;
    cut_depth[i] = cut;
  }
  __syncthreads();

  if (j < C) {
    const int cut = sm.cut;
    uint64_t key = KEY_INELIGIBLE;
    if (gp.static_k > 0) {
      int rank = 0;  // per-request top-static_k by (S desc, node asc) (R:G-15)
      for (int t = 0; t < C; ++t) rank += (sm.S[t] > S) || (sm.S[t] == S && t < j);
      if (rank < gp.static_k) key = make_key(0, 0.0f, gp.cand_base + b + j);
    } else if (gp.schedule == ECHO_SCHED_ALG1) {
      if (d <= cut) {
        int rank = 0;  // position in the level by (S desc, node asc)
        for (int t = 0; t < C; ++t) rank += (sm.d[t] == d) && ((sm.S[t] > S) || (sm.S[t] == S && t < j));
        if (d < cut) key = make_key_alg1(0, d, gp.req_base + i, rank);
        else if (rank < gp.w_max) key = make_key_alg1(1, d, gp.req_base + i, rank);
      }
    } else if (d < cut) {
      key = make_key(0, S, gp.cand_base + b + j);  // tier 0: depth extension
    } else if (d == cut) {
      int rank = 0;  // tier 1: the w_max best nodes of the truncation level (R:G-7, G-8)
      for (int t = 0; t < C; ++t) rank += (sm.d[t] == d) && ((sm.S[t] > S) || (sm.S[t] == S && t < j));
      if (rank < gp.w_max) key = make_key(1, S, gp.cand_base + b + j);
    }
    keys[b + j] = key;
  }
}

__global__ void __launch_bounds__(ECHO_MAX_CAND) k_score_gate(
    const int32_t* __restrict__ cand_offsets, const int32_t* __restrict__ parent, const float* __restrict__ logq,
    const __grid_constant__ GateParams gp, float* __restrict__ path_score, uint8_t* __restrict__ cand_depth,
    int32_t* __restrict__ cut_depth, uint64_t* __restrict__ keys, uint32_t* __restrict__ status) {
  __shared__ ScoreSmem sm;
  pdl_launch_dependents();
  score_gate_request(true, blockIdx.x, threadIdx.x, sm, cand_offsets, parent, logq, gp, path_score, cand_depth, cut_depth,
                     keys, status);
}

constexpr int SEL_THREADS = 1024;
constexpr int SEL_KPT = 16;  // keys per thread kept in registers by the radix select

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += t;
  }
  return v;
}

struct SelectSmem {
  int hist[256];
  int warp[32];
  uint64_t prefix;
  int k;
  int eligible;
  int done;
};

// S3 + the CSR offsets of S4 by one CTA of SEL_THREADS threads.  Returns (in every thread) the threshold: keys below it
// are selected (0 = nothing).
__device__ __forceinline__ uint64_t select_body(
    SelectSmem& sm, const int32_t* __restrict__ cand_offsets, const uint64_t* __restrict__ local_keys, int R,
    const uint64_t* __restrict__ keys, int N, int budget, int32_t* __restrict__ n_selected,
    int32_t* __restrict__ sel_offsets) {
  // `keys` [N] is the whole key population the budget is drawn from (this call's own keys, or the keys of every rank
  // that shares the budget); `local_keys` are this call's candidates, indexed like cand_offsets.
  int (&s_hist)[256] = sm.hist;
  int (&s_warp)[32] = sm.warp;
  uint64_t& s_prefix = sm.prefix;
  int& s_k = sm.k;
  int& s_eligible = sm.eligible;
  int& s_done = sm.done;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  // ---- S3: threshold T = budget-th smallest key (keys are unique => no ties to break) ----
  // Keys stay in registers across the passes when N <= SEL_THREADS * SEL_KPT (every config of BASELINE.json),
  // histogram updates are aggregated per thread and per warp (the top bytes of the keys -- tier, sign, exponent --
  // take one or two values, which would serialise 10 240 shared-memory atomics on one address), and the digit loop
  // stops as soon as the bucket that holds the budget-th key is taken whole.
  const bool cached = N <= SEL_THREADS * SEL_KPT;
  uint64_t rk[SEL_KPT];
#pragma unroll
  for (int i = 0; i < SEL_KPT; ++i) {
    const int g = tid + i * SEL_THREADS;
    rk[i] = (cached && g < N) ? keys[g] : KEY_INELIGIBLE;
  }
  if (tid == 0) s_eligible = 0;
  __syncthreads();
  {
    int e = 0;
    if (cached) {
#pragma unroll
      for (int i = 0; i < SEL_KPT; ++i) e += rk[i] != KEY_INELIGIBLE;
    } else {
      for (int g = tid; g < N; g += SEL_THREADS) e += keys[g] != KEY_INELIGIBLE;
    }
    e = warp_incl_scan(e, lane);
    if (lane == 31 && e) atomicAdd(&s_eligible, e);
  }
  __syncthreads();
  uint64_t T;
  if (budget <= 0) {
    T = 0;  // nothing selected (keys are > 0 unless tier 0, score +inf, g 0: excluded below by budget check)
  } else if (s_eligible <= budget) {
    T = KEY_INELIGIBLE - 1;  // everything eligible (R:G-12)
  } else {
    if (tid == 0) { s_prefix = 0; s_k = budget; s_done = 0; }
    int shift = 56;
    for (int pass = 0; pass < 8; ++pass, shift -= 8) {
      if (tid < 256) s_hist[tid] = 0;
      __syncthreads();
      const uint64_t prefix = s_prefix;
      auto in_prefix = [&](uint64_t key) { return key != KEY_INELIGIBLE && (pass == 0 || (key >> (shift + 8)) == prefix); };
      if (cached) {
        // the thread's keys that share the digit of its first participating key go in as one count; if the whole
        // warp agrees on that digit, as one atomic per warp
        int d0 = -1, cnt0 = 0;
#pragma unroll
        for (int i = 0; i < SEL_KPT; ++i) {
          if (in_prefix(rk[i])) {
            const int digit = (int)((rk[i] >> shift) & 0xff);
            if (d0 < 0) d0 = digit;
            if (digit == d0) ++cnt0;
            else atomicAdd(&s_hist[digit], 1);
          }
        }
        const unsigned have = __ballot_sync(0xffffffffu, d0 >= 0);
        if (have) {
          const int lead = __shfl_sync(0xffffffffu, d0, __ffs(have) - 1);
          if (__all_sync(0xffffffffu, d0 < 0 || d0 == lead)) {
            const int total = __reduce_add_sync(0xffffffffu, cnt0);
            if (lane == 0) atomicAdd(&s_hist[lead], total);
          } else if (d0 >= 0) {
            atomicAdd(&s_hist[d0], cnt0);
          }
        }
      } else {
        for (int g = tid; g < N; g += SEL_THREADS) {
          const uint64_t key = keys[g];
          if (in_prefix(key)) atomicAdd(&s_hist[(int)((key >> shift) & 0xff)], 1);
        }
      }
      __syncthreads();
      if (warp == 0) {  // find the digit that holds the k-th key
        int c[8], sum = 0;
#pragma unroll
        for (int t = 0; t < 8; ++t) { c[t] = s_hist[lane * 8 + t]; sum += c[t]; }
        int incl = warp_incl_scan(sum, lane);
        int excl = incl - sum;
        const int k = s_k;
        if (excl < k && k <= incl) {
          int run = excl;
#pragma unroll
          for (int t = 0; t < 8; ++t) {
            if (run < k && k <= run + c[t]) {
              s_prefix = (prefix << 8) | (uint64_t)(lane * 8 + t);
              s_k = k - run;
              if (k - run == c[t]) s_done = 1;  // the whole bucket is selected: lower digits do not matter
            }
            run += c[t];
          }
        }
      }
      __syncthreads();
      if (s_done) break;
    }
    // keys with the found prefix (and everything below it) are selected; pad the undecided low digits with ones
    T = shift > 0 ? ((s_prefix << shift) | ((1ull << shift) - 1ull)) : s_prefix;
  }
  const bool none = budget <= 0;

  // ---- S4: per-request counts, CSR offsets ----
  for (int r = warp; r < R; r += SEL_THREADS / 32) {
    const int b = cand_offsets[r], C = min(cand_offsets[r + 1] - b, ECHO_MAX_CAND);
    int cnt = 0;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      int j = w * 32 + lane;
      bool s = !none && j < C && local_keys[b + j] <= T;
      cnt += __popc(__ballot_sync(0xffffffffu, s));
    }
    if (lane == 0) sel_offsets[r + 1] = cnt;
  }
  if (tid == 0) sel_offsets[0] = 0;
  __syncthreads();
  {  // in-place inclusive scan of sel_offsets[1..R]
    const int per = (R + SEL_THREADS - 1) / SEL_THREADS;
    const int lo = tid * per, hi = min(R, lo + per);
    int sum = 0;
    for (int r = lo; r < hi; ++r) sum += sel_offsets[r + 1];
    int incl = warp_incl_scan(sum, lane);
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (warp == 0) s_warp[lane] = warp_incl_scan(s_warp[lane], lane);
    __syncthreads();
    int run = incl - sum + (warp ? s_warp[warp - 1] : 0);
    for (int r = lo; r < hi; ++r) { run += sel_offsets[r + 1]; sel_offsets[r + 1] = run; }
    if (tid == SEL_THREADS - 1) *n_selected = s_warp[31];
  }
  __syncthreads();  // the offsets are complete for whoever packs next
  return none ? 0ull : T + 1ull;  // keys < threshold are selected (0 = nothing; T < 2^64 - 1)
}

__global__ void __launch_bounds__(SEL_THREADS) k_select(
    const int32_t* __restrict__ cand_offsets, const uint64_t* __restrict__ local_keys, int R,
    const uint64_t* __restrict__ keys, int N, int budget, int32_t* __restrict__ n_selected,
    int32_t* __restrict__ sel_offsets, uint64_t* __restrict__ threshold) {
  __shared__ SelectSmem sm;
  pdl_launch_dependents();
  pdl_wait();  // keys come from k_score_gate
  const uint64_t thr = select_body(sm, cand_offsets, local_keys, R, keys, N, budget, n_selected, sel_offsets);
  if (threadIdx.x == 0) *threshold = thr;
}

// S4/S5: packed arrays, local parents, ancestor-or-self masks of request r.  One 128-thread group per request, tid =
// candidate; `active` is false for a group without a request (it still takes part in the CTA-wide barriers).
struct PackSmem {
  int par[ECHO_MAX_CAND];  // the request's parent array: the ancestor walks below are chains of dependent reads
  uint32_t bal[4];
};
__device__ __forceinline__ void pack_request(
    bool active, int r, int tid, PackSmem& sm, const int32_t* __restrict__ cand_offsets,
    const int32_t* __restrict__ parent, const uint8_t* __restrict__ cand_depth, const uint64_t* __restrict__ keys,
    uint64_t thr, int capacity, const int32_t* __restrict__ sel_offsets, int32_t* __restrict__ sel_node,
    int32_t* __restrict__ sel_req, int32_t* __restrict__ parent_local, uint8_t* __restrict__ sel_depth,
    uint32_t* __restrict__ anc_mask) {
  const int lane = tid & 31, warp = tid >> 5;
  int b = 0, C = 0, base = 0;
  if (active) {
    b = cand_offsets[r];
    C = min(cand_offsets[r + 1] - b, ECHO_MAX_CAND);
    base = sel_offsets[r];
  }
  {
    const int j = tid;
    const uint32_t mine = __ballot_sync(0xffffffffu, j < C && keys[b + j] < thr);
    if (lane == 0) sm.bal[warp] = mine;
    if (j < C) {
      const int pj = parent[b + j];
      sm.par[j] = pj >= j ? -1 : pj;
    }
  }
  __syncthreads();
  uint32_t bal[4];
#pragma unroll
  for (int w = 0; w < 4; ++w) bal[w] = sm.bal[w];
  auto local_of = [&](int c) -> int {  // packed local index of selected candidate c
    int l = 0;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      if (w < (c >> 5)) l += __popc(bal[w]);
      else if (w == (c >> 5)) l += __popc(bal[w] & ((1u << (c & 31)) - 1u));
    }
    return l;
  };
  const int j = tid;
  if ((bal[warp] >> lane) & 1u) {
    const int l = local_of(j);
    const int k = base + l;
    if (k < capacity) {
      const int p = sm.par[j];
      uint32_t m[4] = {0u, 0u, 0u, 0u};
      m[l >> 5] |= 1u << (l & 31);
      int pl = -1;
      int c = p;
      for (int step = 0; c >= 0 && step < ECHO_MAX_DEPTH; ++step) {
        // ancestor closure (DESIGN.md invariant I2) guarantees every ancestor is selected
        int la = local_of(c);
        if (step == 0) pl = la;
        m[la >> 5] |= 1u << (la & 31);
        c = sm.par[c];
      }
      sel_node[k] = j;
      sel_req[k] = r;
      sel_depth[k] = cand_depth[b + j];
      parent_local[k] = pl;
      reinterpret_cast<uint4*>(anc_mask)[k] = make_uint4(m[0], m[1], m[2], m[3]);
    }
  }
  __syncthreads();  // the group's shared memory may be reused for its next request
}

__global__ void __launch_bounds__(ECHO_MAX_CAND) k_pack(
    const int32_t* __restrict__ cand_offsets, const int32_t* __restrict__ parent,
    const uint8_t* __restrict__ cand_depth, const uint64_t* __restrict__ keys,
    const uint64_t* __restrict__ threshold, int capacity, const int32_t* __restrict__ sel_offsets,
    int32_t* __restrict__ sel_node, int32_t* __restrict__ sel_req, int32_t* __restrict__ parent_local,
    uint8_t* __restrict__ sel_depth, uint32_t* __restrict__ anc_mask) {
  __shared__ PackSmem sm;
  pdl_launch_dependents();
  pdl_wait();  // threshold and offsets come from k_select
  pack_request(true, blockIdx.x, threadIdx.x, sm, cand_offsets, parent, cand_depth, keys, *threshold, capacity,
               sel_offsets, sel_node, sel_req, parent_local, sel_depth, anc_mask);
}

}  // namespace

static GateParams gate_params(const EchoGate* g) {
  GateParams gp;
  gp.depth_mask = g->depth_mask;
  for (int d = 0; d < 32; ++d) gp.log_tau[d] = g->log_tau[d] + 0.0f;  // canonicalise -0 (R:G-13)
  gp.w_max = g->w_max;
  gp.static_k = g->static_k;
  gp.schedule = g->schedule;
  gp.cand_base = g->cand_index_base;
  gp.req_base = g->request_base;
  return gp;
}

int launch_gate_keys(EchoCtx* ctx, const EchoTrees* t, const EchoGate* g, EchoSelection* o, uint64_t* keys,
                     cudaStream_t st) {
  if (t->num_requests > 0) {
    ECHO_COUNT_LAUNCH();
    k_score_gate<<<t->num_requests, ECHO_MAX_CAND, 0, st>>>(t->cand_offsets, t->parent, t->logq, gate_params(g),
                                                            o->path_score, o->cand_depth, o->cut_depth, keys,
                                                            ctx->dev_status);
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}

int launch_gate_select_keys(EchoCtx* ctx, const EchoTrees* t, const EchoGate* g, const uint64_t* local_keys,
                            const uint64_t* all_keys, int64_t n_all, EchoSelection* o, cudaStream_t st) {
  const int R = t->num_requests;
  if (n_all > 0x7fffffffll) return ECHO_ERR_UNSUPPORTED;
  if (256 > ctx->workspace_bytes) return ECHO_ERR_WORKSPACE;
  uint64_t* threshold = reinterpret_cast<uint64_t*>(ctx->workspace);
  const int budget = g->static_k > 0 ? (int)n_all : g->budget;
  ECHO_CUDA_TRY(ctx, launch_pdl(k_select, dim3(1), dim3(SEL_THREADS), 0, st, t->cand_offsets, local_keys, R, all_keys,
                                (int)n_all, budget, o->n_selected, o->sel_offsets, threshold));
  if (R > 0) {
    ECHO_CUDA_TRY(ctx, launch_pdl(k_pack, dim3(R), dim3(ECHO_MAX_CAND), 0, st, t->cand_offsets, t->parent,
                                  o->cand_depth, local_keys, threshold, o->capacity, o->sel_offsets, o->sel_node,
                                  o->sel_req, o->parent_local, o->sel_depth, o->anc_mask));
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}

int launch_gate_select(EchoCtx* ctx, const EchoTrees* t, const EchoGate* g, EchoSelection* o, cudaStream_t st) {
  const int R = t->num_requests, N = t->total_cand;
  uint64_t* keys = reinterpret_cast<uint64_t*>(ctx->workspace);
  const size_t keys_bytes = align_up((size_t)N * sizeof(uint64_t), 256);
  if (keys_bytes + 256 > ctx->workspace_bytes) return ECHO_ERR_WORKSPACE;
  uint64_t* threshold = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(ctx->workspace) + keys_bytes);
  if (R > 0) {
    ECHO_COUNT_LAUNCH();
    k_score_gate<<<R, ECHO_MAX_CAND, 0, st>>>(t->cand_offsets, t->parent, t->logq, gate_params(g), o->path_score,
                                               o->cand_depth, o->cut_depth, keys, ctx->dev_status);
  }
  const int budget = g->static_k > 0 ? N : g->budget;
  ECHO_CUDA_TRY(ctx, launch_pdl(k_select, dim3(1), dim3(SEL_THREADS), 0, st, t->cand_offsets, keys, R, keys, N, budget,
                                o->n_selected, o->sel_offsets, threshold));
  if (R > 0) {
    ECHO_CUDA_TRY(ctx, launch_pdl(k_pack, dim3(R), dim3(ECHO_MAX_CAND), 0, st, t->cand_offsets, t->parent, o->cand_depth,
                                  keys, threshold, o->capacity, o->sel_offsets, o->sel_node, o->sel_req, o->parent_local,
                                  o->sel_depth, o->anc_mask));
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}
