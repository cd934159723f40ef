// echo_gate_select: S1-S5 of the super-tree verify step (include/echo.h).
//   k_gate_cluster: all of it as ONE launch of one thread-block cluster (<= 16 CTAs x 1024 threads, 8 requests per CTA
//                   and round): keys stay in shared memory, the radix select's histograms are summed through
//                   distributed shared memory, the thread that made a key packs its node.  The path echo_gate_select
//                   takes for up to 512 requests.
//   k_score_gate  : one CTA per request -- path scores (Eq. 5), level maxima and the
//                   sparse gate (Eq. 6-7), tier assignment (Alg. 1) and a
//                   unique 64-bit selection key per candidate.
//   k_select      : one CTA -- radix select of the budget-th smallest key (Eq. 4), per-request
//                   counts and CSR offsets.
//   k_pack        : one CTA per request -- Flatten & Pack (Fig. 3(3)) with local parents and 128-bit
//                   ancestor masks.
// The three-kernel chain serves echo_gate_keys / echo_gate_select_keys (several ranks share one budget: the key
// population crosses processes between scoring and selecting), more than 512 requests, and ECHO_OPT_GATE_PATH = 1; it
// shares the scoring and packing device functions with the cluster kernel.
// These steps move < 1 MB and are latency-bound.  (Tried in round 2: scoring in CTAs of eight
// requests whose last one, by a ticket, runs the select -- and the packing too: no gain, 30 us against 28; packing by
// that one CTA is a chain of dependent loads per eight requests, 58 us.)
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

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
// The fields sit at the top of the key (1 + 5 + 24 + 8 bits: depth < 32, request < 2^24 -- checked by the host --,
// rank < 128), so the radix select is through after the first 38 bits.
__device__ __forceinline__ uint64_t make_key_alg1(int phase, int depth, int request, int rank) {
  return ((uint64_t)phase << 63) | ((uint64_t)depth << 58) | ((uint64_t)(uint32_t)request << 34) | ((uint64_t)rank << 26);
}

// Shared memory of one request's scoring (one 128-thread group)
struct ScoreSmem {
  int par[ECHO_MAX_CAND];
  float lq[ECHO_MAX_CAND];
  float S[ECHO_MAX_CAND];
  int d[ECHO_MAX_CAND];
  uint32_t lvlmax[ECHO_MAX_DEPTH];
  uint32_t lvlbal[ECHO_MAX_CAND / 32];
  int cut;
};

// What candidate j of request i reads from global memory (issued ahead of the arithmetic that needs it)
struct CandIn {
  int b, C_all;  // first candidate of the request, its candidate count as given
  int p;
  float lq;
};
__device__ __forceinline__ CandIn load_cand(bool active, int i, int j, const int32_t* __restrict__ cand_offsets,
                                            const int32_t* __restrict__ parent, const float* __restrict__ logq) {
  CandIn in = {0, 0, -1, 0.0f};
  if (active) { in.b = cand_offsets[i]; in.C_all = cand_offsets[i + 1] - in.b; }
  if (j < min(in.C_all, ECHO_MAX_CAND)) { in.p = parent[in.b + j]; in.lq = logq[in.b + j]; }
  return in;
}

// S1-S2 and the selection key of candidate j (= thread in the request's 128-thread group) of request i; the key is
// returned (KEY_INELIGIBLE when j is past the request), the depth goes to d_out.  `active` is false for a group
// without a request (it still takes part in the CTA-wide barriers).
__device__ __forceinline__ uint64_t score_gate_request(
    bool active, int i, int j, const CandIn& in, ScoreSmem& sm, const GateParams& gp, float* __restrict__ path_score,
    uint8_t* __restrict__ cand_depth, int32_t* __restrict__ cut_depth, uint32_t* __restrict__ status, int& d_out) {
  const int b = in.b, C_all = in.C_all;
  const int C = min(C_all, ECHO_MAX_CAND);
  uint32_t bad = 0;
  if (C_all > ECHO_MAX_CAND) bad |= ECHO_DEV_CAND_OVERFLOW;  // more candidates than a request may have (R:G-14)
  if (j < ECHO_MAX_DEPTH) sm.lvlmax[j] = 0u;
  if (j < C) {
    int p = in.p;
    float lq = in.lq;
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

  if (j < ECHO_MAX_DEPTH) {  // the group's first warp, lane = depth: the first gated level that fails Eq. 7
    static_assert(ECHO_MAX_DEPTH == 32, "one lane per depth");
    const uint32_t m = sm.lvlmax[j];
    // ungated or absent levels never fail (R:G-5); the comparison is strict (R:G-4)
    const bool fail = gp.static_k <= 0 && ((gp.depth_mask >> j) & 1u) && m != 0u && !(f32_unordered(m) > gp.log_tau[j]);
    const unsigned fails = __ballot_sync(0xffffffffu, fail);
    if (j == 0 && active) {
      const int cut = fails ? __ffs(fails) - 1 : ECHO_CUT_NEVER;
      sm.cut = cut;
      cut_depth[i] = cut;
    }
  }
  __syncthreads();

  uint64_t key = KEY_INELIGIBLE;
  const int cut = sm.cut;
  if (gp.static_k <= 0 && gp.schedule != ECHO_SCHED_ALG1) {
    // tier 0: depth extension; tier 1: the w_max best nodes of the truncation level by (S desc, node asc)
    // (R:G-7, G-8).  The level's nodes are first gathered into a list (the chain replays are over: lq and
    // d hold the list's scores and node ids from here on), so a rank costs the level's width, not C, compares.
    const bool lvl = j < C && d == cut;
    const unsigned lane = j & 31, wq = j >> 5;
    const unsigned mine = __ballot_sync(0xffffffffu, lvl);
    if (lane == 0) sm.lvlbal[wq] = mine;
    __syncthreads();
    int pos = __popc(mine & ((1u << lane) - 1u)), n_lvl = 0;
#pragma unroll
    for (int w = 0; w < ECHO_MAX_CAND / 32; ++w) {
      const int c = __popc(sm.lvlbal[w]);
      if (w < (int)wq) pos += c;
      n_lvl += c;
    }
    if (lvl) { sm.lq[pos] = S; sm.d[pos] = j; }
    __syncthreads();
    if (j < C && d < cut) {
      key = make_key(0, S, gp.cand_base + b + j);
    } else if (lvl) {
      int rank = 0;
      for (int t = 0; t < n_lvl; ++t) rank += (sm.lq[t] > S) || (sm.lq[t] == S && sm.d[t] < j);
      if (rank < gp.w_max) key = make_key(1, S, gp.cand_base + b + j);
    }
  } else if (j < C) {
    if (gp.static_k > 0) {
      int rank = 0;  // per-request top-static_k by (S desc, node asc) (R:G-15)
      for (int t = 0; t < C; ++t) rank += (sm.S[t] > S) || (sm.S[t] == S && t < j);
      if (rank < gp.static_k) key = make_key(0, 0.0f, gp.cand_base + b + j);
    } else if (d <= cut) {  // ECHO_SCHED_ALG1
      int rank = 0;  // position in the level by (S desc, node asc)
      for (int t = 0; t < C; ++t) rank += (sm.d[t] == d) && ((sm.S[t] > S) || (sm.S[t] == S && t < j));
      if (d < cut) key = make_key_alg1(0, d, gp.req_base + i, rank);
      else if (rank < gp.w_max) key = make_key_alg1(1, d, gp.req_base + i, rank);
    }
  }
  d_out = d;
  return key;
}

__global__ void __launch_bounds__(ECHO_MAX_CAND) k_score_gate(
    const int32_t* __restrict__ cand_offsets, const int32_t* __restrict__ parent, const float* __restrict__ logq,
    const __grid_constant__ GateParams gp, float* __restrict__ path_score, uint8_t* __restrict__ cand_depth,
    int32_t* __restrict__ cut_depth, uint64_t* __restrict__ keys, uint32_t* __restrict__ status) {
  __shared__ ScoreSmem sm;
  pdl_launch_dependents();
  const int i = blockIdx.x, j = threadIdx.x;
  const CandIn in = load_cand(true, i, j, cand_offsets, parent, logq);
  int d;
  const uint64_t key = score_gate_request(true, i, j, in, sm, gp, path_score, cand_depth, cut_depth, status, d);
  if (j < min(in.C_all, ECHO_MAX_CAND)) keys[in.b + j] = key;
  // the excess of an over-long request is ineligible, so that the select never reads an unwritten key
  for (int t = ECHO_MAX_CAND + j; t < in.C_all; t += ECHO_MAX_CAND) keys[in.b + t] = KEY_INELIGIBLE;
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

// S4/S5 for one selected candidate j of request r: its packed slot, local parent and ancestor-or-self mask.  `bal` =
// the request's 128 selection bits, `par(c)` = parent of candidate c (-1 or negative for a root), `base` = the
// request's first packed slot.
template <typename ParFn>
__device__ __forceinline__ void pack_node(
    int r, int j, int depth, const uint32_t (&bal)[4], ParFn par, int base, int capacity,
    int32_t* __restrict__ sel_node, int32_t* __restrict__ sel_req, int32_t* __restrict__ parent_local,
    uint8_t* __restrict__ sel_depth, uint32_t* __restrict__ anc_mask) {
  auto local_of = [&](int c) -> int {  // packed local index of selected candidate c
    int l = 0;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      if (w < (c >> 5)) l += __popc(bal[w]);
      else if (w == (c >> 5)) l += __popc(bal[w] & ((1u << (c & 31)) - 1u));
    }
    return l;
  };
  const int l = local_of(j);
  const int k = base + l;
  if (k >= capacity) return;
  uint32_t m[4] = {0u, 0u, 0u, 0u};
  m[l >> 5] |= 1u << (l & 31);
  int pl = -1;
  int c = par(j);
  for (int step = 0; c >= 0 && step < ECHO_MAX_DEPTH; ++step) {
    // ancestor closure (DESIGN.md invariant I2) guarantees every ancestor is selected
    const int la = local_of(c);
    if (step == 0) pl = la;
    m[la >> 5] |= 1u << (la & 31);
    c = par(c);
  }
  sel_node[k] = j;
  sel_req[k] = r;
  sel_depth[k] = (uint8_t)depth;
  parent_local[k] = pl;
  reinterpret_cast<uint4*>(anc_mask)[k] = make_uint4(m[0], m[1], m[2], m[3]);
}

// One 128-thread group per request, tid = candidate; `active` is false for a group without a request (it still takes
// part in the CTA-wide barriers).
struct PackSmem {
  int par[ECHO_MAX_CAND];  // the request's parent array: the ancestor walks are chains of dependent reads
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
  const int j = tid;
  {
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
  if ((bal[warp] >> lane) & 1u)
    pack_node(r, j, cand_depth[b + j], bal, [&](int c) { return sm.par[c]; }, base, capacity, sel_node, sel_req,
              parent_local, sel_depth, anc_mask);
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

// ---- the whole of echo_gate_select as one launch of one thread-block cluster ----
// The three kernels above cost three launches and two hand-overs through global memory for < 1 MB of data.  Here a
// cluster of CL CTAs of 1024 threads holds everything on chip: CTA c scores requests [c*rpc, (c+1)*rpc) (eight
// 128-thread groups, thread = candidate, up to GC_ROUNDS requests per group), the keys stay in shared memory, the radix
// select takes 11 bits a pass over a 2048-bin histogram that every CTA builds on its own keys and then sums over the
// cluster through distributed shared memory (so every CTA takes the same decisions and nothing is broadcast), and the
// thread that made a key packs its node.  Same arithmetic as the chain: the scoring and packing are the same device
// functions.  Measured (B200, bench.py, cfg2): 21.6 us per echo_gate_select against 28.6 us for the chain.
constexpr int GC_THREADS = 1024;
constexpr int GC_GROUPS = GC_THREADS / ECHO_MAX_CAND;  // 8
constexpr int GC_ROUNDS = 4;
constexpr int GC_SLOTS = GC_GROUPS * GC_ROUNDS;  // requests per CTA
constexpr int GC_BITS = 11;
constexpr int GC_BINS = 1 << GC_BITS;
constexpr int GC_SLICE = 128;                  // bins per slice: one int4 per lane of a warp
constexpr int GC_NSLICE = GC_BINS / GC_SLICE;  // 16
static_assert(GC_BINS == 2 * GC_THREADS, "one thread zeroes two bins");
static_assert(GC_SLOTS == 32, "one warp scans a CTA's request counts");

struct ClusterSmem {
  uint64_t key[GC_SLOTS][ECHO_MAX_CAND];  // selection keys of the CTA's requests (KEY_INELIGIBLE past a request's end)
  ScoreSmem score[GC_GROUPS];
  int8_t par8[GC_SLOTS][ECHO_MAX_CAND];   // validated parents (-1 = root), kept for the packing
  uint8_t dep8[GC_SLOTS][ECHO_MAX_CAND];  // depths
  uint32_t bal[GC_SLOTS][4];              // selection bits per request
  int hist[2][GC_BINS];                   // this CTA's keys by digit, per pass parity; read by every CTA of the cluster
  int slice[2][GC_NSLICE];                // sums of the histogram's slices of GC_SLICE bins; likewise
  int csum[2][GC_NSLICE];                 // the cluster's slice sums
  alignas(16) int tot[2][GC_SLICE];       // the cluster's histogram of the slice that holds the k-th key
  int cnt[GC_SLOTS];  // inclusive count of selected nodes over this CTA's requests
  int cta_total;      // read by every CTA of the cluster
  int base;
  uint64_t found;
};

// Code size is time here: the kernel runs once per step with its instructions cold in every cache (the attention
// kernel has streamed > 1 GB through L2 since), so every loop over a CTA's request slots stays rolled.
__global__ void __launch_bounds__(GC_THREADS, 1) k_gate_cluster(
    const int32_t* __restrict__ cand_offsets, const int32_t* __restrict__ parent, const float* __restrict__ logq,
    const __grid_constant__ GateParams gp, int R, int budget, int capacity, float* __restrict__ path_score,
    uint8_t* __restrict__ cand_depth, int32_t* __restrict__ cut_depth, int32_t* __restrict__ n_selected,
    int32_t* __restrict__ sel_offsets, int32_t* __restrict__ sel_node, int32_t* __restrict__ sel_req,
    int32_t* __restrict__ parent_local, uint8_t* __restrict__ sel_depth, uint32_t* __restrict__ anc_mask,
    uint32_t* __restrict__ status) {
  extern __shared__ __align__(16) unsigned char gc_smem[];
  ClusterSmem& sm = *reinterpret_cast<ClusterSmem*>(gc_smem);
  cg::cluster_group cluster = cg::this_cluster();
  const int CL = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  pdl_launch_dependents();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = tid / ECHO_MAX_CAND, j = tid % ECHO_MAX_CAND;
  const int rpc = (R + CL - 1) / CL;  // requests per CTA (host: <= GC_SLOTS)
  const int rounds = (rpc + GC_GROUPS - 1) / GC_GROUPS;
  const int nslot = rounds * GC_GROUPS;
  // ---- S1-S2 and keys: a round's loads are issued a round ahead of the arithmetic ----
  CandIn nxt = load_cand(g < rpc && rank * rpc + g < R, rank * rpc + g, j, cand_offsets, parent, logq);
  sm.hist[0][2 * tid] = 0;
  sm.hist[0][2 * tid + 1] = 0;
  if (tid < GC_NSLICE) sm.slice[0][tid] = sm.csum[0][tid] = 0;
  if (tid < GC_SLICE) sm.tot[0][tid] = 0;
#pragma unroll 1
  for (int slot = g; slot < nslot; slot += GC_GROUPS) {
    const int i = rank * rpc + slot;
    const CandIn in = nxt;
    {
      const int s2 = slot + GC_GROUPS, i2 = rank * rpc + s2;
      if (s2 < nslot) nxt = load_cand(s2 < rpc && i2 < R, i2, j, cand_offsets, parent, logq);
    }
    int d;
    const uint64_t key =
        score_gate_request(slot < rpc && i < R, i, j, in, sm.score[g], gp, path_score, cand_depth, cut_depth, status, d);
    sm.key[slot][j] = key;
    sm.par8[slot][j] = (int8_t)sm.score[g].par[j];  // (whatever it holds past the request's end is never read)
    sm.dep8[slot][j] = (uint8_t)d;
    __syncthreads();  // the group's scoring buffers are reused by its next request; at the end, all keys are in place
  }

  // ---- S3: threshold T = budget-th smallest key of the cluster's keys (unique => no ties to break) ----
  // A pass: every CTA histograms its own keys (2048 bins, and the sums of the 16 slices of 128 bins); after one
  // cluster barrier every CTA adds up the CL x 16 slice sums, finds the slice that holds the k-th key, adds up that
  // slice's CL x 128 bins and finds the bin -- the same decision everywhere, nothing to broadcast, and 8.5 KB instead
  // of 128 KB through distributed shared memory (which moves ~20 B a cycle per SM).
  const bool none = budget <= 0;
  uint64_t T = 0;
  if (!none) {
    uint64_t prefix = 0;
    int k = budget, shift = 64;
#pragma unroll 1
    for (int pass = 0;; ++pass) {
      const int bits = shift >= GC_BITS ? GC_BITS : shift;  // 11, 11, 11, 11, 11, 9
      const int hi = shift;                                 // bits [hi, 64) are decided: they equal `prefix`
      shift -= bits;
      int* h = sm.hist[pass & 1];
      int* hs = sm.slice[pass & 1];
      int* csum = sm.csum[pass & 1];
      int* tot = sm.tot[pass & 1];
#pragma unroll 1
      for (int slot = g; slot < nslot; slot += GC_GROUPS) {
        const uint64_t key = sm.key[slot][j];
        const bool in_prefix = key != KEY_INELIGIBLE && (pass == 0 || (key >> hi) == prefix);
        const int digit = in_prefix ? (int)((key >> shift) & ((1u << bits) - 1u)) : -1;
        // the top digits take one or two values: a warp that agrees on its digit adds it once
        const int d0 = __shfl_sync(0xffffffffu, digit, 0);
        if (__all_sync(0xffffffffu, digit == d0)) {
          if (lane == 0 && d0 >= 0) { atomicAdd(&h[d0], 32); atomicAdd(&hs[d0 / GC_SLICE], 32); }
        } else if (in_prefix) {
          atomicAdd(&h[digit], 1);
          atomicAdd(&hs[digit / GC_SLICE], 1);
        }
      }
      cluster.sync();  // every CTA's histogram of this pass is complete; the other set of buffers is no longer read
      sm.hist[(pass + 1) & 1][2 * tid] = 0;
      sm.hist[(pass + 1) & 1][2 * tid + 1] = 0;
      if (tid < GC_NSLICE) sm.slice[(pass + 1) & 1][tid] = sm.csum[(pass + 1) & 1][tid] = 0;
      if (tid < GC_SLICE) sm.tot[(pass + 1) & 1][tid] = 0;
      for (int t = tid; t < GC_NSLICE * CL; t += GC_THREADS) {
        const int v = *cluster.map_shared_rank(&hs[t % GC_NSLICE], t / GC_NSLICE);
        if (v) atomicAdd(&csum[t % GC_NSLICE], v);
      }
      __syncthreads();
      // every warp for itself: the slice that holds the k-th key
      const int v = lane < GC_NSLICE ? csum[lane] : 0;
      const int vincl = warp_incl_scan(v, lane);
      if (pass == 0 && __shfl_sync(0xffffffffu, vincl, 31) <= budget) {  // everything eligible (R:G-12)
        T = KEY_INELIGIBLE - 1;
        break;
      }
      const int owner = __ffs(__ballot_sync(0xffffffffu, vincl - v < k && k <= vincl)) - 1;  // exactly one lane
      const int below = __shfl_sync(0xffffffffu, vincl - v, owner);  // keys in the slices below
      for (int t = tid; t < GC_SLICE * CL; t += GC_THREADS) {
        const int c = *cluster.map_shared_rank(&h[owner * GC_SLICE + t % GC_SLICE], t / GC_SLICE);
        if (c) atomicAdd(&tot[t % GC_SLICE], c);
      }
      __syncthreads();
      if (warp == 0) {  // the bin inside the slice, four bins per lane
        const int4 c4 = *reinterpret_cast<const int4*>(&tot[4 * lane]);
        const int c[4] = {c4.x, c4.y, c4.z, c4.w};
        const int sum = c4.x + c4.y + c4.z + c4.w;
        int e = below + warp_incl_scan(sum, lane) - sum;
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          if (e < k && k <= e + c[t])  // exactly one lane and t: (bin << 32 | k inside the bin << 1 | whole bin taken)
            sm.found = ((uint64_t)(owner * GC_SLICE + 4 * lane + t) << 32) | ((uint64_t)(k - e) << 1) |
                       (uint64_t)(k - e == c[t]);
          e += c[t];
        }
      }
      __syncthreads();
      const uint64_t found = sm.found;
      prefix = (prefix << bits) | (found >> 32);
      k = (int)((found & 0xffffffffull) >> 1);
      if ((found & 1ull) || shift == 0) {
        // the whole bin is selected (lower digits do not matter), or every digit is decided: keys with the found
        // prefix and everything below it are selected; pad the undecided low digits with ones
        T = shift > 0 ? ((prefix << shift) | ((1ull << shift) - 1ull)) : prefix;
        break;
      }
    }
  }
  const uint64_t thr = none ? 0ull : T + 1ull;  // keys < thr are selected

  // ---- S4: per-request counts, CSR offsets (a scan over the CTA's requests, then over the cluster's CTAs) ----
#pragma unroll 1
  for (int slot = g; slot < GC_SLOTS; slot += GC_GROUPS) {
    const unsigned b = __ballot_sync(0xffffffffu, slot < nslot && sm.key[slot][j] < thr);
    if (lane == 0) sm.bal[slot][warp & 3] = b;
  }
  __syncthreads();
  if (warp == 0) {
    const int c = __popc(sm.bal[lane][0]) + __popc(sm.bal[lane][1]) + __popc(sm.bal[lane][2]) + __popc(sm.bal[lane][3]);
    const int incl = warp_incl_scan(c, lane);
    sm.cnt[lane] = incl;
    if (lane == 31) sm.cta_total = incl;
  }
  cluster.sync();
  if (warp == 0) {
    const int v = lane < CL ? *cluster.map_shared_rank(&sm.cta_total, lane) : 0;
    const int incl = warp_incl_scan(v, lane);
    const int base = rank ? __shfl_sync(0xffffffffu, incl, (rank + 31) & 31) : 0;
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    const int i = rank * rpc + lane;
    if (lane < rpc && i < R) sel_offsets[i + 1] = base + sm.cnt[lane];
    if (rank == 0 && lane == 0) {
      sel_offsets[0] = 0;
      *n_selected = total;
    }
    if (lane == 0) sm.base = base;
  }
  __syncthreads();
  cluster.barrier_arrive();  // this CTA has read the others' shared memory for the last time

  // ---- S4/S5: Flatten & Pack by the thread that made the key ----
#pragma unroll 1
  for (int slot = g; slot < nslot; slot += GC_GROUPS) {
    if (sm.key[slot][j] < thr) {
      uint32_t bal[4];
#pragma unroll
      for (int w = 0; w < 4; ++w) bal[w] = sm.bal[slot][w];
      const int8_t* par = sm.par8[slot];
      pack_node(rank * rpc + slot, j, sm.dep8[slot][j], bal, [&](int c) { return (int)par[c]; },
                sm.base + (slot ? sm.cnt[slot - 1] : 0), capacity, sel_node, sel_req, parent_local, sel_depth, anc_mask);
    }
  }
  cluster.barrier_wait();  // no CTA leaves while its shared memory may still be read
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

// Largest cluster of k_gate_cluster CTAs this device can place (16 needs the non-portable opt-in), probed once per
// context; 0 = none.
static int gate_cluster_max(EchoCtx* ctx) {
  if (ctx->gate_cluster_max != 0) return ctx->gate_cluster_max > 0 ? ctx->gate_cluster_max : 0;
  ctx->gate_cluster_max = -1;
  if (cudaFuncSetAttribute(k_gate_cluster, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ClusterSmem)) !=
      cudaSuccess) {
    (void)cudaGetLastError();
    return 0;
  }
  const bool np = cudaFuncSetAttribute(k_gate_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess;
  for (int cl = np ? 16 : 8; cl >= 1; cl /= 2) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cl);
    cfg.blockDim = dim3(GC_THREADS);
    cfg.dynamicSmemBytes = sizeof(ClusterSmem);
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cl;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, k_gate_cluster, &cfg) == cudaSuccess && n >= 1) {
      ctx->gate_cluster_max = cl;
      break;
    }
  }
  (void)cudaGetLastError();
  return ctx->gate_cluster_max > 0 ? ctx->gate_cluster_max : 0;
}

// Cluster size for R requests: eight requests per CTA and round; 0 when the cluster kernel cannot take the call.
static int gate_cluster_size(EchoCtx* ctx, int R) {
  const int cl_max = gate_cluster_max(ctx);
  if (cl_max == 0) return 0;
  int cl = 1;
  if (ctx->opt_gate_cluster > 0) cl = (int)ctx->opt_gate_cluster;
  else
    while (cl < cl_max && cl * GC_GROUPS < R) cl *= 2;
  if (cl > cl_max || (R + cl - 1) / cl > GC_SLOTS) return 0;
  return cl;
}

int launch_gate_select(EchoCtx* ctx, const EchoTrees* t, const EchoGate* g, EchoSelection* o, cudaStream_t st) {
  const int R = t->num_requests, N = t->total_cand;
  const int budget = g->static_k > 0 ? N : g->budget;
  const int cl = ctx->opt_gate_path == 1 ? 0 : gate_cluster_size(ctx, R);
  if (cl > 0) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cl);
    cfg.blockDim = dim3(GC_THREADS);
    cfg.dynamicSmemBytes = sizeof(ClusterSmem);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cl;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ECHO_COUNT_LAUNCH();
    ECHO_CUDA_TRY(ctx, cudaLaunchKernelEx(&cfg, k_gate_cluster, t->cand_offsets, t->parent, t->logq, gate_params(g), R,
                                          budget, o->capacity, o->path_score, o->cand_depth, o->cut_depth,
                                          o->n_selected, o->sel_offsets, o->sel_node, o->sel_req, o->parent_local,
                                          o->sel_depth, o->anc_mask, ctx->dev_status));
    return ECHO_OK;
  }
  if (ctx->opt_gate_path == 2) return ECHO_ERR_UNSUPPORTED;
  uint64_t* keys = reinterpret_cast<uint64_t*>(ctx->workspace);
  const size_t keys_bytes = align_up((size_t)N * sizeof(uint64_t), 256);
  if (keys_bytes + 256 > ctx->workspace_bytes) return ECHO_ERR_WORKSPACE;
  uint64_t* threshold = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(ctx->workspace) + keys_bytes);
  if (R > 0) {
    ECHO_COUNT_LAUNCH();
    k_score_gate<<<R, ECHO_MAX_CAND, 0, st>>>(t->cand_offsets, t->parent, t->logq, gate_params(g), o->path_score,
                                               o->cand_depth, o->cut_depth, keys, ctx->dev_status);
  }
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

// ---- echo_gate_select_noalloc (include/echo.h): the three-kernel chain with its scratch in the library image ----
// Scratch layout: [0, 8) the select threshold, [256, 256 + 8 N) the selection keys.  File-scope device array: every
// GPU that loads the library holds ECHO_NOALLOC_SCRATCH_BYTES until the process exits.  In HOST code the name below is
// a host-side stand-in, not a device address: the address a kernel may use comes from cudaGetSymbolAddress, looked up
// once per device with that device current.
static __device__ __align__(256) unsigned char g_noalloc_scratch[ECHO_NOALLOC_SCRATCH_BYTES];

#include <mutex>

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
struct NoallocDevice {
  std::atomic<int> state{0};  // 0 = not set up, 1 = ready, < 0 = the EchoStatus the set-up ended with
  unsigned char* scratch = nullptr;
};
NoallocDevice g_noalloc_dev[NOALLOC_MAX_DEVICES];
std::mutex g_noalloc_mutex;

// Set-up of the current device `dev`: architecture check and the scratch array's device address.  No allocation.
int noalloc_setup(int dev, unsigned char** scratch) {
  NoallocDevice& d = g_noalloc_dev[dev];
  int st = d.state.load(std::memory_order_acquire);
  if (st == 0) {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    st = d.state.load(std::memory_order_acquire);
    if (st == 0) {
      int major = 0, minor = 0;
      void* ptr = nullptr;
      if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
          cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess) {
        st = ECHO_ERR_CUDA;
      } else if (major != 10 || minor != 0) {
        st = ECHO_ERR_ARCH;
      } else if (cudaGetSymbolAddress(&ptr, g_noalloc_scratch) != cudaSuccess || ptr == nullptr) {
        st = ECHO_ERR_CUDA;
      } else {
        d.scratch = static_cast<unsigned char*>(ptr);
        st = 1;
      }
      (void)cudaGetLastError();
      if (st != ECHO_ERR_CUDA) d.state.store(st, std::memory_order_release);  // a CUDA failure may be transient: retried
    }
  }
  if (st != 1) return st;
  *scratch = d.scratch;
  return ECHO_OK;
}
}  // namespace

extern "C" int echo_gate_select_noalloc(const EchoTrees* t, const EchoGate* g, EchoSelection* o, uint32_t* status,
                                        echo_stream_t stream) {
  // the checks of echo_gate_select (api.cu), plus the scratch limit; nothing below allocates
  if (!t || !g || !o || !status) return ECHO_ERR_INVALID_ARG;
  if (t->num_requests < 0 || t->total_cand < 0 || t->max_cand_per_req < 0) return ECHO_ERR_INVALID_ARG;
  if (g->budget < 0 || g->w_max < 0 || g->static_k < 0 || o->capacity < 0) return ECHO_ERR_INVALID_ARG;
  if (g->cand_index_base < 0 || g->request_base < 0) return ECHO_ERR_INVALID_ARG;
  if (g->schedule != ECHO_SCHED_TOPB && g->schedule != ECHO_SCHED_ALG1) return ECHO_ERR_INVALID_ARG;
  if (t->max_cand_per_req > ECHO_MAX_CAND) return ECHO_ERR_UNSUPPORTED;
  if (g->schedule == ECHO_SCHED_ALG1 && (int64_t)g->request_base + t->num_requests > (1 << 24)) return ECHO_ERR_UNSUPPORTED;
  if (!t->cand_offsets || !o->cut_depth || !o->n_selected || !o->sel_offsets) return ECHO_ERR_INVALID_ARG;
  if (t->total_cand > 0 && (!t->parent || !t->logq || !o->path_score || !o->cand_depth)) return ECHO_ERR_INVALID_ARG;
  long need = g->static_k > 0 ? (long)t->num_requests * g->static_k : (long)g->budget;
  if (need > t->total_cand) need = t->total_cand;
  if (o->capacity < need) return ECHO_ERR_INVALID_ARG;
  if (o->capacity > 0 && (!o->sel_node || !o->sel_req || !o->parent_local || !o->sel_depth || !o->anc_mask))
    return ECHO_ERR_INVALID_ARG;
  if (reinterpret_cast<uintptr_t>(o->anc_mask) & 15u) return ECHO_ERR_INVALID_ARG;
  if (t->total_cand > ECHO_NOALLOC_MAX_CAND) return ECHO_ERR_TOO_LARGE;

  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NOALLOC_MAX_DEVICES) return ECHO_ERR_CUDA;
  unsigned char* scratch = nullptr;
  const int rc = noalloc_setup(dev, &scratch);
  if (rc != ECHO_OK) return rc;
  uint64_t* threshold = reinterpret_cast<uint64_t*>(scratch);
  uint64_t* keys = reinterpret_cast<uint64_t*>(scratch + 256);

  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const int R = t->num_requests, N = t->total_cand;
  const int budget = g->static_k > 0 ? N : g->budget;
  if (R > 0) {
    ECHO_COUNT_LAUNCH();
    k_score_gate<<<R, ECHO_MAX_CAND, 0, st>>>(t->cand_offsets, t->parent, t->logq, gate_params(g), o->path_score,
                                               o->cand_depth, o->cut_depth, keys, status);
  }
  if (launch_pdl(k_select, dim3(1), dim3(SEL_THREADS), 0, st, t->cand_offsets, keys, R, keys, N, budget, o->n_selected,
                 o->sel_offsets, threshold) != cudaSuccess)
    return ECHO_ERR_CUDA;
  if (R > 0 &&
      launch_pdl(k_pack, dim3(R), dim3(ECHO_MAX_CAND), 0, st, t->cand_offsets, t->parent, o->cand_depth, keys, threshold,
                 o->capacity, o->sel_offsets, o->sel_node, o->sel_req, o->parent_local, o->sel_depth, o->anc_mask) !=
          cudaSuccess)
    return ECHO_ERR_CUDA;
  return cudaGetLastError() == cudaSuccess ? ECHO_OK : ECHO_ERR_CUDA;
}
