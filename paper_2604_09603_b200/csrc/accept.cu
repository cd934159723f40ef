// echo_accept: S8 (bf16 argmax over the vocabulary), S9 (greedy acceptance = longest accepted
// root-to-leaf path) and S10 (in-place KV-slot compaction, R:C-6).
#include "common.cuh"

namespace {

constexpr int D = 128;
constexpr int PAGE = 16;

__device__ __forceinline__ uint4 ldg_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// (value, index) with "greater value, then lower index" order; -0 == +0 by float compare (R:C-3)
__device__ __forceinline__ void amax_upd(float& bv, int& bi, float v, int i) {
  if (v > bv || (v == bv && i < bi)) { bv = v; bi = i; }
}

__device__ __forceinline__ void amax_chunk(float& bv, int& bi, const uint4 u, int base) {
  // ascending index with strict '>' keeps the first maximum
  const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const float lo = __uint_as_float(w[c] << 16), hi = __uint_as_float(w[c] & 0xffff0000u);
    if (lo > bv) { bv = lo; bi = base + 2 * c; }
    if (hi > bv) { bv = hi; bi = base + 2 * c + 1; }
  }
}

constexpr int AM_THREADS = 256;
constexpr int AM_UNROLL = 4;

// S8: one CTA per packed node row; 16-byte streaming loads, 4 in flight per thread.
__global__ void __launch_bounds__(AM_THREADS) k_argmax_bf16(const int32_t* __restrict__ n_selected,
                                                            const __nv_bfloat16* __restrict__ logits, int64_t ld,
                                                            int vocab, int32_t* __restrict__ target_token) {
  const int row = blockIdx.x;
  if (row >= *n_selected) return;
  const __nv_bfloat16* rp = logits + (size_t)row * ld;
  const uint4* rp4 = reinterpret_cast<const uint4*>(rp);
  const int nvec = vocab / 8;
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  int v = threadIdx.x;
  for (; v + (AM_UNROLL - 1) * AM_THREADS < nvec; v += AM_UNROLL * AM_THREADS) {
    uint4 u[AM_UNROLL];
#pragma unroll
    for (int t = 0; t < AM_UNROLL; ++t) u[t] = ldg_stream(rp4 + v + t * AM_THREADS);
#pragma unroll
    for (int t = 0; t < AM_UNROLL; ++t) amax_chunk(bv, bi, u[t], (v + t * AM_THREADS) * 8);
  }
  for (; v < nvec; v += AM_THREADS) amax_chunk(bv, bi, ldg_stream(rp4 + v), v * 8);
  for (int c = nvec * 8 + threadIdx.x; c < vocab; c += AM_THREADS) {
    const float x = __bfloat162float(rp[c]);
    if (x > bv) { bv = x; bi = c; }
  }
  // an all -inf (or empty) slice leaves bi at INT_MAX; the tie rule then picks any real index
#pragma unroll
  for (int ofs = 16; ofs; ofs >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, bv, ofs);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, ofs);
    amax_upd(bv, bi, ov, oi);
  }
  __shared__ float s_v[AM_THREADS / 32];
  __shared__ int s_i[AM_THREADS / 32];
  if ((threadIdx.x & 31) == 0) { s_v[threadIdx.x >> 5] = bv; s_i[threadIdx.x >> 5] = bi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < AM_THREADS / 32; ++w) amax_upd(bv, bi, s_v[w], s_i[w]);
    if (bi == 0x7fffffff) bi = 0;  // every logit is -inf: first index (all-equal row => 0)
    target_token[row] = bi;
  }
}

// ---- S8 over vocabulary-sharded logits (tensor-parallel ranks) ----
// Each rank holds the columns [vocab_base, vocab_base + vocab_shard) of every logits row.  Its partial result per row
// is ONE 64-bit key = (order-preserving image of the shard's maximum, -0 canonicalised to +0) << 32 | (INT32_MAX -
// global index of its first occurrence): the larger key is the greater value, then the lower index (R:C-3), so the
// argmax over the whole vocabulary is the maximum of the ranks' keys -- one all-gather of rows x 8 B per rank.
__device__ __forceinline__ uint64_t amax_key(float v, int global_index) {
  return ((uint64_t)f32_ordered(v + 0.0f) << 32) | (uint64_t)(uint32_t)(0x7fffffff - global_index);
}

__global__ void __launch_bounds__(AM_THREADS) k_argmax_shard(const int32_t* __restrict__ n_selected,
                                                             const __nv_bfloat16* __restrict__ logits, int64_t ld,
                                                             int vocab_shard, int vocab_base,
                                                             unsigned long long* __restrict__ pairs) {
  const int row = blockIdx.x;
  if (row >= *n_selected) {  // rows past the packed nodes: a defined value in the buffer that is gathered
    if (threadIdx.x == 0) pairs[row] = 0ull;
    return;
  }
  const __nv_bfloat16* rp = logits + (size_t)row * ld;
  const uint4* rp4 = reinterpret_cast<const uint4*>(rp);
  const int nvec = vocab_shard / 8;
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  int v = threadIdx.x;
  for (; v + (AM_UNROLL - 1) * AM_THREADS < nvec; v += AM_UNROLL * AM_THREADS) {
    uint4 u[AM_UNROLL];
#pragma unroll
    for (int t = 0; t < AM_UNROLL; ++t) u[t] = ldg_stream(rp4 + v + t * AM_THREADS);
#pragma unroll
    for (int t = 0; t < AM_UNROLL; ++t) amax_chunk(bv, bi, u[t], (v + t * AM_THREADS) * 8);
  }
  for (; v < nvec; v += AM_THREADS) amax_chunk(bv, bi, ldg_stream(rp4 + v), v * 8);
  for (int c = nvec * 8 + threadIdx.x; c < vocab_shard; c += AM_THREADS) {
    const float x = __bfloat162float(rp[c]);
    if (x > bv) { bv = x; bi = c; }
  }
#pragma unroll
  for (int ofs = 16; ofs; ofs >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, bv, ofs);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, ofs);
    amax_upd(bv, bi, ov, oi);
  }
  __shared__ float s_v[AM_THREADS / 32];
  __shared__ int s_i[AM_THREADS / 32];
  if ((threadIdx.x & 31) == 0) { s_v[threadIdx.x >> 5] = bv; s_i[threadIdx.x >> 5] = bi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < AM_THREADS / 32; ++w) amax_upd(bv, bi, s_v[w], s_i[w]);
    if (bi == 0x7fffffff) bi = 0;  // every logit of the shard is -inf: its first index
    pairs[row] = amax_key(bv, vocab_base + bi);
  }
}

// target_token[row] = index held by the largest of the `world` keys of the row (pairs_all [world][capacity])
constexpr int MG_THREADS = 128;
__global__ void __launch_bounds__(MG_THREADS) k_argmax_merge(const int32_t* __restrict__ n_selected,
                                                             const unsigned long long* __restrict__ pairs_all,
                                                             int world, int capacity,
                                                             int32_t* __restrict__ target_token) {
  const int row = blockIdx.x * MG_THREADS + threadIdx.x;
  if (row >= capacity || row >= *n_selected) return;
  unsigned long long best = 0ull;
  for (int w = 0; w < world; ++w) {
    const unsigned long long k = pairs_all[(size_t)w * capacity + row];
    best = k > best ? k : best;
  }
  target_token[row] = 0x7fffffff - (int)(uint32_t)(best & 0xffffffffull);
}

constexpr int AC_THREADS = 128;

// S9 + S10: one CTA per request.  Warp 0 decides the path; then every thread owns a column of
// 16-byte chunks (layer, K|V, KV head, chunk) and moves it for path node t = 0,1,... in order:
// sources are strictly increasing and src_t >= dst_t, so within a column every read of a slot
// happens before the write that could overwrite it (R:C-6).
__global__ void __launch_bounds__(AC_THREADS) k_accept_compact(
    const int32_t* __restrict__ sel_offsets, const int32_t* __restrict__ parent_local,
    const uint8_t* __restrict__ sel_depth, const uint32_t* __restrict__ anc_mask,
    const int32_t* __restrict__ draft_token, const int32_t* __restrict__ prev_token,
    const int32_t* __restrict__ target_token, const int32_t* __restrict__ page_table,
    const int32_t* __restrict__ prefix_len, int max_pages, int Hkv, int num_pages, int num_layers,
    __nv_bfloat16* __restrict__ k_pool, __nv_bfloat16* __restrict__ v_pool, int32_t* __restrict__ accept_len,
    int32_t* __restrict__ last_node, int32_t* __restrict__ bonus_token, int32_t* __restrict__ new_len,
    int32_t* __restrict__ accept_idx, int32_t* __restrict__ slot_src, int32_t* __restrict__ slot_dst) {
  __shared__ int s_L;
  __shared__ int s_src[ECHO_MAX_ACCEPT], s_dst[ECHO_MAX_ACCEPT];
  const int i = blockIdx.x;
  // what the caller owns (not written by this step's kernels) is loaded while the attention kernel drains
  const int P = prefix_len[i];
  const int prev = prev_token[i];
  pdl_wait();  // the attention kernel before this one reads the pools this kernel compacts in place
  const int b = sel_offsets[i], Ki = min(sel_offsets[i + 1] - b, ECHO_MAX_CAND);
  const int32_t* pt = page_table + (size_t)i * max_pages;
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    // every load of the decision is issued before the first one is used: one memory round trip, then one more for
    // the parents' target tokens
    int pl[4], dr[4], dep[4];
    uint4 am[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const int l = w * 32 + lane;
      pl[w] = -1; dr[w] = 0; dep[w] = 0; am[w] = make_uint4(0u, 0u, 0u, 0u);
      if (l < Ki) {
        pl[w] = parent_local[b + l];
        dr[w] = draft_token[b + l];
        dep[w] = sel_depth[b + l];
        am[w] = reinterpret_cast<const uint4*>(anc_mask)[b + l];
      }
    }
    // match[l]: draft token equals the target's greedy token after the parent (roots: prev_token)
    uint32_t match[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const int l = w * 32 + lane;
      bool mt = false;
      if (l < Ki) mt = dr[w] == (pl[w] < 0 ? prev : target_token[b + pl[w]]);
      match[w] = __ballot_sync(0xffffffffu, mt);
    }
    // acc[l] <=> every ancestor-or-self matches; best = max depth, then lowest l (R:C-4)
    int best_key = -1;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const int l = w * 32 + lane;
      if (l < Ki) {
        const uint4 m = am[w];
        const bool acc = !((m.x & ~match[0]) | (m.y & ~match[1]) | (m.z & ~match[2]) | (m.w & ~match[3]));
        if (acc) best_key = max(best_key, (dep[w] << 8) | (ECHO_MAX_CAND - 1 - l));
      }
    }
#pragma unroll
    for (int ofs = 16; ofs; ofs >>= 1) best_key = max(best_key, __shfl_xor_sync(0xffffffffu, best_key, ofs));
    int L = 0;
    if (best_key >= 0) {
      const int best = ECHO_MAX_CAND - 1 - (best_key & 0xff);
      uint4 m = (best >> 5) == 0 ? am[0] : (best >> 5) == 1 ? am[1] : (best >> 5) == 2 ? am[2] : am[3];  // warp-uniform
      m.x = __shfl_sync(0xffffffffu, m.x, best & 31); m.y = __shfl_sync(0xffffffffu, m.y, best & 31);
      m.z = __shfl_sync(0xffffffffu, m.z, best & 31); m.w = __shfl_sync(0xffffffffu, m.w, best & 31);
      const uint32_t mw[4] = {m.x, m.y, m.z, m.w};
      L = min(__popc(m.x) + __popc(m.y) + __popc(m.z) + __popc(m.w), ECHO_MAX_ACCEPT);
      // lane t finds the t-th set bit (path order = ascending local index, R:P-1)
      int a = -1;
      if (lane < L) {
        int need = lane;
#pragma unroll
        for (int w = 0; w < 4; ++w) {
          const int c = __popc(mw[w]);
          if (a < 0) {
            if (need < c) a = w * 32 + __fns(mw[w], 0, need + 1);
            else need -= c;
          }
        }
      }
      if (lane < ECHO_MAX_ACCEPT) {
        int src = -1, dst = -1, idx = -1;
        if (lane < L) {
          const int sp = P + a, dp = P + lane;
          src = pt[sp / PAGE] * PAGE + sp % PAGE;
          dst = pt[dp / PAGE] * PAGE + dp % PAGE;
          idx = b + a;
        }
        accept_idx[i * ECHO_MAX_ACCEPT + lane] = idx;
        slot_src[i * ECHO_MAX_ACCEPT + lane] = src;
        slot_dst[i * ECHO_MAX_ACCEPT + lane] = dst;
        s_src[lane] = src;
        s_dst[lane] = dst;
      }
      if (lane == 0) { last_node[i] = b + best; bonus_token[i] = target_token[b + best]; }
    } else {
      accept_idx[i * ECHO_MAX_ACCEPT + lane] = -1;
      slot_src[i * ECHO_MAX_ACCEPT + lane] = -1;
      slot_dst[i * ECHO_MAX_ACCEPT + lane] = -1;
      if (lane == 0) { last_node[i] = -1; bonus_token[i] = -1; }
    }
    if (lane == 0) { accept_len[i] = L; new_len[i] = P + L; s_L = L; }
  }
  __syncthreads();
  const int L = s_L;
  if (L == 0 || k_pool == nullptr) return;
  // columns: (layer, kv in {K,V}, head, 16-byte chunk of the 256-byte row)
  const int n_cols = num_layers * 2 * Hkv * (D * 2 / 16);
  for (int col = threadIdx.x; col < n_cols; col += AC_THREADS) {
    const int chunk = col % 16;
    const int head = (col / 16) % Hkv;
    const int kvsel = (col / (16 * Hkv)) % 2;
    const int layer = col / (32 * Hkv);
    __nv_bfloat16* pool = kvsel ? v_pool : k_pool;
    uint4* base = reinterpret_cast<uint4*>(pool + (size_t)layer * num_pages * Hkv * PAGE * D);
    // No destination of an earlier move is the source of a later one (src position P + a_t with a_t >= t, dst
    // position P + t' with t' < t), so the loads of a batch of moves are issued together, then its stores: one
    // memory round trip per 8 moves instead of one per move.
    auto row_ofs = [&](int slot) -> size_t {
      return (((size_t)(slot / PAGE) * Hkv + head) * PAGE + (slot % PAGE)) * (D * 2 / 16) + chunk;
    };
    for (int t0 = 0; t0 < L; t0 += 8) {
      uint4 v[8];
#pragma unroll
      for (int e = 0; e < 8; ++e)
        if (t0 + e < L && s_src[t0 + e] != s_dst[t0 + e]) v[e] = base[row_ofs(s_src[t0 + e])];
#pragma unroll
      for (int e = 0; e < 8; ++e)
        if (t0 + e < L && s_src[t0 + e] != s_dst[t0 + e]) base[row_ofs(s_dst[t0 + e])] = v[e];
    }
  }
}

}  // namespace

int launch_accept(EchoCtx* ctx, const EchoSelection* sel, const EchoVerifyResult* res, int32_t R, EchoPagedKV* kv,
                  EchoAccept* out, cudaStream_t st) {
  const int32_t* tt = res->target_token;
  if (res->target_logits) {
    int32_t* tout = out->target_token_out ? out->target_token_out : reinterpret_cast<int32_t*>(ctx->workspace);
    if (!out->target_token_out && (size_t)sel->capacity * sizeof(int32_t) > ctx->workspace_bytes)
      return ECHO_ERR_WORKSPACE;
    if (sel->capacity > 0) {  // (an empty grid is a launch error)
      ECHO_COUNT_LAUNCH();
      k_argmax_bf16<<<sel->capacity, AM_THREADS, 0, st>>>(
          sel->n_selected, reinterpret_cast<const __nv_bfloat16*>(res->target_logits), res->ld, res->vocab, tout);
    }
    tt = tout;
  }
  if (R > 0) {
    const bool have_pools = kv->k_pool && kv->v_pool;  // NULL pools: slot maps only, no copy
    ECHO_CUDA_TRY(ctx, launch_pdl(k_accept_compact, dim3(R), dim3(AC_THREADS), 0, st,
        sel->sel_offsets, sel->parent_local, sel->sel_depth, sel->anc_mask, res->draft_token, res->prev_token, tt,
        kv->page_table, kv->prefix_len, kv->max_pages_per_req, kv->num_kv_heads, kv->num_pages, kv->num_layers,
        have_pools ? reinterpret_cast<__nv_bfloat16*>(kv->k_pool) : (__nv_bfloat16*)nullptr,
        have_pools ? reinterpret_cast<__nv_bfloat16*>(kv->v_pool) : (__nv_bfloat16*)nullptr, out->accept_len, out->last_node,
        out->bonus_token, out->new_len, out->accept_idx, out->slot_src, out->slot_dst));
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}

int launch_argmax_shard(EchoCtx* ctx, const EchoSelection* sel, const void* logits, int64_t ld, int32_t vocab_shard,
                        int32_t vocab_base, uint64_t* pairs, cudaStream_t st) {
  if (sel->capacity > 0) {
    ECHO_COUNT_LAUNCH();
    k_argmax_shard<<<sel->capacity, AM_THREADS, 0, st>>>(sel->n_selected, reinterpret_cast<const __nv_bfloat16*>(logits), ld,
                                                         vocab_shard, vocab_base,
                                                         reinterpret_cast<unsigned long long*>(pairs));
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}

int launch_argmax_merge(EchoCtx* ctx, const EchoSelection* sel, const uint64_t* pairs_all, int32_t world,
                        int32_t* target_token, cudaStream_t st) {
  if (sel->capacity > 0) {
    ECHO_COUNT_LAUNCH();
    k_argmax_merge<<<(sel->capacity + MG_THREADS - 1) / MG_THREADS, MG_THREADS, 0, st>>>(
        sel->n_selected, reinterpret_cast<const unsigned long long*>(pairs_all), world, sel->capacity, target_token);
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}
