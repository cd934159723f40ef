// echo_accept_stochastic: tree acceptance at temperature > 0 (include/echo.h; paper: "accepting
// a prefix", "speculative sampling acceptance conditions"; readings R:T-1..T-4 of DESIGN.md).
//   k_softmax_stats : one CTA per logits row (the packed nodes' rows and the R root rows): running maximum M and
//                     Z = sum 2^((l - M) c), c = log2(e) / T, in one pass of 16-byte streaming loads.  The second
//                     vocabulary-wide HBM-bound kernel of the library (1.25 GB at cfg4, next to k_argmax_bf16).
//   k_walk_sample   : one CTA per request.  Warp 0 walks the tree: the children of the current node are found by
//                     ballot, their target probabilities gathered in parallel (lane = child), the accept / reject
//                     sequence run in packed order with the rejected mass removed and renormalised.  Then the whole
//                     CTA draws the bonus token from the residual distribution of the last node by inverse CDF in
//                     vocabulary order (segments of 256 tokens reduced by coalesced warp loads, warp 0 scans the
//                     segment sums and resolves the segment), and compacts the accepted KV rows like echo_accept.
#include "common.cuh"

namespace {

constexpr int D = 128;
constexpr int PAGE = 16;
constexpr int ST_THREADS = 256;
constexpr int ST_UNROLL = 4;
constexpr int WS_THREADS = 256;
constexpr int SEG = 256;        // tokens per CDF segment: one coalesced warp load
constexpr int MAX_SEGS = 1024;  // vocabulary <= 262 144

__device__ __forceinline__ uint4 ldg_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ float ex2f(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

// (m, z) <- merge with (om, oz): z counts 2^((l - m) c)
// A side whose maximum is -inf (every logit masked, e.g. banned tokens) holds no mass: without the early return
// (-inf) - (-inf) = NaN would reach ex2 and poison Z.
__device__ __forceinline__ void mz_merge(float& m, float& z, float om, float oz, float c) {
  if (om == -INFINITY) return;
  if (om > m) { z = (m == -INFINITY ? 0.f : z * ex2f((m - om) * c)) + oz; m = om; }
  else if (oz > 0.f) z += oz * ex2f((om - m) * c);
}
__device__ __forceinline__ void mz_chunk(float& m, float& z, const uint4 u, float c) {
  const uint32_t w[4] = {u.x, u.y, u.z, u.w};
  float x[8], cm = -INFINITY;
#pragma unroll
  for (int q = 0; q < 4; ++q) { x[2 * q] = bf16_lo(w[q]); x[2 * q + 1] = bf16_hi(w[q]); }
#pragma unroll
  for (int q = 0; q < 8; ++q) cm = fmaxf(cm, x[q]);
  if (cm == -INFINITY) return;  // eight masked logits add nothing (and (-inf) - (-inf) would be NaN below)
  if (cm > m) { z = m == -INFINITY ? 0.f : z * ex2f((m - cm) * c); m = cm; }
#pragma unroll
  for (int q = 0; q < 8; ++q) z += ex2f((x[q] - m) * c);
}

__global__ void __launch_bounds__(ST_THREADS) k_softmax_stats(const int32_t* __restrict__ n_selected, int cap, int R,
                                                              const __nv_bfloat16* __restrict__ target_logits,
                                                              const __nv_bfloat16* __restrict__ root_logits, int64_t ld,
                                                              int vocab, float c, float2* __restrict__ stats) {
  const int row = blockIdx.x;
  pdl_launch_dependents();
  pdl_wait();
  if (row < cap && row >= *n_selected) return;
  const __nv_bfloat16* rp = row < cap ? target_logits + (size_t)row * ld : root_logits + (size_t)(row - cap) * ld;
  const uint4* rp4 = reinterpret_cast<const uint4*>(rp);
  const int nvec = vocab / 8;
  float m = -INFINITY, z = 0.f;
  int v = threadIdx.x;
  for (; v + (ST_UNROLL - 1) * ST_THREADS < nvec; v += ST_UNROLL * ST_THREADS) {
    uint4 u[ST_UNROLL];
#pragma unroll
    for (int t = 0; t < ST_UNROLL; ++t) u[t] = ldg_stream(rp4 + v + t * ST_THREADS);
#pragma unroll
    for (int t = 0; t < ST_UNROLL; ++t) mz_chunk(m, z, u[t], c);
  }
  for (; v < nvec; v += ST_THREADS) mz_chunk(m, z, ldg_stream(rp4 + v), c);
  for (int q = nvec * 8 + threadIdx.x; q < vocab; q += ST_THREADS) mz_merge(m, z, __bfloat162float(rp[q]), 1.f, c);
#pragma unroll
  for (int ofs = 16; ofs; ofs >>= 1) {
    const float om = __shfl_xor_sync(0xffffffffu, m, ofs), oz = __shfl_xor_sync(0xffffffffu, z, ofs);
    mz_merge(m, z, om, oz, c);
  }
  __shared__ float s_m[ST_THREADS / 32], s_z[ST_THREADS / 32];
  if ((threadIdx.x & 31) == 0) { s_m[threadIdx.x >> 5] = m; s_z[threadIdx.x >> 5] = z; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < ST_THREADS / 32; ++w) mz_merge(m, z, s_m[w], s_z[w], c);
    stats[row] = make_float2(m, z);
  }
}

__global__ void __launch_bounds__(WS_THREADS) k_walk_sample(
    const int32_t* __restrict__ sel_offsets, const int32_t* __restrict__ parent_local,
    const int32_t* __restrict__ draft_token, const __nv_bfloat16* __restrict__ target_logits,
    const __nv_bfloat16* __restrict__ root_logits, int64_t ld, int vocab, int cap, float c, float c_lo,
    const float2* __restrict__ stats, const float* __restrict__ u_accept, const float* __restrict__ u_bonus,
    const int32_t* __restrict__ page_table, const int32_t* __restrict__ prefix_len, int max_pages, int Hkv,
    int num_pages, int num_layers, __nv_bfloat16* __restrict__ k_pool, __nv_bfloat16* __restrict__ v_pool,
    int32_t* __restrict__ accept_len, int32_t* __restrict__ last_node, int32_t* __restrict__ bonus_token,
    int32_t* __restrict__ new_len, int32_t* __restrict__ accept_idx, int32_t* __restrict__ slot_src,
    int32_t* __restrict__ slot_dst) {
  __shared__ int s_path[ECHO_MAX_ACCEPT], s_src[ECHO_MAX_ACCEPT], s_dst[ECHO_MAX_ACCEPT];
  __shared__ int s_removed[ECHO_MAX_CAND];
  __shared__ int s_L, s_cur, s_nrem, s_pick_seg;
  __shared__ double s_prefix, s_target;
  __shared__ float s_seg[MAX_SEGS];
  pdl_wait();  // statistics come from k_softmax_stats; the attention kernel before it reads the pools compacted below
  const int i = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
  const int b = sel_offsets[i], Ki = min(sel_offsets[i + 1] - b, ECHO_MAX_CAND);
  const int P = prefix_len[i];

  if (tid < 32) {
    // ---- the walk (R:T-1..T-3): every lane runs the same control flow, lane = child for the gathers ----
    int cur = -1, L = 0, nrem = 0;
    float remw = 0.f;
    int pl[4], tok[4];  // this lane's four packed nodes: loaded once, so that a level costs one gather round trip
    float ua[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const int l = w * 32 + lane;
      pl[w] = l < Ki ? parent_local[b + l] : -2;
      tok[w] = l < Ki ? draft_token[b + l] : -1;
      ua[w] = l < Ki ? u_accept[b + l] : 2.f;
    }
    while (true) {
      const float2 mz = cur < 0 ? stats[cap + i] : stats[b + cur];
      const __nv_bfloat16* rowp = cur < 0 ? root_logits + (size_t)i * ld : target_logits + (size_t)(b + cur) * ld;
      nrem = 0;
      remw = 0.f;
      int accepted = -1;
      float wgt[4];
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        const bool tok_ok = pl[w] == cur && tok[w] >= 0 && tok[w] < vocab;
        wgt[w] = tok_ok ? ex2f((__bfloat162float(rowp[tok[w]]) - mz.x) * c) : 0.f;
      }
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        if (accepted >= 0) break;
        const bool is_child = pl[w] == cur;
        const int x = is_child ? tok[w] : -1;
        const float u = is_child ? ua[w] : 2.f;
        unsigned cm = __ballot_sync(0xffffffffu, is_child);
        while (cm) {
          const int j = __ffs(cm) - 1;
          cm &= cm - 1;
          const int xj = __shfl_sync(0xffffffffu, x, j);
          const float wj = __shfl_sync(0xffffffffu, wgt[w], j), uj = __shfl_sync(0xffffffffu, u, j);
          bool dup = false;
          for (int r = 0; r < nrem; ++r) dup |= s_removed[r] == xj;
          const float px = dup ? 0.f : wj;
          const float denom = mz.y - remw;
          const float pr = denom > 0.f ? px / denom : 0.f;
          if (uj < pr) { accepted = w * 32 + j; break; }
          if (!dup && xj >= 0 && xj < vocab) {  // a token outside the vocabulary is never accepted and removes nothing
            if (lane == 0) s_removed[nrem] = xj;
            ++nrem;
            remw += wj;
            __syncwarp();
          }
        }
      }
      if (accepted < 0 || L >= ECHO_MAX_ACCEPT) break;
      if (lane == 0) s_path[L] = accepted;
      ++L;
      cur = accepted;
    }
    if (lane == 0) { s_L = L; s_cur = cur; s_nrem = nrem; }
    __syncwarp();
    // slot maps, as echo_accept writes them: path node t moves from position P + a_t to P + t (R:C-6)
    if (lane < ECHO_MAX_ACCEPT) {
      int src = -1, dst = -1, idx = -1;
      if (lane < L) {
        const int32_t* pt = page_table + (size_t)i * max_pages;
        const int a = s_path[lane], sp = P + a, dp = P + lane;
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
    if (lane == 0) { accept_len[i] = L; new_len[i] = P + L; last_node[i] = cur < 0 ? -1 : b + cur; }
  }
  __syncthreads();

  // ---- bonus token from the residual distribution of the last node, inverse CDF in vocabulary order (R:T-4) ----
  // Segments of 256 consecutive tokens: a warp loads one with 32 coalesced 16-byte loads and reduces it to one sum;
  // warp 0 scans the <= 1024 segment sums to the segment that holds the draw and resolves it inside.  The draw is
  // compared with the kernel's OWN total of the residual weights (not with Z of k_softmax_stats, which is summed in
  // another order), the scans run in fp64 and the exponent argument uses c split in two floats, so that the CDF the
  // draw is inverted on is within ~3e-7 of the exact one (ex2.approx: 2^-22 per weight, pseudo-random in sign).
  {
    const int cur = s_cur, nrem = s_nrem, warp = tid >> 5;
    const float2 mz = cur < 0 ? stats[cap + i] : stats[b + cur];
    const __nv_bfloat16* rowp = cur < 0 ? root_logits + (size_t)i * ld : target_logits + (size_t)(b + cur) * ld;
    const int nseg = (vocab + SEG - 1) / SEG;
    auto wgt = [&](float x) { const float d = x - mz.x; return ex2f(fmaf(d, c, d * c_lo)); };
    auto load8 = [&](int base, float (&w)[8]) {  // weights of tokens base .. base+7 (0 past the vocabulary)
      if (base + 8 <= vocab) {
        const uint4 u = ldg_stream(reinterpret_cast<const uint4*>(rowp + base));
        const uint32_t q[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          w[2 * e] = wgt(bf16_lo(q[e]));
          w[2 * e + 1] = wgt(bf16_hi(q[e]));
        }
      } else {
#pragma unroll
        for (int e = 0; e < 8; ++e) w[e] = base + e < vocab ? wgt(__bfloat162float(rowp[base + e])) : 0.f;
      }
    };
    constexpr int NW = WS_THREADS / 32, UNR = 8;
    for (int s0 = warp; s0 < nseg; s0 += UNR * NW) {  // eight segments' loads in flight per warp
      uint4 u[UNR];
#pragma unroll
      for (int t = 0; t < UNR; ++t) {
        const int base = (s0 + t * NW) * SEG + lane * 8;
        u[t] = make_uint4(0u, 0u, 0u, 0u);
        if (base + 8 <= vocab) u[t] = ldg_stream(reinterpret_cast<const uint4*>(rowp + base));
      }
#pragma unroll
      for (int t = 0; t < UNR; ++t) {
        const int sgm = s0 + t * NW, base = sgm * SEG + lane * 8;
        if (sgm >= nseg) break;  // warp-uniform
        float w[8];
        if (base + 8 <= vocab) {
          const uint32_t q[4] = {u[t].x, u[t].y, u[t].z, u[t].w};
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            w[2 * e] = wgt(bf16_lo(q[e]));
            w[2 * e + 1] = wgt(bf16_hi(q[e]));
          }
        } else {
          load8(base, w);
        }
        float sum = ((w[0] + w[1]) + (w[2] + w[3])) + ((w[4] + w[5]) + (w[6] + w[7]));
#pragma unroll
        for (int ofs = 16; ofs; ofs >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, ofs);
        if (lane == 0) s_seg[sgm] = sum;
      }
    }
    __syncthreads();
    if (tid < nrem) atomicAdd(&s_seg[s_removed[tid] / SEG], -wgt(__bfloat162float(rowp[s_removed[tid]])));
    __syncthreads();
    if (tid < 32) {  // lane = a run of consecutive segments; warp scan of the runs, then the owning lane walks its run
      const int per = (nseg + 31) / 32, l0 = min(nseg, lane * per), l1 = min(nseg, l0 + per);
      double mine = 0.0;
      for (int sgm = l0; sgm < l1; ++sgm) mine += (double)fmaxf(s_seg[sgm], 0.f);
      double incl = mine;
#pragma unroll
      for (int ofs = 1; ofs < 32; ofs <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, incl, ofs);
        if (lane >= ofs) incl += t;
      }
      const double total = __shfl_sync(0xffffffffu, incl, 31);
      const double target = (double)u_bonus[i] * total;
      const double before = incl - mine;
      const unsigned hit = __ballot_sync(0xffffffffu, mine > 0.0 && before + mine > target);
      const unsigned pos = __ballot_sync(0xffffffffu, mine > 0.0);
      const int owner = hit ? __ffs(hit) - 1 : (pos ? 31 - __clz(pos) : 0);  // past the end by rounding: last mass
      if (lane == owner) {
        double run = before;
        int pick = -1, last_pos = l0;
        for (int sgm = l0; sgm < l1; ++sgm) {
          const double w = (double)fmaxf(s_seg[sgm], 0.f);
          if (w > 0.0) last_pos = sgm;
          if (run + w > target) { pick = sgm; break; }
          run += w;
        }
        s_prefix = pick >= 0 ? run : -INFINITY;
        s_pick_seg = pick >= 0 ? pick : last_pos;
        s_target = target;
      }
    }
    __syncthreads();
    if (tid < 32) {
      const int base = s_pick_seg * SEG + lane * 8;
      const double target = s_target;
      float w[8];
      load8(base, w);
#pragma unroll
      for (int e = 0; e < 8; ++e)
        for (int r = 0; r < nrem; ++r)
          if (s_removed[r] == base + e) w[e] = 0.f;
      const double mine = (double)(((w[0] + w[1]) + (w[2] + w[3])) + ((w[4] + w[5]) + (w[6] + w[7])));
      double incl = mine;
#pragma unroll
      for (int ofs = 1; ofs < 32; ofs <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, incl, ofs);
        if (lane >= ofs) incl += t;
      }
      const double before = s_prefix + (incl - mine);
      int pick = -1, last_nz = -1;
      double acc = before;
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        if (w[e] > 0.f) last_nz = base + e;
        acc += (double)w[e];
        if (pick < 0 && w[e] > 0.f && acc > target) pick = base + e;
      }
      const unsigned found = __ballot_sync(0xffffffffu, pick >= 0);
      const unsigned nz = __ballot_sync(0xffffffffu, last_nz >= 0);
      int out_tok;
      if (found) out_tok = __shfl_sync(0xffffffffu, pick, __ffs(found) - 1);
      else out_tok = nz ? __shfl_sync(0xffffffffu, last_nz, 31 - __clz(nz)) : 0;
      if (lane == 0) bonus_token[i] = out_tok;
    }
  }

  // ---- compaction of the accepted KV rows (same moves as k_accept_compact) ----
  const int L = s_L;
  if (L == 0 || k_pool == nullptr) return;
  const int n_cols = num_layers * 2 * Hkv * (D * 2 / 16);
  for (int col = tid; col < n_cols; col += WS_THREADS) {
    const int chunk = col % 16;
    const int head = (col / 16) % Hkv;
    const int kvsel = (col / (16 * Hkv)) % 2;
    const int layer = col / (32 * Hkv);
    __nv_bfloat16* pool = kvsel ? v_pool : k_pool;
    uint4* base = reinterpret_cast<uint4*>(pool + (size_t)layer * num_pages * Hkv * PAGE * D);
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

int launch_accept_stochastic(EchoCtx* ctx, const EchoSelection* sel, const EchoSampleInputs* in, int32_t R,
                             EchoPagedKV* kv, EchoAccept* out, cudaStream_t st) {
  const int cap = sel->capacity;
  const size_t need = (size_t)(cap + R) * sizeof(float2);
  if (need > ctx->workspace_bytes) return ECHO_ERR_WORKSPACE;
  float2* stats = reinterpret_cast<float2*>(ctx->workspace);
  const double c_exact = 1.4426950408889634 / (double)in->temperature;
  const float c = (float)c_exact, c_lo = (float)(c_exact - (double)c);  // log2(e) / T in two floats (bonus-draw CDF)
  if (cap + R > 0) {
    ECHO_CUDA_TRY(ctx, launch_pdl(k_softmax_stats, dim3(cap + R), dim3(ST_THREADS), 0, st, sel->n_selected, cap, R,
                                  reinterpret_cast<const __nv_bfloat16*>(in->target_logits),
                                  reinterpret_cast<const __nv_bfloat16*>(in->root_logits), in->ld, in->vocab, c, stats));
  }
  if (R > 0) {
    const bool have_pools = kv->k_pool && kv->v_pool;
    ECHO_CUDA_TRY(ctx, launch_pdl(k_walk_sample, dim3(R), dim3(WS_THREADS), 0, st, sel->sel_offsets, sel->parent_local,
                                  in->draft_token, reinterpret_cast<const __nv_bfloat16*>(in->target_logits),
                                  reinterpret_cast<const __nv_bfloat16*>(in->root_logits), in->ld, in->vocab, cap, c, c_lo,
                                  stats, in->u_accept, in->u_bonus, kv->page_table, kv->prefix_len,
                                  kv->max_pages_per_req, kv->num_kv_heads, kv->num_pages, kv->num_layers,
                                  have_pools ? reinterpret_cast<__nv_bfloat16*>(kv->k_pool) : (__nv_bfloat16*)nullptr,
                                  have_pools ? reinterpret_cast<__nv_bfloat16*>(kv->v_pool) : (__nv_bfloat16*)nullptr,
                                  out->accept_len, out->last_node, out->bonus_token, out->new_len, out->accept_idx,
                                  out->slot_src, out->slot_dst));
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}
