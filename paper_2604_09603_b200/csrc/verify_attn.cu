// echo_verify_attn: S6 (split-KV tree-masked paged GQA attention) + S7 (LSE merge).
//   k_attn_smallrow : CUDA-core kernel, one CTA per (packed node, KV head, split), one warp per query
//                     head of the GQA group.  Used when node rows x group cannot fill a tensor-core
//                     tile (and as the on-device cross-check of the tcgen05 kernel).
//   k_lse_merge     : combines split partials (S7).
//   the tcgen05/TMA kernel lives in verify_attn_tc.cu.
// Definition of the operator: include/echo.h, R:A-1..A-8 (the paper only names it).
#include "common.cuh"

namespace {

constexpr int D = 128;
constexpr int PAGE = 16;
constexpr int TILE = 128;  // split granularity in tokens (same as the tcgen05 kernel's KV tile)
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;

__device__ __forceinline__ float bf16lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

__global__ void k_attn_smallrow(const int32_t* __restrict__ n_selected, const int32_t* __restrict__ sel_offsets,
                                const int32_t* __restrict__ sel_req, const uint32_t* __restrict__ anc_mask,
                                const __nv_bfloat16* __restrict__ k_pool, const __nv_bfloat16* __restrict__ v_pool,
                                const int32_t* __restrict__ page_table, const int32_t* __restrict__ prefix_len,
                                int max_pages, int Hkv, int Hq, const __nv_bfloat16* __restrict__ q,
                                __nv_bfloat16* __restrict__ out, float* __restrict__ lse, float scale_log2,
                                int splits, float* __restrict__ part_o, float* __restrict__ part_lse,
                                uint32_t* __restrict__ status) {
  extern __shared__ float s_q[];  // [G][128]
  const int k = blockIdx.x, kvh = blockIdx.y, split = blockIdx.z;
  if (k >= *n_selected) return;
  const int G = Hq / Hkv;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int h = kvh * G + warp;
  const int i = sel_req[k];
  const int Ki = sel_offsets[i + 1] - sel_offsets[i];
  const int P = prefix_len[i];
  const uint4 mk = reinterpret_cast<const uint4*>(anc_mask)[k];
  const uint32_t mw[4] = {mk.x, mk.y, mk.z, mk.w};
  const int total = P + Ki;
  if (threadIdx.x == 0 && (total + PAGE - 1) / PAGE > max_pages) atomicOr(status, ECHO_DEV_PAGE_OVERFLOW);
  const int n_tiles = (total + TILE - 1) / TILE;
  const int tps = (n_tiles + splits - 1) / splits;
  const int t_lo = min(total, split * tps * TILE), t_hi = min(total, (split + 1) * tps * TILE);

  float* myq = s_q + warp * D;
  {
    const __nv_bfloat16* qp = q + ((size_t)k * Hq + h) * D;
    for (int c = lane; c < D; c += 32) myq[c] = __bfloat162float(qp[c]);
  }
  __syncwarp();

  float m = -INFINITY, lsum = 0.f;
  float o[4] = {0.f, 0.f, 0.f, 0.f};  // lane owns dims 4*lane .. 4*lane+3
  const int32_t* pt = page_table + (size_t)i * max_pages;
  for (int t0 = t_lo; t0 < t_hi; t0 += 32) {
    const int t = t0 + lane;
    bool vis = t < t_hi;
    if (vis && t >= P) { const int a = t - P; vis = (mw[a >> 5] >> (a & 31)) & 1u; }
    float s = -INFINITY;
    size_t row = 0;
    if (t < t_hi) row = (((size_t)pt[t / PAGE] * Hkv + kvh) * PAGE + (t % PAGE)) * D;
    if (vis) {
      const uint4* kp = reinterpret_cast<const uint4*>(k_pool + row);
      float acc = 0.f;
#pragma unroll
      for (int c = 0; c < D / 8; ++c) {
        const uint4 u = kp[c];
        const float* qq = myq + c * 8;
        acc = fmaf(bf16lo(u.x), qq[0], acc); acc = fmaf(bf16hi(u.x), qq[1], acc);
        acc = fmaf(bf16lo(u.y), qq[2], acc); acc = fmaf(bf16hi(u.y), qq[3], acc);
        acc = fmaf(bf16lo(u.z), qq[4], acc); acc = fmaf(bf16hi(u.z), qq[5], acc);
        acc = fmaf(bf16lo(u.w), qq[6], acc); acc = fmaf(bf16hi(u.w), qq[7], acc);
      }
      s = acc * scale_log2;
    }
    float cm = s;
#pragma unroll
    for (int ofs = 16; ofs; ofs >>= 1) cm = fmaxf(cm, __shfl_xor_sync(0xffffffffu, cm, ofs));
    const float m_new = fmaxf(m, cm);
    if (m_new == -INFINITY) continue;  // nothing visible so far (warp-uniform)
    const float corr = exp2f(m - m_new);
    const float p = vis ? exp2f(s - m_new) : 0.f;
    float ps = p;
#pragma unroll
    for (int ofs = 16; ofs; ofs >>= 1) ps += __shfl_xor_sync(0xffffffffu, ps, ofs);
    lsum = lsum * corr + ps;
#pragma unroll
    for (int c = 0; c < 4; ++c) o[c] *= corr;
    m = m_new;
    const uint32_t vmask = __ballot_sync(0xffffffffu, vis);
    for (int tt = 0; tt < 32; ++tt) {
      if (!((vmask >> tt) & 1u)) continue;  // invisible slots are never read (R:A-7)
      const float pp = __shfl_sync(0xffffffffu, p, tt);
      const size_t vrow = __shfl_sync(0xffffffffu, (unsigned long long)row, tt);
      const uint2 u = *reinterpret_cast<const uint2*>(v_pool + vrow + lane * 4);
      o[0] = fmaf(pp, bf16lo(u.x), o[0]); o[1] = fmaf(pp, bf16hi(u.x), o[1]);
      o[2] = fmaf(pp, bf16lo(u.y), o[2]); o[3] = fmaf(pp, bf16hi(u.y), o[3]);
    }
  }
  const float inv = lsum > 0.f ? 1.f / lsum : 0.f;
  const float my_lse = lsum > 0.f ? (m + log2f(lsum)) * LN2 : -INFINITY;
  const size_t rowi = (size_t)k * Hq + h;
  if (splits == 1) {
    __nv_bfloat162 a = __floats2bfloat162_rn(o[0] * inv, o[1] * inv), b2 = __floats2bfloat162_rn(o[2] * inv, o[3] * inv);
    uint2 w;
    w.x = *reinterpret_cast<uint32_t*>(&a);
    w.y = *reinterpret_cast<uint32_t*>(&b2);
    *reinterpret_cast<uint2*>(out + rowi * D + lane * 4) = w;
    if (lane == 0) lse[rowi] = my_lse;
  } else {
    const size_t n_rows = (size_t)gridDim.x * Hq;
    float4 w = make_float4(o[0] * inv, o[1] * inv, o[2] * inv, o[3] * inv);
    *reinterpret_cast<float4*>(part_o + ((size_t)split * n_rows + rowi) * D + lane * 4) = w;
    if (lane == 0) part_lse[(size_t)split * n_rows + rowi] = my_lse;
  }
}

// S7: lse = ln sum_s exp(lse_s), O = sum_s exp(lse_s - lse) O_s; one warp per (node, head) row.
__global__ void k_lse_merge(const int32_t* __restrict__ n_selected, const int32_t* __restrict__ sel_req,
                            const int32_t* __restrict__ sel_offsets, const int32_t* __restrict__ prefix_len, int Hq,
                            size_t n_rows_cap, int splits_cap, const float* __restrict__ part_o, const float* __restrict__ part_lse,
                            __nv_bfloat16* __restrict__ out, float* __restrict__ lse) {
  const size_t row = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (row >= (size_t)(*n_selected) * Hq) return;
  // splits that hold no KV tile of this request were never written: same rule as the planners
  const int i = sel_req[row / Hq];
  const int n_tiles = (prefix_len[i] + sel_offsets[i + 1] - sel_offsets[i] + TILE - 1) / TILE;
  const int tps = (n_tiles + splits_cap - 1) / splits_cap;
  const int splits = (n_tiles + tps - 1) / tps;
  float mx = -INFINITY;
  for (int s = 0; s < splits; ++s) mx = fmaxf(mx, part_lse[(size_t)s * n_rows_cap + row]);
  float den = 0.f;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int s = 0; s < splits; ++s) {
    const float ls = part_lse[(size_t)s * n_rows_cap + row];
    if (ls == -INFINITY) continue;
    const float w = exp2f((ls - mx) * LOG2E);
    const float4 v = *reinterpret_cast<const float4*>(part_o + ((size_t)s * n_rows_cap + row) * D + lane * 4);
    den += w;
    acc.x = fmaf(w, v.x, acc.x); acc.y = fmaf(w, v.y, acc.y);
    acc.z = fmaf(w, v.z, acc.z); acc.w = fmaf(w, v.w, acc.w);
  }
  const float inv = 1.f / den;
  __nv_bfloat162 a = __floats2bfloat162_rn(acc.x * inv, acc.y * inv), b = __floats2bfloat162_rn(acc.z * inv, acc.w * inv);
  uint2 w;
  w.x = *reinterpret_cast<uint32_t*>(&a);
  w.y = *reinterpret_cast<uint32_t*>(&b);
  *reinterpret_cast<uint2*>(out + row * D + lane * 4) = w;
  if (lane == 0) lse[row] = mx + logf(den);
}

}  // namespace

int launch_verify_attn(EchoCtx* ctx, const EchoSelection* sel, const EchoPagedKV* kv, int32_t layer, int32_t Hq,
                       int32_t R, const void* q, void* out, float* lse, float sm_scale, cudaStream_t st) {
  const int Hkv = kv->num_kv_heads, G = Hq / Hkv, cap = sel->capacity;
  if (cap <= 0 || R <= 0) return ECHO_OK;
  const size_t layer_elems = (size_t)kv->num_pages * Hkv * PAGE * D;
  const __nv_bfloat16* kp = reinterpret_cast<const __nv_bfloat16*>(kv->k_pool) + (size_t)layer * layer_elems;
  const __nv_bfloat16* vp = reinterpret_cast<const __nv_bfloat16*>(kv->v_pool) + (size_t)layer * layer_elems;

  // split policy: the host knows only capacities (P_i, K_i are device-side).  Split the KV range only when there
  // are fewer (request, KV head) streams than SMs, and then just enough to give every SM one: every split level
  // costs per-item set-up, the fp32 partials and the merge launch, and the planner already balances whole items.
  // Measured: cfg1 (256 streams) one split 0.068 ms, two 0.107 ms; cfg3 (512 streams) one 0.256 ms, two 0.312 ms.
  const int splits = attn_split_policy(ctx, R, Hkv);
  const size_t n_rows = (size_t)cap * Hq;
  // workspace layout: [keys: unused here][part_o: splits*n_rows*128 f32][part_lse: splits*n_rows f32]
  float* part_o = reinterpret_cast<float*>(ctx->workspace);
  float* part_lse = part_o + (size_t)splits * n_rows * D;
  if (splits > 1 && (size_t)splits * n_rows * (D + 1) * sizeof(float) > ctx->workspace_bytes) return ECHO_ERR_WORKSPACE;

  const bool tc_ok = (G >= 1 && G <= 128 && (128 % G) == 0);
  int path = (int)ctx->opt_attn_path;
  if (path == 0) path = tc_ok ? 2 : 1;
  if (path == 2 && !tc_ok) return ECHO_ERR_UNSUPPORTED;
  const float scale_log2 = sm_scale * LOG2E;
  if (path == 2) {
    int rc = launch_verify_attn_tc(ctx, sel, kv, layer, Hq, R, q, out, lse, sm_scale, splits, part_o, part_lse, st);
    if (rc != ECHO_OK) return rc;
  } else {
    if (G > 32) return ECHO_ERR_UNSUPPORTED;
    dim3 grid(cap, Hkv, splits);
    ECHO_COUNT_LAUNCH();
    k_attn_smallrow<<<grid, G * 32, G * D * sizeof(float), st>>>(
        sel->n_selected, sel->sel_offsets, sel->sel_req, sel->anc_mask, kp, vp, kv->page_table, kv->prefix_len,
        kv->max_pages_per_req, Hkv, Hq, reinterpret_cast<const __nv_bfloat16*>(q),
        reinterpret_cast<__nv_bfloat16*>(out), lse, scale_log2, splits, part_o, part_lse, ctx->dev_status);
  }
  if (splits > 1) {
    const int wpb = 8;
    const unsigned blocks = (unsigned)((n_rows + wpb - 1) / wpb);
    ECHO_COUNT_LAUNCH();
    k_lse_merge<<<blocks, wpb * 32, 0, st>>>(sel->n_selected, sel->sel_req, sel->sel_offsets, kv->prefix_len, Hq,
                                             n_rows, splits, part_o, part_lse,
                                             reinterpret_cast<__nv_bfloat16*>(out), lse);
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}
