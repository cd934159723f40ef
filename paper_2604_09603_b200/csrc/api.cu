// C-ABI entry points of libecho.so (include/echo.h): argument validation and launch only.
#include "common.cuh"

#include <new>

static bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) != 0; }

// A context belongs to one device: every compute entry point makes it current for the duration of the call, so that a
// caller whose current device differs (or a second context on another GPU) launches where the context's memory lives.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(const EchoCtx* ctx) {
    if (ctx && cudaGetDevice(&prev) == cudaSuccess && prev != ctx->device) switched = cudaSetDevice(ctx->device) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

// SM clock seen by a kernel right now: one thread spins ~20 us and divides its cycle counter by the global timer.
// NVML / nvidia-smi sample every 20-100 ms at best and read 1965 MHz between kernels; under the verify step the SMs
// run at 1.25-1.5 GHz, and a kernel bound by SM cycles scales with that.
__global__ void k_clock_probe(float* out) {
  unsigned long long t0, t1;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
  const long long c0 = clock64();
  do {
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
  } while (t1 - t0 < 20000ull);
  const long long c1 = clock64();
  *out = (float)((double)(c1 - c0) * 1000.0 / (double)(t1 - t0));
}

extern "C" {

uint64_t echo_launch_count(void) { return g_echo_launches.load(std::memory_order_relaxed); }

int echo_probe_sm_clock(EchoCtx* ctx, float* mhz_dev, echo_stream_t stream) {
  if (!ctx || !mhz_dev) return ECHO_ERR_INVALID_ARG;
  DeviceGuard dg(ctx);
  k_clock_probe<<<1, 1, 0, reinterpret_cast<cudaStream_t>(stream)>>>(mhz_dev);
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}

const char* echo_strerror(int code) {
  switch (code) {
    case ECHO_OK: return "ok";
    case ECHO_ERR_INVALID_ARG: return "invalid argument";
    case ECHO_ERR_UNSUPPORTED: return "unsupported shape";
    case ECHO_ERR_WORKSPACE: return "workspace too small";
    case ECHO_ERR_ARCH: return "device is not sm_100 (B200)";
    case ECHO_ERR_CUDA: return "CUDA error (see echo_last_error)";
    case ECHO_ERR_TOO_LARGE: return "more candidates than the fixed scratch of echo_gate_select_noalloc holds (ECHO_NOALLOC_MAX_CAND)";
    default: return "unknown error";
  }
}

size_t echo_workspace_bytes(int32_t R, int32_t N, int32_t capacity, int32_t Hq, int32_t max_splits) {
  if (R < 0 || N < 0 || capacity < 0 || Hq < 0) return 0;
  const size_t splits = max_splits <= 0 || max_splits > 16 ? 16 : (size_t)max_splits;
  const size_t keys = align_up((size_t)N * sizeof(uint64_t), 256) + 256;  // select keys + threshold
  // split-KV partials exist only when a stream is split; the work list sits behind them: <= R * Hkv * row tiles *
  // splits records of 32 B, and Hkv * row tiles <= 2 Hq (row tiles = ceil(min(capacity, 128) * G / 128))
  const size_t parts = splits > 1 ? align_up(splits * capacity * Hq * (128 + 1) * sizeof(float), 256) : 0;
  const size_t plan = 256 + (size_t)R * 2 * (Hq > 0 ? Hq : 1) * splits * 32;
  const size_t stats = ((size_t)capacity + R) * 8;  // echo_accept_stochastic: (max, Z) per logits row
  size_t m = keys > parts + plan ? keys : parts + plan;
  if (stats > m) m = stats;
  return align_up(m, 256) + 4096;
}

int echo_attn_splits(EchoCtx* ctx, int32_t R, int32_t Hkv) {
  if (!ctx || R < 0 || Hkv <= 0) return ECHO_ERR_INVALID_ARG;
  return attn_split_policy(ctx, R, Hkv);
}

int echo_create(EchoCtx** out, int device, size_t workspace_bytes) {
  if (!out) return ECHO_ERR_INVALID_ARG;
  *out = nullptr;
  int n = 0;
  if (cudaGetDeviceCount(&n) != cudaSuccess || device < 0 || device >= n) return ECHO_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return ECHO_ERR_CUDA;
  if (prop.major != 10 || prop.minor != 0) return ECHO_ERR_ARCH;
  EchoCtx* c = new (std::nothrow) EchoCtx();
  if (!c) return ECHO_ERR_CUDA;
  memset(c, 0, sizeof(*c));
  c->device = device;
  c->num_sms = prop.multiProcessorCount;
  int prev = 0;
  cudaGetDevice(&prev);
  cudaSetDevice(device);
  c->workspace_bytes = align_up(workspace_bytes ? workspace_bytes : 256, 256);
  cudaError_t e = cudaMalloc(&c->workspace, c->workspace_bytes);
  if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&c->dev_status), 256);
  if (e == cudaSuccess) e = cudaMemset(c->dev_status, 0, 256);
  cudaSetDevice(prev);
  if (e != cudaSuccess) {
    if (c->workspace) cudaFree(c->workspace);
    delete c;
    return ECHO_ERR_CUDA;
  }
  *out = c;
  return ECHO_OK;
}

int echo_destroy(EchoCtx* ctx) {
  if (!ctx) return ECHO_ERR_INVALID_ARG;
  DeviceGuard dg(ctx);
  cudaFree(ctx->workspace);
  cudaFree(ctx->dev_status);
  free_tmap_cache(ctx->tmaps);
  delete ctx;
  return ECHO_OK;
}

const char* echo_last_error(EchoCtx* ctx) { return ctx ? ctx->last_error : "null context"; }

int echo_device_status(EchoCtx* ctx, uint32_t* flags, echo_stream_t stream) {
  DeviceGuard dg(ctx);
  if (!ctx || !flags) return ECHO_ERR_INVALID_ARG;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  ECHO_CUDA_TRY(ctx, cudaMemcpyAsync(flags, ctx->dev_status, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
  ECHO_CUDA_TRY(ctx, cudaMemsetAsync(ctx->dev_status, 0, sizeof(uint32_t), st));
  ECHO_CUDA_TRY(ctx, cudaStreamSynchronize(st));
  return ECHO_OK;
}

int echo_set_option(EchoCtx* ctx, int key, int64_t value) {
  if (!ctx) return ECHO_ERR_INVALID_ARG;
  switch (key) {
    case ECHO_OPT_FORCE_SPLITS:
      if (value < 0 || value > 16) return ECHO_ERR_INVALID_ARG;
      ctx->opt_force_splits = value;
      return ECHO_OK;
    case ECHO_OPT_ATTN_PATH:
      if (value < 0 || value > 2) return ECHO_ERR_INVALID_ARG;
      ctx->opt_attn_path = value;
      return ECHO_OK;
    case ECHO_OPT_NUM_CTAS:
      if (value < 0 || value > 4096) return ECHO_ERR_INVALID_ARG;
      ctx->opt_num_ctas = value;
      return ECHO_OK;
    case ECHO_OPT_ATTN_SAFE:
      if (value < 0 || value > 1) return ECHO_ERR_INVALID_ARG;
      ctx->opt_attn_safe = value;
      return ECHO_OK;
    case ECHO_OPT_GATE_PATH:
      if (value < 0 || value > 2) return ECHO_ERR_INVALID_ARG;
      ctx->opt_gate_path = value;
      return ECHO_OK;
    case ECHO_OPT_ATTN_PLAN:
      if (value < 0 || value > 1) return ECHO_ERR_INVALID_ARG;
      ctx->opt_attn_plan = value;
      return ECHO_OK;
    case ECHO_OPT_GATE_CLUSTER:
      if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8 && value != 16) return ECHO_ERR_INVALID_ARG;
      ctx->opt_gate_cluster = value;
      return ECHO_OK;
    default: return ECHO_ERR_INVALID_ARG;
  }
}

static int check_gate(EchoCtx* ctx, const EchoTrees* t, const EchoGate* g, EchoSelection* o, bool need_packed) {
  if (!ctx || !t || !g || !o) return ECHO_ERR_INVALID_ARG;
  if (t->num_requests < 0 || t->total_cand < 0 || t->max_cand_per_req < 0) return ECHO_ERR_INVALID_ARG;
  if (g->budget < 0 || g->w_max < 0 || g->static_k < 0 || o->capacity < 0) return ECHO_ERR_INVALID_ARG;
  if (g->cand_index_base < 0 || g->request_base < 0) return ECHO_ERR_INVALID_ARG;
  if (g->schedule != ECHO_SCHED_TOPB && g->schedule != ECHO_SCHED_ALG1) return ECHO_ERR_INVALID_ARG;
  if (t->max_cand_per_req > ECHO_MAX_CAND) return ECHO_ERR_UNSUPPORTED;
  // ECHO_SCHED_ALG1 keys carry the global request index in 24 bits
  if (g->schedule == ECHO_SCHED_ALG1 && (int64_t)g->request_base + t->num_requests > (1 << 24)) return ECHO_ERR_UNSUPPORTED;
  if (!t->cand_offsets || !o->cut_depth) return ECHO_ERR_INVALID_ARG;
  if (t->total_cand > 0 && (!t->parent || !t->logq || !o->path_score || !o->cand_depth)) return ECHO_ERR_INVALID_ARG;
  if (!need_packed) return ECHO_OK;
  if (!o->n_selected || !o->sel_offsets) return ECHO_ERR_INVALID_ARG;
  long need = g->static_k > 0 ? (long)t->num_requests * g->static_k : (long)g->budget;
  if (need > t->total_cand) need = t->total_cand;
  if (o->capacity < need) return ECHO_ERR_INVALID_ARG;
  if (o->capacity > 0 && (!o->sel_node || !o->sel_req || !o->parent_local || !o->sel_depth || !o->anc_mask))
    return ECHO_ERR_INVALID_ARG;
  if (misaligned(o->anc_mask, 16)) return ECHO_ERR_INVALID_ARG;
  return ECHO_OK;
}

int echo_gate_select(EchoCtx* ctx, const EchoTrees* t, const EchoGate* g, EchoSelection* o, echo_stream_t stream) {
  DeviceGuard dg(ctx);
  const int rc = check_gate(ctx, t, g, o, true);
  if (rc != ECHO_OK) return rc;
  return launch_gate_select(ctx, t, g, o, reinterpret_cast<cudaStream_t>(stream));
}

int echo_gate_keys(EchoCtx* ctx, const EchoTrees* t, const EchoGate* g, EchoSelection* o, uint64_t* keys,
                   echo_stream_t stream) {
  DeviceGuard dg(ctx);
  const int rc = check_gate(ctx, t, g, o, false);
  if (rc != ECHO_OK) return rc;
  if (t->total_cand > 0 && (!keys || misaligned(keys, 8))) return ECHO_ERR_INVALID_ARG;
  return launch_gate_keys(ctx, t, g, o, keys, reinterpret_cast<cudaStream_t>(stream));
}

int echo_gate_select_keys(EchoCtx* ctx, const EchoTrees* t, const EchoGate* g, const uint64_t* local_keys,
                          const uint64_t* all_keys, int64_t n_all, EchoSelection* o, echo_stream_t stream) {
  DeviceGuard dg(ctx);
  const int rc = check_gate(ctx, t, g, o, true);
  if (rc != ECHO_OK) return rc;
  if (n_all < 0 || (n_all > 0 && !all_keys) || (t->total_cand > 0 && !local_keys)) return ECHO_ERR_INVALID_ARG;
  if (misaligned(all_keys, 8) || misaligned(local_keys, 8)) return ECHO_ERR_INVALID_ARG;
  return launch_gate_select_keys(ctx, t, g, local_keys, all_keys, n_all, o, reinterpret_cast<cudaStream_t>(stream));
}

static int check_kv(const EchoPagedKV* kv, bool need_pools) {
  if (!kv) return ECHO_ERR_INVALID_ARG;
  if (kv->head_dim != 128 || kv->page_size != 16) return ECHO_ERR_UNSUPPORTED;
  if (kv->num_kv_heads <= 0 || kv->num_pages < 0 || kv->max_pages_per_req < 0 || kv->num_layers <= 0)
    return ECHO_ERR_INVALID_ARG;
  if (!kv->page_table || !kv->prefix_len) return ECHO_ERR_INVALID_ARG;
  if (need_pools && (!kv->k_pool || !kv->v_pool)) return ECHO_ERR_INVALID_ARG;
  if (misaligned(kv->k_pool, 16) || misaligned(kv->v_pool, 16)) return ECHO_ERR_INVALID_ARG;
  return ECHO_OK;
}

int echo_verify_attn(EchoCtx* ctx, const EchoSelection* sel, const EchoPagedKV* kv, int32_t layer, int32_t Hq,
                     int32_t R, const void* q, void* out, float* lse, float sm_scale, echo_stream_t stream) {
  DeviceGuard dg(ctx);
  if (!ctx || !sel) return ECHO_ERR_INVALID_ARG;
  int rc = check_kv(kv, true);
  if (rc != ECHO_OK) return rc;
  if (R < 0 || Hq <= 0 || sel->capacity < 0 || layer < 0 || layer >= kv->num_layers) return ECHO_ERR_INVALID_ARG;
  if (Hq % kv->num_kv_heads != 0) return ECHO_ERR_UNSUPPORTED;
  if (!sel->n_selected || !sel->sel_offsets) return ECHO_ERR_INVALID_ARG;
  if (sel->capacity > 0 && (!q || !out || !lse || !sel->sel_req || !sel->anc_mask)) return ECHO_ERR_INVALID_ARG;
  if (misaligned(q, 16) || misaligned(out, 16) || misaligned(sel->anc_mask, 16)) return ECHO_ERR_INVALID_ARG;
  return launch_verify_attn(ctx, sel, kv, layer, Hq, R, q, out, lse, sm_scale, reinterpret_cast<cudaStream_t>(stream));
}

int echo_accept_stochastic(EchoCtx* ctx, const EchoSelection* sel, const EchoSampleInputs* in, int32_t R, EchoPagedKV* kv,
                           EchoAccept* out, echo_stream_t stream) {
  DeviceGuard dg(ctx);
  if (!ctx || !sel || !in || !out) return ECHO_ERR_INVALID_ARG;
  int rc = check_kv(kv, false);
  if (rc != ECHO_OK) return rc;
  if (R < 0 || sel->capacity < 0 || in->vocab <= 0 || in->ld < in->vocab || !(in->temperature > 0.f)) return ECHO_ERR_INVALID_ARG;
  if (in->ld % 8 != 0 || in->vocab > 262144) return ECHO_ERR_UNSUPPORTED;
  if (!sel->sel_offsets || !sel->n_selected || !in->root_logits || !in->u_bonus) return ECHO_ERR_INVALID_ARG;
  if (sel->capacity > 0 && (!sel->parent_local || !in->draft_token || !in->target_logits || !in->u_accept))
    return ECHO_ERR_INVALID_ARG;
  if (misaligned(in->target_logits, 16) || misaligned(in->root_logits, 16)) return ECHO_ERR_INVALID_ARG;
  if (!out->accept_len || !out->last_node || !out->bonus_token || !out->new_len || !out->accept_idx || !out->slot_src ||
      !out->slot_dst)
    return ECHO_ERR_INVALID_ARG;
  return launch_accept_stochastic(ctx, sel, in, R, kv, out, reinterpret_cast<cudaStream_t>(stream));
}

int echo_draft_expand(EchoCtx* ctx, const EchoDraftLevel* l, EchoTrees* t, int32_t* token, float* score_out,
                      echo_stream_t stream) {
  DeviceGuard dg(ctx);
  if (!ctx || !l || !t) return ECHO_ERR_INVALID_ARG;
  if (t->num_requests < 0 || l->level < 0 || l->topk < 1) return ECHO_ERR_INVALID_ARG;
  if (l->level >= ECHO_MAX_DEPTH || l->topk > ECHO_MAX_TOPK) return ECHO_ERR_UNSUPPORTED;
  if (t->num_requests > 0 && (!t->cand_offsets || !t->parent || !t->logq || !token || !score_out || !l->parent_score ||
                              !l->child_logq || !l->child_token))
    return ECHO_ERR_INVALID_ARG;
  return launch_draft_expand(ctx, l, t, token, score_out, reinterpret_cast<cudaStream_t>(stream));
}

int echo_calibrate(EchoCtx* ctx, const EchoTraces* t, double delta, EchoCalibration* o, echo_stream_t stream) {
  DeviceGuard dg(ctx);
  if (!ctx || !t || !o) return ECHO_ERR_INVALID_ARG;
  if (t->num_samples < 0 || !(delta == delta)) return ECHO_ERR_INVALID_ARG;
  if (t->num_samples > 0 && (!t->depth || !t->conf || !t->accepted)) return ECHO_ERR_INVALID_ARG;
  if (!o->auc || !o->tau || !o->n_pos || !o->n_neg || !o->depth_mask) return ECHO_ERR_INVALID_ARG;
  if (misaligned(o->auc, 8) || misaligned(t->conf, 4)) return ECHO_ERR_INVALID_ARG;
  return launch_calibrate(ctx, t, delta, o, reinterpret_cast<cudaStream_t>(stream));
}

int echo_argmax_shard(EchoCtx* ctx, const EchoSelection* sel, const void* logits_shard, int64_t ld, int32_t vocab_shard,
                      int32_t vocab_base, uint64_t* pairs_out, echo_stream_t stream) {
  DeviceGuard dg(ctx);
  if (!ctx || !sel || !logits_shard || !pairs_out || !sel->n_selected || sel->capacity < 0) return ECHO_ERR_INVALID_ARG;
  if (vocab_shard <= 0 || vocab_base < 0 || ld < vocab_shard || (int64_t)vocab_base + vocab_shard > INT32_MAX)
    return ECHO_ERR_INVALID_ARG;
  if (ld % 8 != 0) return ECHO_ERR_UNSUPPORTED;
  if (misaligned(logits_shard, 16) || misaligned(pairs_out, 8)) return ECHO_ERR_INVALID_ARG;
  return launch_argmax_shard(ctx, sel, logits_shard, ld, vocab_shard, vocab_base, pairs_out,
                             reinterpret_cast<cudaStream_t>(stream));
}

int echo_argmax_merge(EchoCtx* ctx, const EchoSelection* sel, const uint64_t* pairs_all, int32_t world,
                      int32_t* target_token_out, echo_stream_t stream) {
  DeviceGuard dg(ctx);
  if (!ctx || !sel || !pairs_all || !target_token_out || !sel->n_selected || sel->capacity < 0 || world < 1)
    return ECHO_ERR_INVALID_ARG;
  if (misaligned(pairs_all, 8)) return ECHO_ERR_INVALID_ARG;
  return launch_argmax_merge(ctx, sel, pairs_all, world, target_token_out, reinterpret_cast<cudaStream_t>(stream));
}

int echo_accept(EchoCtx* ctx, const EchoSelection* sel, const EchoVerifyResult* res, int32_t R, EchoPagedKV* kv,
                EchoAccept* out, echo_stream_t stream) {
  DeviceGuard dg(ctx);
  if (!ctx || !sel || !res || !out) return ECHO_ERR_INVALID_ARG;
  int rc = check_kv(kv, false);
  if (rc != ECHO_OK) return rc;
  if (R < 0 || sel->capacity < 0) return ECHO_ERR_INVALID_ARG;
  if ((res->target_token != nullptr) == (res->target_logits != nullptr)) return ECHO_ERR_INVALID_ARG;
  if (res->target_logits) {
    if (res->vocab <= 0 || res->ld < res->vocab) return ECHO_ERR_INVALID_ARG;
    if (res->ld % 8 != 0) return ECHO_ERR_UNSUPPORTED;
    if (misaligned(res->target_logits, 16)) return ECHO_ERR_INVALID_ARG;
  }
  if (!sel->sel_offsets || !sel->n_selected) return ECHO_ERR_INVALID_ARG;
  if (R > 0 && (!res->prev_token || !out->accept_len || !out->last_node || !out->bonus_token || !out->new_len ||
                !out->accept_idx || !out->slot_src || !out->slot_dst))
    return ECHO_ERR_INVALID_ARG;
  if (sel->capacity > 0 && (!res->draft_token || !sel->parent_local || !sel->sel_depth || !sel->anc_mask))
    return ECHO_ERR_INVALID_ARG;
  if (misaligned(sel->anc_mask, 16)) return ECHO_ERR_INVALID_ARG;
  return launch_accept(ctx, sel, res, R, kv, out, reinterpret_cast<cudaStream_t>(stream));
}

}  // extern "C"
