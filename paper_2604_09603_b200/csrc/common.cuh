// Shared internals of libecho.so (CUDA path only; the CPU oracle shares nothing with this).
#pragma once
#include <climits>
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/echo.h"

struct TmapCache;  // TMA tensor maps this context has encoded (verify_attn_tc.cu)
void free_tmap_cache(TmapCache*);

struct EchoCtx {
  int device;
  int num_sms;
  void* workspace;
  size_t workspace_bytes;
  uint32_t* dev_status;  // device status word (inside its own allocation)
  int64_t opt_force_splits;
  int64_t opt_attn_path;
  int64_t opt_num_ctas;
  int64_t opt_attn_safe;
  int64_t opt_gate_path, opt_gate_cluster;
  int64_t opt_attn_plan;
  int gate_cluster_max;  // 0 = not probed yet, -1 = no cluster launch on this device
  TmapCache* tmaps;
  bool attn_attr_set, calib_attr_set;  // cudaFuncSetAttribute is per device, i.e. per context
  char last_error[256];
};

// split policy of echo_verify_attn (verify_attn.cu): the host knows only capacities (P_i, K_i are device-side)
static inline int attn_split_policy(const EchoCtx* ctx, long R, long Hkv) {
  int splits = 1;
  if (ctx->opt_force_splits > 0) splits = (int)ctx->opt_force_splits;
  else
    while (splits < 8 && R * Hkv * splits < (long)ctx->num_sms) splits *= 2;
  return splits > 16 ? 16 : splits;
}

#define ECHO_CUDA_TRY(ctx, expr)                                                              \
  do {                                                                                        \
    cudaError_t _e = (expr);                                                                  \
    if (_e != cudaSuccess) {                                                                  \
      snprintf((ctx)->last_error, sizeof((ctx)->last_error), "%s:%d %s: %s", __FILE__, __LINE__, \
               #expr, cudaGetErrorString(_e));                                                \
      return ECHO_ERR_CUDA;                                                                   \
    }                                                                                         \
  } while (0)

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// kernels launched by this library in this process (echo_launch_count): bench.py's `gpu_launches` is this counter's
// increase over the timed region, not arithmetic
#include <atomic>
inline std::atomic<uint64_t> g_echo_launches{0};
#define ECHO_COUNT_LAUNCH() (g_echo_launches.fetch_add(1, std::memory_order_relaxed))

// launchers implemented by the .cu files
// Programmatic dependent launch: the kernel may start while its predecessor on the stream is still running; it
// must call pdl_wait() before touching anything the predecessor writes (or reads and this kernel overwrites).
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                     Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  ECHO_COUNT_LAUNCH();
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
#endif

int launch_gate_select(EchoCtx*, const EchoTrees*, const EchoGate*, EchoSelection*, cudaStream_t);
int launch_gate_keys(EchoCtx*, const EchoTrees*, const EchoGate*, EchoSelection*, uint64_t* keys, cudaStream_t);
int launch_gate_select_keys(EchoCtx*, const EchoTrees*, const EchoGate*, const uint64_t* local_keys,
                            const uint64_t* all_keys, int64_t n_all, EchoSelection*, cudaStream_t);
int launch_draft_expand(EchoCtx*, const EchoDraftLevel*, EchoTrees*, int32_t* token, float* score_out, cudaStream_t);
int launch_accept_stochastic(EchoCtx*, const EchoSelection*, const EchoSampleInputs*, int32_t R, EchoPagedKV*, EchoAccept*,
                             cudaStream_t);
int launch_calibrate(EchoCtx*, const EchoTraces*, double delta, EchoCalibration*, cudaStream_t);
int launch_verify_attn(EchoCtx*, const EchoSelection*, const EchoPagedKV*, int32_t layer, int32_t Hq, int32_t R,
                       const void* q, void* out, float* lse, float sm_scale, cudaStream_t);
int launch_accept(EchoCtx*, const EchoSelection*, const EchoVerifyResult*, int32_t R, EchoPagedKV*, EchoAccept*,
                  cudaStream_t);
int launch_argmax_shard(EchoCtx*, const EchoSelection*, const void* logits, int64_t ld, int32_t vocab_shard,
                        int32_t vocab_base, uint64_t* pairs, cudaStream_t);
int launch_argmax_merge(EchoCtx*, const EchoSelection*, const uint64_t* pairs_all, int32_t world, int32_t* target_token,
                        cudaStream_t);
// tcgen05 path (verify_attn_tc.cu); returns ECHO_ERR_UNSUPPORTED when the shape cannot use it
int launch_verify_attn_tc(EchoCtx*, const EchoSelection*, const EchoPagedKV*, int32_t layer, int32_t Hq, int32_t R,
                          const void* q, void* out, float* lse, float sm_scale, int splits, float* part_o,
                          float* part_ml, cudaStream_t);

// order-preserving map fp32 -> u32 (ascending float <=> ascending unsigned)
__host__ __device__ static inline uint32_t f32_ordered(float f) {
#ifdef __CUDA_ARCH__
  uint32_t u = __float_as_uint(f);
#else
  uint32_t u;
  memcpy(&u, &f, 4);
#endif
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
