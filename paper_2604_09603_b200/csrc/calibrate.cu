// echo_calibrate: warm-up calibration of the sparse gates (include/echo.h; paper: "Offline Calibration", P:115,
// "Adaptive Calibration"; readings R:K-1..K-3 of DESIGN.md section 3).
//   k_calib_partition : appends every (confidence, accepted) sample to the segment of its depth as one 32-bit key
//                       (confidence bits << 1 | accepted): confidences lie in [0, 1], so the sign bit is free
//   k_calib_depth     : one CTA per depth -- stable LSD radix sort of the segment in shared memory (4-bit digits,
//                       thread = contiguous chunk, so a scan over [digit][thread] counters gives stable positions),
//                       then, on the sorted keys, the Mann-Whitney statistic (AUC) and the observed value that
//                       maximises Youden's J, both in exact integer arithmetic
//   k_calib_finish    : sweet-spot mask D_sig = {d : AUC_d > delta}
// A sort / scan workload of a few hundred thousand samples: latency-bound, no roofline claim.
#include "common.cuh"

namespace {

constexpr int CAP = ECHO_CALIB_MAX_PER_DEPTH;  // samples of one depth that fit the shared-memory sort
constexpr int NT = 1024;
constexpr int PER = CAP / NT;  // 24 contiguous keys per thread
constexpr int SM_KEYS_A = 0;
constexpr int SM_KEYS_B = SM_KEYS_A + CAP * 4;
constexpr int SM_CNT = SM_KEYS_B + CAP * 4;  // uint16 cnt[16][NT], later reused for reductions
constexpr int SM_TOTAL = SM_CNT + 16 * NT * 2;
static_assert(CAP % NT == 0 && SM_TOTAL <= 227 * 1024, "shared-memory budget");

__global__ void __launch_bounds__(256) k_calib_partition(const uint8_t* __restrict__ depth, const float* __restrict__ conf,
                                                         const uint8_t* __restrict__ accepted, long long M,
                                                         int32_t* __restrict__ g_cnt, uint32_t* __restrict__ seg,
                                                         uint32_t* __restrict__ status) {
  __shared__ int s_cnt[32], s_base[32];
  if (threadIdx.x < 32) s_cnt[threadIdx.x] = 0;
  __syncthreads();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int d = -1, rank = 0;
  uint32_t key = 0;
  if (i < M) {
    const float c = conf[i];
    d = depth[i];
    if (d >= ECHO_MAX_DEPTH || !(c >= 0.0f && c <= 1.0f)) {  // also NaN
      atomicOr(status, ECHO_DEV_BAD_TRACE);
      d = -1;
    } else {
      key = (__float_as_uint(c + 0.0f) << 1) | (accepted[i] ? 1u : 0u);  // + 0: -0 -> +0
      rank = atomicAdd(&s_cnt[d], 1);
    }
  }
  __syncthreads();
  if (threadIdx.x < 32 && s_cnt[threadIdx.x]) s_base[threadIdx.x] = atomicAdd(&g_cnt[threadIdx.x], s_cnt[threadIdx.x]);
  __syncthreads();
  if (d >= 0) {
    const int pos = s_base[d] + rank;
    if (pos < CAP) seg[(size_t)d * CAP + pos] = key;
    else atomicOr(status, ECHO_DEV_CALIB_OVERFLOW);
  }
}

__device__ __forceinline__ int block_excl_scan(int v, int* s_warp, int& total) {  // NT threads, returns exclusive prefix
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  __syncthreads();  // s_warp may still be read from a previous call
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    int w = s_warp[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += t;
    }
    s_warp[lane] = w;
  }
  __syncthreads();
  total = s_warp[31];
  return incl - v + (warp ? s_warp[warp - 1] : 0);
}

__global__ void __launch_bounds__(NT, 1) k_calib_depth(const int32_t* __restrict__ g_cnt, const uint32_t* __restrict__ seg,
                                                       double* __restrict__ auc, float* __restrict__ tau,
                                                       int32_t* __restrict__ n_pos_out, int32_t* __restrict__ n_neg_out) {
  extern __shared__ __align__(16) uint8_t sm[];
  uint32_t* src = reinterpret_cast<uint32_t*>(sm + SM_KEYS_A);
  uint32_t* dst = reinterpret_cast<uint32_t*>(sm + SM_KEYS_B);
  uint16_t* cnt = reinterpret_cast<uint16_t*>(sm + SM_CNT);
  __shared__ int s_warp[32];
  __shared__ unsigned long long s_two_u;
  __shared__ long long s_best;
  const int d = blockIdx.x, tid = threadIdx.x, lane = tid & 31;
  const int n = min(g_cnt[d], CAP);
  const int per = (n + NT - 1) / NT;  // keys per thread (<= PER); keys [n, per * NT) are padding that sorts last
  const int lo = tid * per;
  for (int i = tid; i < per * NT; i += NT) src[i] = i < n ? seg[(size_t)d * CAP + i] : 0xffffffffu;
  if (tid == 0) { s_two_u = 0ull; s_best = LLONG_MIN; }
  __syncthreads();

  // ---- stable LSD radix sort, 8 passes of 4 bits ----
  for (int shift = 0; shift < 32; shift += 4) {
#pragma unroll
    for (int dg = 0; dg < 16; ++dg) cnt[dg * NT + tid] = 0;
    for (int e = 0; e < per; ++e) ++cnt[((src[lo + e] >> shift) & 15u) * NT + tid];
    __syncthreads();
    {  // exclusive scan of the flattened [digit][thread] counters; this thread owns entries [16 tid, 16 tid + 16)
      uint16_t* mine = cnt + 16 * tid;
      int v[16], sum = 0;
#pragma unroll
      for (int q = 0; q < 16; ++q) { v[q] = mine[q]; sum += v[q]; }
      int total;
      int run = block_excl_scan(sum, s_warp, total);
#pragma unroll
      for (int q = 0; q < 16; ++q) { mine[q] = (uint16_t)run; run += v[q]; }
    }
    __syncthreads();
    for (int e = 0; e < per; ++e) {
      const uint32_t k = src[lo + e];
      const int pos = cnt[((k >> shift) & 15u) * NT + tid]++;
      dst[pos] = k;
    }
    __syncthreads();
    uint32_t* t = src; src = dst; dst = t;
  }
  // sorted keys are in `src` (8 swaps); `dst` becomes cum_neg[idx] = rejected samples before idx
  int my_neg = 0;
  for (int e = 0; e < per; ++e) my_neg += (lo + e < n) && !(src[lo + e] & 1u);
  int n_neg;
  int run = block_excl_scan(my_neg, s_warp, n_neg);
  for (int e = 0; e < per; ++e) {
    dst[lo + e] = (uint32_t)run;
    run += (lo + e < n) && !(src[lo + e] & 1u);
  }
  __syncthreads();
  const int n_pos = n - n_neg;

  unsigned long long two_u = 0ull;  // 2 x Mann-Whitney U = sum over accepted samples of (2 #neg below + #neg equal)
  long long best = LLONG_MIN;       // (J(v) n_pos n_neg) << 32 | (2^32 - 1 - index): largest J, then smallest v
  for (int e = 0; e < per; ++e) {
    const int idx = lo + e;
    if (idx >= n) break;
    const uint32_t k = src[idx];
    if (k & 1u) {
      int a = 0, b = idx;  // first index whose confidence equals this one: lower bound of (confidence << 1)
      const uint32_t want = k & ~1u;
      while (a < b) {
        const int m = (a + b) >> 1;
        if (src[m] < want) a = m + 1; else b = m;
      }
      two_u += (unsigned long long)dst[a] + dst[idx];
    }
    if (idx == n - 1 || (src[idx + 1] >> 1) != (k >> 1)) {  // last sample of a confidence value v: candidate tau = v
      const int neg_le = (idx + 1 < n) ? (int)dst[idx + 1] : n_neg;
      const int pos_le = idx + 1 - neg_le;
      const long long num = (long long)(n_pos - pos_le) * n_neg - (long long)(n_neg - neg_le) * n_pos;
      const long long cand = num * 4294967296ll + (long long)(0xffffffffu - (uint32_t)idx);
      best = max(best, cand);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    two_u += __shfl_xor_sync(0xffffffffu, two_u, o);
    best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
  }
  if (lane == 0) {
    atomicAdd(&s_two_u, two_u);
    atomicMax(&s_best, best);
  }
  __syncthreads();
  if (tid == 0) {
    n_pos_out[d] = n_pos;
    n_neg_out[d] = n_neg;
    if (n_pos == 0 || n_neg == 0) {
      auc[d] = 0.5;
      tau[d] = 0.0f;
    } else {
      auc[d] = (double)s_two_u / (double)(2ll * n_pos * n_neg);
      const uint32_t idx = 0xffffffffu - (uint32_t)(s_best & 0xffffffffll);
      tau[d] = __uint_as_float(src[idx] >> 1);
    }
  }
}

__global__ void k_calib_finish(const double* __restrict__ auc, const int32_t* __restrict__ n_pos,
                               const int32_t* __restrict__ n_neg, double delta, uint32_t* __restrict__ depth_mask) {
  const int d = threadIdx.x;
  const unsigned m = __ballot_sync(0xffffffffu, n_pos[d] > 0 && n_neg[d] > 0 && auc[d] > delta);
  if (d == 0) *depth_mask = m;
}

}  // namespace

int launch_calibrate(EchoCtx* ctx, const EchoTraces* t, double delta, EchoCalibration* o, cudaStream_t st) {
  const size_t need = 256 + (size_t)ECHO_MAX_DEPTH * CAP * sizeof(uint32_t);
  if (need > ctx->workspace_bytes) return ECHO_ERR_WORKSPACE;
  int32_t* g_cnt = reinterpret_cast<int32_t*>(ctx->workspace);
  uint32_t* seg = reinterpret_cast<uint32_t*>(reinterpret_cast<uint8_t*>(ctx->workspace) + 256);
  ECHO_CUDA_TRY(ctx, cudaMemsetAsync(g_cnt, 0, 256, st));
  const long long M = t->num_samples;
  if (M > 0) {
    const long long blocks = (M + 255) / 256;
    if (blocks > 0x7fffffffll) return ECHO_ERR_UNSUPPORTED;
    ECHO_COUNT_LAUNCH();
    k_calib_partition<<<(unsigned)blocks, 256, 0, st>>>(t->depth, t->conf, t->accepted, M, g_cnt, seg, ctx->dev_status);
  }
  if (!ctx->calib_attr_set) {  // per context: the attribute is a per-device property of the function
    ECHO_CUDA_TRY(ctx, cudaFuncSetAttribute(k_calib_depth, cudaFuncAttributeMaxDynamicSharedMemorySize, SM_TOTAL));
    ctx->calib_attr_set = true;
  }
  ECHO_COUNT_LAUNCH();
  k_calib_depth<<<ECHO_MAX_DEPTH, NT, SM_TOTAL, st>>>(g_cnt, seg, o->auc, o->tau, o->n_pos, o->n_neg);
  ECHO_COUNT_LAUNCH();
  k_calib_finish<<<1, 32, 0, st>>>(o->auc, o->n_pos, o->n_neg, delta, o->depth_mask);
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}
