// echo_draft_expand: one level of every request's draft tree from the draft model's top-k outputs, written straight
// into the EchoTrees arrays on the device (include/echo.h; paper: "G_i.append(topk tokens)",
// P:144, trees of depth x top-k; readings R:D-1..D-3).
//   k_draft_expand : one CTA per request, thread = candidate (parent slot p, child rank c): cumulative score
//                    fl32(S_parent + logq) (Eq. 5), rank among the k_prev x k candidates by (score desc, p asc,
//                    c asc) by counting, the k best written to the level's node slots in that order.
// Kilobytes per call, latency-bound: no roofline claim.
#include "common.cuh"

namespace {

constexpr int MAXK = ECHO_MAX_TOPK;

__global__ void __launch_bounds__(MAXK * MAXK) k_draft_expand(
    int level, int k, int k_prev, const int32_t* __restrict__ cand_offsets, const float* __restrict__ parent_score,
    const float* __restrict__ child_logq, const int32_t* __restrict__ child_token, int32_t* __restrict__ parent,
    float* __restrict__ logq, int32_t* __restrict__ token, float* __restrict__ score_out,
    uint32_t* __restrict__ status) {
  __shared__ float s_S[MAXK * MAXK];
  const int i = blockIdx.x, t = threadIdx.x, n = k_prev * k;
  pdl_launch_dependents();
  pdl_wait();
  float S = 0.f;
  if (t < n) {
    const int p = t / k;
    S = __fadd_rn(parent_score[(size_t)i * k_prev + p], child_logq[(size_t)i * n + t]);  // no contraction (R:G-3)
    s_S[t] = S;
  }
  __syncthreads();
  if (t >= n) return;
  int rank = 0;  // candidates are numbered p * k + c: index order is (parent slot asc, child rank asc)
  for (int u = 0; u < n; ++u) rank += (s_S[u] > S) || (s_S[u] == S && u < t);
  if (rank >= k) return;
  const int b = cand_offsets[i];
  if (b + (level + 1) * k > cand_offsets[i + 1]) {  // the request's tree has no room for this level
    atomicOr(status, ECHO_DEV_TREE_OVERFLOW);
    return;
  }
  const int node = b + level * k + rank;
  parent[node] = level == 0 ? -1 : (level - 1) * k + t / k;
  logq[node] = child_logq[(size_t)i * n + t];
  token[node] = child_token[(size_t)i * n + t];
  score_out[(size_t)i * k + rank] = S;
}

}  // namespace

int launch_draft_expand(EchoCtx* ctx, const EchoDraftLevel* l, EchoTrees* trees, int32_t* token, float* score_out,
                        cudaStream_t st) {
  const int k = l->topk, k_prev = l->level == 0 ? 1 : l->topk;
  if (trees->num_requests > 0) {
    ECHO_CUDA_TRY(ctx, launch_pdl(k_draft_expand, dim3(trees->num_requests), dim3(MAXK * MAXK), 0, st, l->level, k,
                                  k_prev, trees->cand_offsets, l->parent_score, l->child_logq, l->child_token,
                                  const_cast<int32_t*>(trees->parent), const_cast<float*>(trees->logq), token, score_out,
                                  ctx->dev_status));
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}
