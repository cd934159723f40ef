/* echo.h -- C ABI of libecho.so: the batch-wide "super-tree" verify step of ECHO
 * (arxiv 2604.09603) as hand-written CUDA for one B200 (sm_100a).
 *
 * Citations: `P:<n>` = line <n> of the paper text; `R:<id>` = a reading of a
 * point the paper leaves open, listed in DESIGN.md section 3.
 *
 * Conventions
 *   - Every pointer marked "dev" is DEVICE memory owned by the caller; it must stay valid
 *     until the work queued on `stream` has finished.  Structs themselves are HOST memory,
 *     read during the call only.
 *   - The hot path is three calls -- echo_gate_select, echo_verify_attn, echo_accept; beside them
 *     echo_gate_keys / echo_gate_select_keys (one budget shared by several ranks), echo_argmax_shard /
 *     echo_argmax_merge (S8 over vocabulary-sharded logits),
 *     echo_accept_stochastic (temperature > 0), echo_calibrate (warm-up calibration of the gates)
 *     and echo_draft_expand (draft-side tree construction).  Every compute call is asynchronous
 *     on `stream`, never synchronises, never reads a device result on the host (CUDA-graph
 *     capturable).  Data-dependent sizes (n_selected, K_i, P_i) live on the device only.
 *   - Return value: ECHO_OK (0) or a negative EchoStatus.  Data-dependent precondition
 *     violations cannot be seen by the host; they set bits in the device status word
 *     (echo_device_status) and leave outputs unspecified.  Nothing traps.
 *   - A context belongs to one device; every call makes that device current for its duration and restores
 *     the caller's.
 *   - There is no CPU fallback and no dispatch on architecture: echo_create fails with
 *     ECHO_ERR_ARCH unless the device has compute capability 10.0.
 *   - R = number of requests (the paper's batch size B); the paper's budget K_max
 *     (Eq. 4) is `budget`.
 */
#ifndef ECHO_H_
#define ECHO_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct EchoCtx EchoCtx;  /* opaque; owns the workspace and the TMA tensor maps it has encoded */
typedef void* echo_stream_t;     /* a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream */

typedef enum {
  ECHO_OK = 0,
  ECHO_ERR_INVALID_ARG = -1, /* NULL pointer, negative size, capacity too small, misaligned pointer */
  ECHO_ERR_UNSUPPORTED = -2, /* head_dim != 128, page_size != 16, Hq % Hkv != 0, max_cand_per_req > 128, ECHO_SCHED_ALG1 with more
                                than 2^24 requests over the ranks sharing a budget */
  ECHO_ERR_WORKSPACE = -3,   /* ctx workspace smaller than echo_workspace_bytes(...) for this call */
  ECHO_ERR_ARCH = -4,        /* device is not sm_100 */
  ECHO_ERR_CUDA = -5,        /* a CUDA runtime / driver call failed; text via echo_last_error */
  ECHO_ERR_TOO_LARGE = -6    /* echo_gate_select_noalloc: total_cand > ECHO_NOALLOC_MAX_CAND (its fixed scratch array) */
} EchoStatus;

/* bits of the device status word */
#define ECHO_DEV_BAD_PARENT 1u   /* parent[j] >= j or < -1 */
#define ECHO_DEV_BAD_LOGQ 2u     /* logq > 0 or NaN */
#define ECHO_DEV_DEPTH_OVERFLOW 4u /* a candidate deeper than 31 */
#define ECHO_DEV_PAGE_OVERFLOW 8u  /* P_i + K_i needs more than max_pages_per_req pages */
#define ECHO_DEV_BAD_TRACE 16u     /* echo_calibrate: depth >= 32 or a confidence outside [0, 1] / NaN (sample skipped) */
#define ECHO_DEV_TREE_OVERFLOW 64u  /* echo_draft_expand: level * topk nodes do not fit the request's candidate range */
#define ECHO_DEV_CALIB_OVERFLOW 32u /* echo_calibrate: more than ECHO_CALIB_MAX_PER_DEPTH samples at one depth (rest dropped) */
#define ECHO_DEV_CAND_OVERFLOW 128u /* a request with more than ECHO_MAX_CAND candidates / packed nodes (the rest is ignored) */
#define ECHO_DEV_INTERNAL 256u      /* a kernel found its own set-up violated (e.g. misaligned shared memory); outputs unspecified */

/* test / tuning hooks for echo_set_option */
#define ECHO_OPT_FORCE_SPLITS 1   /* >0: split every KV stream into exactly this many parts (<= 16) */
#define ECHO_OPT_ATTN_PATH 2      /* 0 = auto, 1 = CUDA-core small-row kernel, 2 = tcgen05 kernel */
#define ECHO_OPT_NUM_CTAS 3       /* >0: persistent grid size of the tcgen05 kernel (default: #SMs) */
#define ECHO_OPT_ATTN_SAFE 4      /* 1: the tcgen05 kernel takes every item in its safe form (running row maximum) */
#define ECHO_OPT_GATE_PATH 5      /* echo_gate_select: 0 = auto, 1 = three kernels (score, select, pack), 2 = one
                                     thread-block cluster (ECHO_ERR_UNSUPPORTED past 32 requests per CTA) */
#define ECHO_OPT_ATTN_PLAN 7      /* tcgen05 kernel's work list: 0 = auto (planned inside the kernel for up to 512 (request,
                                     split) pairs, else by a planner kernel in front of it), 1 = always the planner kernel */
#define ECHO_OPT_GATE_CLUSTER 6   /* >0: cluster size of that kernel (1, 2, 4, 8, 16; default: one CTA per 8 requests) */

#define ECHO_MAX_CAND 128   /* C_i <= 128 candidates per request (R:G-14) */
#define ECHO_MAX_DEPTH 32   /* depth < 32 (R:G-14) */
#define ECHO_MAX_TOPK 16    /* echo_draft_expand: draft top-k per node (the configs use 8, 10, 16) */
#define ECHO_CALIB_MAX_PER_DEPTH 24576 /* echo_calibrate sorts one depth's samples in shared memory */
#define ECHO_CALIB_WORKSPACE_BYTES (256 + (size_t)ECHO_MAX_DEPTH * ECHO_CALIB_MAX_PER_DEPTH * 4)
#define ECHO_MAX_ACCEPT 32  /* an accepted path has <= 32 nodes (one per depth) */
#define ECHO_CUT_NEVER 0x7fffffff

/* ---- lifetime ------------------------------------------------------------------------ */
/* Creates a context on `device` with a workspace of `workspace_bytes` (device memory, owned by
 * the context, freed by echo_destroy).  ECHO_ERR_ARCH unless compute capability is 10.0. */
int echo_create(EchoCtx** out, int device, size_t workspace_bytes);
int echo_destroy(EchoCtx* ctx);
/* Workspace needed by any call with at most these sizes: select keys [total_cand]; split-KV partials
 * [max_splits][capacity][num_q_heads] x (128+1) fp32 (max_splits = the largest split count echo_verify_attn may
 * use: 1 when num_requests * num_kv_heads >= #SMs, else up to 8, or the ECHO_OPT_FORCE_SPLITS value; <= 0 means 16,
 * the upper limit); the work list; (capacity + num_requests) x 8 bytes of echo_accept_stochastic statistics. */
size_t echo_workspace_bytes(int32_t num_requests, int32_t total_cand, int32_t capacity, int32_t num_q_heads,
                            int32_t max_splits);
/* The number of KV splits echo_verify_attn uses for a batch of num_requests requests x num_kv_heads KV heads on this
 * context (its device's SM count and ECHO_OPT_FORCE_SPLITS): the max_splits to size the workspace with. */
int echo_attn_splits(EchoCtx* ctx, int32_t num_requests, int32_t num_kv_heads);
const char* echo_strerror(int code);
const char* echo_last_error(EchoCtx* ctx);  /* text of the last ECHO_ERR_CUDA on this context */
/* Copies the device status word to *flags with a blocking 4-byte copy on `stream` and clears it. */
int echo_device_status(EchoCtx* ctx, uint32_t* flags, echo_stream_t stream);
int echo_set_option(EchoCtx* ctx, int key, int64_t value);
/* Measurement helpers (bench.py).  echo_launch_count: kernels this library has launched in this process so far (a
 * host-side counter).  echo_probe_sm_clock: queues a one-thread kernel on `stream` that spins ~20 us and writes the SM
 * clock it ran at, in MHz, to the DEVICE float *mhz_dev (cycle counter / global timer): the clock under load, which
 * NVML does not show for kernels shorter than its sampling period. */
uint64_t echo_launch_count(void);
int echo_probe_sm_clock(EchoCtx* ctx, float* mhz_dev, echo_stream_t stream);

/* ---- problem statement ----------------------------------- */
/* Candidate draft trees G_i with parent function pa(j) and draft log-probabilities (Eq. 5). */
typedef struct {
  int32_t num_requests;     /* R >= 0 */
  int32_t total_cand;       /* N = sum C_i */
  int32_t max_cand_per_req; /* max C_i, <= ECHO_MAX_CAND */
  const int32_t* cand_offsets; /* dev [R+1], CSR, cand_offsets[0] = 0 */
  const int32_t* parent;       /* dev [N], request-local, -1 = root, parent[j] < j (topological) */
  const float* logq;           /* dev [N], natural log of the draft confidence q(x|h), <= 0 (R:G-2) */
} EchoTrees;

#define ECHO_SCHED_TOPB 0
#define ECHO_SCHED_ALG1 1

/* Gate and scheduler parameters: Alg. 1 inputs (K_max, D_sig, tau, W_max). */
typedef struct {
  uint32_t depth_mask; /* bit d set <=> d in D_sig (Eq. 7) */
  float log_tau[32];   /* natural log of tau_d; compared as max_j S > log_tau[d], strict (R:G-4) */
  int32_t w_max;       /* Phase-2 width cap per truncated request; 0 = no widening */
  int32_t budget;      /* K_max >= 0 (Eq. 4) */
  int32_t static_k;    /* 0 = elastic global top-B; >0 = per-request top-static_k, gates off (R:G-15) */
  int32_t schedule;    /* ECHO_SCHED_TOPB: global top-B by path score inside a tier (north_star, R:G-10);
                          ECHO_SCHED_ALG1: Algorithm 1 as printed, P:127-160 -- Phase 1 depth by depth, request order
                          inside a depth, a level best-first by (S desc, node asc); Phase 2 over the truncated
                          requests in truncation order (R:L-1..L-4).  Ignored when static_k > 0. */
  int32_t cand_index_base; /* 0, or -- when several ranks share one budget (echo_gate_keys / echo_gate_select_keys) --
                              the number of candidates of the ranks before this one: keys carry the global candidate
                              index, so ties break by (rank, request, node) and keys stay unique across ranks */
  int32_t request_base;    /* likewise the number of requests of the ranks before this one (ECHO_SCHED_ALG1 keys) */
} EchoGate;

/* Packed ragged batch ("Flatten & Pack", Fig. 3(3)): request asc, node asc (R:P-1). */
typedef struct {
  int32_t capacity;       /* >= budget (elastic) or >= min(N, R*static_k) (static) */
  int32_t* n_selected;    /* dev [1] */
  int32_t* sel_offsets;   /* dev [R+1] CSR over packed nodes; K_i = sel_offsets[i+1]-sel_offsets[i] */
  int32_t* sel_node;      /* dev [capacity] request-local candidate id */
  int32_t* sel_req;       /* dev [capacity] */
  int32_t* parent_local;  /* dev [capacity] packed request-local parent index, -1 = root */
  uint8_t* sel_depth;     /* dev [capacity] */
  uint32_t* anc_mask;     /* dev [capacity][4] ancestor-or-self bits over packed local indices */
  float* path_score;      /* dev [N]  S (Eq. 5) */
  uint8_t* cand_depth;    /* dev [N] */
  int32_t* cut_depth;     /* dev [R] first failing gated depth, ECHO_CUT_NEVER if none */
} EchoSelection;

/* Paged KV cache (R:A-2, A-3): pools bf16 [num_layers][num_pages][num_kv_heads][16][128];
 * token position t of request i lives in page page_table[i][t/16], slot t%16.  The packed tree
 * node with local index l is tentatively appended at position prefix_len[i] + l. */
typedef struct {
  int32_t num_kv_heads, head_dim /* 128 */, page_size /* 16 */, num_pages, max_pages_per_req, num_layers;
  void* k_pool;              /* dev, 16-byte aligned */
  void* v_pool;              /* dev, 16-byte aligned */
  const int32_t* page_table; /* dev [R][max_pages_per_req] */
  const int32_t* prefix_len; /* dev [R]  P_i >= 0 */
} EchoPagedKV;

/* What the target model said (greedy): tokens directly, or bf16 logits to argmax. */
typedef struct {
  const int32_t* draft_token;  /* dev [capacity] packed order */
  const int32_t* prev_token;   /* dev [R] target's greedy token after the committed prefix (R:C-2) */
  const int32_t* target_token; /* dev [capacity] target's greedy token AFTER each packed node, or NULL */
  const void* target_logits;   /* dev bf16 [capacity][ld], 16-byte aligned, or NULL; exactly one of the two */
  int32_t vocab;               /* V (argmax over columns < V) */
  int64_t ld;                  /* row stride in elements, >= V, multiple of 8 */
} EchoVerifyResult;

typedef struct {
  int32_t* accept_len;   /* dev [R] accepted draft nodes on the chosen path (R:C-5) */
  int32_t* last_node;    /* dev [R] packed index of the deepest accepted node, -1 if none */
  int32_t* bonus_token;  /* dev [R] target token after last_node, -1 if none */
  int32_t* new_len;      /* dev [R] P_i + accept_len */
  int32_t* accept_idx;   /* dev [R][32] packed indices along the path, -1 padded */
  int32_t* slot_src;     /* dev [R][32] KV slot (page*16+offset) each path node is read from */
  int32_t* slot_dst;     /* dev [R][32] KV slot it is moved to (position P_i + t) */
  int32_t* target_token_out; /* dev [capacity] argmax result (logits form), may be NULL */
} EchoAccept;

/* ---- the three calls of the hot path ------------------------------------------------------ */

/* S1-S5: fp32 path scores accumulated root->leaf (Eq. 5), layer confidence and sparse
 * gate in the log domain (Eq. 6-7), budgeted global top-B selection with depth
 * extension (tier 0) strictly before width expansion (tier 1) (Eq. 4, Alg. 1, priority
 * P:162-167), ties by (score desc, request, node); then packing and 128-bit ancestor masks.
 * Writes every field of `out`.  Needs workspace >= echo_workspace_bytes(R, N, capacity, 0). */
int echo_gate_select(EchoCtx* ctx, const EchoTrees* trees, const EchoGate* gate, EchoSelection* out,
                     echo_stream_t stream);

/* S6-S7: ragged tree-masked paged GQA attention (the "specialized operators for irregular batch
 * shapes"; definition R:A-1..A-8).  For packed node k = (i,l) and query head h
 * (KV head h / (Hq/Hkv)): softmax over positions [0,P_i) and P_i + a for every set bit a of
 * anc_mask[k], logits sm_scale * <q, k_t>; out = sum p_t v_t (bf16, RNE), lse = ln sum exp.
 * q/out: dev bf16 [capacity][num_q_heads][128], 16-byte aligned; lse: dev f32 [capacity][num_q_heads].
 * Rows k >= n_selected are not written.  Slots past P_i + K_i may hold any bits, NaN included. */
int echo_verify_attn(EchoCtx* ctx, const EchoSelection* sel, const EchoPagedKV* kv, int32_t layer,
                     int32_t num_q_heads, int32_t num_requests, const void* q, void* out, float* lse,
                     float sm_scale, echo_stream_t stream);

/* S8-S10: optional fused argmax over bf16 target logits (lowest index wins ties, R:C-3), greedy
 * acceptance = longest accepted root-to-leaf path (max depth, then lowest local index; P:52,
 * P:199, R:C-1..C-5), and in-place compaction of the accepted KV rows of all layers to positions
 * P_i .. P_i+L-1, every read before any write to the same slot column (R:C-6). */
int echo_accept(EchoCtx* ctx, const EchoSelection* sel, const EchoVerifyResult* res, int32_t num_requests,
                EchoPagedKV* kv, EchoAccept* out, echo_stream_t stream);

/* ---- one budget shared by several ranks (request-sharded multi-GPU) ---------- */
/* echo_gate_select in two halves around the one exchange the path has: every rank computes S1-S2 and the 64-bit
 * selection keys of its own candidates (echo_gate_keys; keys[total_cand] device, caller-owned; ~0 = not eligible),
 * the ranks all-gather their keys (N x 8 B each, e.g. ncclAllGather; ranks with fewer candidates pad with ~0), and
 * every rank selects against the whole population and packs its own requests (echo_gate_select_keys: the budget-th
 * smallest of all_keys[n_all] is the threshold; local_keys are this rank's, indexed like cand_offsets).  With
 * all_keys == local_keys the pair equals echo_gate_select.  gate->cand_index_base / request_base must be the exclusive
 * prefix sums of total_cand / num_requests over the ranks, and gate->budget the global K_max on every rank. */
int echo_gate_keys(EchoCtx* ctx, const EchoTrees* trees, const EchoGate* gate, EchoSelection* out, uint64_t* keys,
                   echo_stream_t stream);
int echo_gate_select_keys(EchoCtx* ctx, const EchoTrees* trees, const EchoGate* gate, const uint64_t* local_keys,
                          const uint64_t* all_keys, int64_t n_all, EchoSelection* out, echo_stream_t stream);

/* ---- S8 over vocabulary-sharded logits (tensor-parallel ranks) ----------------- */
/* When the ranks shard the KV heads (attention needs no collective), the target logits are sharded over the
 * vocabulary: rank r holds logits_shard = dev bf16 [capacity][ld], columns [vocab_base, vocab_base + vocab_shard) of
 * every packed node's row (ld >= vocab_shard, ld % 8 == 0, 16-byte aligned; vocab_base + vocab_shard < 2^31).  The
 * greedy target token (first maximum, -0 == +0, R:C-3) then needs the one exchange this split has:
 *   echo_argmax_shard: pairs_out[k] (dev u64 [capacity], caller-owned) = (order-preserving image of the shard's
 *     maximum, -0 taken as +0) << 32 | (2^31 - 1 - global index of its first occurrence) for k < n_selected, 0 for
 *     the rows behind: a greater key is a greater value, then a lower index;
 *   the ranks all-gather their pairs (capacity x 8 B each, e.g. ncclAllGather) into pairs_all = dev u64
 *     [world][capacity];
 *   echo_argmax_merge: target_token_out[k] (dev i32 [capacity]) = the index in the greatest of the row's `world` keys,
 *     k < n_selected -- what echo_accept computes from the unsharded logits -- to be handed to echo_accept as
 *     EchoVerifyResult.target_token.
 * A shard whose logits are all -inf reports its first index, so an all -inf row yields token 0 like echo_accept. */
int echo_argmax_shard(EchoCtx* ctx, const EchoSelection* sel, const void* logits_shard, int64_t ld, int32_t vocab_shard,
                      int32_t vocab_base, uint64_t* pairs_out, echo_stream_t stream);
int echo_argmax_merge(EchoCtx* ctx, const EchoSelection* sel, const uint64_t* pairs_all, int32_t world,
                      int32_t* target_token_out, echo_stream_t stream);

/* ---- a call that allocates nothing -------------------------------------------------------- */
/* echo_gate_select for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid it): no context, no workspace.  The scratch the selection needs -- the 64-bit selection keys
 * [total_cand] and the threshold, which echo_gate_select keeps in the context's workspace -- lives in a fixed array of
 * ECHO_NOALLOC_SCRATCH_BYTES (256 + 8 * ECHO_NOALLOC_MAX_CAND = 512.25 KB) that is part of the library image: every
 * GPU that loads libecho.so holds it until the process exits.  The call makes no cudaMalloc / cudaFree and calls no
 * allocating library routine; it runs the three-kernel form of the step (score + keys, radix select, pack), results
 * identical to echo_gate_select.
 *   - Runs on the calling thread's CURRENT device (compute capability 10.0, else ECHO_ERR_ARCH); `stream` and every
 *     dev pointer must belong to it.  The first call on a device looks up the array's device address (once per
 *     device): make that first call outside stream capture.
 *   - trees / gate / out: as for echo_gate_select; out->capacity >= min(budget, total_cand) (static_k: num_requests *
 *     static_k).  `status`: dev [1], caller-owned; the ECHO_DEV_* bits of data-dependent violations are OR-ed into it
 *     (the caller zeroes it when it wants to).
 *   - total_cand > ECHO_NOALLOC_MAX_CAND -> ECHO_ERR_TOO_LARGE, nothing is launched.
 *   - Every call on a device shares the one array, which keeps the last call's contents; nothing in it has to start
 *     at zero (every word a call reads it has written before).  Calls that overlap on the GPU -- two streams, two
 *     threads, two processes' worth of graphs replayed at once -- RACE on it: serialise them on one stream. */
#define ECHO_NOALLOC_MAX_CAND 65536
#define ECHO_NOALLOC_SCRATCH_BYTES (256 + 8 * (size_t)ECHO_NOALLOC_MAX_CAND)
int echo_gate_select_noalloc(const EchoTrees* trees, const EchoGate* gate, EchoSelection* out, uint32_t* status,
                             echo_stream_t stream);

/* ---- acceptance at temperature > 0 ----------------------------------- */
typedef struct {
  const int32_t* draft_token; /* dev [capacity], packed order */
  const void* target_logits;  /* dev bf16 [capacity][ld]: the target's logits after each packed node */
  const void* root_logits;    /* dev bf16 [R][ld]: the target's logits after the last committed token of each request */
  int32_t vocab;
  int64_t ld;                 /* row pitch in elements, multiple of 8; rows 16-byte aligned */
  float temperature;          /* > 0 */
  const float* u_accept;      /* dev [capacity]: uniform [0,1) draws, one per packed node (used when the node is tried) */
  const float* u_bonus;       /* dev [R]: uniform [0,1) draws for the bonus tokens */
} EchoSampleInputs;
/* Tree acceptance under the speculative-sampling conditions in the multi-round form of tree drafters
 * whose proposals are their deterministic top-k (q = 1 on a proposed token; readings R:T-1..T-4): from the
 * distribution p = softmax(root_logits / T) of a request, the children of the current node are tried in packed order;
 * child c with token x is accepted iff u_accept[c] < p'(x), where p' is p with the tokens already rejected at this
 * node removed and renormalised; an accepted child becomes the current node (p = softmax(target_logits[c] / T)); when
 * none is accepted, bonus_token is drawn from p' by inverse CDF in vocabulary order with u_bonus.  Every emitted token
 * is distributed exactly as the target's p.  Probabilities are fp32 (ex2.approx), so a draw within ~1e-5 of its
 * threshold may fall either way.  Outputs and KV compaction as echo_accept (target_token_out unused).  Needs
 * (capacity + R) * 8 bytes of context workspace. */
int echo_accept_stochastic(EchoCtx* ctx, const EchoSelection* sel, const EchoSampleInputs* in, int32_t num_requests,
                           EchoPagedKV* kv, EchoAccept* out, echo_stream_t stream);

/* ---- draft-side tree construction ------------------------------------ */
/* The draft model's outputs for one level: every node of the previous level (one virtual root with score 0 at level 0,
 * else topk nodes in their slot order) proposes its topk most likely next tokens with their log-probabilities. */
typedef struct {
  int32_t level, topk;        /* 0 <= level < 32, 1 <= topk <= ECHO_MAX_TOPK */
  const float* parent_score;  /* dev [R][k_prev]: cumulative scores of the previous level (zeros at level 0) */
  const float* child_logq;    /* dev [R][k_prev][topk], natural log, <= 0 */
  const int32_t* child_token; /* dev [R][k_prev][topk] */
} EchoDraftLevel;
/* Appends level `level` to every request's candidate tree in place ("G_i.append(topk tokens)", Alg. 1 l.10):
 * the topk candidates with the best cumulative score fl32(S_parent + logq) (Eq. 5), ties by (parent slot, child rank),
 * become nodes cand_offsets[i] + level*topk + slot with parent (level-1)*topk + parent slot (-1 at level 0), their logq
 * and token; score_out [R][topk] is the next call's parent_score.  trees->parent / logq (written here, hence not
 * const in effect) and token [total_cand] are caller-owned device arrays with room for (level+1)*topk nodes per request
 * (status bit otherwise).  Readings R:D-1..D-3. */
int echo_draft_expand(EchoCtx* ctx, const EchoDraftLevel* draft, EchoTrees* trees, int32_t* token, float* score_out,
                      echo_stream_t stream);

/* ---- warm-up calibration of the gates ------------------------------ */
/* Traces collected during warm-up: one sample per (request, depth) with the layer confidence
 * c_{i,d} (Eq. 6, a probability in [0, 1]) and whether the node the target then took at that depth was accepted. */
typedef struct {
  int64_t num_samples;     /* M >= 0 */
  const uint8_t* depth;    /* dev [M], < 32 */
  const float* conf;       /* dev [M], in [0, 1], no NaN */
  const uint8_t* accepted; /* dev [M], 0 / 1 */
} EchoTraces;
typedef struct {
  double* auc;          /* dev [32]: AUC_d, 0.5 where a class is missing */
  float* tau;           /* dev [32]: tau_d (an observed confidence), 0 where a class is missing */
  int32_t* n_pos;       /* dev [32]: accepted samples at depth d */
  int32_t* n_neg;       /* dev [32]: rejected samples at depth d */
  uint32_t* depth_mask; /* dev [1]: bit d <=> d in D_sig */
} EchoCalibration;
/* "Offline Calibration": per depth, AUC_d of the confidences of accepted vs rejected samples
 * (Hanley & McNeil 1982: (#{c+ > c-} + 0.5 #{c+ == c-}) / (n+ n-), computed exactly on integers and divided once in
 * fp64); D_sig = {d : both classes present and AUC_d > delta}; tau_d = the smallest observed confidence v that
 * maximises J(v) = #{c+ > v}/n+ - #{c- > v}/n- (the gate is c > tau, Eq. 7; readings R:K-1..K-3).  The caller turns
 * tau into EchoGate.log_tau on the host (R:G-2).  Needs a context workspace of ECHO_CALIB_WORKSPACE_BYTES; at most
 * ECHO_CALIB_MAX_PER_DEPTH samples per depth (more: status bit, the excess is dropped).  Asynchronous on `stream`. */
int echo_calibrate(EchoCtx* ctx, const EchoTraces* traces, double delta, EchoCalibration* out, echo_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* ECHO_H_ */
