// S6 on the 5th-gen tensor cores: persistent, warp-specialised split-KV verify attention.
//
//   work item   = (request i, KV head, 128-row tile of (node, head-in-group) rows, KV split); KV tile = 128 tokens
//   warp 12     = K producer, warp 14 = V producer (all lanes walk the loop, one elected lane issues): one 4-D TMA
//                 box per page (16 tokens x 128 d of one KV head), pages looked up in the page table one tile ahead.
//                 "Stage empty" is S-full (K) / S-free (V) of the same tile index, not a barrier of its own.
//                 The Q tile (3-D tensor map over [node][head][d]) is loaded by the QK^T issuer, warp 13.
//   warp 13     = issuer of S = Q K^T (SS, K-major x K-major) into one of three S buffers in TMEM
//   warp 15     = issuer of O += P V (TS: P read from TMEM where the softmax wrote it over S, V as the MN-major B
//                 operand straight from its TMA layout); accumulators never leave TMEM
//   warps 0-7   = softmax, two warpgroups that take ALTERNATE KV tiles (thread = one whole row of 128 columns): while
//                 one warpgroup waits for its S tile, loads it from TMEM or hands P back, the other one computes, so
//                 the two warps of an SM sub-partition are never stalled together.  Weights are taken against the
//                 fixed reference 0 (fp32 and bf16 share the exponent range, so no running maximum is needed while
//                 the row sums stay inside [2^-90, 2^100]); tree mask only in tiles that touch positions >= P_i; every
//                 2^x on MUFU (ex2.approx), packed f32x2 FMA / ADD; P written back to TMEM as bf16 over S.
//   warps 8-11  = epilogue: O / l -> bf16 out + lse (or the fp32 split partial) while the softmax is on the next item;
//                 it also checks the row sums: an item with a sum outside the window is flagged and redone at the end
//                 by the same CTA in the SAFE form (running row maximum, O rescaled in TMEM; warpgroup 0 alone).
//   setmaxnreg  : softmax 192, epilogue 80, producer / issuer warps 40 registers
// Each KV page is read once per (KV head, row tile) and serves all rows of the tile.
// Operator definition: include/echo.h (paper: P:39, P:85 names it only; readings R:A-1..A-8).
#include <cuda.h>

#include "common.cuh"
#include "tc_ptx.cuh"

namespace {

constexpr int D = 128;
constexpr int PAGE = 16;
constexpr int TILE_M = 128;
constexpr int TILE_N = 128;
constexpr int NSTAGE = 3;
constexpr int HALF_BYTES = TILE_N * 128;     // Q tile: [128 rows][64 bf16] per d-half, 128-byte rows, SW128
constexpr int TILE_BYTES = 2 * HALF_BYTES;   // both d-halves: 32 KB
constexpr int PAGE_BYTES = PAGE * D * 2;  // one TMA box: [2 token groups][2 d-halves][8 tokens][64 d], 4 KB
constexpr int GROUP_BYTES = 2048;         // 8 tokens x 128 d: d-half 0 (1 KB SW128 atom), then d-half 1
constexpr int SMEM_Q = 0;
constexpr int SMEM_K = SMEM_Q + TILE_BYTES;
constexpr int SMEM_V = SMEM_K + NSTAGE * TILE_BYTES;
// float stats[5][128] of the item just finished: warpgroup 0's weight sum (exact), normaliser, reference; warpgroup
// 1's weight sum and normaliser (single-buffered: the epilogue hands it back through B_STATFREE as soon as it is read)
constexpr int SMEM_STATS = SMEM_V + NSTAGE * TILE_BYTES;
constexpr int ST_L0 = 0, ST_N0 = 1, ST_M0 = 2, ST_L1 = 3, ST_N1 = 4;
constexpr int SMEM_BAR = SMEM_STATS + 5 * TILE_M * 4;
constexpr int BAR_BYTES = 256;                      // up to 32 mbarriers
constexpr int SMEM_TMEM_SLOT = SMEM_BAR + BAR_BYTES;  // 16 bytes
constexpr int SMEM_REDO = SMEM_TMEM_SLOT + 16;        // bitmap over this CTA's items: redo in the safe form
constexpr int REDO_WORDS = 60;
constexpr int REDO_CAP = REDO_WORDS * 32;  // items of a CTA beyond this take the safe form at once
constexpr int SMEM_TOTAL = SMEM_REDO + REDO_WORDS * 4;  // = 227 KB exactly; dynamic smem is declared 1024-byte aligned
static_assert(SMEM_TOTAL <= 232448, "shared memory budget");
// warpgroups 0 and 1 (warps 0-3, 4-7) softmax; warpgroup 2 (warps 8-11) epilogue; warpgroup 3: warp 12 K producer,
// 13 QK^T MMA issuer, 14 V + Q producer, 15 PV MMA issuer
constexpr int NTHREADS = 512;
constexpr int W_EPI = 8, W_PROD_K = 12, W_MMA_QK = 13, W_PROD_V = 14, W_MMA_PV = 15;
constexpr int REGS_SOFTMAX = 192, REGS_EPILOGUE = 80, REGS_AUX = 40;  // 128 * (2 * 192 + 80 + 40) <= 512 * 128, the launch allocation
static_assert(NSTAGE == 3, "K / V stage g % NSTAGE and S buffer g % NSBUF must be the same index");
constexpr int NSBUF = 3;        // S / P buffers in TMEM: the QK^T of tile j+2 is issued before the PV of tile j
constexpr int TMEM_O = NSBUF * TILE_N;
constexpr int TMEM_COLS = 512;  // S_b [128 b, 128 b + 128) for b < 3, O [384,512); P_b aliases S_b[0,64)
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;
// The fast form takes every weight as 2^(s * scale * log2e) with no reference subtracted.  fp32 sums and bf16 weights
// both carry 8 exponent bits, so the result is the same as with a running maximum as long as nothing overflows and
// what underflows is negligible: an item whose row sum ends inside [2^-90, 2^100] has every weight <= 2^100 and has
// lost at most 2^-126 per key to flush-to-zero (< 2^-21 of the sum over 32 768 keys).  Anything else -- inf, NaN
// included -- sends the item to the safe form.
constexpr float SUM_LO = 8.0779356694631609e-28f;  // 2^-90
constexpr float SUM_HI = 1.2676506002282294e30f;   // 2^100

constexpr uint32_t IDESC_QK = tc::idesc_bf16(TILE_M, TILE_N, 0, 0);
constexpr uint32_t IDESC_PV = tc::idesc_bf16(TILE_M, D, 0, 1);

// barrier indices (8 bytes each)
enum { B_QFULL = 0, B_QEMPTY = 1, B_KFULL = 2, B_VFULL = 5, B_SFULL = 8, B_PFULL = 11, B_SFREE = 14, B_OFULL = 17,
       B_OFREE = 18, B_STATS = 19, B_STATFREE = 20, B_PHASE = 21, B_COUNT = 22 };
static_assert(B_COUNT * 8 <= BAR_BYTES, "barrier region");

struct AttnParams {
  const int4* items;
  const int32_t* n_items;
  const int32_t* sel_offsets;
  const uint4* anc_mask;
  const int32_t* page_table;
  const int32_t* prefix_len;
  int max_pages, Hkv, Hq, G, log2G;
  int page_row_base;  // layer * num_pages
  __nv_bfloat16* out;
  float* lse;
  float scale_log2;
  int splits;
  int force_safe;  // test hook: every item takes the safe form
  float* part_o;
  float* part_lse;
  size_t n_rows_cap;
  uint32_t* status;
  // in-kernel planning (plan_in_kernel != 0): every CTA builds the work list itself and writes its own records
  int plan_in_kernel, R, max_items, max_rt;
  int4* items_w;
  int32_t* n_items_w;
};
// Up to INPLAN_MAX (request, split) entries are planned inside the attention kernel (one entry per thread, NTHREADS);
// tile counts above INPLAN_BUCKETS - 1 share the last bucket (as in k_plan).
constexpr int INPLAN_MAX = 512;
constexpr int INPLAN_BUCKETS = 1024;

// Optional wait-time profile (build with -DECHO_WAIT_PROF): cycles each role spends blocked on each mbarrier,
// per CTA, read back with echo_debug_wait_prof (csrc/debug_prof.h).  Compiled out otherwise.
#ifdef ECHO_WAIT_PROF
#include "debug_prof.h"
__device__ unsigned long long g_wait_prof[ECHO_PROF_CTAS][ECHO_PROF_SLOTS];
__device__ long long g_trace[256][8];
#define PROF_T0() const long long prof_t0_ = clock64()
#define PROF_ADD(slot) prof_[slot] += clock64() - prof_t0_
#define PROF_WAIT(slot, b, ph) do { const long long t_ = clock64(); tc::mbar_wait(b, ph); prof_[slot] += clock64() - t_; } while (0)
#define PROF_WAIT_RELAXED(slot, b, ph) do { const long long t_ = clock64(); tc::mbar_wait_relaxed(b, ph); prof_[slot] += clock64() - t_; } while (0)
#define PROF_WAIT_BACKOFF(slot, b, ph) do { const long long t_ = clock64(); tc::mbar_wait_backoff(b, ph); prof_[slot] += clock64() - t_; } while (0)
#define PROF_DECL(n) unsigned long long prof_[n] = {}
#define PROF_FLUSH(base, n) do { if (blockIdx.x < ECHO_PROF_CTAS) for (int q_ = 0; q_ < n; ++q_) g_wait_prof[blockIdx.x][(base) + q_] = prof_[q_]; } while (0)
#define PROF_SPAN_BEGIN() const long long span_t_ = clock64()
#define PROF_SPAN_END(slot) prof_[slot] += clock64() - span_t_
#define PROF_COUNT(slot) prof_[slot] += 1
#define TRACE(gg, ev) do { if (blockIdx.x == 0 && (gg) < 256 && lane == 0) g_trace[gg][ev] = clock64(); } while (0)
#define TRACE_K(ev) do { if (blockIdx.x == 0 && threadIdx.x == 0) g_trace[255][ev] = clock64(); } while (0)
#define PROF_SPAN2_BEGIN() const long long span2_t_ = clock64()
#define PROF_SPAN2_END(slot) prof_[slot] += clock64() - span2_t_
#else
#define PROF_T0() do {} while (0)
#define PROF_ADD(slot) do {} while (0)
#define PROF_WAIT(slot, b, ph) tc::mbar_wait(b, ph)
#define PROF_WAIT_RELAXED(slot, b, ph) tc::mbar_wait_relaxed(b, ph)
#define PROF_WAIT_BACKOFF(slot, b, ph) tc::mbar_wait_backoff(b, ph)
#define PROF_DECL(n) do {} while (0)
#define PROF_FLUSH(base, n) do {} while (0)
#define PROF_SPAN_BEGIN() do {} while (0)
#define PROF_SPAN_END(slot) do {} while (0)
#define PROF_COUNT(slot) do {} while (0)
#define PROF_SPAN2_BEGIN() do {} while (0)
#define PROF_SPAN2_END(slot) do {} while (0)
#define TRACE(gg, ev) do {} while (0)
#define TRACE_K(ev) do {} while (0)
#endif

// work item record written by k_plan: two int4 = {req, kvh | rt<<8 | split<<16, jt0, jt1} {P_i, sel_offsets[i], K_i, 0}
struct Item { int req, kvh, rt, split, jt0, jt1, P, off, Ki; };
__device__ __forceinline__ Item decode(const int4 v, const int4 w) {
  Item it;
  it.req = v.x; it.kvh = v.y & 0xff; it.rt = (v.y >> 8) & 0xff; it.split = (v.y >> 16) & 0xff; it.jt0 = v.z; it.jt1 = v.w;
  it.P = w.x; it.off = w.y; it.Ki = w.z;
  return it;
}
// snake order over the length-sorted work list: round k of CTA c takes k*G+c (k even) or (k+1)*G-1-c (k odd)
__device__ __forceinline__ int item_index(int k, int cta, int grid) {
  return (k & 1) ? (k + 1) * grid - 1 - cta : k * grid + cta;
}

// Work-list records without a global load per item: every lane of a warp holds the record of one of the CTA's items
// k with k / 32 == blk (lane = k % 32), fetched 32 at a time, and an item's fields are broadcast by shuffles.  Under a
// saturated memory system a dependent global load costs 2500-3500 cycles; per-item loads at the item boundaries, in
// six roles one after another, were a third of the kernel (event trace, round 2).  A prefetch held in registers does
// not help: ptxas spills it right behind the load, which then waits for it.
struct ItemFeed {
  int4 r0, r1;
  int blk;
  __device__ __forceinline__ void init() { blk = -1; r0 = r1 = make_int4(0, 0, 0, 0); }
  __device__ __forceinline__ void ensure(const int4* items, int k, int cta, int grid, int n_items, int lane) {
    if ((k >> 5) != blk) {  // warp-uniform
      blk = k >> 5;
      const int idx = item_index((k & ~31) + lane, cta, grid);
      r0 = r1 = make_int4(0, 0, 0, 0);  // past the end of the list: an item without nodes or tiles
      if (idx < n_items) { r0 = items[2 * idx]; r1 = items[2 * idx + 1]; }
    }
  }
  // record of item k (any k of the block held), the same in every lane
  __device__ __forceinline__ Item get(const int4* items, int k, int cta, int grid, int n_items, int lane) {
    ensure(items, k, cta, grid, n_items, lane);
    const int src = k & 31;
    int4 a, b;
    a.x = __shfl_sync(0xffffffffu, r0.x, src); a.y = __shfl_sync(0xffffffffu, r0.y, src);
    a.z = __shfl_sync(0xffffffffu, r0.z, src); a.w = __shfl_sync(0xffffffffu, r0.w, src);
    b.x = __shfl_sync(0xffffffffu, r1.x, src); b.y = __shfl_sync(0xffffffffu, r1.y, src);
    b.z = __shfl_sync(0xffffffffu, r1.z, src); b.w = 0;
    return decode(a, b);
  }
};

// Every role walks the same sequence of items: first the CTA's share of the work list (phase 0; the items past
// REDO_CAP in the safe form), then -- once the epilogue has seen the last row sums (B_PHASE) -- the items it flagged,
// in the safe form.  fn(k, safe), k = the item's ordinal in the CTA's list.
template <typename Fn, typename Between>
__device__ __forceinline__ void walk_items(int cta, int grid, int n_items, bool force_safe, const volatile uint32_t* redo,
                                           uint32_t bar_phase, Between&& between, Fn&& fn) {
  // ONE call site of fn for both phases: the per-item code is cold (it runs once per ~14 KV tiles), and instruction
  // fetches that miss under a saturated memory system cost hundreds of cycles per 128-byte line -- every duplicate
  // of the item body is paid for at every item boundary.
  for (int ph = 0; ph < 2; ++ph) {
    if (ph == 1) {
      between();
      tc::mbar_wait_relaxed(bar_phase, 0);
      uint32_t any = 0;
#pragma unroll 4
      for (int w = 0; w < REDO_WORDS; ++w) any |= redo[w];
      if (!any) break;
    }
    for (int k = 0; item_index(k, cta, grid) < n_items; ++k) {  // item indices grow with k
      if (ph == 1 && (k >= REDO_CAP || !((redo[k >> 5] >> (k & 31)) & 1u))) continue;
      fn(k, ph, ph == 1 || force_safe || k >= REDO_CAP);
    }
  }
}

__device__ __forceinline__ uint32_t mask_word(const uint4& m, int w) {
  return w == 0 ? m.x : w == 1 ? m.y : w == 2 ? m.z : w == 3 ? m.w : 0u;
}
// visibility of tokens t0..t0+31 for a row with ancestor mask m: t < P, or bit (t - P) of m (R:A-1, A-2)
__device__ __forceinline__ uint32_t visible_word(const uint4& m, int P, int t0) {
  const int npref = P - t0;
  uint32_t bits = npref >= 32 ? 0xffffffffu : npref <= 0 ? 0u : ((1u << npref) - 1u);
  const int a0 = t0 - P;
  if (a0 >= 0) {
    if (a0 < 128) bits |= __funnelshift_r(mask_word(m, a0 >> 5), mask_word(m, (a0 >> 5) + 1), a0 & 31);
  } else if (a0 > -32) {
    bits |= m.x << (-a0);
  }
  return bits;
}

__device__ __forceinline__ void mask_chunk(uint32_t (&s)[32], uint32_t vis) {
#pragma unroll
  for (int e = 0; e < 32; ++e)
    if (!((vis >> e) & 1u)) s[e] = 0xff800000u;  // -inf
}

// weights p = 2^(s*scale_log2 + neg_m) of one 32-column chunk of a row: packed to bf16 in pk, added to the exact fp32
// partial sums in acc.  Packed f32x2 FMA / ADD halve the issue slots: straight-line FFMA2 / MUFU.EX2 / F2FP / FADD2.  A
// masked key arrives as -inf and MUFU turns it into 0.  (Round 1-2 took every fourth pair's 2^x on the FMA pipe by a
// degree-3 polynomial to relieve MUFU; with the present structure that costs 2.5 % -- A/B on one box, cfg2 0.2630 vs
// 0.2563 ms, static-60 0.656 vs 0.642 -- XU is at 42 % of its peak without it.)
__device__ __forceinline__ void weights_chunk(const uint32_t (&sc)[32], uint64_t sc2, uint64_t nm2, uint32_t (&pk)[16],
                                              uint64_t (&acc)[4]) {
#pragma unroll
  for (int e = 0; e < 32; e += 2) {
    const uint64_t x2 = tc::fma_f32x2(tc::pack_f32x2(__uint_as_float(sc[e]), __uint_as_float(sc[e + 1])), sc2, nm2);
    float x0, x1;
    tc::unpack_f32x2(x2, x0, x1);
    const float p0 = tc::ex2(x0), p1 = tc::ex2(x1);
    pk[e >> 1] = tc::pack_bf16(p0, p1);
    acc[(e >> 1) & 3] = tc::add_f32x2(acc[(e >> 1) & 3], tc::pack_f32x2(p0, p1));
  }
}

__device__ __forceinline__ float acc_total(const uint64_t (&acc)[4]) {
  float a0, a1;
  tc::unpack_f32x2(tc::add_f32x2(tc::add_f32x2(acc[0], acc[1]), tc::add_f32x2(acc[2], acc[3])), a0, a1);
  return a0 + a1;
}

// One S row (128 fp32 columns in TMEM at tS) -> bf16 P over its first 64 columns, four 32-column chunks, the load of
// chunk c+1 in flight while chunk c is processed.  ts = exact sum of the weights.  This is the hot loop of the kernel:
// every key inside the prefix, no visibility logic, fully unrolled.
__device__ __forceinline__ void tile_weights_fast(uint32_t tS, float scale_log2, float neg_m, float& ts) {
  const uint64_t sc2 = tc::pack_f32x2(scale_log2, scale_log2), nm2 = tc::pack_f32x2(neg_m, neg_m);
  uint64_t acc[4] = {0ull, 0ull, 0ull, 0ull};  // 8 independent fp32 partial sums
  uint32_t s0[32], s1[32];
  tc::tmem_ld32(tS, s0);
  // two chunks per trip (the two register buffers by name), the loop itself rolled: half the code of the kernel's
  // hottest path -- the whole kernel has to live in a 32 KB instruction cache next to the per-item code
#pragma unroll 1
  for (int c = 0; c < 4; c += 2) {
    uint32_t pk[16];
    tc::tmem_wait_ld();
    tc::reg_fence32(s0);
    tc::tmem_ld32(tS + 32 * (c + 1), s1);
    weights_chunk(s0, sc2, nm2, pk, acc);
    tc::tmem_st16(tS + 16 * c, pk);  // P columns [16c, 16c+16) lie inside S chunks already read (c/2 <= c)
    tc::tmem_wait_ld();
    tc::reg_fence32(s1);
    if (c == 0) tc::tmem_ld32(tS + 64, s0);
    weights_chunk(s1, sc2, nm2, pk, acc);
    tc::tmem_st16(tS + 16 * (c + 1), pk);
  }
  ts = acc_total(acc);
}

// A tile that touches the tree or the ragged end (once or twice per item) goes through the SAME hot loop: first the
// invisible keys of the row are overwritten with -inf in TMEM (chunks every row of the warp sees whole are skipped),
// afterwards the bf16 weights just stored are summed for the normaliser (few visible keys: O must stay an exact convex
// combination of V rows; lse always takes the exact sum).  Both passes are small rolled loops on purpose: code that
// runs once per item is fetched from L2 every time, and a separate unrolled masked instantiation of the tile body
// cost ~3000 cycles per item in instruction misses (event trace, round 2).
__device__ __forceinline__ void mask_tile_in_tmem(uint32_t tS, const uint32_t (&vis)[4]) {
#pragma unroll 1
  for (int c = 0; c < 4; ++c) {
    const uint32_t v = c == 0 ? vis[0] : c == 1 ? vis[1] : c == 2 ? vis[2] : vis[3];
    if (__all_sync(0xffffffffu, v == 0xffffffffu)) continue;  // warp-uniform
    uint32_t s[32];
    tc::tmem_ld32(tS + 32 * c, s);
    tc::tmem_wait_ld();
    tc::reg_fence32(s);
    mask_chunk(s, v);
    tc::tmem_st32(tS + 32 * c, s);
  }
  tc::tmem_wait_st();
}
__device__ __forceinline__ float rounded_sum_of_p(uint32_t tS) {  // P = bf16 pairs in columns [0,64)
  float r0 = 0.f, r1 = 0.f;
  tc::tmem_wait_st();
#pragma unroll 1
  for (int c = 0; c < 2; ++c) {
    uint32_t pk[32];
    tc::tmem_ld32(tS + 32 * c, pk);
    tc::tmem_wait_ld();
    tc::reg_fence32(pk);
#pragma unroll
    for (int e = 0; e < 32; ++e) {
      r0 += __uint_as_float(pk[e] << 16);
      r1 += __uint_as_float(pk[e] & 0xffff0000u);
    }
  }
  return r0 + r1;
}

// row maximum of S (masked keys already hold -inf), for the safe form
__device__ __forceinline__ float row_max_pass(uint32_t tS) {
  float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll 1
  for (int c = 0; c < 4; ++c) {
    uint32_t s[32];
    tc::tmem_ld32(tS + 32 * c, s);
    tc::tmem_wait_ld();
    tc::reg_fence32(s);
#pragma unroll
    for (int e = 0; e < 32; e += 4) {
      mx0 = tc::max3(mx0, __uint_as_float(s[e]), __uint_as_float(s[e + 1]));
      mx1 = tc::max3(mx1, __uint_as_float(s[e + 2]), __uint_as_float(s[e + 3]));
    }
  }
  return fmaxf(mx0, mx1);
}

__global__ void __launch_bounds__(NTHREADS, 1) k_verify_attn_tc(const __grid_constant__ CUtensorMap tmap_q,
                                                                const __grid_constant__ CUtensorMap tmap_k,
                                                                const __grid_constant__ CUtensorMap tmap_v,
                                                                const AttnParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t sbase = tc::smem_u32(smem_raw);
  const uint32_t sQ = sbase + SMEM_Q, sK = sbase + SMEM_K, sV = sbase + SMEM_V, sBar = sbase + SMEM_BAR;
  uint8_t* gen_base = smem_raw;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(gen_base + SMEM_TMEM_SLOT);
  volatile uint32_t* redo = reinterpret_cast<volatile uint32_t*>(gen_base + SMEM_REDO);
  float* stats = reinterpret_cast<float*>(gen_base + SMEM_STATS);
  auto bar = [&](int i) -> uint32_t { return sBar + 8u * i; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cta = blockIdx.x, grid = gridDim.x;
  TRACE_K(0);
  pdl_launch_dependents();  // echo_accept's kernel may queue behind this one (it waits for our completion itself)

  if (threadIdx.x == 0) {
    if (sbase & 1023u) atomicOr(p.status, ECHO_DEV_INTERNAL);  // SW128 operand tiles need 1024-byte alignment
    for (int i = 0; i < B_COUNT; ++i) {
      const uint32_t cnt = (i >= B_PFULL && i < B_PFULL + NSBUF) ? 4u  /* one arrival per warp of the owning warpgroup */
                           : (i == B_OFREE || i == B_STATFREE || i == B_PHASE) ? 128u
                           : (i == B_STATS) ? 256u : 1u;
      tc::mbar_init(bar(i), cnt);
    }
    tc::fence_barrier_init();
    tc::prefetch_tmap(&tmap_q);
    tc::prefetch_tmap(&tmap_k);
    tc::prefetch_tmap(&tmap_v);
  }
  if (threadIdx.x < REDO_WORDS) redo[threadIdx.x] = 0u;
  if (warp == W_MMA_QK) tc::tmem_alloc(sbase + SMEM_TMEM_SLOT, TMEM_COLS);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  TRACE_K(1);
  // Programmatic dependent launch: everything above (barrier init, TMEM allocation, descriptor prefetch) overlaps
  // the kernel before (k_plan, or the gate's); sel_offsets / the work list are read only after it has completed.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  TRACE_K(2);
  int n_items;
  if (p.plan_in_kernel) {
    // The work list without a launch of its own (k_plan: ~5 us in front of every attention call, 10 % of cfg1): every
    // CTA computes the whole placement -- entries (request, split) bucketed by tile count, longest first, ties by
    // entry index, so that all CTAs agree -- and writes only the records the snake order gives to itself.  Scratch:
    // the K ring, which no TMA has written yet.
    static_assert(NTHREADS == INPLAN_MAX && INPLAN_BUCKETS == 2 * NTHREADS, "one entry and two buckets per thread");
    int* s_bkt = reinterpret_cast<int*>(gen_base + SMEM_K);
    int* s_cnt = s_bkt + INPLAN_MAX;
    int* s_hist = s_cnt + INPLAN_MAX;
    int* s_wsum = s_hist + INPLAN_BUCKETS;
    const int t = threadIdx.x;
    s_hist[2 * t] = 0;
    s_hist[2 * t + 1] = 0;
    int bkt = -1, cnt = 0, r = 0, sp = 0, j0 = 0, j1 = 0, n_rt = 1, P = 0, off = 0, Ki = 0;
    if (t < p.R * p.splits) {
      r = t / p.splits;
      sp = t - r * p.splits;
      off = p.sel_offsets[r];
      P = p.prefix_len[r];
      Ki = p.sel_offsets[r + 1] - off;
      if (Ki > ECHO_MAX_CAND) {  // more packed nodes than a request can have: clamp and flag (never silently truncate)
        if (cta == 0) atomicOr(p.status, ECHO_DEV_CAND_OVERFLOW);
        Ki = ECHO_MAX_CAND;
      }
      if (Ki > 0) {
        const int n_tiles = (P + Ki + TILE_N - 1) / TILE_N;
        n_rt = min((Ki * p.G + TILE_M - 1) / TILE_M, p.max_rt);
        const int tps = (n_tiles + p.splits - 1) / p.splits;
        j0 = sp * tps;
        j1 = min(n_tiles, j0 + tps);
        if (j0 < n_tiles) {
          cnt = p.Hkv * n_rt;
          bkt = INPLAN_BUCKETS - 1 - min(j1 - j0, INPLAN_BUCKETS - 1);
        }
      }
    }
    s_bkt[t] = bkt;
    s_cnt[t] = cnt;
    __syncthreads();
    if (cnt > 0) atomicAdd(&s_hist[bkt], cnt);
    __syncthreads();
    const int h0 = s_hist[2 * t], h1 = s_hist[2 * t + 1];
    int incl = h0 + h1;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int v = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += v;
    }
    if (lane == 31) s_wsum[warp] = incl;
    __syncthreads();  // (also: every bucket count has been read)
    if (warp == 0) {
      int w = lane < NTHREADS / 32 ? s_wsum[lane] : 0;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, w, o);
        if (lane >= o) w += v;
      }
      s_wsum[lane] = w;
    }
    __syncthreads();
    const int base = incl - (h0 + h1) + (warp ? s_wsum[warp - 1] : 0);
    s_hist[2 * t] = base;  // first position of the bucket (bucket 0 = longest)
    s_hist[2 * t + 1] = base + h0;
    n_items = min(s_wsum[31], p.max_items);
    __syncthreads();
    if (cnt > 0) {
      int pos = s_hist[bkt];
      for (int e = 0; e < t; ++e)
        if (s_bkt[e] == bkt) pos += s_cnt[e];
      for (int q = 0; q < cnt; ++q) {
        const int idx = pos + q;
        const int rnd = idx / grid, pp = idx - rnd * grid;
        if (((rnd & 1) ? grid - 1 - pp : pp) == cta && idx < p.max_items) {  // item_index(rnd, cta, grid) == idx
          const int kvh = q / n_rt, rt = q - kvh * n_rt;
          p.items_w[2 * idx] = make_int4(r, kvh | (rt << 8) | (sp << 16), j0, j1);
          p.items_w[2 * idx + 1] = make_int4(P, off, Ki, 0);
        }
      }
    }
    if (cta == 0 && t == 0) *p.n_items_w = n_items;
    tc::fence_proxy_async();  // the scratch is done with before the TMA writes the K ring
    __threadfence_block();
    __syncthreads();          // this CTA's records are in place for its own readers
  } else {
    n_items = *p.n_items;
  }
  const bool force_safe = p.force_safe != 0;

  if (warp >= 12) tc::setmaxnreg_dec<REGS_AUX>();
  if (warp == W_PROD_K || warp == W_PROD_V) {
    // ============================== TMA producers: K ring, V ring + Q ==============================
    // A page (16 tokens x 128 d of one KV head, 4 KB contiguous in the pool) is one 4-D box {64 d, 8 tokens, 2 d-halves,
    // 2 token groups}; a 128-token tile is eight of them, their ids read from the page table by lanes 0-7 one tile
    // ahead.  All 32 lanes walk the loop (same addresses, same values: every TMA operand is provably warp-uniform),
    // one elected lane issues.  (The Q tile is loaded by the QK^T issuer itself.)
    {
      const bool is_k = warp == W_PROD_K;
      const uint32_t s_dst = is_k ? sK : sV;
      const CUtensorMap* tmap = is_k ? &tmap_k : &tmap_v;
      // "stage empty" is not a barrier of its own: K stage g % 3 is free when QK^T of tile g has completed, which is
      // what B_SFULL[g % 3] says, and V stage g % 3 when PV of tile g has, which is B_SFREE[g % 3] (NSTAGE == NSBUF, one
      // tile counter).  Every tcgen05.commit costs the issuing thread ~150 cycles in the queue it shares with the MMAs
      // (`mio` stalls on UTCBAR, ncu source page): two commits per tile less.
      const int b_full = is_k ? B_KFULL : B_VFULL, b_empty = is_k ? B_SFULL : B_SFREE;
      int g = 0, itc = 0;
      PROF_DECL(3);
      PROF_T0();
      ItemFeed feed;
      feed.init();
      auto fetch = [&](int k) {  // record of item k with every field provably warp-uniform (TMA operands)
        const Item t = feed.get(p.items, k, cta, grid, n_items, lane);
        Item it;
        it.req = tc::uniform(t.req); it.kvh = tc::uniform(t.kvh); it.rt = tc::uniform(t.rt); it.split = 0;
        it.jt0 = tc::uniform(t.jt0); it.jt1 = tc::uniform(t.jt1); it.P = tc::uniform(t.P); it.off = tc::uniform(t.off);
        it.Ki = tc::uniform(t.Ki);
        return it;
      };
      auto n_pages = [&](const Item& it) { return min((it.P + it.Ki + PAGE - 1) / PAGE, p.max_pages); };
      auto tile_page = [&](const Item& it, int j) -> int {  // lane e < 8: id of page e of tile j (0 past the end)
        const int pi = j * 8 + (lane & 7);
        return pi < n_pages(it) ? p.page_table[(size_t)it.req * p.max_pages + pi] : 0;
      };
      int cur = 0;            // page ids of the tile about to be issued, fetched one tile ahead -- across items too
      bool cur_valid = false;
      // `ahead`: the item after this one in the list (phase 0), whose first tile's page ids are requested before this
      // item ends, or nullptr
      auto produce = [&](const Item& it, const Item* ahead) {
        const int total = it.P + it.Ki;
        if ((total + PAGE - 1) / PAGE > p.max_pages && is_k && lane == 0)
          atomicOr(p.status, ECHO_DEV_PAGE_OVERFLOW);  // page table too short: flag, load what exists
        const int npages = n_pages(it);
        if (!cur_valid) cur = tile_page(it, it.jt0);
        for (int j = it.jt0; j < it.jt1; ++j, ++g) {
          int nxt = 0;
          cur_valid = false;
          if (j + 1 < it.jt1) nxt = tile_page(it, j + 1);
          else if (ahead && ahead->jt1 > ahead->jt0) { nxt = tile_page(*ahead, ahead->jt0); cur_valid = true; }
          const int slot = g % NSTAGE, ph = (g / NSTAGE) & 1;
          const int npv = max(0, min(8, npages - j * 8));  // pages of this tile that hold tokens
          const uint32_t dst = s_dst + slot * TILE_BYTES;
          const uint32_t fb = bar(b_full + slot);
          int pg[8];
#pragma unroll
          for (int e = 0; e < 8; ++e) pg[e] = __shfl_sync(0xffffffffu, cur, e);
          PROF_WAIT_BACKOFF(1, bar(b_empty + slot), ph ^ 1);
          if (tc::elect_one()) {
            tc::mbar_expect_tx(fb, npv * PAGE_BYTES);
#pragma unroll
            for (int e = 0; e < 8; ++e) {
              if (e < npv) {
                const int grp = ((p.page_row_base + pg[e]) * p.Hkv + it.kvh) * (PAGE / 8);  // 8-token group index
                tc::tma_load_4d(dst + e * PAGE_BYTES, tmap, fb, 0, 0, 0, grp);
              }
            }
          }
          __syncwarp();
          cur = nxt;
        }
        ++itc;
      };
      walk_items(cta, grid, n_items, force_safe, redo, bar(B_PHASE), [&]() { cur_valid = false; }, [&](int k, int ph, bool) {
        const Item it = fetch(k);
        const bool more = ph == 0 && item_index(k + 1, cta, grid) < n_items;
        Item nx = it;
        if (more) nx = fetch(k + 1);  // same 32-block except once in 32 items
        if (ph == 1) cur_valid = false;
        produce(it, more ? &nx : nullptr);
      });
      PROF_ADD(0);
      if (lane == 0) PROF_FLUSH(is_k ? 0 : 4, 3);
    }
  } else if (warp == W_MMA_QK) {
    // ============================== MMA issuer for S = Q K^T (one lane) ==============================
    // Two issuing threads, one per product: a single thread retires a 128x128x16 tcgen05.mma only every ~110
    // cycles, two threads keep the tensor pipe at 70-85 cycles per instruction (measured).  This thread runs up to
    // NSBUF tiles ahead of the PV issuer; S/P buffer b is handed back through B_SFREE when the PV that read P_b is done.
    // All 32 lanes walk the loop (every operand warp-uniform), one elected lane issues.
    {
      int g = 0, itc = 0;
      PROF_DECL(6);
      PROF_T0();
      const uint32_t tmem_u = (uint32_t)tc::uniform((int)tmem);
      const uint64_t qdesc = tc::smem_desc_sw128(sQ, 16, 1024);
      ItemFeed feed;
      feed.init();
      // This warp also loads the Q tile: it is the one that knows when the last QK^T of the previous item has read
      // it (its own commit), so the load goes out the moment the buffer is free instead of when a producer warp gets
      // there (1300 cycles later on average); and three tiles before an item ends it pulls the next item's Q tile
      // into L2, which turns the 2600-cycle load at the boundary into an L2 hit (a prefetch a whole item ahead is
      // evicted again: the KV stream turns the L2 over every ~20 us).
      auto q_coords = [&](const Item& t, int& h0, int& node0) {
        h0 = tc::uniform(t.kvh) * p.G;
        node0 = tc::uniform(t.off) + tc::uniform(t.rt) * (TILE_M >> p.log2G);
      };
      auto issue = [&](int k, int ph, bool) {
        const Item rec = feed.get(p.items, k, cta, grid, n_items, lane);
        const int n = tc::uniform(rec.jt1 - rec.jt0);
        int h0, node0;
        q_coords(rec, h0, node0);
        PROF_WAIT(3, bar(B_QEMPTY), (itc & 1) ^ 1);
        if (tc::elect_one()) {
          tc::mbar_expect_tx(bar(B_QFULL), TILE_BYTES);
          tc::tma_load_3d(sQ, &tmap_q, bar(B_QFULL), 0, h0, node0);
          tc::tma_load_3d(sQ + HALF_BYTES, &tmap_q, bar(B_QFULL), 64, h0, node0);
        }
        __syncwarp();
        const bool more = ph == 0 && item_index(k + 1, cta, grid) < n_items;
        int h1 = 0, node1 = 0;
        if (more) q_coords(feed.get(p.items, k + 1, cta, grid, n_items, lane), h1, node1);
        PROF_WAIT(3, bar(B_QFULL), itc & 1);
        TRACE(g, 7);
        for (int j = 0; j < n; ++j, ++g) {
          if (more && j == max(0, n - 4)) {
            if (tc::elect_one()) {
              tc::tma_prefetch_3d(&tmap_q, 0, h1, node1);
              tc::tma_prefetch_3d(&tmap_q, 64, h1, node1);
            }
            __syncwarp();
          }
          const int slot = g % NSTAGE;
          PROF_WAIT(1, bar(B_KFULL + slot), (g / NSTAGE) & 1);
          const int b = g % NSBUF;
          PROF_WAIT(2, bar(B_SFREE + b), ((g / NSBUF) & 1) ^ 1);  // PV of tile g - NSBUF has read P_b
          tc::tc_fence_after();
          // K tile: 8-token groups GROUP_BYTES apart (SBO), d-half at +1 KB inside a group
          const uint64_t kdesc = tc::smem_desc_sw128(sK + slot * TILE_BYTES, 16, GROUP_BYTES);
          TRACE(g, 0);
          if (tc::elect_one()) {
#pragma unroll
            for (int kk = 0; kk < D / 16; ++kk) {
              const uint32_t q16 = ((kk & 3) * 32 + (kk >> 2) * HALF_BYTES) >> 4;
              const uint32_t k16 = ((kk & 3) * 32 + (kk >> 2) * 1024) >> 4;
              tc::mma_ss(tmem_u + b * TILE_N, qdesc + q16, kdesc + k16, IDESC_QK, kk > 0);
            }
            tc::mma_commit(bar(B_SFULL + b));  // S_b is complete and K stage `slot` (== b) is free
            if (j == n - 1) tc::mma_commit(bar(B_QEMPTY));
          }
          __syncwarp();
          TRACE(g, 1);
        }
        ++itc;
      };
      walk_items(cta, grid, n_items, force_safe, redo, bar(B_PHASE), []() {}, issue);
      PROF_ADD(0);
      if (lane == 0) PROF_FLUSH(8, 4);
    }
    __syncwarp();
  } else if (warp == W_MMA_PV) {
    // ============================== MMA issuer for O += P V (one lane) ==============================
    {
      int g = 0, itc = 0;
      const uint32_t tmem_u = (uint32_t)tc::uniform((int)tmem);
      const uint32_t tO = tmem_u + TMEM_O;
      ItemFeed feed;
      feed.init();
      auto issue = [&](int k, int, bool) {
        const Item rec = feed.get(p.items, k, cta, grid, n_items, lane);
        const int n = tc::uniform(rec.jt1 - rec.jt0);
        for (int j = 0; j < n; ++j, ++g) {
          const int b = g % NSBUF, slot = g % NSTAGE;
          tc::mbar_wait(bar(B_PFULL + b), (g / NSBUF) & 1);
          tc::mbar_wait(bar(B_VFULL + slot), (g / NSTAGE) & 1);
          if (j == 0) tc::mbar_wait(bar(B_OFREE), (itc & 1) ^ 1);  // epilogue of the previous item has read O
          tc::tc_fence_after();
          // V tile as MN-major B: 64-wide d atoms 1 KB apart (LBO), 8-token groups GROUP_BYTES apart (SBO).
          // P (bf16 pairs) sits in columns [0,64) of S_b: 16 tokens = 8 columns per MMA.
          const uint64_t vdesc = tc::smem_desc_sw128(sV + slot * TILE_BYTES, 1024, GROUP_BYTES);
          TRACE(g, 4);
          if (tc::elect_one()) {
#pragma unroll
            for (int kk = 0; kk < TILE_N / 16; ++kk)
              tc::mma_ts(tO, tmem_u + b * TILE_N + kk * 8, vdesc + ((kk * 2 * GROUP_BYTES) >> 4), IDESC_PV, (j > 0) || (kk > 0));
            tc::mma_commit(bar(B_SFREE + b));  // P_b has been read and V stage `slot` (== b) is free
            if (j == n - 1) tc::mma_commit(bar(B_OFULL));
          }
          __syncwarp();
          TRACE(g, 5);
        }
        ++itc;
      };
      walk_items(cta, grid, n_items, force_safe, redo, bar(B_PHASE), []() {}, issue);
    }
    __syncwarp();
  } else if (warp < W_EPI) {
    // ============================== softmax (warpgroups 0 and 1, thread = row) ==============================
    // Warpgroup w takes the KV tiles with g & 1 == w (g counted over the CTA's whole run), thread = row.  The two warps
    // of an SM sub-partition are then on different tiles and out of step: one computes while the other waits for S,
    // loads it from TMEM or hands P back.  (Tried: both warpgroups on the two token halves of one tile, separate
    // barriers per half -- they run in lockstep and 64 columns cost 1380 cycles instead of 800; halves of 64 tokens
    // with their own QK^T products -- the N = 64 product re-reads Q for half the work and is bound by shared-memory
    // reads.)  In the safe form warpgroup 0 takes every tile and keeps the running row maximum.  Each warpgroup adds
    // up the weights of its tiles and publishes them once per item; the epilogue adds the two.
    tc::setmaxnreg_inc<REGS_SOFTMAX>();
    int wg = warp >> 2;
    asm volatile("" : "+r"(wg));  // keep it in a register: recomputing it from %tid (S2R) in every loop costs ~5 %
    const int wq = warp & 3;   // TMEM lane quarter this warp may access
    const int row = wq * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(wq * 32) << 16;
    int g = 0, itc = 0;
    PROF_DECL(7);
    PROF_T0();
#ifdef ECHO_WAIT_PROF
    long long gap_t_ = clock64();
#endif
    auto do_item = [&](const Item& it, const uint4& mk, const bool safe) {
      const int P = it.P, total = it.P + it.Ki;
      // A warp none of whose 32 rows belongs to a node (the last row tile of a request is ragged: a quarter to a third
      // of all row-warps at the configs of BASELINE.json) computes nothing -- whatever its TMEM lanes hold goes through
      // PV into O rows that are never stored -- but keeps every barrier's pace: it waits for S like the others (so it
      // cannot run a phase ahead of P-full), helps zero the ragged V rows, and arrives.
      const bool idle = ((it.rt * TILE_M + wq * 32) >> p.log2G) >= it.Ki;
      float m_used = safe ? -INFINITY : 0.f, lsum = 0.f, lnorm = 0.f;
      const uint32_t tO = tmem + TMEM_O + lane_addr;
      // fast form: warpgroup w takes the tiles with g & 1 == w; safe form: warpgroup 0 takes all of them
      const int n_t = it.jt1 - it.jt0, g_first = g, g_end = g + n_t;
      const int first = safe ? (wg ? n_t : 0) : ((g ^ wg) & 1), step = safe ? 1 : 2;
      g += first;
      for (int j = it.jt0 + first; j < it.jt1; j += step, g += step) {
        const int b = g % NSBUF;
        const uint32_t tS = tmem + b * TILE_N + lane_addr;
#ifdef ECHO_WAIT_PROF
        prof_[4] += clock64() - gap_t_;
#endif
        PROF_WAIT(1, bar(B_SFULL + b), (g / NSBUF) & 1);
        PROF_SPAN_BEGIN();
        if (wq == 0) TRACE(g, 2);
        const int tile0 = j * TILE_N;
        if (!idle) {
        tc::tc_fence_after();
        const bool masked = tile0 + TILE_N > P;  // the tile touches tree positions or the ragged end
        uint32_t vis[4] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu};
        if (masked) {
#pragma unroll
          for (int c = 0; c < 4; ++c) vis[c] = visible_word(mk, P, tile0 + 32 * c);
        }
        float ts = 0.f, tr = 0.f;  // this tile's exact weight sum / share of the normaliser
        if (masked) mask_tile_in_tmem(tS, vis);
        float neg_ref = 0.f;
        if (safe) {
          // safe form: row maximum first, O rescaled in TMEM when the reference moves (all lanes take the same path:
          // the TMEM instructions are warp-wide)
          const float mx = row_max_pass(tS);
          const float m_new = fmaxf(m_used, mx * p.scale_log2);
          float alpha = 1.f;
          if (m_new > m_used) {
            alpha = (m_used == -INFINITY) ? 0.f : tc::ex2(m_used - m_new);
            m_used = m_new;
          }
          lsum *= alpha;
          lnorm *= alpha;
          if (g > g_first && __any_sync(0xffffffffu, alpha != 1.f)) {  // O holds PV of earlier tiles
            // every PV issued so far must have landed: the last one is PV(g-1), whose commit frees its S buffer.  That
            // barrier is at most one phase behind here (QK(g) was issued after PV(g-3), hence PV(g-4), was done), so
            // the parity wait is unambiguous -- one shared "PV done" barrier can lag by two phases and let O be
            // rescaled under a running PV.
            PROF_WAIT(3, bar(B_SFREE + (g - 1) % NSBUF), ((g - 1) / NSBUF) & 1);
            tc::tc_fence_after();
#pragma unroll 1
            for (int c = 0; c < 4; ++c) {
              uint32_t o[32];
              tc::tmem_ld32(tO + c * 32, o);
              tc::tmem_wait_ld();
              tc::reg_fence32(o);
#pragma unroll
              for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * alpha);
              tc::tmem_st32(tO + c * 32, o);
            }
            tc::tmem_wait_st();
          }
          neg_ref = (m_used == -INFINITY) ? 0.f : -m_used;
        }
        tile_weights_fast(tS, p.scale_log2, neg_ref, ts);
        tr = (masked || safe) ? rounded_sum_of_p(tS) : ts;
        lsum += ts;
        lnorm += tr;
        tc::tmem_wait_st();
        }
        if (tile0 + TILE_N > total) {  // ragged end: V rows past the last token may hold anything (R:A-7)
          const int slot = g % NSTAGE;
          PROF_WAIT(4, bar(B_VFULL + slot), (g / NSTAGE) & 1);
          if (row >= total - tile0) {  // both d-halves of V row `row`
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              uint4* z = reinterpret_cast<uint4*>(gen_base + SMEM_V + slot * TILE_BYTES + (row >> 3) * GROUP_BYTES + h * 1024 +
                                                 (row & 7) * 128);
#pragma unroll
              for (int e = 0; e < 8; ++e) z[e] = make_uint4(0u, 0u, 0u, 0u);
            }
          }
          tc::fence_proxy_async();
        }
        tc::tc_fence_before();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(bar(B_PFULL + b));
        if (wq == 0) TRACE(g, 3);
        PROF_SPAN_END(5);
        PROF_COUNT(6);
#ifdef ECHO_WAIT_PROF
        gap_t_ = clock64();
#endif
      }
      g = g_end;
      // ---- publish this warpgroup's sums (and warpgroup 0's reference) for the epilogue ----
      PROF_SPAN2_BEGIN();
      PROF_WAIT(2, bar(B_STATFREE), (itc & 1) ^ 1);  // the epilogue has read the statistics of the previous item
      stats[(wg ? ST_L1 : ST_L0) * TILE_M + row] = lsum;
      stats[(wg ? ST_N1 : ST_N0) * TILE_M + row] = lnorm;
      if (wg == 0) stats[ST_M0 * TILE_M + row] = (m_used == -INFINITY) ? 0.f : m_used;
      tc::mbar_arrive(bar(B_STATS));
      PROF_SPAN2_END(3);
      ++itc;
    };
    // Records come from the lane-distributed feed; the rows' ancestor masks likewise: the 32 rows of a warp belong to
    // npw = 32 / G nodes, so the 32 lanes hold the masks of `slots` = 32 / npw consecutive items (lane = slot * npw +
    // node), fetched together every `slots` items -- one exposed load latency per block instead of one per item.
    ItemFeed feed;
    feed.init();
    const int npw = p.log2G < 5 ? (32 >> p.log2G) : 1, slots = 32 / npw;
    uint4 mblk = make_uint4(0u, 0u, 0u, 0u);
    int mblk_k0 = -(1 << 30);
    auto item_mask = [&](int k, bool stream) -> uint4 {
      if (!stream) {  // redo phase: items come out of order, one load per item
        const Item t = feed.get(p.items, k, cta, grid, n_items, lane);
        const int l = (t.rt * TILE_M + row) >> p.log2G;
        return l < t.Ki ? p.anc_mask[t.off + l] : make_uint4(0u, 0u, 0u, 0u);
      }
      if (k - mblk_k0 >= slots) {  // warp-uniform
        mblk_k0 = k - (k % slots);
        const int kk = mblk_k0 + lane / npw;  // same 32-block as k: slots divides 32
        feed.ensure(p.items, k, cta, grid, n_items, lane);
        const int rt = (__shfl_sync(0xffffffffu, feed.r0.y, kk & 31) >> 8) & 0xff;
        const int off = __shfl_sync(0xffffffffu, feed.r1.y, kk & 31), Ki = __shfl_sync(0xffffffffu, feed.r1.z, kk & 31);
        const int l = ((rt * TILE_M + wq * 32) >> p.log2G) + lane % npw;
        mblk = l < Ki ? p.anc_mask[off + l] : make_uint4(0u, 0u, 0u, 0u);
      }
      const int src = (k - mblk_k0) * npw + (p.log2G < 5 ? (lane >> p.log2G) : 0);
      uint4 m;
      m.x = __shfl_sync(0xffffffffu, mblk.x, src); m.y = __shfl_sync(0xffffffffu, mblk.y, src);
      m.z = __shfl_sync(0xffffffffu, mblk.z, src); m.w = __shfl_sync(0xffffffffu, mblk.w, src);
      return m;
    };
    walk_items(cta, grid, n_items, force_safe, redo, bar(B_PHASE), []() {}, [&](int k, int ph, bool safe) {
      const Item it = feed.get(p.items, k, cta, grid, n_items, lane);
      const uint4 mk = item_mask(k, ph == 0);
      do_item(it, mk, safe);
    });
    PROF_ADD(0);
    if ((warp & 3) == 0 && lane == 0) PROF_FLUSH(16 + 8 * wg, 7);
  } else if (warp < W_PROD_K) {
    // ============================== epilogue (warpgroup 2, thread = row) ==============================
    // O of item n is normalised and stored here while the softmax warpgroups are already on item n+1.  The row sums
    // of the fast form are checked here: outside the window -> the item's bit in the redo bitmap.
    tc::setmaxnreg_dec<REGS_EPILOGUE>();
    const int wq = warp & 3;
    const int row = wq * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(wq * 32) << 16;
    int itc = 0;
    PROF_DECL(3);
    PROF_T0();
    ItemFeed feed;
    feed.init();
    auto finish = [&](int k, int, bool safe) {
      const Item it = feed.get(p.items, k, cta, grid, n_items, lane);
      const int r_glob = it.rt * TILE_M + row;
      const int l = r_glob >> p.log2G, gq = r_glob & (p.G - 1);
      const bool valid = l < it.Ki;
      const uint32_t tO = tmem + TMEM_O + lane_addr;
      const size_t rowg = (size_t)(it.off + l) * p.Hq + it.kvh * p.G + gq;
      PROF_WAIT_RELAXED(1, bar(B_STATS), itc & 1);
      const float lsum = stats[ST_L0 * TILE_M + row] + stats[ST_L1 * TILE_M + row];
      const float lnorm = stats[ST_N0 * TILE_M + row] + stats[ST_N1 * TILE_M + row];
      const float m_ref = stats[ST_M0 * TILE_M + row];
      tc::mbar_arrive(bar(B_STATFREE));
      if (!safe) {
        const bool bad = valid && !(lsum >= SUM_LO && lsum <= SUM_HI);
        if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(const_cast<uint32_t*>(redo) + (k >> 5), 1u << (k & 31));
      }
      const float inv = lnorm > 0.f ? 1.f / lnorm : 0.f;
      const float lse_v = lsum > 0.f ? (m_ref + log2f(lsum)) * LN2 : -INFINITY;
      PROF_WAIT(2, bar(B_OFULL), itc & 1);
      tc::tc_fence_after();
      // rolled on purpose (this code runs once per item and is fetched from L2 every time); O is handed back to the
      // PV issuer as soon as its last chunk is in registers, before that chunk is converted and stored
#pragma unroll 1
      for (int c = 0; c < 4; ++c) {
        uint32_t oc[32];
        tc::tmem_ld32(tO + c * 32, oc);
        tc::tmem_wait_ld();
        tc::reg_fence32(oc);
        if (c == 3) {
          tc::tc_fence_before();
          tc::mbar_arrive(bar(B_OFREE));
        }
        if (valid) {
          if (p.splits == 1) {
            uint4* dst = reinterpret_cast<uint4*>(p.out + rowg * D + c * 32);
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              uint4 w;
              w.x = tc::pack_bf16(__uint_as_float(oc[8 * e + 0]) * inv, __uint_as_float(oc[8 * e + 1]) * inv);
              w.y = tc::pack_bf16(__uint_as_float(oc[8 * e + 2]) * inv, __uint_as_float(oc[8 * e + 3]) * inv);
              w.z = tc::pack_bf16(__uint_as_float(oc[8 * e + 4]) * inv, __uint_as_float(oc[8 * e + 5]) * inv);
              w.w = tc::pack_bf16(__uint_as_float(oc[8 * e + 6]) * inv, __uint_as_float(oc[8 * e + 7]) * inv);
              dst[e] = w;
            }
          } else {
            float4* dst = reinterpret_cast<float4*>(p.part_o + ((size_t)it.split * p.n_rows_cap + rowg) * D + c * 32);
#pragma unroll
            for (int e = 0; e < 8; ++e)
              dst[e] = make_float4(__uint_as_float(oc[4 * e + 0]) * inv, __uint_as_float(oc[4 * e + 1]) * inv,
                                   __uint_as_float(oc[4 * e + 2]) * inv, __uint_as_float(oc[4 * e + 3]) * inv);
          }
        }
      }
      if (valid) {
        if (p.splits == 1) p.lse[rowg] = lse_v;
        else p.part_lse[(size_t)it.split * p.n_rows_cap + rowg] = lse_v;
      }
      ++itc;
    };
    // between the phases: the bitmap is final (release); every role, this one included, then reads it
    walk_items(cta, grid, n_items, force_safe, redo, bar(B_PHASE), [&]() { tc::mbar_arrive(bar(B_PHASE)); }, finish);
    PROF_ADD(0);
    if (warp == W_EPI && lane == 0) PROF_FLUSH(12, 3);
  }

  // ---- teardown ----
  tc::tc_fence_before();
  __syncthreads();
  TRACE_K(3);
  if (warp == W_MMA_QK) tc::tmem_dealloc(tmem, TMEM_COLS);
}

// Device-side planner: P_i and K_i exist only on the device, so the work list is built there.
// Items are bucketed by KV-tile count (descending) so that the snake assignment balances CTAs.
constexpr int PLAN_THREADS = 256;   // one request per thread and pass at the batch sizes of BASELINE.json; a small CTA syncs faster
constexpr int PLAN_BUCKETS = 1024;  // tile counts above 1023 (131 k tokens) share the last bucket
__global__ void __launch_bounds__(PLAN_THREADS) k_plan(const int32_t* __restrict__ sel_offsets,
                                                       const int32_t* __restrict__ prefix_len, int R, int Hkv, int G,
                                                       int splits, int max_items, int max_rt, int4* __restrict__ items,
                                                       int32_t* __restrict__ n_items, uint32_t* __restrict__ status) {
  __shared__ int s_cnt[PLAN_BUCKETS];
  __shared__ int s_warp[32];
  pdl_launch_dependents();  // let k_verify_attn_tc set itself up meanwhile
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int b = tid; b < PLAN_BUCKETS; b += PLAN_THREADS) s_cnt[b] = 0;
  if (tid < 32) s_warp[tid] = 0;
  const int P_first = tid < R ? prefix_len[tid] : 0;  // the caller's: loaded while the kernel before this one drains
  pdl_wait();                                        // sel_offsets come from echo_gate_select's kernels
  __syncthreads();
  auto for_items = [&](auto&& fn) {
    for (int r = tid; r < R; r += PLAN_THREADS) {
      const int off = sel_offsets[r], P = r == tid ? P_first : prefix_len[r];
      int Ki = sel_offsets[r + 1] - off;
      if (Ki <= 0) continue;
      if (Ki > ECHO_MAX_CAND) {  // more packed nodes than a request can have: clamp and flag (never silently truncate)
        atomicOr(status, ECHO_DEV_CAND_OVERFLOW);
        Ki = ECHO_MAX_CAND;
      }
      const int n_tiles = (P + Ki + TILE_N - 1) / TILE_N;
      const int n_rt = min((Ki * G + TILE_M - 1) / TILE_M, max_rt);
      const int tps = (n_tiles + splits - 1) / splits;
      for (int s = 0; s * tps < n_tiles; ++s) {
        const int j0 = s * tps, j1 = min(n_tiles, j0 + tps);
        fn(r, s, j0, j1, n_rt, P, off, Ki);
      }
    }
  };
  for_items([&](int, int, int j0, int j1, int n_rt, int, int, int) {
    atomicAdd(&s_cnt[PLAN_BUCKETS - 1 - min(j1 - j0, PLAN_BUCKETS - 1)], Hkv * n_rt);
  });
  __syncthreads();
  {  // exclusive scan over buckets (bucket 0 = longest)
    const int per = PLAN_BUCKETS / PLAN_THREADS;
    int loc[per], sum = 0;
    for (int t = 0; t < per; ++t) { loc[t] = s_cnt[tid * per + t]; sum += loc[t]; }
    int incl = sum;
    for (int o = 1; o < 32; o <<= 1) { int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      int w = s_warp[lane];
      for (int o = 1; o < 32; o <<= 1) { int v = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += v; }
      s_warp[lane] = w;
    }
    __syncthreads();
    int run = incl - sum + (warp ? s_warp[warp - 1] : 0);
    for (int t = 0; t < per; ++t) { s_cnt[tid * per + t] = run; run += loc[t]; }
    if (tid == PLAN_THREADS - 1) *n_items = min(run, max_items);
  }
  __syncthreads();
  for_items([&](int r, int s, int j0, int j1, int n_rt, int P, int off, int Ki) {
    const int pos0 = atomicAdd(&s_cnt[PLAN_BUCKETS - 1 - min(j1 - j0, PLAN_BUCKETS - 1)], Hkv * n_rt);
    int pos = pos0;
    for (int kvh = 0; kvh < Hkv; ++kvh)
      for (int rt = 0; rt < n_rt; ++rt, ++pos)
        if (pos < max_items) {
          items[2 * pos] = make_int4(r, kvh | (rt << 8) | (s << 16), j0, j1);
          items[2 * pos + 1] = make_int4(P, off, Ki, 0);
        }
  });
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

}  // namespace

// Tensor maps are a pure function of (base pointer, shape): the context keeps the few it has encoded (the Q buffers of
// a double-buffered serving loop, the K and V pools) instead of calling the driver three times per launch.
struct TmapCache {
  struct Entry {
    const void* base;
    uint64_t a, b, c;  // shape key
    CUtensorMap map;
  };
  static constexpr int N = 16;
  Entry e[N];
  int used = 0, next = 0;
};

void free_tmap_cache(TmapCache* c) { delete c; }

// Copies the map out: a later insertion of the same call may recycle the slot a hit was found in.
static int cached_tmap(EchoCtx* ctx, CUtensorMap* out, const void* base, uint64_t a, uint64_t b, uint64_t c,
                       int (*encode)(EchoCtx*, CUtensorMap*, const void*, uint64_t, uint64_t, uint64_t)) {
  if (!ctx->tmaps) ctx->tmaps = new TmapCache();
  TmapCache* tc_ = ctx->tmaps;
  for (int i = 0; i < tc_->used; ++i)
    if (tc_->e[i].base == base && tc_->e[i].a == a && tc_->e[i].b == b && tc_->e[i].c == c) {
      *out = tc_->e[i].map;
      return ECHO_OK;
    }
  TmapCache::Entry& ent = tc_->e[tc_->next];
  ent.base = nullptr;
  const int rc = encode(ctx, &ent.map, base, a, b, c);
  if (rc != ECHO_OK) return rc;
  ent.base = base; ent.a = a; ent.b = b; ent.c = c;
  tc_->next = (tc_->next + 1) % TmapCache::N;
  if (tc_->used < TmapCache::N) ++tc_->used;
  *out = ent.map;
  return ECHO_OK;
}

// Q / out [cap][Hq][128] bf16 as a 3-D map, box = {64 d, G heads, 128/G nodes}
static int encode_q(EchoCtx* ctx, CUtensorMap* m, const void* q, uint64_t cap, uint64_t Hq, uint64_t G) {
  EncodeTiledFn enc = get_encode();
  cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)Hq, (cuuint64_t)cap};
  cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)Hq * D * 2};
  cuuint32_t box[3] = {64, (cuuint32_t)G, (cuuint32_t)(TILE_M / G)};
  cuuint32_t es[3] = {1, 1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(q), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(ctx->last_error, sizeof(ctx->last_error), "cuTensorMapEncodeTiled(Q) failed: %d", (int)r);
    return ECHO_ERR_CUDA;
  }
  return ECHO_OK;
}
// pool rows [token][128 d] seen as [8-token group][d-half][token in group][64 d]: one box = one page
static int encode_pool(EchoCtx* ctx, CUtensorMap* m, const void* pool, uint64_t total_rows, uint64_t, uint64_t) {
  EncodeTiledFn enc = get_encode();
  cuuint64_t dims[4] = {64, 8, 2, (cuuint64_t)(total_rows / 8)};
  cuuint64_t strides[3] = {(cuuint64_t)D * 2, 128, (cuuint64_t)D * 2 * 8};
  cuuint32_t box[4] = {64, 8, 2, (cuuint32_t)(PAGE / 8)};
  cuuint32_t es[4] = {1, 1, 1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(pool), dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(ctx->last_error, sizeof(ctx->last_error), "cuTensorMapEncodeTiled(KV) failed: %d", (int)r);
    return ECHO_ERR_CUDA;
  }
  return ECHO_OK;
}

#ifdef ECHO_WAIT_PROF
static const int4* g_dbg_items = nullptr;     // the last launch's work list (debug build only)
static const int32_t* g_dbg_n_items = nullptr;
extern "C" int echo_debug_wait_prof(EchoCtx* ctx, uint64_t* host_out, int32_t n_ctas) {
  if (ctx && host_out && n_ctas <= -3) {  // the work list of the last launch: up to -n_ctas records of 8 int32; returns n_items
    int32_t n = 0;
    ECHO_CUDA_TRY(ctx, cudaDeviceSynchronize());
    ECHO_CUDA_TRY(ctx, cudaMemcpy(&n, g_dbg_n_items, 4, cudaMemcpyDeviceToHost));
    const int m = n < -n_ctas ? n : -n_ctas;
    ECHO_CUDA_TRY(ctx, cudaMemcpy(host_out, g_dbg_items, (size_t)m * 32, cudaMemcpyDeviceToHost));
    return n;
  }
  if (ctx && host_out && n_ctas == -1) {  // event trace of CTA 0: [256 tiles][8 events] clock64
    ECHO_CUDA_TRY(ctx, cudaDeviceSynchronize());
    ECHO_CUDA_TRY(ctx, cudaMemcpyFromSymbol(host_out, g_trace, sizeof(long long) * 256 * 8));
    return 256;
  }
  if (!ctx || !host_out || n_ctas <= 0) return ECHO_ERR_INVALID_ARG;
  if (n_ctas > ECHO_PROF_CTAS) n_ctas = ECHO_PROF_CTAS;
  ECHO_CUDA_TRY(ctx, cudaDeviceSynchronize());
  ECHO_CUDA_TRY(ctx, cudaMemcpyFromSymbol(host_out, g_wait_prof, sizeof(unsigned long long) * ECHO_PROF_SLOTS * n_ctas));
  return n_ctas;
}
#endif

int launch_verify_attn_tc(EchoCtx* ctx, const EchoSelection* sel, const EchoPagedKV* kv, int32_t layer, int32_t Hq,
                          int32_t R, const void* q, void* out, float* lse, float sm_scale, int splits, float* part_o,
                          float* part_lse, cudaStream_t st) {
  const int Hkv = kv->num_kv_heads, G = Hq / Hkv, cap = sel->capacity;
  int log2G = 0;
  while ((1 << log2G) < G) ++log2G;
  if ((1 << log2G) != G || G > 128 || !(sm_scale > 0.f)) return ECHO_ERR_UNSUPPORTED;
  if (!get_encode()) {
    snprintf(ctx->last_error, sizeof(ctx->last_error), "cuTensorMapEncodeTiled entry point not found");
    return ECHO_ERR_CUDA;
  }
  const size_t total_rows = (size_t)kv->num_layers * kv->num_pages * Hkv * PAGE;
  if (total_rows >= (1ull << 31)) return ECHO_ERR_UNSUPPORTED;
  CUtensorMap tq, tk, tv;
  if (cached_tmap(ctx, &tq, q, (uint64_t)cap, (uint64_t)Hq, (uint64_t)G, encode_q) != ECHO_OK ||
      cached_tmap(ctx, &tk, kv->k_pool, total_rows, 0, 0, encode_pool) != ECHO_OK ||
      cached_tmap(ctx, &tv, kv->v_pool, total_rows, 0, 0, encode_pool) != ECHO_OK)
    return ECHO_ERR_CUDA;
  // plan region sits behind the split partials in the workspace
  const size_t n_rows = (size_t)cap * Hq;
  const size_t part_bytes = splits > 1 ? align_up((size_t)splits * n_rows * (D + 1) * sizeof(float), 256) : 0;
  const int max_rt = (int)(((size_t)(cap < ECHO_MAX_CAND ? cap : ECHO_MAX_CAND) * G + TILE_M - 1) / TILE_M);
  const size_t max_items = (size_t)R * Hkv * max_rt * splits;
  const size_t plan_bytes = 256 + max_items * 2 * sizeof(int4);
  if (part_bytes + plan_bytes > ctx->workspace_bytes) return ECHO_ERR_WORKSPACE;
  uint8_t* plan = reinterpret_cast<uint8_t*>(ctx->workspace) + part_bytes;
  int32_t* n_items = reinterpret_cast<int32_t*>(plan);
  int4* items = reinterpret_cast<int4*>(plan + 256);
#ifdef ECHO_WAIT_PROF
  g_dbg_items = items;
  g_dbg_n_items = n_items;
#endif
  const bool plan_in_kernel = (long)R * splits <= INPLAN_MAX && ctx->opt_attn_plan != 1;
  if (!plan_in_kernel)
    ECHO_CUDA_TRY(ctx, launch_pdl(k_plan, dim3(1), dim3(PLAN_THREADS), 0, st, sel->sel_offsets, kv->prefix_len, R, Hkv, G,
                                  splits, (int)max_items, max_rt, items, n_items, ctx->dev_status));

  if (!ctx->attn_attr_set) {  // per context, i.e. per device (the attribute is a per-device property of the function)
    ECHO_CUDA_TRY(ctx, cudaFuncSetAttribute(k_verify_attn_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_TOTAL));
    ctx->attn_attr_set = true;
  }
  AttnParams p;
  p.items = items; p.n_items = n_items; p.sel_offsets = sel->sel_offsets;
  p.anc_mask = reinterpret_cast<const uint4*>(sel->anc_mask);
  p.page_table = kv->page_table; p.prefix_len = kv->prefix_len; p.max_pages = kv->max_pages_per_req;
  p.Hkv = Hkv; p.Hq = Hq; p.G = G; p.log2G = log2G; p.page_row_base = layer * kv->num_pages;
  p.out = reinterpret_cast<__nv_bfloat16*>(out); p.lse = lse; p.scale_log2 = sm_scale * LOG2E; p.splits = splits;
  p.force_safe = ctx->opt_attn_safe ? 1 : 0;
  p.part_o = part_o; p.part_lse = part_lse; p.n_rows_cap = n_rows; p.status = ctx->dev_status;
  p.plan_in_kernel = plan_in_kernel ? 1 : 0; p.R = R; p.max_items = (int)max_items; p.max_rt = max_rt;
  p.items_w = items; p.n_items_w = n_items;
  int grid = ctx->opt_num_ctas > 0 ? (int)ctx->opt_num_ctas : ctx->num_sms;
  if ((size_t)grid > max_items) grid = (int)(max_items ? max_items : 1);
  {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(NTHREADS);
    cfg.dynamicSmemBytes = SMEM_TOTAL;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ECHO_COUNT_LAUNCH();
    ECHO_CUDA_TRY(ctx, cudaLaunchKernelEx(&cfg, k_verify_attn_tc, tq, tk, tv, p));
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}
