// S6 on the 5th-gen tensor cores: persistent, warp-specialised split-KV verify attention.
//
//   work item   = (request i, KV head, 128-row tile of (node, head-in-group) rows, KV split); KV tile = 128 tokens
//   warps 12,16 = K producers, warps 14,17 = V producers (one lane each): one 4-D TMA box per page (16 tokens x 128 d
//                 of one KV head), pages looked up in the page table; warp 12 also loads the Q tile (3-D tensor map
//                 over [node][head][d]).  Two issuing threads per ring because one cp.async.bulk.tensor costs its
//                 thread 110-170 cycles whatever the box size.
//   warp 13     = issuer of S = Q K^T (SS, K-major x K-major) into one of three S buffers in TMEM
//   warp 15     = issuer of O += P V (TS: P read from TMEM where the softmax wrote it over S, V as the MN-major B
//                 operand straight from its TMA layout); accumulators never leave TMEM
//   warps 0-7   = softmax, two warpgroups, thread = half a row (64 columns): weights against a running reference
//                 without a row maximum first, two-pass fallback on a vote of the two warps of a row quarter; tree
//                 mask only in tiles that touch positions >= P_i; a quarter of the prefix-tile weights take 2^x on
//                 the FMA pipe; P written back to TMEM as bf16 over the first 32 columns of the thread's S half
//   warps 8-11  = epilogue: O / l -> bf16 out + lse (or the fp32 split partial) while the softmax is on the next item
//   setmaxnreg  : softmax 160, epilogue 80, single-lane warps 40 registers
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
constexpr int SMEM_STATS = SMEM_V + NSTAGE * TILE_BYTES;  // float stats[2][128]: 1 / l_rounded, lse of the item just finished
constexpr int SMEM_XCHG = SMEM_STATS + 2 * TILE_M * 4;  // float xchg[2 warpgroups][128]: half-row maxima / sums
constexpr int SMEM_BAR = SMEM_XCHG + 2 * TILE_M * 4;
constexpr int SMEM_TOTAL = SMEM_BAR + 256;  // dynamic smem is declared 1024-byte aligned: no slack
// warpgroups 0 and 1 (warps 0-3, 4-7) softmax: warpgroup w takes columns [64 w, 64 w + 64) of every S row, so each
// SM sub-partition has two softmax warps to issue from; warpgroup 2 (warps 8-11) epilogue; warpgroup 3: warp 12 Q+K
// producer, 13 QK^T MMA issuer, 14 V producer, 15 PV MMA issuer; warpgroup 4: warps 16 / 17 second K / V producer,
// 18-19 idle (they pad the warpgroup so that setmaxnreg applies)
constexpr int NTHREADS = 640;
constexpr int W_EPI = 8, W_PROD_K0 = 12, W_MMA_QK = 13, W_PROD_V0 = 14, W_MMA_PV = 15, W_PROD_K1 = 16, W_PROD_V1 = 17;
constexpr int REGS_SOFTMAX = 160, REGS_EPILOGUE = 80, REGS_AUX = 40;  // 128 * (2 * 160 + 80 + 2 * 40) = 640 * 96, the launch allocation
constexpr int NSBUF = 3;        // S / P buffers in TMEM: the QK^T of tile j+2 is issued before the PV of tile j
constexpr int TMEM_O = NSBUF * TILE_N;
constexpr int TMEM_COLS = 512;  // S_b [128 b, 128 b + 128) for b < 3, O [384,512); P_b aliases S_b[0,64)
// of every POLY_PERIOD weight pairs in a prefix tile, POLY_COUNT take 2^x on the FMA pipe, the rest on MUFU
#ifndef ECHO_POLY_COUNT
#define ECHO_POLY_COUNT 1
#endif
constexpr int POLY_PERIOD = 4, POLY_COUNT = ECHO_POLY_COUNT;  // measured best: 1 of 4 (2 of 4 and 3 of 8 are slower)
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;
constexpr float WEIGHT_SUM_LIMIT = 4294967296.f;  // a tile whose weight sum exceeds 2^32 is redone against its own maximum
// Every item starts from the reference 0 instead of the first tile's row maxima: weights are floating point, so any
// reference within 2^-64 .. 2^32 of the true one gives the same O and lse; a first tile whose weight sum falls outside
// that range is redone in the two-pass form, which takes the reference from the data.
constexpr float WEIGHT_SUM_FLOOR = 5.421010862427522e-20f;  // 2^-64

constexpr uint32_t IDESC_QK = tc::idesc_bf16(TILE_M, TILE_N, 0, 0);
constexpr uint32_t IDESC_PV = tc::idesc_bf16(TILE_M, D, 0, 1);

// barrier indices (8 bytes each)
enum { B_QFULL = 0, B_QEMPTY = 1, B_KFULL = 2, B_KEMPTY = 5, B_VFULL = 8, B_VEMPTY = 11, B_SFULL = 14, B_PFULL = 17,
       B_PVDONE = 20, B_OFULL = 21, B_OFREE = 22, B_STATS = 23, B_SFREE = 24, B_COUNT = 27 };

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
  float* part_o;
  float* part_lse;
  size_t n_rows_cap;
  uint32_t* status;
};

// Optional wait-time profile (build with -DECHO_WAIT_PROF): cycles each role spends blocked on each mbarrier,
// per CTA, read back with echo_debug_wait_prof.  Compiled out otherwise.
#ifdef ECHO_WAIT_PROF
__device__ unsigned long long g_wait_prof[ECHO_PROF_CTAS][ECHO_PROF_SLOTS];
#define PROF_T0() const long long prof_t0_ = clock64()
#define PROF_ADD(slot) prof_[slot] += clock64() - prof_t0_
#define PROF_WAIT(slot, b, ph) do { const long long t_ = clock64(); tc::mbar_wait(b, ph); prof_[slot] += clock64() - t_; } while (0)
#define PROF_WAIT_RELAXED(slot, b, ph) do { const long long t_ = clock64(); tc::mbar_wait_relaxed(b, ph); prof_[slot] += clock64() - t_; } while (0)
#define PROF_WAIT_BACKOFF(slot, b, ph) do { const long long t_ = clock64(); tc::mbar_wait_backoff(b, ph); prof_[slot] += clock64() - t_; } while (0)
#define PROF_DECL(n) unsigned long long prof_[n] = {}
#define PROF_FLUSH(base, n) do { if (blockIdx.x < ECHO_PROF_CTAS) for (int q_ = 0; q_ < n; ++q_) g_wait_prof[blockIdx.x][(base) + q_] = prof_[q_]; } while (0)
#define PROF_SPAN_BEGIN() const long long span_t_ = clock64()
#define PROF_SPAN_END(slot) prof_[slot] += clock64() - span_t_
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
#endif

// work item record written by k_plan: two int4 = {req, kvh | rt<<8 | split<<16, jt0, jt1} {P_i, sel_offsets[i], K_i, 0}
struct Item { int req, kvh, rt, split, jt0, jt1, P, off, Ki; };
__device__ __forceinline__ Item decode(const int4 v, const int4 w) {
  Item it;
  it.req = v.x; it.kvh = v.y & 0xff; it.rt = (v.y >> 8) & 0xff; it.split = (v.y >> 16) & 0xff; it.jt0 = v.z; it.jt1 = v.w;
  it.P = w.x; it.off = w.y; it.Ki = w.z;
  return it;
}
__device__ __forceinline__ Item load_item(const int4* items, int idx) { return decode(items[2 * idx], items[2 * idx + 1]); }
// snake order over the length-sorted work list: round k of CTA c takes k*G+c (k even) or (k+1)*G-1-c (k odd)
__device__ __forceinline__ int item_index(int k, int cta, int grid) {
  return (k & 1) ? (k + 1) * grid - 1 - cta : k * grid + cta;
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

// ---- softmax passes over this thread's half of an S row (64 fp32 columns in TMEM), two 32-column tcgen05.ld, the
// second in flight while the first is processed ----
__device__ __forceinline__ void mask_chunk(uint32_t (&s)[32], uint32_t vis) {
#pragma unroll
  for (int e = 0; e < 32; ++e)
    if (!((vis >> e) & 1u)) s[e] = 0xff800000u;  // -inf
}

// 2^x for a pair of finite x on the FMA pipe instead of MUFU (16 ex2 per clock per SM, the busiest pipe of the
// softmax): n = round(x) by the 1.5*2^23 trick, f = x - n in [-0.5, 0.5], 2^f by a degree-3 minimax polynomial
// (relative error 7.5e-5, far below the bf16 rounding of P), then n is added to the exponent field.  x is clamped
// to [-125, 126]: 2^-125 instead of less is negligible against the reference weight 1 (so this form is used only
// where no key is masked), and 2^126 sends the tile to the two-pass fallback.
__device__ __forceinline__ void ex2_poly_x2(uint64_t x2, float& p0, float& p1) {
  float x0, x1;
  tc::unpack_f32x2(x2, x0, x1);
  x2 = tc::pack_f32x2(fminf(fmaxf(x0, -125.f), 126.f), fminf(fmaxf(x1, -125.f), 126.f));
  const uint64_t magic = tc::pack_f32x2(12582912.f, 12582912.f), nmagic = tc::pack_f32x2(-12582912.f, -12582912.f);
  const uint64_t t = tc::add_f32x2(x2, magic);
  const uint64_t n = tc::add_f32x2(t, nmagic);
  const uint64_t f = tc::fma_f32x2(n, tc::pack_f32x2(-1.f, -1.f), x2);
  uint64_t q = tc::fma_f32x2(f, tc::pack_f32x2(0x1.c3f76p-5f, 0x1.c3f76p-5f), tc::pack_f32x2(0x1.f0de1ap-3f, 0x1.f0de1ap-3f));
  q = tc::fma_f32x2(q, f, tc::pack_f32x2(0x1.62f31ap-1f, 0x1.62f31ap-1f));
  q = tc::fma_f32x2(q, f, tc::pack_f32x2(0x1.fff692p-1f, 0x1.fff692p-1f));
  float q0, q1, t0, t1;
  tc::unpack_f32x2(q, q0, q1);
  tc::unpack_f32x2(t, t0, t1);
  p0 = __uint_as_float(__float_as_uint(q0) + (__float_as_uint(t0) << 23));
  p1 = __uint_as_float(__float_as_uint(q1) + (__float_as_uint(t1) << 23));
}

// weights p = 2^(s*scale_log2 + neg_m) for 64 columns: packed to bf16 in pk, exact fp32 sum in ts and (tail tiles
// only) the sum of the bf16-rounded weights in tr.  Packed f32x2 FMA / ADD halve the issue slots.
// TAIL = false (all 64 keys inside the prefix) compiles to straight-line FFMA2 / MUFU / F2FP / FADD2 with no
// visibility selects and no rounded sum: 2.5 issue slots per weight.
template <bool TAIL>
__device__ __forceinline__ void weights_pass(uint32_t tSh, const uint32_t (&vis)[2], float scale_log2, float neg_m,
                                             uint32_t (&pk)[32], float& ts, float& tr) {
  const uint64_t sc2 = tc::pack_f32x2(scale_log2, scale_log2), nm2 = tc::pack_f32x2(neg_m, neg_m);
  uint64_t acc[4] = {0ull, 0ull, 0ull, 0ull};  // 8 independent fp32 partial sums
  float trr[2] = {0.f, 0.f};
  uint32_t s[2][32];
  tc::tmem_ld32(tSh, s[0]);
  tc::tmem_wait_ld();
  tc::tmem_ld32(tSh + 32, s[1]);
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    if (c == 1) tc::tmem_wait_ld();
    uint32_t(&sc)[32] = s[c];
    if (TAIL) mask_chunk(sc, vis[c]);
#pragma unroll
    for (int e = 0; e < 32; e += 2) {
      const uint64_t x2 = tc::fma_f32x2(tc::pack_f32x2(__uint_as_float(sc[e]), __uint_as_float(sc[e + 1])), sc2, nm2);
      float p0, p1;
      if (!TAIL && ((e >> 1) % POLY_PERIOD) < POLY_COUNT) {
        ex2_poly_x2(x2, p0, p1);
      } else {
        float x0, x1;
        tc::unpack_f32x2(x2, x0, x1);
        p0 = tc::ex2(x0);
        p1 = tc::ex2(x1);
      }
      const uint32_t w = tc::pack_bf16(p0, p1);
      pk[c * 16 + (e >> 1)] = w;
      acc[(e >> 1) & 3] = tc::add_f32x2(acc[(e >> 1) & 3], tc::pack_f32x2(p0, p1));
      // tiles that touch the tree / ragged end may have a handful of visible keys: there O is normalised by the
      // sum of the bf16-rounded weights the tensor core multiplies with, so that O stays an exact convex
      // combination of V rows; lse always uses the exact fp32 sum
      if (TAIL) trr[(e >> 1) & 1] += __uint_as_float(w << 16) + __uint_as_float(w & 0xffff0000u);
    }
  }
  float a0, a1;
  tc::unpack_f32x2(tc::add_f32x2(tc::add_f32x2(acc[0], acc[1]), tc::add_f32x2(acc[2], acc[3])), a0, a1);
  ts = a0 + a1;
  tr = TAIL ? trr[0] + trr[1] : ts;
}

__device__ __forceinline__ float row_max_pass(uint32_t tSh, const uint32_t (&vis)[2]) {
  float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
  uint32_t s[2][32];
  tc::tmem_ld32(tSh, s[0]);
  tc::tmem_ld32(tSh + 32, s[1]);
  tc::tmem_wait_ld();
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    mask_chunk(s[c], vis[c]);
#pragma unroll
    for (int e = 0; e < 32; e += 2)
      mx[(e >> 1) & 3] = tc::max3(mx[(e >> 1) & 3], __uint_as_float(s[c][e]), __uint_as_float(s[c][e + 1]));
  }
  return fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3]));
}

// named barrier over the two warps that share a TMEM lane quarter (one per softmax warpgroup), ids 1-4
__device__ __forceinline__ bool pair_or(int quarter, bool pred) {
  uint32_t r;
  asm volatile(
      "{\n\t.reg .pred p, q;\n\tsetp.ne.u32 p, %1, 0;\n\t"
      "barrier.cta.red.or.pred q, %2, 64, p;\n\t"
      "selp.u32 %0, 1, 0, q;\n\t}"
      : "=r"(r)
      : "r"((uint32_t)pred), "r"(quarter + 1)
      : "memory");
  return r != 0;
}
__device__ __forceinline__ void pair_sync(int quarter) {
  asm volatile("barrier.cta.sync %0, 64;" ::"r"(quarter + 1) : "memory");
}

__global__ void __launch_bounds__(NTHREADS, 1) k_verify_attn_tc(const __grid_constant__ CUtensorMap tmap_q,
                                                                const __grid_constant__ CUtensorMap tmap_k,
                                                                const __grid_constant__ CUtensorMap tmap_v,
                                                                const AttnParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t sbase = tc::smem_u32(smem_raw);
  const uint32_t sQ = sbase + SMEM_Q, sK = sbase + SMEM_K, sV = sbase + SMEM_V, sBar = sbase + SMEM_BAR;
  uint8_t* gen_base = smem_raw;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(gen_base + SMEM_BAR + B_COUNT * 8);
  float* stats = reinterpret_cast<float*>(gen_base + SMEM_STATS);
  float* xchg = reinterpret_cast<float*>(gen_base + SMEM_XCHG);
  auto bar = [&](int i) -> uint32_t { return sBar + 8u * i; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int cta = blockIdx.x, grid = gridDim.x;
  pdl_launch_dependents();  // echo_accept's kernel may queue behind this one (it waits for our completion itself)

  if (threadIdx.x == 0) {
    if (sbase & 1023u) __trap();  // SW128 operand tiles need 1024-byte alignment
    for (int i = 0; i < B_COUNT; ++i) {
      const uint32_t cnt = (i >= B_KFULL && i < B_KFULL + NSTAGE) || (i >= B_VFULL && i < B_VFULL + NSTAGE) ? 2u
                           : (i >= B_PFULL && i < B_PFULL + NSBUF) ? 8u  /* one arrival per softmax warp */
                           : (i == B_OFREE || i == B_STATS) ? 128u : 1u;
      tc::mbar_init(bar(i), cnt);
    }
    tc::fence_barrier_init();
    tc::prefetch_tmap(&tmap_q);
    tc::prefetch_tmap(&tmap_k);
    tc::prefetch_tmap(&tmap_v);
  }
  if (warp == W_MMA_QK) tc::tmem_alloc(sBar + B_COUNT * 8, TMEM_COLS);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  // Programmatic dependent launch: everything above (barrier init, TMEM allocation, descriptor prefetch) overlaps
  // k_plan; the work list is read only after k_plan has completed.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const int n_items = *p.n_items;

  if (warp >= 12) tc::setmaxnreg_dec<REGS_AUX>();
  if (warp == W_PROD_K0 || warp == W_PROD_V0 || warp == W_PROD_K1 || warp == W_PROD_V1) {
    // ============================== TMA producers: Q + K ring, V ring ==============================
    // One cp.async.bulk.tensor costs its issuing thread 110-170 cycles whatever the box size (measured), so a page
    // (16 tokens x 128 d of one KV head, 4 KB contiguous in the pool) is one 4-D box {64 d, 8 tokens, 2 d-halves,
    // 2 token groups} and each ring has two issuing threads in different warps: thread h takes pages 4h..4h+3 of
    // every 128-token tile.  The whole loop runs in one lane so that every TMA operand is warp-uniform; page ids of
    // tile j+1 are fetched while tile j is being issued.
    if (lane == 0) {
      const bool is_k = warp == W_PROD_K0 || warp == W_PROD_K1;
      const int half = (warp == W_PROD_K1 || warp == W_PROD_V1) ? 1 : 0;
      const bool loads_q = warp == W_PROD_K0;
      const uint32_t s_dst = is_k ? sK : sV;
      const CUtensorMap* tmap = is_k ? &tmap_k : &tmap_v;
      const int b_full = is_k ? B_KFULL : B_VFULL, b_empty = is_k ? B_KEMPTY : B_VEMPTY;
      int g = 0, itc = 0;
      PROF_DECL(3);
      PROF_T0();
      Item nx = {};
      bool more = item_index(0, cta, grid) < n_items;  // item indices grow with k
      if (more) nx = load_item(p.items, item_index(0, cta, grid));
      for (int k = 1; more; ++k) {
        const Item it = nx;
        more = item_index(k, cta, grid) < n_items;
        if (more) nx = load_item(p.items, item_index(k, cta, grid));
        const int total = it.P + it.Ki;
        if (loads_q) {
          PROF_WAIT_BACKOFF(2, bar(B_QEMPTY), (itc & 1) ^ 1);
          tc::mbar_expect_tx(bar(B_QFULL), TILE_BYTES);
          const int node0 = it.off + it.rt * (TILE_M >> p.log2G);
          tc::tma_load_3d(sQ, &tmap_q, bar(B_QFULL), 0, it.kvh * p.G, node0);
          tc::tma_load_3d(sQ + HALF_BYTES, &tmap_q, bar(B_QFULL), 64, it.kvh * p.G, node0);
        }
        const int32_t* pt = p.page_table + (size_t)it.req * p.max_pages;
        int npages = (total + PAGE - 1) / PAGE;
        if (npages > p.max_pages) {  // page table too short: flag, load what exists
          if (loads_q) atomicOr(p.status, ECHO_DEV_PAGE_OVERFLOW);
          npages = p.max_pages;
        }
        int cur[4], nxt[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int pi = it.jt0 * 8 + half * 4 + e;
          cur[e] = pi < npages ? pt[pi] : 0;
        }
        for (int j = it.jt0; j < it.jt1; ++j, ++g) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int pi = (j + 1) * 8 + half * 4 + e;
            nxt[e] = (j + 1 < it.jt1 && pi < npages) ? pt[pi] : 0;
          }
          const int slot = g % NSTAGE, ph = (g / NSTAGE) & 1;
          const int npv = max(0, min(4, npages - j * 8 - half * 4));  // my pages of this tile that hold tokens
          const uint32_t dst = s_dst + slot * TILE_BYTES + half * 4 * PAGE_BYTES;
          const uint32_t fb = bar(b_full + slot);
          PROF_WAIT_BACKOFF(1, bar(b_empty + slot), ph ^ 1);
          tc::mbar_expect_tx(fb, npv * PAGE_BYTES);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            if (e < npv) {
              const int grp = ((p.page_row_base + cur[e]) * p.Hkv + it.kvh) * (PAGE / 8);  // 8-token group index
              tc::tma_load_4d(dst + e * PAGE_BYTES, tmap, fb, 0, 0, 0, grp);
            }
          }
#pragma unroll
          for (int e = 0; e < 4; ++e) cur[e] = nxt[e];
        }
        ++itc;
      }
      PROF_ADD(0);
      if (half == 0) PROF_FLUSH(is_k ? 0 : 4, 3);
    }
    __syncwarp();
  } else if (warp == W_MMA_QK) {
    // ============================== MMA issuer for S = Q K^T (one lane) ==============================
    // Two issuing threads, one per product: a single thread retires a 128x128x16 tcgen05.mma only every ~110
    // cycles, two threads keep the tensor pipe at 70-85 cycles per instruction (measured).  This thread runs up to
    // NSBUF tiles ahead of the PV issuer; S/P buffer b is handed back through B_SFREE when the PV that read P_b is done.
    if (lane == 0) {
      int g = 0, itc = 0;
      PROF_DECL(6);
      PROF_T0();
      const uint64_t qdesc = tc::smem_desc_sw128(sQ, 16, 1024);
      for (int k = 0;; ++k) {
        const int idx = item_index(k, cta, grid);
        if (idx >= n_items) break;  // item indices grow with k
        const int4 rec = p.items[2 * idx];
        const int n = rec.w - rec.z;
        PROF_WAIT(5, bar(B_QFULL), itc & 1);
        for (int j = 0; j < n; ++j, ++g) {
          const int slot = g % NSTAGE, b = g % NSBUF;
          PROF_WAIT(1, bar(B_KFULL + slot), (g / NSTAGE) & 1);
          PROF_WAIT(2, bar(B_SFREE + b), ((g / NSBUF) & 1) ^ 1);  // PV of tile g - NSBUF has read P_b
          tc::tc_fence_after();
          // K tile: 8-token groups GROUP_BYTES apart (SBO), d-half h at +1 KB inside a group
          const uint64_t kdesc = tc::smem_desc_sw128(sK + slot * TILE_BYTES, 16, GROUP_BYTES);
#pragma unroll
          for (int kk = 0; kk < D / 16; ++kk) {
            const uint32_t q16 = ((kk & 3) * 32 + (kk >> 2) * HALF_BYTES) >> 4;
            const uint32_t k16 = ((kk & 3) * 32 + (kk >> 2) * 1024) >> 4;
            tc::mma_ss(tmem + b * TILE_N, qdesc + q16, kdesc + k16, IDESC_QK, kk > 0);
          }
          tc::mma_commit(bar(B_SFULL + b));
          tc::mma_commit(bar(B_KEMPTY + slot));
          if (j == n - 1) tc::mma_commit(bar(B_QEMPTY));
        }
        ++itc;
      }
      PROF_ADD(0);
      PROF_FLUSH(8, 6);
    }
    __syncwarp();
  } else if (warp == W_MMA_PV) {
    // ============================== MMA issuer for O += P V (one lane) ==============================
    if (lane == 0) {
      int g = 0, itc = 0;
      const uint32_t tO = tmem + TMEM_O;
      for (int k = 0;; ++k) {
        const int idx = item_index(k, cta, grid);
        if (idx >= n_items) break;
        const int4 rec = p.items[2 * idx];
        const int n = rec.w - rec.z;
        for (int j = 0; j < n; ++j, ++g) {
          const int b = g % NSBUF, slot = g % NSTAGE;
          tc::mbar_wait(bar(B_PFULL + b), (g / NSBUF) & 1);
          tc::mbar_wait(bar(B_VFULL + slot), (g / NSTAGE) & 1);
          if (j == 0) tc::mbar_wait(bar(B_OFREE), (itc & 1) ^ 1);  // epilogue of the previous item has read O
          tc::tc_fence_after();
          // V tile as MN-major B: 64-wide d atoms 1 KB apart (LBO), 8-token groups GROUP_BYTES apart (SBO).
          // P of tokens [0,64) sits in columns [0,32) of S_b, P of tokens [64,128) in columns [64,96): each softmax
          // warpgroup overwrites only columns of its own half of S.
          const uint64_t vdesc = tc::smem_desc_sw128(sV + slot * TILE_BYTES, 1024, GROUP_BYTES);
#pragma unroll
          for (int kk = 0; kk < TILE_N / 16; ++kk)
            tc::mma_ts(tO, tmem + b * TILE_N + (kk >> 2) * 64 + (kk & 3) * 8, vdesc + ((kk * 2 * GROUP_BYTES) >> 4), IDESC_PV,
                       (j > 0) || (kk > 0));
          tc::mma_commit(bar(B_VEMPTY + slot));
          tc::mma_commit(bar(B_SFREE + b));
          tc::mma_commit(bar(B_PVDONE));
          if (j == n - 1) tc::mma_commit(bar(B_OFULL));
        }
        ++itc;
      }
    }
    __syncwarp();
  } else if (warp < W_EPI) {
    // ============================== softmax (warpgroups 0 and 1, thread = half of a row) ==============================
    // Both halves of a row keep the same running reference m_used (it changes only in the pair-synchronised
    // two-pass branch) and their own partial weight sums, added up once per item.
    tc::setmaxnreg_inc<REGS_SOFTMAX>();
    const int wg = warp >> 2;  // which 64 columns of every S row
    const int wq = warp & 3;   // TMEM lane quarter this warp may access
    const int row = wq * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(wq * 32) << 16;
    float* xchg_mine = xchg + wg * TILE_M + row;
    const float* xchg_other = xchg + (wg ^ 1) * TILE_M + row;
    int g = 0, itc = 0;
    PROF_DECL(7);
    PROF_T0();
    // Item records are fetched two items ahead and the row's ancestor mask one item ahead, so that no global-load
    // latency sits between the last tile of one item and the first tile of the next.
    auto row_mask = [&](const int4& r0, const int4& r1) -> uint4 {
      const int l = ((((r0.y >> 8) & 0xff) * TILE_M + row) >> p.log2G);
      return l < r1.z ? p.anc_mask[r1.y + l] : make_uint4(0u, 0u, 0u, 0u);
    };
    const int4 zero4 = make_int4(0, 0, 0, 0);
    int4 a0 = zero4, a1 = zero4, b0 = zero4, b1 = zero4;  // records of the next item (a) and the one after (b)
    uint4 mk_next = make_uint4(0u, 0u, 0u, 0u);
    bool more = item_index(0, cta, grid) < n_items;
    if (more) { a0 = p.items[2 * item_index(0, cta, grid)]; a1 = p.items[2 * item_index(0, cta, grid) + 1]; }
    if (item_index(1, cta, grid) < n_items) { b0 = p.items[2 * item_index(1, cta, grid)]; b1 = p.items[2 * item_index(1, cta, grid) + 1]; }
    if (more) mk_next = row_mask(a0, a1);
    for (int k = 0; more; ++k) {
      const Item it = decode(a0, a1);
      const uint4 mk = mk_next;
      more = item_index(k + 1, cta, grid) < n_items;
      a0 = b0; a1 = b1;
      if (item_index(k + 2, cta, grid) < n_items) { b0 = p.items[2 * item_index(k + 2, cta, grid)]; b1 = p.items[2 * item_index(k + 2, cta, grid) + 1]; }
      if (more) mk_next = row_mask(a0, a1);
      const int P = it.P, total = it.P + it.Ki;
      float m_used = 0.f, lsum = 0.f, lsum_r = 0.f;
      const uint32_t tOh = tmem + TMEM_O + wg * 64 + lane_addr;

      for (int j = it.jt0; j < it.jt1; ++j, ++g) {
        const int b = g % NSBUF;
        const uint32_t tSh = tmem + b * TILE_N + wg * 64 + lane_addr;  // my 64 columns of S; P goes to their first 32
        PROF_WAIT(1, bar(B_SFULL + b), (g / NSBUF) & 1);
        tc::tc_fence_after();
        const int tile0 = j * TILE_N, tok0 = tile0 + wg * 64;
        const bool tail = tok0 + 64 > P;  // my keys touch tree positions or the ragged end: apply visibility
        uint32_t vis[2] = {0xffffffffu, 0xffffffffu};
        if (tail) {
          vis[0] = visible_word(mk, P, tok0);
          vis[1] = visible_word(mk, P, tok0 + 32);
        }
        uint32_t pk[32];  // my half of the bf16 P row
        float ts = 0.f, tr = 0.f;  // this tile's exact / bf16-rounded weight sums
        // Fast path: the weights are taken against the running reference m_used without looking at this tile's
        // maximum first; only if a weight sum leaves [0, 2^32] (reference too low, or no reference yet) do the
        // two warps of the row quarter fall back to the two-pass form (row maximum, rescale, weights).  P is
        // stored only after that check, so S is still intact for the second pass.
        bool slow = __any_sync(0xffffffffu, m_used == -INFINITY);  // the same in both halves
        if (!slow) {
          PROF_SPAN_BEGIN();
          if (tail) weights_pass<true>(tSh, vis, p.scale_log2, -m_used, pk, ts, tr);
          else weights_pass<false>(tSh, vis, p.scale_log2, -m_used, pk, ts, tr);
          slow = pair_or(wq, !(ts <= WEIGHT_SUM_LIMIT) || (j == it.jt0 && ts < WEIGHT_SUM_FLOOR));
          PROF_SPAN_END(5);
        }
        if (slow) {
          if (j == it.jt0) m_used = -INFINITY;  // nothing accumulated yet: drop the guessed reference
          float mx = row_max_pass(tSh, vis);
          *xchg_mine = mx;
          pair_sync(wq);
          mx = fmaxf(mx, *xchg_other);
          pair_sync(wq);  // both halves have read before the slots are written again
          const float m_new = fmaxf(m_used, mx * p.scale_log2);
          float alpha = 1.f;
          if (m_new > m_used) {
            alpha = (m_used == -INFINITY) ? 0.f : tc::ex2(m_used - m_new);
            m_used = m_new;
          }
          lsum *= alpha;
          lsum_r *= alpha;
          if (j > it.jt0) {  // O holds PV of earlier tiles: wait for the last one, rescale my 64 columns in TMEM
            PROF_WAIT(3, bar(B_PVDONE), (g - 1) & 1);
            tc::tc_fence_after();
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              uint32_t o[32];
              tc::tmem_ld32(tOh + c * 32, o);
              tc::tmem_wait_ld();
#pragma unroll
              for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * alpha);
              tc::tmem_st32(tOh + c * 32, o);
            }
            tc::tmem_wait_st();
          }
          const float m_eff = (m_used == -INFINITY) ? 0.f : m_used;
          weights_pass<true>(tSh, vis, p.scale_log2, -m_eff, pk, ts, tr);  // vis is all ones off the tail
        }
        lsum += ts;
        lsum_r += tr;
        PROF_SPAN_BEGIN();
        tc::tmem_st32(tSh, pk);
        tc::tmem_wait_st();
        if (tile0 + TILE_N > total) {  // ragged end: V rows past the last token may hold anything (R:A-7)
          const int slot = g % NSTAGE;
          PROF_WAIT(4, bar(B_VFULL + slot), (g / NSTAGE) & 1);
          if (row >= total - tile0) {  // warpgroup w clears d-half w of V row `row`
            uint4* z = reinterpret_cast<uint4*>(gen_base + SMEM_V + slot * TILE_BYTES + (row >> 3) * GROUP_BYTES + wg * 1024 +
                                               (row & 7) * 128);
#pragma unroll
            for (int e = 0; e < 8; ++e) z[e] = make_uint4(0u, 0u, 0u, 0u);
          }
          tc::fence_proxy_async();
        }
        tc::tc_fence_before();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(bar(B_PFULL + b));
        PROF_SPAN_END(6);
      }

      // ---- add the two halves' sums; warpgroup 0 hands 1 / l_rounded and lse = ln2 * (m + log2 l) to the epilogue ----
      if (wg == 1) {
        xchg_mine[0] = lsum;
        // the rounded sum travels in warpgroup 0's slot, which warpgroup 0 itself does not write here
        const_cast<float*>(xchg_other)[0] = lsum_r;
      }
      pair_sync(wq);
      if (wg == 0) {
        lsum += *xchg_other;
        lsum_r += *xchg_mine;
        const float inv = lsum_r > 0.f ? 1.f / lsum_r : 0.f;
        const float m_eff = (m_used == -INFINITY) ? 0.f : m_used;
        const float lse_v = lsum > 0.f ? (m_eff + log2f(lsum)) * LN2 : -INFINITY;
        tc::mbar_wait(bar(B_OFREE), (itc & 1) ^ 1);  // epilogue of item itc-1 has read its statistics
        stats[row] = inv;
        stats[TILE_M + row] = lse_v;
        tc::mbar_arrive(bar(B_STATS));
      }
      pair_sync(wq);  // the exchange slots are free again
      ++itc;
    }
    PROF_ADD(0);
    if (warp == 0 && lane == 0) PROF_FLUSH(16, 7);
  } else if (warp < W_PROD_K0) {
    // ============================== epilogue (warpgroup 2, thread = row) ==============================
    // O of item n is normalised and stored here while the softmax warpgroup is already on item n+1 (O and the
    // statistics are double buffered by item parity).
    tc::setmaxnreg_dec<REGS_EPILOGUE>();
    const int wq = warp & 3;
    const int row = wq * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(wq * 32) << 16;
    int itc = 0;
    PROF_DECL(3);
    PROF_T0();
    for (int k = 0;; ++k) {
      const int idx = item_index(k, cta, grid);
      if (idx >= n_items) break;
      const Item it = load_item(p.items, idx);
      const int r_glob = it.rt * TILE_M + row;
      const int l = r_glob >> p.log2G, gq = r_glob & (p.G - 1);
      const bool valid = l < it.Ki;
      const int opar = itc & 1;
      const uint32_t tO = tmem + TMEM_O + lane_addr;
      const size_t rowg = (size_t)(it.off + l) * p.Hq + it.kvh * p.G + gq;
      PROF_WAIT_RELAXED(1, bar(B_STATS), itc & 1);
      const float inv = stats[row];
      const float lse_v = stats[TILE_M + row];
      PROF_WAIT(2, bar(B_OFULL), itc & 1);
      tc::tc_fence_after();
      uint32_t o[2][32];
      tc::tmem_ld32(tO, o[0]);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        tc::tmem_wait_ld();
        if (c < 3) tc::tmem_ld32(tO + (c + 1) * 32, o[(c + 1) & 1]);
        uint32_t(&oc)[32] = o[c & 1];
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
      tc::tc_fence_before();
      tc::mbar_arrive(bar(B_OFREE));
      ++itc;
    }
    PROF_ADD(0);
    if (warp == W_EPI && lane == 0) PROF_FLUSH(24, 3);
  }

  // ---- teardown ----
  tc::tc_fence_before();
  __syncthreads();
  if (warp == W_MMA_QK) tc::tmem_dealloc(tmem, TMEM_COLS);
}

// Device-side planner: P_i and K_i exist only on the device, so the work list is built there.
// Items are bucketed by KV-tile count (descending) so that the snake assignment balances CTAs.
constexpr int PLAN_THREADS = 256;   // one request per thread and pass at the batch sizes of BASELINE.json; a small CTA syncs faster
constexpr int PLAN_BUCKETS = 1024;  // tile counts above 1023 (131 k tokens) share the last bucket
__global__ void __launch_bounds__(PLAN_THREADS) k_plan(const int32_t* __restrict__ sel_offsets,
                                                       const int32_t* __restrict__ prefix_len, int R, int Hkv, int G,
                                                       int splits, int max_items, int4* __restrict__ items,
                                                       int32_t* __restrict__ n_items) {
  __shared__ int s_cnt[PLAN_BUCKETS];
  __shared__ int s_warp[32];
  pdl_launch_dependents();  // let k_verify_attn_tc set itself up meanwhile
  pdl_wait();               // sel_offsets come from echo_gate_select's kernels
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int b = tid; b < PLAN_BUCKETS; b += PLAN_THREADS) s_cnt[b] = 0;
  if (tid < 32) s_warp[tid] = 0;
  __syncthreads();
  auto for_items = [&](auto&& fn) {
    for (int r = tid; r < R; r += PLAN_THREADS) {
      const int off = sel_offsets[r], Ki = sel_offsets[r + 1] - off, P = prefix_len[r];
      if (Ki <= 0) continue;
      const int n_tiles = (P + Ki + TILE_N - 1) / TILE_N;
      const int n_rt = (Ki * G + TILE_M - 1) / TILE_M;
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

int debug_wait_prof(unsigned long long* host_out, int n_ctas) {
#ifdef ECHO_WAIT_PROF
  if (n_ctas > ECHO_PROF_CTAS) n_ctas = ECHO_PROF_CTAS;
  return cudaMemcpyFromSymbol(host_out, g_wait_prof, sizeof(unsigned long long) * ECHO_PROF_SLOTS * n_ctas) == cudaSuccess
             ? n_ctas : ECHO_ERR_CUDA;
#else
  (void)host_out; (void)n_ctas;
  return ECHO_ERR_UNSUPPORTED;
#endif
}

int launch_verify_attn_tc(EchoCtx* ctx, const EchoSelection* sel, const EchoPagedKV* kv, int32_t layer, int32_t Hq,
                          int32_t R, const void* q, void* out, float* lse, float sm_scale, int splits, float* part_o,
                          float* part_lse, cudaStream_t st) {
  const int Hkv = kv->num_kv_heads, G = Hq / Hkv, cap = sel->capacity;
  int log2G = 0;
  while ((1 << log2G) < G) ++log2G;
  if ((1 << log2G) != G || G > 128 || !(sm_scale > 0.f)) return ECHO_ERR_UNSUPPORTED;
  EncodeTiledFn enc = get_encode();
  if (!enc) {
    snprintf(ctx->last_error, sizeof(ctx->last_error), "cuTensorMapEncodeTiled entry point not found");
    return ECHO_ERR_CUDA;
  }
  const size_t total_rows = (size_t)kv->num_layers * kv->num_pages * Hkv * PAGE;
  if (total_rows >= (1ull << 31)) return ECHO_ERR_UNSUPPORTED;
  CUtensorMap tq, tk, tv;
  {
    cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)Hq, (cuuint64_t)cap};
    cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)Hq * D * 2};
    cuuint32_t box[3] = {64, (cuuint32_t)G, (cuuint32_t)(TILE_M / G)};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = enc(&tq, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(q), dims, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
      snprintf(ctx->last_error, sizeof(ctx->last_error), "cuTensorMapEncodeTiled(Q) failed: %d", (int)r);
      return ECHO_ERR_CUDA;
    }
  }
  for (int which = 0; which < 2; ++which) {
    // pool rows [token][128 d] seen as [8-token group][d-half][token in group][64 d]: one box = one page
    cuuint64_t dims[4] = {64, 8, 2, (cuuint64_t)(total_rows / 8)};
    cuuint64_t strides[3] = {(cuuint64_t)D * 2, 128, (cuuint64_t)D * 2 * 8};
    cuuint32_t box[4] = {64, 8, 2, (cuuint32_t)(PAGE / 8)};
    cuuint32_t es[4] = {1, 1, 1, 1};
    CUresult r = enc(which ? &tv : &tk, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, which ? kv->v_pool : kv->k_pool, dims,
                     strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
      snprintf(ctx->last_error, sizeof(ctx->last_error), "cuTensorMapEncodeTiled(KV) failed: %d", (int)r);
      return ECHO_ERR_CUDA;
    }
  }
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
  ECHO_CUDA_TRY(ctx, launch_pdl(k_plan, dim3(1), dim3(PLAN_THREADS), 0, st, sel->sel_offsets, kv->prefix_len, R, Hkv, G,
                                splits, (int)max_items, items, n_items));

  static bool attr_set = false;
  if (!attr_set) {
    ECHO_CUDA_TRY(ctx, cudaFuncSetAttribute(k_verify_attn_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_TOTAL));
    attr_set = true;
  }
  AttnParams p;
  p.items = items; p.n_items = n_items; p.sel_offsets = sel->sel_offsets;
  p.anc_mask = reinterpret_cast<const uint4*>(sel->anc_mask);
  p.page_table = kv->page_table; p.prefix_len = kv->prefix_len; p.max_pages = kv->max_pages_per_req;
  p.Hkv = Hkv; p.Hq = Hq; p.G = G; p.log2G = log2G; p.page_row_base = layer * kv->num_pages;
  p.out = reinterpret_cast<__nv_bfloat16*>(out); p.lse = lse; p.scale_log2 = sm_scale * LOG2E; p.splits = splits;
  p.part_o = part_o; p.part_lse = part_lse; p.n_rows_cap = n_rows; p.status = ctx->dev_status;
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
    ECHO_CUDA_TRY(ctx, cudaLaunchKernelEx(&cfg, k_verify_attn_tc, tq, tk, tv, p));
  }
  ECHO_CUDA_TRY(ctx, cudaGetLastError());
  return ECHO_OK;
}
