/* CPU ORACLE for S6-S7 (verify attention) in plain C -- TEST INFRASTRUCTURE ONLY.
 *
 * The same definition as `verify_attn` in oracle/echo_oracle.py, written as loops so that the whole of a
 * BASELINE.json configuration (131 072 (node, head) rows at cfg2) can be checked row by row and timed on all host
 * cores: for packed node k = (request i, local node l) and query head h (KV head h / (Hq / Hkv), S:A-5)
 *
 *     visible set  T = [0, P_i)  U  { P_i + a : bit a of anc_mask[k] set }            (S:A-1, A-2)
 *     s_t   = sm_scale * <q[k][h], K[t]>                                  t in T, fp64, d ascending
 *     M     = max_t s_t,   Z = sum_t exp(s_t - M)                                   t ascending
 *     out   = (sum_t exp(s_t - M) V[t]) / Z,   lse = M + ln Z                                      (S:A-4)
 *
 * with K[t], V[t] the rows of the paged pools [layer][page][Hkv][16][128] (S:A-3) at page page_table[i][t / 16],
 * slot t % 16.  bf16 inputs are widened exactly; there is no online softmax, no splitting, no blocking: one row is
 * computed start to finish by one thread, rows are shared out over `threads` POSIX threads (the result does not depend
 * on their number).  No code, header, table or constant is shared with the CUDA path (paper_2604_09603_b200/csrc).
 *
 * Pins (tests/test_oracle_attn_c_pins.py, -m "not gpu"): every row of cfg0 and samples of cfg1 / cfg3 / cfg4 against
 * the numpy oracle (itself pinned by closed forms and a brute-force dense softmax); Q = 0 => out = mean of the visible
 * V rows and lse = ln |T|, from a gather written in the test; a one-hot K / q construction whose softmax is known;
 * thread-count invariance (bit-identical).  The paper prints no numeric example of this operator: parity with the
 * paper's own values is unpinned, as for every function of the oracle.
 *
 * Built by oracle/attn_c.py (and __graft_entry__.build()):  gcc -O2 -shared -fPIC -pthread ... -lm   (no -ffast-math:
 * the sums run in source order).
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define D 128
#define PAGE 16

typedef struct {
  const int32_t* sel_offsets; /* [R + 1] */
  const int32_t* sel_req;     /* [n_selected] */
  const uint32_t* anc_mask;   /* [n_selected][4] */
  const uint16_t* q;          /* bf16 bits [cap][Hq][128] */
  const uint16_t* k_pool;     /* bf16 bits [layers][pages][Hkv][16][128] */
  const uint16_t* v_pool;
  const int32_t* page_table;  /* [R][max_pages] */
  const int32_t* prefix_len;  /* [R] */
  int max_pages, num_pages, Hq, Hkv, layer;
  double scale;
  const int32_t* rows;        /* [n_rows][2] = (packed node, head), or NULL: all rows of nodes [0, n_selected) */
  int64_t n_rows;
  double* out;                /* [n_rows][128] */
  double* lse;                /* [n_rows] */
  int64_t max_visible;
} problem_t;

typedef struct {
  const problem_t* p;
  int64_t first, step; /* rows first, first + step, ... : interleaved so that long and short prefixes mix */
  int failed;
} job_t;

static double bf16_bits_to_f64(uint16_t b) {
  const uint32_t u = (uint32_t)b << 16;
  float f;
  memcpy(&f, &u, 4);
  return (double)f;
}

/* row of token position t of request i, KV head kvh, in a pool */
static const uint16_t* pool_row(const problem_t* p, const uint16_t* pool, int i, int kvh, int64_t t) {
  const int64_t page = p->page_table[(int64_t)i * p->max_pages + t / PAGE];
  return pool + ((((int64_t)p->layer * p->num_pages + page) * p->Hkv + kvh) * PAGE + t % PAGE) * D;
}

static void one_row(const problem_t* p, int k, int h, int64_t* pos, double* s, double* out, double* lse) {
  const int i = p->sel_req[k];
  const int64_t P = p->prefix_len[i];
  const int kvh = h / (p->Hq / p->Hkv);
  int64_t n = 0;
  for (int64_t t = 0; t < P; ++t) pos[n++] = t;
  for (int a = 0; a < 128; ++a)
    if ((p->anc_mask[(int64_t)k * 4 + a / 32] >> (a % 32)) & 1u) pos[n++] = P + a;
  double qv[D];
  const uint16_t* qrow = p->q + ((int64_t)k * p->Hq + h) * D;
  for (int d = 0; d < D; ++d) qv[d] = bf16_bits_to_f64(qrow[d]);
  double M = -INFINITY;
  for (int64_t j = 0; j < n; ++j) {
    const uint16_t* kr = pool_row(p, p->k_pool, i, kvh, pos[j]);
    double dot = 0.0;
    for (int d = 0; d < D; ++d) dot += bf16_bits_to_f64(kr[d]) * qv[d];
    s[j] = p->scale * dot;
    if (s[j] > M) M = s[j];
  }
  double Z = 0.0, acc[D];
  for (int d = 0; d < D; ++d) acc[d] = 0.0;
  for (int64_t j = 0; j < n; ++j) {
    const double e = exp(s[j] - M);
    const uint16_t* vr = pool_row(p, p->v_pool, i, kvh, pos[j]);
    Z += e;
    for (int d = 0; d < D; ++d) acc[d] += e * bf16_bits_to_f64(vr[d]);
  }
  for (int d = 0; d < D; ++d) out[d] = acc[d] / Z;
  *lse = M + log(Z);
}

static void* worker(void* arg) {
  job_t* job = (job_t*)arg;
  const problem_t* p = job->p;
  int64_t* pos = (int64_t*)malloc(sizeof(int64_t) * (size_t)p->max_visible);
  double* s = (double*)malloc(sizeof(double) * (size_t)p->max_visible);
  if (!pos || !s) {
    job->failed = 1;
  } else {
    for (int64_t r = job->first; r < p->n_rows; r += job->step) {
      const int k = p->rows ? p->rows[2 * r] : (int)(r / p->Hq);
      const int h = p->rows ? p->rows[2 * r + 1] : (int)(r % p->Hq);
      one_row(p, k, h, pos, s, p->out + r * D, p->lse + r);
    }
  }
  free(pos);
  free(s);
  return NULL;
}

/* Returns 0, or -1 on a bad argument / failed allocation.  rows == NULL: all n_selected * Hq rows in (node, head)
 * order (then n_rows must be n_selected * Hq). */
int oracle_verify_attn(const int32_t* sel_offsets, const int32_t* sel_req, const uint32_t* anc_mask, int32_t n_selected,
                       int32_t num_requests, const uint16_t* q, const uint16_t* k_pool, const uint16_t* v_pool,
                       const int32_t* page_table, const int32_t* prefix_len, int32_t max_pages, int32_t num_pages,
                       int32_t Hq, int32_t Hkv, int32_t layer, float sm_scale, const int32_t* rows, int64_t n_rows,
                       double* out, double* lse, int32_t threads) {
  if (!sel_offsets || !sel_req || !anc_mask || !q || !k_pool || !v_pool || !page_table || !prefix_len || !out || !lse)
    return -1;
  if (Hq <= 0 || Hkv <= 0 || Hq % Hkv || n_rows < 0 || threads < 1 || (!rows && n_rows != (int64_t)n_selected * Hq))
    return -1;
  problem_t p;
  p.sel_offsets = sel_offsets; p.sel_req = sel_req; p.anc_mask = anc_mask; p.q = q; p.k_pool = k_pool; p.v_pool = v_pool;
  p.page_table = page_table; p.prefix_len = prefix_len; p.max_pages = max_pages; p.num_pages = num_pages;
  p.Hq = Hq; p.Hkv = Hkv; p.layer = layer; p.scale = (double)sm_scale; p.rows = rows; p.n_rows = n_rows;
  p.out = out; p.lse = lse;
  int64_t maxP = 0;
  for (int i = 0; i < num_requests; ++i)
    if (prefix_len[i] > maxP) maxP = prefix_len[i];
  p.max_visible = maxP + 128;
  if (threads > n_rows) threads = n_rows > 0 ? (int32_t)n_rows : 1;
  pthread_t* th = (pthread_t*)malloc(sizeof(pthread_t) * (size_t)threads);
  job_t* jobs = (job_t*)malloc(sizeof(job_t) * (size_t)threads);
  if (!th || !jobs) { free(th); free(jobs); return -1; }
  int rc = 0, started = 0;
  for (int t = 0; t < threads; ++t) {
    jobs[t].p = &p;
    jobs[t].first = t;
    jobs[t].step = threads;
    jobs[t].failed = 0;
    if (pthread_create(&th[t], NULL, worker, &jobs[t]) != 0) { rc = -1; break; }
    ++started;
  }
  for (int t = 0; t < started; ++t) {
    pthread_join(th[t], NULL);
    if (jobs[t].failed) rc = -1;
  }
  free(th);
  free(jobs);
  return rc;
}
