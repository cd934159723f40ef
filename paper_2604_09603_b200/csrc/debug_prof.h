/* Private debug hook of libecho.so, NOT part of the product ABI (include/echo.h): only a library built with
 * -DECHO_WAIT_PROF (ECHO_WAIT_PROF=1 python -m paper_2604_09603_b200.build --force) exports it.
 * Copies the per-CTA mbarrier wait-cycle counters of the last tcgen05 verify-attention launch to HOST memory
 * host_out[n_ctas][ECHO_PROF_SLOTS] (uint64) after a device synchronise.  Slots: K producer 0 total, 1 wait K-empty,
 * 2 wait Q-empty; V producer 4 total, 5 wait V-empty; QK^T issuer 8 total, 9 K-full, 10 S-free, 11 Q-full; epilogue
 * 12 total, 13 stats, 14 O-full; softmax warpgroup w: 16+8w total, +1 S-full, +2 stats-free, +3 PV-done, +4 V-full
 * (ragged tile).  Returns the number of rows written or a negative EchoStatus. */
#ifndef ECHO_DEBUG_PROF_H_
#define ECHO_DEBUG_PROF_H_
#include <stdint.h>
#define ECHO_PROF_CTAS 256 /* rows (persistent CTAs) ... */
#define ECHO_PROF_SLOTS 32 /* ... x counters per CTA */
#ifdef __cplusplus
extern "C"
#endif
int echo_debug_wait_prof(struct EchoCtx* ctx, uint64_t* host_out, int32_t n_ctas);
#endif
