// tcgen05 / TMA verify-attention kernel -- placeholder until the real kernel lands.
#include "common.cuh"
int launch_verify_attn_tc(EchoCtx*, const EchoSelection*, const EchoPagedKV*, int32_t, int32_t, int32_t, const void*,
                          void*, float*, float, int, float*, float*, cudaStream_t) {
  return ECHO_ERR_UNSUPPORTED;
}
