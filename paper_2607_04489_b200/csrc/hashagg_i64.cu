// hash aggregation kernels for 64-bit and fused / generic keys (whole-input mode); see hashagg.cuh
#include "hashagg.cuh"

namespace eiger {
int launch_hash_agg_i64(const HashAggLaunch& L, cudaStream_t s) {
  return L.key_kind == KK_I64 ? launch_sig<KK_I64>(L, s) : launch_sig<KK_GEN>(L, s);
}
}  // namespace eiger
