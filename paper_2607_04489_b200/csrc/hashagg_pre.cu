// hash aggregation kernels of the partition mode (rebased keys written by partition.cu); see hashagg.cuh
#include "hashagg.cuh"

namespace eiger {
int launch_hash_agg_pre(const HashAggLaunch& L, cudaStream_t s) {
  return L.key_kind == KK_U32PRE ? launch_sig<KK_U32PRE>(L, s) : launch_sig<KK_U64PRE>(L, s);
}
}  // namespace eiger
