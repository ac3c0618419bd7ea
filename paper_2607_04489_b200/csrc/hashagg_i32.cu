// hash aggregation kernels for a single int32 key column (whole-input mode); see hashagg.cuh
#include "hashagg.cuh"

namespace eiger {
int launch_hash_agg_i32(const HashAggLaunch& L, cudaStream_t s) { return launch_sig<KK_I32>(L, s); }
}  // namespace eiger
