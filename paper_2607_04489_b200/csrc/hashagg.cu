// Step A6b / A6c / second half of A6d: dispatch of the hash aggregation kernels (hashagg.cuh) to
// the translation units that instantiate them.
#include "hashagg.cuh"

namespace eiger {

size_t hash_agg_slot_bytes(const AggPlan& p, int key_kind) {
  size_t w = (key_kind == KK_I32 || key_kind == KK_U32PRE || key_kind == KK_GEN32) ? 4 : 8;
  for (int j = 0; j < p.n_acc; ++j) w += p.op[j] == EIGER_COUNT ? 4 : 8;
  return w;
}

int launch_hash_agg(const HashAggLaunch& L, cudaStream_t s) {
  if (L.threads < 32 || L.threads > kMaxThreads || (L.threads & 31) || L.slots < 64) return EIGER_ERR_ARG;
  switch (L.key_kind) {
    case KK_I32: return launch_hash_agg_i32(L, s);
    case KK_I64: case KK_GEN: return launch_hash_agg_i64(L, s);
    case KK_U32PRE: case KK_U64PRE: return launch_hash_agg_pre(L, s);
    default: return EIGER_ERR_ARG;
  }
}

}  // namespace eiger
