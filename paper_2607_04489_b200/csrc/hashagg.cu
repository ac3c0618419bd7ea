// Step A6b / A6c / second half of A6d: dispatch of the hash aggregation kernels (hashagg.cuh) to
// the translation units that instantiate them.
#include "hashagg.cuh"

namespace eiger {

size_t hash_agg_slot_bytes(const AggPlan& p, int key_kind) {
  size_t w = (key_kind == KK_I32 || key_kind == KK_U32PRE || key_kind == KK_GEN32) ? 4 : 8;
  for (int j = 0; j < p.n_acc; ++j) w += p.op[j] == EIGER_COUNT ? 4 : 8;
  return w;
}

HashAggSmem hash_agg_smem_layout(const KeyDesc& key, const AggPlan& plan, int key_kind, int threads, bool hot, int stages) {
  HashAggSmem m{};
  const bool pre = key_kind == KK_U32PRE || key_kind == KK_U64PRE;
  const uint32_t chunk = 2u * (uint32_t)(pre ? threads - 32 : threads);    // partition mode: the last warp only produces
  auto up = [](uint32_t x) { return (x + 127u) & ~127u; };
  uint32_t off = 0;
  m.n_src = pre ? 1 : key.ncols;
  for (int c = 0; c < m.n_src; ++c) {
    const int w = pre ? (key_kind == KK_U32PRE ? 4 : 8) : (key.dtype[c] == EIGER_I8 ? 1 : key.dtype[c] == EIGER_I32 ? 4 : 8);
    m.kw[c] = (uint8_t)w; m.koff[c] = off; off += up(chunk * (uint32_t)w);
  }
  for (int c = 0; c < plan.n_vals; ++c) { m.vw[c] = plan.vw[c] ? plan.vw[c] : (uint8_t)8; m.voff[c] = off; off += up(chunk * (uint32_t)m.vw[c]); }
  m.stage_bytes = off;
  m.stages = stages > 0 ? std::min(stages, kMaxStages) : kDefaultStages;
  m.hot_off = m.stages * m.stage_bytes;
  const uint32_t hot_bytes = hot ? (uint32_t)((kMaxThreads / 32) * kMaxHot * (kMaxAcc * 8 + 4)) : 0u;
  m.table_off = up(m.hot_off + hot_bytes);
  return m;
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
