// Pieces shared by the two row-moving kernels (partition.cu: radix partition by hash bits;
// sortagg.cu: stable radix-sort passes by key digits): the shared-memory layout of a tile whose
// rows arrive through the bulk-copy ring (ring.cuh) and are staged column by column.
#pragma once
#include <algorithm>

#include "internal.h"
#include "ring.cuh"
#include "rows.cuh"

namespace eiger {
namespace {

struct ScatterSmem {
  uint32_t koff[kMaxKeyCols], voff[kMaxVals];   // columns inside a ring stage
  uint8_t kw[kMaxKeyCols], vw[kMaxVals];
  int n_src;
  uint32_t stage_bytes, out_off, pid_off, total;
  int stages;
};
__device__ __forceinline__ uint64_t stage_elem(const unsigned char* col, int w, uint32_t r) {
  if (w == 8) return *reinterpret_cast<const uint64_t*>(col + 8 * (size_t)r);
  if (w == 4) return (uint64_t)(int64_t)*reinterpret_cast<const int32_t*>(col + 4 * (size_t)r);
  return (uint64_t)(int64_t)*reinterpret_cast<const int8_t*>(col + r);
}
template <int KK>
__device__ __forceinline__ typename KeyTraits<KK>::U stage_key(const KeyDesc& key, const ScatterSmem& sm, const unsigned char* st, uint32_t r) {
  using U = typename KeyTraits<KK>::U;
  if constexpr (KK == KK_I32) return *reinterpret_cast<const uint32_t*>(st + sm.koff[0] + 4 * (size_t)r) - (uint32_t)key.base[0];
  else if constexpr (KK == KK_U32PRE) return *reinterpret_cast<const uint32_t*>(st + sm.koff[0] + 4 * (size_t)r);
  else if constexpr (KK == KK_I64) return *reinterpret_cast<const uint64_t*>(st + sm.koff[0] + 8 * (size_t)r) - key.base[0];
  else if constexpr (KK == KK_U64PRE) return *reinterpret_cast<const uint64_t*>(st + sm.koff[0] + 8 * (size_t)r);
  else {
    uint64_t d[kMaxKeyCols];
#pragma unroll
    for (int c = 0; c < kMaxKeyCols; ++c) d[c] = c < key.ncols ? stage_elem(st + sm.koff[c], sm.kw[c], r) - key.base[c] : 0ull;
    return (U)fuse_cols(key, d);
  }
}

// shared-memory layout of the scatter kernel for a tile of `tile` rows
inline ScatterSmem scatter_smem_layout(const KeyDesc& key, int key_kind, const uint8_t* vw, int n_vals, uint32_t tile, int stages, size_t out_key_bytes) {
  ScatterSmem m{};
  auto up = [](uint32_t x) { return (x + 127u) & ~127u; };
  uint32_t off = 0;
  const bool pre = key_kind == KK_U32PRE || key_kind == KK_U64PRE;
  m.n_src = pre ? 1 : key.ncols;
  for (int c = 0; c < m.n_src; ++c) {
    const int w = pre ? (key_kind == KK_U32PRE ? 4 : 8) : (key.dtype[c] == EIGER_I8 ? 1 : key.dtype[c] == EIGER_I32 ? 4 : 8);
    m.kw[c] = (uint8_t)w; m.koff[c] = off; off += up(tile * (uint32_t)w);
  }
  for (int c = 0; c < n_vals; ++c) { m.vw[c] = vw[c] ? vw[c] : (uint8_t)8; m.voff[c] = off; off += up(tile * (uint32_t)m.vw[c]); }
  m.stage_bytes = off;
  m.stages = stages;
  m.out_off = (uint32_t)stages * m.stage_bytes;
  m.pid_off = m.out_off + up(tile * (uint32_t)std::max<size_t>(8, out_key_bytes));
  m.total = m.pid_off + up(tile * 2u);
  return m;
}


}  // namespace
}  // namespace eiger
