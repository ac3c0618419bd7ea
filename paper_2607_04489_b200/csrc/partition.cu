// Step A6d, first half: radix partition of the rows by the top bits of the table hash
// ("applies a hash function to the keys before partitioning to ensure more even partition
// sizes", §3.3; best for g > 2^20).  Keys leave this pass
// already rebased and fused (KK_U32PRE / KK_U64PRE); value columns travel with their keys
// (the paper's GFTR).
//
// One level = histogram (keys only) -> exclusive scan -> scatter.  The scatter stages every
// tile in shared memory in partition order first, so that what leaves the SM are runs of
// consecutive rows of one partition, not one 8-byte store per lane.  Two levels (fan-out
// P1 x P2) are chained when the final partition count exceeds what one staged pass writes
// efficiently; level 2 runs per level-1 partition (blockIdx.y) over the level-1 output.
#include <algorithm>

#include <cstdlib>

#include "internal.h"
#include "ring.cuh"
#include "rows.cuh"
#include "scatter.cuh"

namespace eiger {
namespace {

#ifndef EIGER_SCATTER_PT
#define EIGER_SCATTER_PT 512
#endif
#ifndef EIGER_SCATTER_PR
#define EIGER_SCATTER_PR 8
#endif
constexpr int kPT = EIGER_SCATTER_PT;     // threads per CTA
constexpr int kPR = EIGER_SCATTER_PR;     // rows per thread per tile
constexpr int kTile = kPT * kPR;          // 4096 rows staged per tile
constexpr int kMaxFan = 1024;             // partitions per level
#ifndef EIGER_SCATTER_CTAS
#define EIGER_SCATTER_CTAS 2
#endif
constexpr int kScatterCtas = EIGER_SCATTER_CTAS;

template <int KK> struct SrcKey { using U = typename KeyTraits<KK>::U; };

struct LevelArgs {
  KeyDesc key;                              // source keys (original columns or a partitioned copy)
  const void* vals[kMaxVals];             // value columns, sm.vw[c] bytes per element
  void* out_vals[kMaxVals];
  void* out_keys;                           // UO[n]
  const unsigned long long* seg_off;        // nullptr: one segment [0, n); else [gridDim.y + 1]
  uint32_t* hist;                           // [segments * fan]
  unsigned long long* cursor;               // [segments * fan]
  int64_t n;
  int32_t n_vals, fan, shift;
};

template <int KK>
__global__ void __launch_bounds__(kPT)
part_hist_kernel(const __grid_constant__ LevelArgs a) {
  using U = typename SrcKey<KK>::U;
  __shared__ uint32_t s_hist[kMaxFan];
  const int tid = threadIdx.x, seg = blockIdx.y;
  for (int p = tid; p < a.fan; p += kPT) s_hist[p] = 0;
  __syncthreads();
  const int64_t r0 = a.seg_off ? (int64_t)a.seg_off[seg] : 0, r1 = a.seg_off ? (int64_t)a.seg_off[seg + 1] : a.n;
  const uint32_t mask = (uint32_t)a.fan - 1u;
  const int64_t stride = (int64_t)gridDim.x * kPT;
  int64_t i = r0 + (int64_t)blockIdx.x * kPT + tid;
  for (; i + 3 * stride < r1; i += 4 * stride) {
    U u[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) u[k] = load_u<KK>(a.key, i + k * stride);
#pragma unroll
    for (int k = 0; k < 4; ++k) atomicAdd(&s_hist[part_id<U>(u[k], a.shift, mask)], 1u);
  }
  for (; i < r1; i += stride) atomicAdd(&s_hist[part_id<U>(load_u<KK>(a.key, i), a.shift, mask)], 1u);
  __syncthreads();
  for (int p = tid; p < a.fan; p += kPT) if (s_hist[p]) atomicAdd(&a.hist[(size_t)seg * a.fan + p], s_hist[p]);
}

// level-1 histogram from one already taken at a larger fan-out: ids are top bits of the hash,
// so partition p of `fan` is partitions [p * g, (p + 1) * g) of `pre_fan`, g = pre_fan / fan
__global__ void part_fold_kernel(const uint32_t* __restrict__ pre, int pre_fan, uint32_t* __restrict__ hist, int fan) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= fan) return;
  const int g = pre_fan / fan;
  uint32_t c = 0;
  for (int k = 0; k < g; ++k) c += pre[p * g + k];
  hist[p] = c;
}

// exclusive prefix sum of `count` 32-bit counts -> 64-bit offsets [count + 1] and cursors [count]
// (single CTA; count <= 2^20: a few microseconds)
__global__ void __launch_bounds__(1024)
part_scan_kernel(const uint32_t* __restrict__ hist, unsigned long long* __restrict__ off,
                 unsigned long long* __restrict__ cursor, int count) {
  __shared__ unsigned long long s_part[1024];
  const int tid = threadIdx.x;
  const int per = (count + 1023) / 1024;
  const int b = tid * per, e = min(count, b + per);
  unsigned long long local = 0;
  for (int p = b; p < e; ++p) local += hist[p];
  s_part[tid] = local;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const unsigned long long v = tid >= o ? s_part[tid - o] : 0ull;
    __syncthreads();
    s_part[tid] += v;
    __syncthreads();
  }
  unsigned long long run = s_part[tid] - local;
  for (int p = b; p < e; ++p) { off[p] = run; cursor[p] = run; run += hist[p]; }
  if (tid == 1023) off[count] = s_part[1023];
}

// Work items of the per-partition aggregation pass: a partition much larger than the average (a
// hot key: C3's top key owns 12 % of the rows) is cut into several items so that one CTA is not
// left with it; item_off[p] .. item_off[p + 1] are partition p's items (exclusive prefix sum).
__global__ void __launch_bounds__(1024)
part_items_kernel(const unsigned long long* __restrict__ off, unsigned long long* __restrict__ item_off,
                  uint32_t* __restrict__ item_part, int count, unsigned long long chunk_rows) {
  __shared__ unsigned long long s_part[1024];
  const int tid = threadIdx.x;
  const int per = (count + 1023) / 1024;
  const int b = tid * per, e = min(count, b + per);
  auto items = [&](int p) -> unsigned long long {
    const unsigned long long rows = off[p + 1] - off[p];
    return rows == 0 ? 0ull : (rows > 2 * chunk_rows ? (rows + chunk_rows - 1) / chunk_rows : 1ull);
  };
  unsigned long long local = 0;
  for (int p = b; p < e; ++p) local += items(p);
  s_part[tid] = local;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const unsigned long long v = tid >= o ? s_part[tid - o] : 0ull;
    __syncthreads();
    s_part[tid] += v;
    __syncthreads();
  }
  unsigned long long run = s_part[tid] - local;
  // item -> partition map: the aggregation pass reads its partition with one broadcast load
  for (int p = b; p < e; ++p) {
    item_off[p] = run;
    const unsigned long long k = items(p);
    for (unsigned long long i = 0; i < k; ++i) item_part[run + i] = (uint32_t)p;
    run += k;
  }
  if (tid == 1023) item_off[count] = s_part[1023];
}

// ---- scatter ---------------------------------------------------------------------------------
// The rows of a tile arrive through a shared-memory ring filled by bulk copies (ring.cuh): the read
// stream does not stop while the CTA ranks, stages and writes (the round-1 kernel, whose threads
// loaded their own rows, moved 3.4-3.9 TB/s with half of its stall samples on those loads).  A tile
// is RPT x blockDim rows; each column is staged in partition order in shared memory and leaves
// the SM as runs of consecutive rows of one partition (measured, eiger_probe("store_warp"): random
// 256-byte runs are written at 6.0 TB/s, 128-byte runs at 4.4 TB/s).
struct ScatterArgs {
  LevelArgs lv;
  ScatterSmem sm;
  uint32_t tile;
};

template <int KK, class UO, int RPT>
__global__ void __launch_bounds__(1024, 1)
part_scatter_kernel(const __grid_constant__ ScatterArgs A) {
  using U = typename SrcKey<KK>::U;
  const LevelArgs& a = A.lv;
  const ScatterSmem& sm = A.sm;
  extern __shared__ __align__(128) unsigned char dsm[];      // [ring stages][s_out: tile x 8][s_pid: tile x 2]
  __shared__ __align__(8) uint64_t s_full[kMaxStages], s_empty[kMaxStages];
  __shared__ long long s_delta[kMaxFan];
  __shared__ uint32_t s_cnt[kMaxFan], s_loff[kMaxFan];
  __shared__ uint32_t s_warp[32];
  unsigned char* s_out = dsm + sm.out_off;
  uint16_t* s_pid = reinterpret_cast<uint16_t*>(dsm + sm.pid_off);
  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5, seg = blockIdx.y;
  const int fan = a.fan;
  const uint32_t mask = (uint32_t)fan - 1u, tile = A.tile;
  const int64_t r0 = a.seg_off ? (int64_t)a.seg_off[seg] : 0, r1 = a.seg_off ? (int64_t)a.seg_off[seg + 1] : a.n;
  unsigned long long* cursor = a.cursor + (size_t)seg * fan;
  UO* out_keys = static_cast<UO*>(a.out_keys);
  for (int p = tid; p < fan; p += T) s_cnt[p] = 0;
  if (tid == 0) {
    for (int s = 0; s < sm.stages; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], (uint32_t)(T >> 5)); }
    mbar_fence_init();
  }
  __syncthreads();
  // tiles of this segment: tile t covers rows [A0 + t * tile, + tile), A0 = r0 rounded down to 32 rows
  // (every bulk copy then starts 16-byte aligned); rows outside [r0, r1) are masked.  Only tiles that
  // end inside the column(s) travel by bulk copy: the last, ragged one of a caller's column is loaded
  // by the threads (a bulk copy must be a multiple of 16 bytes and may not run past the allocation).
  const int64_t A0 = r0 & ~(int64_t)31;
  const int64_t n_tiles = r1 > r0 ? (r1 - A0 + tile - 1) / tile : 0;
  const bool padded = a.seg_off != nullptr;                  // level 2 reads the library's own padded copy
  const int64_t n_bulk = padded ? n_tiles : (r1 - A0) / tile;
  const int64_t mine = n_bulk > blockIdx.x ? (n_bulk - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const uint64_t policy = policy_evict_first();
  uint32_t g_issued = 0;
  auto issue = [&](uint32_t g) {                             // thread 0
    const int64_t row0 = A0 + ((int64_t)blockIdx.x + (int64_t)g * gridDim.x) * tile;
    int64_t rows = ((r1 - row0) + 31) & ~(int64_t)31;
    if (rows > (int64_t)tile) rows = tile;
    const uint32_t s = g % (uint32_t)sm.stages;
    if (g >= (uint32_t)sm.stages) mbar_wait(&s_empty[s], ((g / (uint32_t)sm.stages) - 1u) & 1u);
    unsigned char* st = dsm + (size_t)s * sm.stage_bytes;
    uint32_t bytes = 0;
    for (int c = 0; c < sm.n_src; ++c) bytes += (uint32_t)rows * sm.kw[c];
    for (int c = 0; c < a.n_vals; ++c) bytes += (uint32_t)rows * sm.vw[c];
    mbar_expect_tx(&s_full[s], bytes);
    for (int c = 0; c < sm.n_src; ++c)
      bulk_g2s_hint(st + sm.koff[c], static_cast<const unsigned char*>(a.key.ptr[c]) + row0 * sm.kw[c], (uint32_t)rows * sm.kw[c], &s_full[s], policy);
    for (int c = 0; c < a.n_vals; ++c)
      bulk_g2s_hint(st + sm.voff[c], reinterpret_cast<const unsigned char*>(a.vals[c]) + row0 * sm.vw[c], (uint32_t)rows * sm.vw[c], &s_full[s], policy);
  };
  if (tid == 0) for (; g_issued < (uint32_t)sm.stages && (int64_t)g_issued < mine; ++g_issued) issue(g_issued);

  // one tile whose rows sit in stage `st`: rows [row0, row0 + tile) of the segment, valid where in [r0, r1)
  auto process = [&](const unsigned char* st, int64_t row0, int ring_stage) {
    const uint32_t lo = (uint32_t)(r0 > row0 ? r0 - row0 : 0), hi = (uint32_t)(r1 - row0 < (int64_t)tile ? r1 - row0 : (int64_t)tile);
    // A: keys -> partition ids and ranks inside the tile
    U u[RPT];
    uint32_t pos[RPT];
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
      const uint32_t i = (uint32_t)(r * T + tid);
      if (i >= lo && i < hi) {
        u[r] = stage_key<KK>(a.key, sm, st, i);
        const uint32_t q = part_id<U>(u[r], a.shift, mask);
        pos[r] = (q << 16) | atomicAdd(&s_cnt[q], 1u);       // rank < tile <= 8192 fits 16 bits
      }
    }
    __syncthreads();
    // B: exclusive scan of the per-partition counts (one counter per thread: fan <= blockDim); claim global space
    {
      const uint32_t c = tid < fan ? s_cnt[tid] : 0u;
      uint32_t inc = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
      if (lane == 31) s_warp[warp] = inc;
      __syncthreads();
      if (warp == 0) {
        const uint32_t w = lane < (T >> 5) ? s_warp[lane] : 0u;
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += y; }
        s_warp[lane] = winc - w;
      }
      __syncthreads();
      if (tid < fan) {
        const uint32_t run = s_warp[warp] + inc - c;
        s_loff[tid] = run;
        s_delta[tid] = c ? (long long)atomicAdd(&cursor[tid], (unsigned long long)c) - (long long)run : 0ll;
        s_cnt[tid] = 0;
      }
    }
    __syncthreads();
    // C/D per column: stage in partition order, then write runs.  Keys first (they are in registers).
    UO* ko = reinterpret_cast<UO*>(s_out);
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
      const uint32_t i = (uint32_t)(r * T + tid);
      if (i >= lo && i < hi) {
        const uint32_t q = pos[r] >> 16;
        pos[r] = s_loff[q] + (pos[r] & 0xFFFFu);
        ko[pos[r]] = (UO)u[r];
        s_pid[pos[r]] = (uint16_t)q;
      }
    }
    __syncthreads();
    const uint32_t m = hi - lo;                              // rows of this tile
    // write-out, unrolled: the destination of staged position j = r * T + tid is the same for every
    // column, so it is computed once (all partition-id loads, then all offset loads: independent
    // shared-memory loads in flight together instead of one dependent chain per position)
    long long dstp[RPT];
    {
      uint32_t pid[RPT];
#pragma unroll
      for (int r = 0; r < RPT; ++r) { const uint32_t j = (uint32_t)(r * T + tid); pid[r] = j < m ? s_pid[j] : 0u; }
#pragma unroll
      for (int r = 0; r < RPT; ++r) { const uint32_t j = (uint32_t)(r * T + tid); dstp[r] = j < m ? s_delta[pid[r]] + (long long)j : -1ll; }
      UO kv[RPT];
#pragma unroll
      for (int r = 0; r < RPT; ++r) { const uint32_t j = (uint32_t)(r * T + tid); if (j < m) kv[r] = ko[j]; }
#pragma unroll
      for (int r = 0; r < RPT; ++r) if (dstp[r] >= 0) out_keys[dstp[r]] = kv[r];
    }
    for (int c = 0; c < a.n_vals; ++c) {
      __syncthreads();                                       // s_out is read by the previous column's write-out
      const unsigned char* col = st + sm.voff[c];
      if (sm.vw[c] == 8) {
        uint64_t* vo = reinterpret_cast<uint64_t*>(s_out);
#pragma unroll
        for (int r = 0; r < RPT; ++r) { const uint32_t i = (uint32_t)(r * T + tid); if (i >= lo && i < hi) vo[pos[r]] = *reinterpret_cast<const uint64_t*>(col + 8 * (size_t)i); }
        if (c == a.n_vals - 1 && ring_stage >= 0) { __syncwarp(); if (lane == 0) mbar_arrive(&s_empty[ring_stage]); }
        __syncthreads();
        uint64_t* dst = static_cast<uint64_t*>(a.out_vals[c]);
        uint64_t vv[RPT];
#pragma unroll
        for (int r = 0; r < RPT; ++r) { const uint32_t j = (uint32_t)(r * T + tid); if (j < m) vv[r] = vo[j]; }
#pragma unroll
        for (int r = 0; r < RPT; ++r) if (dstp[r] >= 0) dst[dstp[r]] = vv[r];
      } else {
        uint32_t* vo = reinterpret_cast<uint32_t*>(s_out);
#pragma unroll
        for (int r = 0; r < RPT; ++r) { const uint32_t i = (uint32_t)(r * T + tid); if (i >= lo && i < hi) vo[pos[r]] = *reinterpret_cast<const uint32_t*>(col + 4 * (size_t)i); }
        if (c == a.n_vals - 1 && ring_stage >= 0) { __syncwarp(); if (lane == 0) mbar_arrive(&s_empty[ring_stage]); }
        __syncthreads();
        uint32_t* dst = static_cast<uint32_t*>(a.out_vals[c]);
        uint32_t vv[RPT];
#pragma unroll
        for (int r = 0; r < RPT; ++r) { const uint32_t j = (uint32_t)(r * T + tid); if (j < m) vv[r] = vo[j]; }
#pragma unroll
        for (int r = 0; r < RPT; ++r) if (dstp[r] >= 0) dst[dstp[r]] = vv[r];
      }
    }
    if (a.n_vals == 0 && ring_stage >= 0) { __syncwarp(); if (lane == 0) mbar_arrive(&s_empty[ring_stage]); }
    __syncthreads();                                         // s_out / s_pid / s_delta are reused by the next tile
  };

  for (int64_t k = 0; k < mine; ++k) {
    const uint32_t g = (uint32_t)k, s = g % (uint32_t)sm.stages;
    mbar_wait(&s_full[s], (g / (uint32_t)sm.stages) & 1u);
    process(dsm + (size_t)s * sm.stage_bytes, A0 + ((int64_t)blockIdx.x + k * gridDim.x) * tile, (int)s);
    if (tid == 0 && (int64_t)g_issued < mine) { issue(g_issued); ++g_issued; }
  }
  // the ragged last tile of a caller's column: loaded by the threads into stage 0 (every bulk copy of
  // this CTA has landed and been consumed by now)
  if (!padded && n_tiles > n_bulk && (int)(n_bulk % gridDim.x) == (int)blockIdx.x) {
    const int64_t row0 = A0 + n_bulk * tile;
    const uint32_t rows = (uint32_t)(r1 - row0);
    unsigned char* st = dsm;
    for (int c = 0; c < sm.n_src; ++c) {
      const unsigned char* src = static_cast<const unsigned char*>(a.key.ptr[c]) + row0 * sm.kw[c];
      for (uint32_t o = tid; o < rows * sm.kw[c]; o += T) st[sm.koff[c] + o] = src[o];
    }
    for (int c = 0; c < a.n_vals; ++c) {
      const uint32_t* src = reinterpret_cast<const uint32_t*>(reinterpret_cast<const unsigned char*>(a.vals[c]) + row0 * sm.vw[c]);
      uint32_t* d = reinterpret_cast<uint32_t*>(st + sm.voff[c]);
      for (uint32_t o = tid; o < rows * (sm.vw[c] / 4u); o += T) d[o] = src[o];
    }
    __syncthreads();
    process(st, row0, -1);
  }
}

// ---- the round-1 scatter: the threads load their own rows (8 per thread, 4096-row tiles, two CTAs
// per SM, the next tile prefetched into L2); 8-byte value columns only.  Kept selectable
// (EIGER_SCATTER_RING=0) for same-box comparisons with the ring version above. ----
template <int KK, class UO>
__global__ void __launch_bounds__(kPT, kScatterCtas)
part_scatter_ldg_kernel(const __grid_constant__ LevelArgs a) {
  using U = typename SrcKey<KK>::U;
  // dynamic shared memory (above the 48 KB static limit): staging buffers, then the counters
  extern __shared__ __align__(16) unsigned char dsm[];
  uint64_t* s_val = reinterpret_cast<uint64_t*>(dsm);
  UO* s_key = reinterpret_cast<UO*>(dsm + sizeof(uint64_t) * kTile);
  long long* s_delta = reinterpret_cast<long long*>(dsm + (sizeof(uint64_t) + sizeof(UO)) * kTile);
  uint32_t* s_cnt = reinterpret_cast<uint32_t*>(s_delta + kMaxFan);
  uint32_t* s_loff = s_cnt + kMaxFan;
  uint16_t* s_pid = reinterpret_cast<uint16_t*>(s_loff + kMaxFan);
  __shared__ uint32_t s_warp[kPT / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, seg = blockIdx.y;
  const int fan = a.fan;
  const uint32_t mask = (uint32_t)fan - 1u;
  const int64_t r0 = a.seg_off ? (int64_t)a.seg_off[seg] : 0, r1 = a.seg_off ? (int64_t)a.seg_off[seg + 1] : a.n;
  unsigned long long* cursor = a.cursor + (size_t)seg * fan;
  UO* out_keys = static_cast<UO*>(a.out_keys);
  for (int p = tid; p < fan; p += kPT) s_cnt[p] = 0;
  __syncthreads();
  const int64_t n_tiles = (r1 - r0 + kTile - 1) / kTile;
  constexpr int kPer = kMaxFan / kPT;       // counters per thread in the scan (consecutive)
  for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    const int64_t base = r0 + t * kTile;
    const int m = (int)min((int64_t)kTile, r1 - base);
    // the CTA's next tile is pulled into L2 now: its loads are what this kernel waits for most
    // (ncu: long_scoreboard 49 % of stall samples with one tile in flight per CTA)
    {
      const int64_t nb = base + (int64_t)gridDim.x * kTile;
      if constexpr (KK != KK_GEN && KK != KK_GEN32) {
       if (nb < r1 && a.key.ncols == 1) {
        const int64_t nm = min((int64_t)kTile, r1 - nb);
        const int64_t kbytes = nm * (int64_t)sizeof(U), vbytes = nm * 8;
        const char* kp = static_cast<const char*>(a.key.ptr[0]) + nb * (int64_t)sizeof(U);
        for (int64_t o = (int64_t)tid * 128; o < kbytes; o += (int64_t)kPT * 128) prefetch_l2(kp + o);
        for (int c = 0; c < a.n_vals; ++c) {
          const char* vp = reinterpret_cast<const char*>(static_cast<const uint64_t*>(a.vals[c]) + nb);
          for (int64_t o = (int64_t)tid * 128; o < vbytes; o += (int64_t)kPT * 128) prefetch_l2(vp + o);
        }
       }
      } else if (nb < r1) {
        // several key columns (level 1 of a fused key): each column at its own width
        const int64_t nm = min((int64_t)kTile, r1 - nb);
        for (int kc = 0; kc < a.key.ncols; ++kc) {
          const int64_t w = a.key.dtype[kc] == EIGER_I8 ? 1 : (a.key.dtype[kc] == EIGER_I32 ? 4 : 8);
          const char* kp = static_cast<const char*>(a.key.ptr[kc]) + nb * w;
          for (int64_t o = (int64_t)tid * 128; o < nm * w; o += (int64_t)kPT * 128) prefetch_l2(kp + o);
        }
        for (int c = 0; c < a.n_vals; ++c) {
          const char* vp = reinterpret_cast<const char*>(static_cast<const uint64_t*>(a.vals[c]) + nb);
          for (int64_t o = (int64_t)tid * 128; o < nm * 8; o += (int64_t)kPT * 128) prefetch_l2(vp + o);
        }
      }
    }
    // A: keys -> partition ids and ranks inside the tile
    U u[kPR];
    uint32_t pos[kPR];
    uint64_t v0[kPR];
#pragma unroll
    for (int r = 0; r < kPR; ++r) {
      const int i = r * kPT + tid;
      if (i < m) {
        u[r] = load_u<KK>(a.key, base + i);
        if (a.n_vals > 0) v0[r] = ldg_stream_u64(static_cast<const uint64_t*>(a.vals[0]) + base + i);
      }
    }
#pragma unroll
    for (int r = 0; r < kPR; ++r) {
      const int i = r * kPT + tid;
      if (i < m) {
        const uint32_t q = part_id<U>(u[r], a.shift, mask);
        pos[r] = (q << 16) | atomicAdd(&s_cnt[q], 1u);      // rank < 4096 fits 16 bits
      }
    }
    __syncthreads();
    // B: exclusive scan of the per-partition counts; claim global space per partition
    long long gclaim[kPer];
    uint32_t gcnt[kPer];
#pragma unroll
    for (int k = 0; k < kPer; ++k) { gclaim[k] = 0; gcnt[k] = 0; }
    {
      uint32_t c[kPer], sum = 0;
#pragma unroll
      for (int k = 0; k < kPer; ++k) { const int p = tid * kPer + k; c[k] = p < fan ? s_cnt[p] : 0u; sum += c[k]; }
      uint32_t inc = sum;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
      if (lane == 31) s_warp[warp] = inc;
      __syncthreads();
      if (warp == 0) {
        uint32_t w = lane < kPT / 32 ? s_warp[lane] : 0u;
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += y; }
        if (lane < kPT / 32) s_warp[lane] = winc - w;
      }
      __syncthreads();
      uint32_t run = s_warp[warp] + inc - sum;
      // the claims' round trips to L2 overlap the staging below: their results are first needed in D
#pragma unroll
      for (int k = 0; k < kPer; ++k) {
        const int p = tid * kPer + k;
        if (p < fan) {
          s_loff[p] = run;
          gclaim[k] = c[k] ? (long long)atomicAdd(&cursor[p], (unsigned long long)c[k]) - (long long)run : 0ll;
          gcnt[k] = c[k];
          s_cnt[p] = 0;
          run += c[k];
        }
      }
    }
    __syncthreads();
    // C: stage keys (and the first value column) in partition order
#pragma unroll
    for (int r = 0; r < kPR; ++r) {
      const int i = r * kPT + tid;
      if (i < m) {
        const uint32_t q = pos[r] >> 16;
        pos[r] = s_loff[q] + (pos[r] & 0xFFFFu);
        s_key[pos[r]] = (UO)u[r];
        s_pid[pos[r]] = (uint16_t)q;
        if (a.n_vals > 0) s_val[pos[r]] = v0[r];
      }
    }
#pragma unroll
    for (int k = 0; k < kPer; ++k) { const int p = tid * kPer + k; if (p < fan && gcnt[k]) s_delta[p] = gclaim[k]; }
    __syncthreads();
    // D: write runs
#pragma unroll
    for (int r = 0; r < kPR; ++r) {
      const int j = r * kPT + tid;
      if (j < m) {
        const long long dst = s_delta[s_pid[j]] + j;
        out_keys[dst] = s_key[j];
        if (a.n_vals > 0) static_cast<uint64_t*>(a.out_vals[0])[dst] = s_val[j];
      }
    }
    // remaining value columns, one staged at a time
    for (int c = 1; c < a.n_vals; ++c) {
      __syncthreads();
#pragma unroll
      for (int r = 0; r < kPR; ++r) {
        const int i = r * kPT + tid;
        if (i < m) s_val[pos[r]] = ldg_stream_u64(static_cast<const uint64_t*>(a.vals[c]) + base + i);
      }
      __syncthreads();
#pragma unroll
      for (int r = 0; r < kPR; ++r) {
        const int j = r * kPT + tid;
        if (j < m) static_cast<uint64_t*>(a.out_vals[c])[s_delta[s_pid[j]] + j] = s_val[j];
      }
    }
    __syncthreads();
  }
}

template <int KK, class UO, int RPT>
int launch_scatter(const LevelArgs& a, const uint8_t* vw, int threads, int stages, int gx, int segments, cudaStream_t s) {
  ScatterArgs A{};
  A.lv = a;
  A.tile = (uint32_t)(RPT * threads);
  A.sm = scatter_smem_layout(a.key, KK, vw, a.n_vals, A.tile, stages, sizeof(UO));
  auto kern = part_scatter_kernel<KK, UO, RPT>;
  EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)A.sm.total));
  kern<<<dim3(gx, segments), threads, A.sm.total, s>>>(A);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

template <int KK>
int run_level(LevelArgs a, const uint8_t* vw, int segments, unsigned long long* off, int sm_count, size_t smem_optin, cudaStream_t s, const uint32_t* pre_hist = nullptr) {
  using UO = typename SrcKey<KK>::U;
  // tile shape: the largest of (1024 x 6), (1024 x 4), (512 x 6), (512 x 4), (256 x 4) rows whose ring
  // (two stages) + staging buffer fit one CTA's shared memory
  static const int cand[][2] = {{1024, 6}, {1024, 4}, {512, 6}, {512, 4}, {256, 4}};
  int threads = 256, rpt = 4;
  const int stages = 2;
  {
    const char* et = std::getenv("EIGER_SCATTER_T"); const char* er = std::getenv("EIGER_SCATTER_RPT");
    bool found = false;
    for (auto& c : cand) {
      if (et && std::atoi(et) != c[0]) continue;
      if (er && std::atoi(er) != c[1]) continue;
      if (c[0] < a.fan) continue;                            // one counter per thread in the scan
      const ScatterSmem m = scatter_smem_layout(a.key, KK, vw, a.n_vals, (uint32_t)(c[0] * c[1]), stages, sizeof(UO));
      if ((size_t)m.total + 20 * 1024 <= smem_optin) { threads = c[0]; rpt = c[1]; found = true; break; }
    }
    if (!found) { threads = std::max(256, a.fan); rpt = 4; }
  }
  const int64_t tile = (int64_t)threads * rpt;
  const int64_t avg_rows = a.n / segments + 1;
  const int64_t tiles = std::max<int64_t>(1, (avg_rows + tile - 1) / tile);
  const int64_t want = segments == 1 ? (int64_t)sm_count : std::max<int64_t>(1, ((int64_t)sm_count * 2 + segments - 1) / segments);
  const int gx = (int)std::min<int64_t>(tiles, want);
  if (pre_hist && segments == 1 && a.fan <= kPreFan) {
    part_fold_kernel<<<(a.fan + 255) / 256, 256, 0, s>>>(pre_hist, kPreFan, a.hist, a.fan);
  } else {
    EIGER_CUDA(cudaMemsetAsync(a.hist, 0, sizeof(uint32_t) * (size_t)segments * a.fan, s));
    const int64_t htiles = std::max<int64_t>(1, (avg_rows + kTile - 1) / kTile);
    const int64_t hwant = segments == 1 ? (int64_t)sm_count * 8 : std::max<int64_t>(1, ((int64_t)sm_count * 8 + segments - 1) / segments);
    part_hist_kernel<KK><<<dim3((int)std::min<int64_t>(htiles, hwant), segments), kPT, 0, s>>>(a);
  }
  count_launch();
  part_scan_kernel<<<1, 1024, 0, s>>>(a.hist, off, a.cursor, segments * a.fan);
  count_launch();
  bool all8 = true;
  for (int c = 0; c < a.n_vals; ++c) all8 = all8 && (vw[c] == 0 || vw[c] == 8);
  const char* er = std::getenv("EIGER_SCATTER_RING");
  // measured on one box (C5 2^16 / 2^20 / C4, ms per partition pass): per-thread loads 1.85 / 2.01 / 9.22, ring 1.89 / 1.95 / 10.67:
  // the ring version is kept for 4-byte value columns and as the EIGER_SCATTER_RING=1 experiment
  if (all8 && !(er && std::atoi(er) == 1)) {
    const int64_t otiles = std::max<int64_t>(1, (avg_rows + kTile - 1) / kTile);
    const int64_t owant = segments == 1 ? (int64_t)sm_count * 8 : std::max<int64_t>(1, ((int64_t)sm_count * 8 + segments - 1) / segments);
    const int ogx = (int)std::min<int64_t>(otiles, owant);
    constexpr size_t osmem = (sizeof(uint64_t) + sizeof(UO) + sizeof(uint16_t)) * kTile + (8 + 4 + 4) * kMaxFan;
    auto kern = part_scatter_ldg_kernel<KK, UO>;
    EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)osmem));
    kern<<<dim3(ogx, segments), kPT, osmem, s>>>(a);
    count_launch();
    EIGER_CUDA(cudaGetLastError());
    return EIGER_OK;
  }
  if (rpt == 6) return launch_scatter<KK, UO, 6>(a, vw, threads, stages, gx, segments, s);
  return launch_scatter<KK, UO, 4>(a, vw, threads, stages, gx, segments, s);
}

template <int KK, int KK2>
int run_levels(PartitionLaunch& L, int sm_count, size_t smem_optin, cudaStream_t s) {
  using U = typename SrcKey<KK>::U;
  const int W = 8 * (int)sizeof(U);
  LevelArgs a{};
  a.key = L.key; a.n = L.n; a.n_vals = L.plan.n_vals;
  for (int c = 0; c < kMaxVals; ++c) { a.vals[c] = L.plan.vals[c]; a.out_vals[c] = L.valsA[c]; }
  a.out_keys = L.keysA; a.seg_off = nullptr; a.hist = L.hist; a.cursor = L.cur1;
  a.fan = 1 << L.bits1; a.shift = W - L.bits1;
  int rc = run_level<KK>(a, L.plan.vw, 1, L.off1, sm_count, smem_optin, s, L.pre_hist);
  if (rc) return rc;
  L.out_keys = L.keysA; L.out_vals = L.valsA; L.out_off = L.off1; L.n_parts = 1 << L.bits1;
  if (L.bits2 > 0) {
    LevelArgs b{};
    b.key = L.key; b.key.ptr[0] = L.keysA; b.key.ncols = 1;      // one pre-fused column from here on
    for (int k = 1; k < kMaxKeyCols; ++k) b.key.ptr[k] = nullptr;
    b.n = L.n; b.n_vals = L.plan.n_vals;
    for (int c = 0; c < kMaxVals; ++c) { b.vals[c] = L.valsA[c]; b.out_vals[c] = L.valsB[c]; }
    b.out_keys = L.keysB; b.seg_off = L.off1; b.hist = L.hist; b.cursor = L.cur2;
    b.fan = 1 << L.bits2; b.shift = W - L.bits1 - L.bits2;
    rc = run_level<KK2>(b, L.plan.vw, 1 << L.bits1, L.off2, sm_count, smem_optin, s);
    if (rc) return rc;
    L.out_keys = L.keysB; L.out_vals = L.valsB; L.out_off = L.off2; L.n_parts = 1 << (L.bits1 + L.bits2);
  }
  part_items_kernel<<<1, 1024, 0, s>>>(L.out_off, L.item_off, L.item_part, L.n_parts, (unsigned long long)L.chunk_rows);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

}  // namespace

int partition_max_bits_per_level() { int b = 0; while ((1 << (b + 1)) <= kMaxFan) ++b; return b; }

int launch_partition(PartitionLaunch& L, int sm_count, size_t smem_optin, cudaStream_t s) {
  const int mb = partition_max_bits_per_level();
  if (L.bits1 < 1 || L.bits1 > mb || L.bits2 < 0 || L.bits2 > mb) return EIGER_ERR_ARG;
  switch (L.key_kind) {
    case KK_I32: return run_levels<KK_I32, KK_U32PRE>(L, sm_count, smem_optin, s);
    case KK_I64: return run_levels<KK_I64, KK_U64PRE>(L, sm_count, smem_optin, s);
    case KK_GEN: case KK_I8I8: return run_levels<KK_GEN, KK_U64PRE>(L, sm_count, smem_optin, s);
    case KK_GEN32: return run_levels<KK_GEN32, KK_U32PRE>(L, sm_count, smem_optin, s);
    case KK_U64PRE: return run_levels<KK_U64PRE, KK_U64PRE>(L, sm_count, smem_optin, s);   // a spill buffer: keys already rebased and fused
    default: return EIGER_ERR_ARG;
  }
}

}  // namespace eiger
