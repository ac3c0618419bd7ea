// EIGER_SORT: sort-based group-by, the third algorithm of the paper (§3.3 "sort-based,
// hash-based, and partition-hash-based"; SORT/TR, stable across group
// cardinalities, the winner between 2^14 and 2^20 groups on A100 / GH200).  Payload columns travel
// with the keys (the paper's GFTR).
//
//   1. LSD radix sort of the rows on the rebased, fused key u (rows.cuh), 8 bits per pass and only
//      the ceil(log2 R) bits the key range R needs (the range comes from the statistics pass:
//      a dense 2^16-key column sorts in two passes, a full-range int32 column in four).  One pass =
//      per-tile digit histograms -> column-wise scan -> STABLE scatter: the rows of a tile arrive
//      through the bulk-copy ring (ring.cuh), every warp ranks a contiguous block of the tile with
//      match.any (equal digits keep their order), and the tile leaves the SM as runs of consecutive
//      rows per digit.  Pass 0 reads the caller's columns and fuses the key on the fly.
//   2. Segmented reduce over the sorted rows: group index = number of run heads before the row
//      (per-tile head counts, scanned); inside a warp the rows of a run are combined with shuffles,
//      run heads merge into a per-tile shared-memory array, tiles merge into the output columns.
//      The groups come out in ascending key order.
#include <algorithm>
#include <cstdlib>

#include "scatter.cuh"

namespace eiger {
namespace {

constexpr int kDigitBits = 8, kDigits = 1 << kDigitBits;

struct SortPassArgs {
  KeyDesc key;                       // source keys (pass 0: the caller's columns; later: one pre-fused column)
  const void* vals[kMaxVals];
  void* out_vals[kMaxVals];
  void* out_keys;
  int64_t n;
  int32_t n_vals, shift;
  uint32_t digit_mask;
  uint32_t* tile_hist;               // [n_tiles][kDigits]: after the scan, rows of this digit in earlier tiles
  const unsigned long long* digit_base;   // [kDigits]: rows with a smaller digit
  ScatterSmem sm;
  uint32_t tile, wcnt_off;           // wcnt: [warps][kDigits] uint16 in dynamic shared memory
  int32_t padded;                    // the source is the library's own padded copy (passes after the first)
};

template <class U> __device__ __forceinline__ uint32_t digit_of(U u, int shift, uint32_t mask) { return (uint32_t)(u >> shift) & mask; }

// per-tile digit histogram (tile = the scatter kernel's tile)
template <int KK>
__global__ void __launch_bounds__(256) sort_hist_kernel(const __grid_constant__ SortPassArgs a) {
  using U = typename KeyTraits<KK>::U;
  __shared__ uint32_t h[kDigits];
  const int tid = threadIdx.x;
  const int64_t n_tiles = (a.n + a.tile - 1) / a.tile;
  for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    h[tid] = 0;
    __syncthreads();
    const int64_t r0 = t * a.tile, r1 = r0 + a.tile < a.n ? r0 + a.tile : a.n;
    int64_t i = r0 + tid;
    for (; i + 3 * 256 < r1; i += 4 * 256) {
      U u[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) u[k] = load_u<KK>(a.key, i + k * 256);
#pragma unroll
      for (int k = 0; k < 4; ++k) atomicAdd(&h[digit_of<U>(u[k], a.shift, a.digit_mask)], 1u);
    }
    for (; i < r1; i += 256) atomicAdd(&h[digit_of<U>(load_u<KK>(a.key, i), a.shift, a.digit_mask)], 1u);
    __syncthreads();
    a.tile_hist[t * kDigits + tid] = h[tid];
    __syncthreads();
  }
}

// column d of the [n_tiles][kDigits] matrix -> exclusive prefix over the tiles; total[d]
__global__ void __launch_bounds__(1024) sort_colscan_kernel(uint32_t* __restrict__ m, int64_t n_tiles, unsigned long long* __restrict__ total) {
  __shared__ unsigned long long s_part[1024];
  const int d = blockIdx.x, tid = threadIdx.x;
  const int64_t per = (n_tiles + 1023) / 1024;
  const int64_t b = tid * per, e = b + per < n_tiles ? b + per : n_tiles;
  unsigned long long local = 0;
  for (int64_t t = b; t < e; ++t) local += m[t * kDigits + d];
  s_part[tid] = local;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const unsigned long long v = tid >= o ? s_part[tid - o] : 0ull;
    __syncthreads();
    s_part[tid] += v;
    __syncthreads();
  }
  unsigned long long run = s_part[tid] - local;
  for (int64_t t = b; t < e; ++t) { const uint32_t c = m[t * kDigits + d]; m[t * kDigits + d] = (uint32_t)run; run += c; }   // n < 2^32
  if (tid == 1023) total[d] = s_part[1023];
}
__global__ void sort_digit_base_kernel(const unsigned long long* __restrict__ total, unsigned long long* __restrict__ base) {
  if (threadIdx.x == 0) { unsigned long long run = 0; for (int d = 0; d < kDigits; ++d) { base[d] = run; run += total[d]; } }
}

// STABLE scatter of one radix pass.  Warp w ranks rows [w * 32 * RPT, (w + 1) * 32 * RPT) of the tile.
template <int KK, class UO, int RPT>
__global__ void __launch_bounds__(1024, 1)
sort_scatter_kernel(const __grid_constant__ SortPassArgs a) {
  using U = typename KeyTraits<KK>::U;
  const ScatterSmem& sm = a.sm;
  extern __shared__ __align__(128) unsigned char dsm[];      // [ring stages][s_out][s_pid][wcnt]
  __shared__ __align__(8) uint64_t s_full[kMaxStages], s_empty[kMaxStages];
  __shared__ long long s_delta[kDigits];
  __shared__ uint32_t s_loff[kDigits], s_tot[kDigits];
  __shared__ uint32_t s_warp[32];
  unsigned char* s_out = dsm + sm.out_off;
  uint8_t* s_pid = dsm + sm.pid_off;
  uint16_t* wcnt = reinterpret_cast<uint16_t*>(dsm + a.wcnt_off);
  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5, nw = T >> 5;
  const uint32_t tile = a.tile;
  UO* out_keys = static_cast<UO*>(a.out_keys);
  if (tid == 0) {
    for (int s = 0; s < sm.stages; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], (uint32_t)nw); }
    mbar_fence_init();
  }
  __syncthreads();
  const int64_t n_tiles = (a.n + tile - 1) / tile;
  const bool padded = a.padded != 0;                         // later passes read the library's padded copy
  const int64_t n_bulk = padded ? n_tiles : a.n / tile;
  const int64_t mine = n_bulk > blockIdx.x ? (n_bulk - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const uint64_t policy = policy_evict_first();
  uint32_t g_issued = 0;
  auto issue = [&](uint32_t g) {
    const int64_t row0 = ((int64_t)blockIdx.x + (int64_t)g * gridDim.x) * tile;
    int64_t rows = ((a.n - row0) + 31) & ~(int64_t)31;
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
      bulk_g2s_hint(st + sm.voff[c], static_cast<const unsigned char*>(a.vals[c]) + row0 * sm.vw[c], (uint32_t)rows * sm.vw[c], &s_full[s], policy);
  };
  if (tid == 0) for (; g_issued < (uint32_t)sm.stages && (int64_t)g_issued < mine; ++g_issued) issue(g_issued);

  auto process = [&](const unsigned char* st, int64_t t, int ring_stage) {
    const int64_t row0 = t * tile;
    const uint32_t hi = (uint32_t)(a.n - row0 < (int64_t)tile ? a.n - row0 : (int64_t)tile);
    for (int i = tid; i < nw * kDigits; i += T) wcnt[i] = 0;
    __syncthreads();
    // A: stable ranks inside the warp's block of the tile
    U u[RPT];
    uint32_t pos[RPT];
    const uint32_t wbase = (uint32_t)warp * 32u * RPT;
    uint16_t* myc = wcnt + warp * kDigits;
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
      const uint32_t i = wbase + (uint32_t)r * 32u + (uint32_t)lane;
      const bool valid = i < hi;
      u[r] = valid ? stage_key<KK>(a.key, sm, st, i) : (U)0;
      const uint32_t d = valid ? digit_of<U>(u[r], a.shift, a.digit_mask) : (uint32_t)kDigits;
      const uint32_t peers = __match_any_sync(0xffffffffu, d);
      const int leader = __ffs((int)peers) - 1;
      uint32_t old = 0;
      if (valid && lane == leader) { old = myc[d]; myc[d] = (uint16_t)(old + __popc(peers)); }
      old = __shfl_sync(0xffffffffu, old, leader);
      pos[r] = (d << 16) | (old + __popc(peers & ((1u << lane) - 1u)));
      __syncwarp();
    }
    __syncthreads();
    // B: per digit, exclusive prefix over the warps (rows of warp w precede those of warp w + 1)
    if (tid < kDigits) {
      uint32_t run = 0;
      for (int w = 0; w < nw; ++w) { const uint32_t x = wcnt[w * kDigits + tid]; wcnt[w * kDigits + tid] = (uint16_t)run; run += x; }
      s_tot[tid] = run;
    }
    __syncthreads();
    {
      const uint32_t c = tid < kDigits ? s_tot[tid] : 0u;
      uint32_t inc = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
      if (lane == 31) s_warp[warp] = inc;
      __syncthreads();
      if (warp == 0) {
        const uint32_t w = lane < nw ? s_warp[lane] : 0u;
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += y; }
        s_warp[lane] = winc - w;
      }
      __syncthreads();
      if (tid < kDigits) {
        const uint32_t run = s_warp[warp] + inc - c;
        s_loff[tid] = run;
        s_delta[tid] = (long long)(a.digit_base[tid] + a.tile_hist[t * kDigits + tid]) - (long long)run;
      }
    }
    __syncthreads();
    // C/D: stage each column in digit order (stable), write runs
    UO* ko = reinterpret_cast<UO*>(s_out);
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
      const uint32_t d = pos[r] >> 16;
      if (d < (uint32_t)kDigits) {
        pos[r] = s_loff[d] + myc[d] + (pos[r] & 0xFFFFu);
        ko[pos[r]] = (UO)u[r];
        s_pid[pos[r]] = (uint8_t)d;
      } else {
        pos[r] = 0xFFFFFFFFu;
      }
    }
    __syncthreads();
    for (uint32_t j = tid; j < hi; j += T) out_keys[s_delta[s_pid[j]] + j] = ko[j];
    for (int c = 0; c < a.n_vals; ++c) {
      __syncthreads();
      const unsigned char* col = st + sm.voff[c];
      if (sm.vw[c] == 8) {
        uint64_t* vo = reinterpret_cast<uint64_t*>(s_out);
#pragma unroll
        for (int r = 0; r < RPT; ++r) if (pos[r] != 0xFFFFFFFFu) vo[pos[r]] = *reinterpret_cast<const uint64_t*>(col + 8 * (size_t)(wbase + r * 32 + lane));
        if (c == a.n_vals - 1 && ring_stage >= 0) { __syncwarp(); if (lane == 0) mbar_arrive(&s_empty[ring_stage]); }
        __syncthreads();
        uint64_t* dst = static_cast<uint64_t*>(a.out_vals[c]);
        for (uint32_t j = tid; j < hi; j += T) dst[s_delta[s_pid[j]] + j] = vo[j];
      } else {
        uint32_t* vo = reinterpret_cast<uint32_t*>(s_out);
#pragma unroll
        for (int r = 0; r < RPT; ++r) if (pos[r] != 0xFFFFFFFFu) vo[pos[r]] = *reinterpret_cast<const uint32_t*>(col + 4 * (size_t)(wbase + r * 32 + lane));
        if (c == a.n_vals - 1 && ring_stage >= 0) { __syncwarp(); if (lane == 0) mbar_arrive(&s_empty[ring_stage]); }
        __syncthreads();
        uint32_t* dst = static_cast<uint32_t*>(a.out_vals[c]);
        for (uint32_t j = tid; j < hi; j += T) dst[s_delta[s_pid[j]] + j] = vo[j];
      }
    }
    if (a.n_vals == 0 && ring_stage >= 0) { __syncwarp(); if (lane == 0) mbar_arrive(&s_empty[ring_stage]); }
    __syncthreads();
  };

  for (int64_t k = 0; k < mine; ++k) {
    const uint32_t g = (uint32_t)k, s = g % (uint32_t)sm.stages;
    mbar_wait(&s_full[s], (g / (uint32_t)sm.stages) & 1u);
    process(dsm + (size_t)s * sm.stage_bytes, (int64_t)blockIdx.x + k * gridDim.x, (int)s);
    if (tid == 0 && (int64_t)g_issued < mine) { issue(g_issued); ++g_issued; }
  }
  if (!padded && n_tiles > n_bulk && (int)(n_bulk % gridDim.x) == (int)blockIdx.x) {
    // the ragged last tile of the caller's columns: loaded by the threads into stage 0
    const int64_t row0 = n_bulk * tile;
    const uint32_t rows = (uint32_t)(a.n - row0);
    unsigned char* st = dsm;
    for (int c = 0; c < sm.n_src; ++c) {
      const unsigned char* src = static_cast<const unsigned char*>(a.key.ptr[c]) + row0 * sm.kw[c];
      for (uint32_t o = tid; o < rows * sm.kw[c]; o += T) st[sm.koff[c] + o] = src[o];
    }
    for (int c = 0; c < a.n_vals; ++c) {
      const uint32_t* src = reinterpret_cast<const uint32_t*>(static_cast<const unsigned char*>(a.vals[c]) + row0 * sm.vw[c]);
      uint32_t* d = reinterpret_cast<uint32_t*>(st + sm.voff[c]);
      for (uint32_t o = tid; o < rows * (sm.vw[c] / 4u); o += T) d[o] = src[o];
    }
    __syncthreads();
    process(st, n_bulk, -1);
  }
}

// ---- segmented reduce over the sorted rows -------------------------------------------------------
constexpr int kRedThreads = 512, kRedRows = 4;              // tile = 2048 sorted rows
constexpr int kRedTile = kRedThreads * kRedRows;

struct ReduceArgs {
  KeyDesc key;                       // for un-fusing the group keys
  AggPlan plan;                      // vals[] = the sorted value columns
  const void* keys;                  // sorted rebased keys (UO)
  int64_t n;
  uint32_t* tile_heads;              // [n_tiles + 1]: run heads per tile -> exclusive scan
  void* out_keys[kMaxKeyCols]; uint64_t* out_aggs[kMaxAggs]; int32_t n_out; int64_t out_capacity;
  CallDev* call;
};

template <class UO>
__global__ void __launch_bounds__(kRedThreads) sort_heads_kernel(const __grid_constant__ ReduceArgs a) {
  __shared__ uint32_t s_w[kRedThreads / 32];
  const UO* k = static_cast<const UO*>(a.keys);
  const int tid = threadIdx.x;
  const int64_t n_tiles = (a.n + kRedTile - 1) / kRedTile;
  for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    uint32_t c = 0;
#pragma unroll
    for (int r = 0; r < kRedRows; ++r) {
      const int64_t i = t * kRedTile + r * kRedThreads + tid;
      if (i < a.n) c += (i == 0 || k[i] != k[i - 1]) ? 1u : 0u;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((tid & 31) == 0) s_w[tid >> 5] = c;
    __syncthreads();
    if (tid == 0) { uint32_t tot = 0; for (int w = 0; w < kRedThreads / 32; ++w) tot += s_w[w]; a.tile_heads[t] = tot; }
    __syncthreads();
  }
}
// exclusive scan of up to 2^21 tile counts (single CTA); the total goes to call->n_groups
__global__ void __launch_bounds__(1024) sort_heads_scan_kernel(uint32_t* __restrict__ h, int64_t count, CallDev* call) {
  __shared__ unsigned long long s_part[1024];
  const int tid = threadIdx.x;
  const int64_t per = (count + 1023) / 1024;
  const int64_t b = tid * per, e = b + per < count ? b + per : count;
  unsigned long long local = 0;
  for (int64_t p = b; p < e; ++p) local += h[p];
  s_part[tid] = local;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const unsigned long long v = tid >= o ? s_part[tid - o] : 0ull;
    __syncthreads();
    s_part[tid] += v;
    __syncthreads();
  }
  unsigned long long run = s_part[tid] - local;
  for (int64_t p = b; p < e; ++p) { const uint32_t c = h[p]; h[p] = (uint32_t)run; run += c; }
  if (tid == 1023) call->n_groups = s_part[1023];
}
__global__ void sort_out_init_kernel(ReduceArgs a, int64_t g) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < g; i += stride)
    for (int j = 0; j < a.n_out; ++j) a.out_aggs[j][i] = acc_identity(a.plan.op[j]);
}

template <class UO, int SIG>
__global__ void __launch_bounds__(kRedThreads) sort_reduce_kernel(const __grid_constant__ ReduceArgs a) {
  using S = Sig<SIG>;
  constexpr int NV = S::kVals, NA = S::kAcc;
  // per-tile accumulators: one cell per (local group, accumulator); a tile has at most kRedTile groups
  extern __shared__ __align__(16) uint64_t s_acc[];          // [n_acc][kRedTile]
  __shared__ uint32_t s_wheads[kRedThreads / 32];
  const int n_acc = S::kStatic ? NA : a.plan.n_acc, n_vals = S::kStatic ? NV : a.plan.n_vals;
  const UO* k = static_cast<const UO*>(a.keys);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t n_tiles = (a.n + kRedTile - 1) / kRedTile;
  for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    const int64_t row0 = t * kRedTile;
    const uint32_t m = (uint32_t)(a.n - row0 < kRedTile ? a.n - row0 : kRedTile);
    for (int i = tid; i < n_acc * kRedTile; i += kRedThreads) s_acc[i] = acc_identity(sig_op<SIG>(a.plan, i / kRedTile));
    // warp w owns rows [w * 32 * kRedRows, ...), round r = 32 consecutive rows: heads, local group ids
    uint32_t heads[kRedRows];
    uint32_t wcount = 0;
    const uint32_t wbase = (uint32_t)warp * 32u * kRedRows;
    UO key[kRedRows];
    bool valid[kRedRows], head[kRedRows];
#pragma unroll
    for (int r = 0; r < kRedRows; ++r) {
      const uint32_t i = wbase + r * 32u + lane;
      valid[r] = i < m;
      key[r] = valid[r] ? k[row0 + i] : (UO)0;
      const int64_t gi = row0 + i;
      head[r] = valid[r] && (gi == 0 || key[r] != k[gi - 1]);
      heads[r] = __ballot_sync(0xffffffffu, head[r]);
      wcount += __popc(heads[r]);
    }
    if (lane == 0) s_wheads[warp] = wcount;
    __syncthreads();
    uint32_t lg = 0;                                         // heads of the tile before this warp's block
    for (int w = 0; w < warp; ++w) lg += s_wheads[w];
    const unsigned long long gbase = a.tile_heads[t];        // groups that start before this tile
    // a row's local group = heads up to and including it, minus one; a tile whose first row is not a
    // head continues the previous tile's last group: local group "-1" = global group gbase - 1
    for (int r = 0; r < kRedRows; ++r) {
      const uint32_t i = wbase + r * 32u + lane;
      const uint32_t before = lg + __popc(heads[r] & ((2u << lane) - 1u));     // heads at rows <= this one
      lg += __popc(heads[r]);
      // segmented warp reduction: run of a row = up to the next head (exclusive) inside these 32 rows
      uint64_t part[NA];
#pragma unroll
      for (int j = 0; j < NA; ++j) {
        if (!S::kStatic && j >= n_acc) { part[j] = 0; continue; }
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        const int c = sig_col<SIG>(a.plan, j);
        uint64_t raw = 0;
        if (valid[r] && op != EIGER_COUNT) raw = global_val(a.plan, c, sig_vw<SIG>(a.plan, c), row0 + i);
        part[j] = valid[r] ? row_partial(op, f, raw) : acc_identity(op);
      }
      // end of this lane's run: the next head after it, or 32
      const uint32_t later = heads[r] & ~((2u << lane) - 1u);
      const int run_end = later ? __ffs((int)later) - 1 : 32;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
        for (int j = 0; j < NA; ++j) {
          if (!S::kStatic && j >= n_acc) continue;
          const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
          const uint64_t other = __shfl_down_sync(0xffffffffu, part[j], o);
          if (lane + o < run_end) part[j] = combine(op, f, part[j], other);
        }
      }
      // the first lane of each run inside these 32 rows holds the run's total: a head, or lane 0
      const bool first = valid[r] && (head[r] || lane == 0);
      if (first) {
        const uint32_t g_local = before;                    // 0 = continues the previous tile's group
        if (g_local == 0) {
#pragma unroll
          for (int j = 0; j < NA; ++j) {
            if (!S::kStatic && j >= n_acc) continue;
            if (j < a.n_out && gbase > 0 && (int64_t)(gbase - 1) < a.out_capacity)
              atomic_merge(a.out_aggs[j] + (gbase - 1), sig_op<SIG>(a.plan, j), sig_f64<SIG>(a.plan, j), part[j]);
          }
        } else {
#pragma unroll
          for (int j = 0; j < NA; ++j) {
            if (!S::kStatic && j >= n_acc) continue;
            atomic_merge(s_acc + (size_t)j * kRedTile + (g_local - 1), sig_op<SIG>(a.plan, j), sig_f64<SIG>(a.plan, j), part[j]);
          }
        }
        if (head[r]) {                                      // the group's key: written once, by its head row
          const unsigned long long g = gbase + g_local - 1;
          if ((int64_t)g < a.out_capacity) store_group_key(a.key, a.out_keys, (uint64_t)key[r], g);
        }
      }
    }
    __syncthreads();
    // flush the tile's groups: the last one may continue in the next tile -> atomic; the others are complete
    uint32_t tile_groups = 0;
    for (int w = 0; w < kRedThreads / 32; ++w) tile_groups += s_wheads[w];
    for (uint32_t g = tid; g < tile_groups; g += kRedThreads) {
      const unsigned long long gg = gbase + g;
      if ((int64_t)gg >= a.out_capacity) continue;
      for (int j = 0; j < a.n_out; ++j) {
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        atomic_merge(a.out_aggs[j] + gg, op, f, s_acc[(size_t)j * kRedTile + g]);
      }
    }
    __syncthreads();
  }
}
// partial -> final form (fp64 MIN / MAX are kept as order-preserving integers while merging)
__global__ void sort_finalize_kernel(ReduceArgs a, int64_t g) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < g; i += stride)
    for (int j = 0; j < a.n_out; ++j)
      if (a.plan.f64[j] && (a.plan.op[j] == EIGER_MIN || a.plan.op[j] == EIGER_MAX)) a.out_aggs[j][i] = acc_finalize(a.plan.op[j], true, a.out_aggs[j][i]);
}

template <int KK, class UO>
int run_pass(SortPassArgs a, int threads, int rpt, int sm_count, cudaStream_t s) {
  const int64_t n_tiles = (a.n + a.tile - 1) / a.tile;
  sort_hist_kernel<KK><<<(int)std::min<int64_t>(n_tiles, (int64_t)sm_count * 8), 256, 0, s>>>(a);
  count_launch();
  unsigned long long* total = const_cast<unsigned long long*>(a.digit_base) + kDigits;
  sort_colscan_kernel<<<kDigits, 1024, 0, s>>>(a.tile_hist, n_tiles, total);
  sort_digit_base_kernel<<<1, 32, 0, s>>>(total, const_cast<unsigned long long*>(a.digit_base));
  count_launch(2);
  const size_t smem = (size_t)a.wcnt_off + (size_t)(threads / 32) * kDigits * 2;
  const int gx = (int)std::min<int64_t>(n_tiles, sm_count);
  if (rpt == 6) {
    auto kern = sort_scatter_kernel<KK, UO, 6>;
    EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<gx, threads, smem, s>>>(a);
  } else {
    auto kern = sort_scatter_kernel<KK, UO, 4>;
    EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<gx, threads, smem, s>>>(a);
  }
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

// tile shape of a pass: as in partition.cu, the largest candidate whose shared memory fits
template <class UO>
void pick_tile(const KeyDesc& key, int kk, const AggPlan& plan, size_t smem_optin, int* threads, int* rpt, ScatterSmem* m, uint32_t* wcnt_off) {
  static const int cand[][2] = {{1024, 6}, {1024, 4}, {512, 6}, {512, 4}, {256, 4}};
  for (auto& c : cand) {
    const ScatterSmem l = scatter_smem_layout(key, kk, plan.vw, plan.n_vals, (uint32_t)(c[0] * c[1]), 2, sizeof(UO));
    const size_t total = (size_t)l.total + (size_t)(c[0] / 32) * kDigits * 2 + 8 * 1024;
    if (total <= smem_optin || (c[0] == 256 && c[1] == 4)) { *threads = c[0]; *rpt = c[1]; *m = l; *wcnt_off = l.total; return; }
  }
}

template <class UO, int KK0, int KKN>
int sort_groupby(SortLaunch& L, int sm_count, size_t smem_optin, cudaStream_t s) {
  const int passes = (L.bits + kDigitBits - 1) / kDigitBits;
  const void* cur_keys = nullptr;
  void* const* cur_vals = nullptr;
  for (int p = 0; p < std::max(passes, 1); ++p) {
    SortPassArgs a{};
    const bool first = p == 0;
    a.key = L.key;
    if (!first) { a.key.ptr[0] = cur_keys; a.key.ncols = 1; for (int k = 1; k < kMaxKeyCols; ++k) a.key.ptr[k] = cur_keys; }
    void* dk = (p & 1) ? L.keysB : L.keysA;
    void* const* dv = (p & 1) ? L.valsB : L.valsA;
    for (int c = 0; c < kMaxVals; ++c) { a.vals[c] = first ? L.plan.vals[c] : cur_vals[c]; a.out_vals[c] = dv[c]; }
    a.out_keys = dk; a.n = L.n; a.n_vals = L.plan.n_vals;
    a.shift = p * kDigitBits;
    const int left = L.bits - p * kDigitBits;
    a.digit_mask = left >= kDigitBits ? (uint32_t)kDigits - 1u : (left > 0 ? (1u << left) - 1u : 0u);
    a.tile_hist = L.tile_hist; a.digit_base = L.digit_base; a.padded = first ? 0 : 1;
    int threads, rpt;
    const int kk = first ? KK0 : KKN;
    pick_tile<UO>(a.key, kk, L.plan, smem_optin, &threads, &rpt, &a.sm, &a.wcnt_off);
    a.tile = (uint32_t)(threads * rpt);
    const int rc = first ? run_pass<KK0, UO>(a, threads, rpt, sm_count, s) : run_pass<KKN, UO>(a, threads, rpt, sm_count, s);
    if (rc) return rc;
    cur_keys = dk; cur_vals = dv;
  }
  // segmented reduce
  ReduceArgs r{};
  r.key = L.key; r.plan = L.plan;
  for (int c = 0; c < kMaxVals; ++c) r.plan.vals[c] = cur_vals[c];
  r.keys = cur_keys; r.n = L.n; r.tile_heads = L.tile_hist;
  for (int k = 0; k < kMaxKeyCols; ++k) r.out_keys[k] = L.out_keys[k];
  for (int j = 0; j < kMaxAggs; ++j) r.out_aggs[j] = static_cast<uint64_t*>(L.out_aggs[j]);
  r.n_out = L.n_out_aggs; r.out_capacity = L.out_capacity; r.call = L.call;
  const int64_t n_tiles = (L.n + kRedTile - 1) / kRedTile;
  const int grid = (int)std::min<int64_t>(n_tiles, (int64_t)sm_count * 4);
  sort_heads_kernel<UO><<<grid, kRedThreads, 0, s>>>(r);
  sort_heads_scan_kernel<<<1, 1024, 0, s>>>(L.tile_hist, n_tiles, L.call);
  count_launch(2);
  // the output cells start as identities: tiles merge into them (a group may span tiles)
  const int64_t gcap = std::min<int64_t>(L.out_capacity, L.n);
  sort_out_init_kernel<<<(int)std::min<int64_t>((gcap + 255) / 256 + 1, (int64_t)sm_count * 8), 256, 0, s>>>(r, gcap);
  count_launch();
  auto launch_red = [&](auto kern, int n_acc) -> int {
    const size_t sm = (size_t)n_acc * kRedTile * 8;
    EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    kern<<<grid, kRedThreads, sm, s>>>(r);
    count_launch();
    return EIGER_OK;
  };
  int rc;
  switch (L.sig) {
    case SIG_SC: rc = launch_red(sort_reduce_kernel<UO, SIG_SC>, 2); break;
    case SIG_SC32: rc = launch_red(sort_reduce_kernel<UO, SIG_SC32>, 2); break;
    default: rc = launch_red(sort_reduce_kernel<UO, SIG_GENERIC>, L.plan.n_acc); break;
  }
  if (rc) return rc;
  bool any_fmm = false;
  for (int j = 0; j < L.n_out_aggs; ++j) any_fmm = any_fmm || (L.plan.f64[j] && (L.plan.op[j] == EIGER_MIN || L.plan.op[j] == EIGER_MAX));
  if (any_fmm) { sort_finalize_kernel<<<(int)std::min<int64_t>((gcap + 255) / 256 + 1, (int64_t)sm_count * 8), 256, 0, s>>>(r, gcap); count_launch(); }
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

}  // namespace

int launch_sort_groupby(SortLaunch& L, int sm_count, size_t smem_optin, cudaStream_t s) {
  if (L.n <= 0 || L.n >= (1ll << 32) || L.bits < 0 || L.bits > 64) return EIGER_ERR_ARG;
  const bool k32 = L.bits <= 32;
  switch (L.key_kind) {
    case KK_I32: return sort_groupby<uint32_t, KK_I32, KK_U32PRE>(L, sm_count, smem_optin, s);
    case KK_I64: return k32 ? sort_groupby<uint32_t, KK_I64, KK_U32PRE>(L, sm_count, smem_optin, s)
                            : sort_groupby<uint64_t, KK_I64, KK_U64PRE>(L, sm_count, smem_optin, s);
    case KK_GEN32: return sort_groupby<uint32_t, KK_GEN32, KK_U32PRE>(L, sm_count, smem_optin, s);
    case KK_GEN: return sort_groupby<uint64_t, KK_GEN, KK_U64PRE>(L, sm_count, smem_optin, s);
    default: return EIGER_ERR_ARG;
  }
}

}  // namespace eiger
