// Step A6a for key ranges between one CTA's shared memory and the L2-atomics regime
// (2^13 .. 2^17 slots): the direct-index array is SPLIT over C co-operating CTAs.
//
// CTA b owns the slots u with u mod C = b mod C and keeps them in a shared-memory array of
// ceil(R / C) slots; the C CTAs of a group walk the SAME tiles of the input: each reads every key
// of the tile (the first reader pulls it from HBM, the other C - 1 hit in L2), keeps the rows it
// owns - compacted per warp with a ballot into a small queue, so that the value loads and the three
// shared-memory atomics per row run with full warps - and ignores the rest.  HBM traffic stays B per
// row; what grows with C is the key scan (a load, a mask and a ballot per key and CTA) and the L2 -> SM
// traffic.
//
// Why not distributed shared memory (one array spread over a thread-block cluster, remote atomics):
// measured with eiger_probe("dsmem_red" / "dsmem_atom") on the B200, remote shared-memory atomics run
// at 23-25 G rows/s chip-wide for clusters of 8 / 16 against 1240 G rows/s for local ones - 50 times
// slower, slower even than L2 atomics (92 G rows/s) - and plain remote 8-byte stores reach 85-93 G
// rows/s (profiles/r2_probe.md).  Moving the KEYS to every owner through L2 and keeping all atomics
// local is what the hardware is fast at.  PAPER.md:219 (range test), PAPER.md:304-306 (the crossover
// region between the small-table and the partitioned regime).
#include <algorithm>

#include "hashagg.cuh"

namespace eiger {
namespace {

constexpr int kSplitThreads = 1024;
constexpr int kQueue = 64;                       // queue entries per warp (flushed 32 at a time)


// Keys of one tile, kVec vector loads per thread, all issued before the first use: a CTA scans C times
// its share of the input, so the scan must keep many bytes in flight (the first version, two 8-byte
// loads per thread and no prefetch, scanned at 16 GB/s per SM: 0.65 ms per 2^28 keys and group size).
// Element e of vector v of thread t is row v * (E * 1024) + E * t + e of the tile.
template <int KK> struct TileKeys {
  using U = typename KeyTraits<KK>::U;
  static constexpr int E = (KK == KK_I32) ? 4 : 2;             // keys per vector load
  static constexpr int kVec = 4;
  static constexpr int KR = E * kVec;                          // keys per thread and tile
  static constexpr int64_t kTileRows = (int64_t)KR * kSplitThreads;
  __device__ static __forceinline__ uint32_t row_of(int r, int tid) { return (uint32_t)((r / E) * (E * kSplitThreads) + E * tid + (r % E)); }
  __device__ static __forceinline__ void load(const KeyDesc& key, int64_t base, int tid, U (&u)[KR]) {
#pragma unroll
    for (int v = 0; v < kVec; ++v) {
      const int64_t i = base + (int64_t)v * (E * kSplitThreads) + E * tid;
      if constexpr (KK == KK_I32) {
        const uint4 x = ldg_stream_16(static_cast<const int32_t*>(key.ptr[0]) + i);
        const uint32_t b = (uint32_t)key.base[0];
        u[4 * v] = x.x - b; u[4 * v + 1] = x.y - b; u[4 * v + 2] = x.z - b; u[4 * v + 3] = x.w - b;
      } else {
        load_u2<KK>(key, i, *reinterpret_cast<U(*)[2]>(&u[2 * v]));
      }
    }
  }
};

struct SplitArgs {
  KeyDesc key;
  AggPlan plan;
  int64_t n;
  uint64_t cap;                                  // R: keys u >= cap are outside the planned range
  uint32_t local_slots;                          // ceil(R / C)
  int32_t lgC, spec;
  void* table;                                   // global [R][n_acc] cells
  CallDev* call;
};

template <int KK, int SIG>
__global__ void __launch_bounds__(kSplitThreads, 1)
split_direct_kernel(const __grid_constant__ SplitArgs a) {
  using U = typename KeyTraits<KK>::U;
  using S = Sig<SIG>;
  constexpr int NV = S::kVals, NA = S::kAcc;
  extern __shared__ __align__(16) unsigned char smem[];     // [accumulator planes: n_acc x local_slots x 8][queues]
  const int n_acc = S::kStatic ? NA : a.plan.n_acc;
  const int n_vals = S::kStatic ? NV : a.plan.n_vals;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t C = 1u << a.lgC, me = blockIdx.x & (C - 1);
  const uint32_t L = a.local_slots;
  for (int j = 0; j < n_acc; ++j) smem_init_plane(smem, L, j, sig_op<SIG>(a.plan, j), sig_f64<SIG>(a.plan, j), tid, kSplitThreads);
  uint32_t* q_slot = reinterpret_cast<uint32_t*>(smem + (size_t)n_acc * 8 * L) + warp * 2 * kQueue;
  uint32_t* q_row = q_slot + kQueue;
  __syncthreads();

  // the rows a full warp pops from its queue: value loads (gather) + shared-memory accumulation
  auto consume = [&](uint32_t slot, int64_t row) {
    uint64_t raw[NV];
#pragma unroll
    for (int c = 0; c < NV; ++c) raw[c] = (S::kStatic || c < n_vals) ? global_val(a.plan, c, sig_vw<SIG>(a.plan, c), row) : 0ull;
#pragma unroll
    for (int j = 0; j < NA; ++j) {
      if (!S::kStatic && j >= n_acc) break;
      const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
      smem_merge(smem, L, j, slot, op, f, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
    }
  };

  // group g = blockIdx.x >> lgC of gridDim.x >> lgC groups walks tiles g, g + groups, ..; the next tile's
  // keys are requested before the current tile is processed
  using TK = TileKeys<KK>;
  constexpr int KR = TK::KR;
  const int64_t tile = TK::kTileRows;
  const int64_t groups = gridDim.x >> a.lgC;
  const int64_t n_full = a.n / tile;
  int cnt = 0;                                   // entries waiting in this warp's queue (warp-uniform)
  bool bad = false;
  const uint32_t lt = (1u << lane) - 1u;
  auto scan_row = [&](U ur, bool okr, uint32_t off, int64_t base) {
    const bool mine = okr && ((uint32_t)ur & (C - 1)) == me;
    const uint32_t m = __ballot_sync(0xffffffffu, mine);
    if (mine) {
      const int p = cnt + __popc(m & lt);
      q_slot[p] = (uint32_t)((uint64_t)ur >> a.lgC);
      q_row[p] = off;
    }
    cnt += __popc(m);
    if (cnt >= 32) {
      __syncwarp();
      cnt -= 32;
      consume(q_slot[cnt + lane], base + q_row[cnt + lane]);
      __syncwarp();
    }
  };
  auto drain = [&](int64_t base) {               // the queue is drained at the end of every tile (row offsets are relative to it)
    __syncwarp();
    if (lane < cnt) consume(q_slot[lane], base + q_row[lane]);
    cnt = 0;
    __syncwarp();
  };
  {
    U cur[KR], nxt[KR];
    int64_t t = blockIdx.x >> a.lgC;
    if (t < n_full) TK::load(a.key, t * tile, tid, cur);
    for (; t < n_full; t += groups) {
      const bool more = t + groups < n_full;
      if (more) TK::load(a.key, (t + groups) * tile, tid, nxt);
      const int64_t base = t * tile;
      // one range check per thread and tile (the largest of its keys): a key outside the planned range
      // (speculative run / caller's statistics) discards the whole result, so the thread's keys of this
      // tile are simply not queued
      U umax = cur[0];
#pragma unroll
      for (int r = 1; r < KR; ++r) umax = cur[r] > umax ? cur[r] : umax;
      const bool in_range = (uint64_t)umax < a.cap;
      bad = bad || !in_range;
#pragma unroll
      for (int r = 0; r < KR; ++r) scan_row(cur[r], in_range, TK::row_of(r, tid), base);
      drain(base);
      if (a.spec && __any_sync(0xffffffffu, bad)) break;
      if (more) {
#pragma unroll
        for (int r = 0; r < KR; ++r) cur[r] = nxt[r];
      }
    }
  }
  // the ragged last tile, by the group that would have taken it: row at a time
  if (n_full * tile < a.n && (n_full % groups) == (blockIdx.x >> a.lgC)) {
    const int64_t base = n_full * tile;
    for (int64_t o = tid - lane; base + o < a.n; o += kSplitThreads) {          // warp-uniform trip count
      const int64_t i = base + o + lane;
      bool okr = i < a.n;
      const U ur = okr ? load_u<KK>(a.key, i) : (U)0;
      if (okr && (uint64_t)ur >= a.cap) { bad = true; okr = false; }
      scan_row(ur, okr, (uint32_t)(o + lane), base);
    }
    drain(base);
  }
  if (bad) atomicOr(&a.call->abort, 1u);
  __syncthreads();
  // flush: local slot s of owner `me` is global slot s * C + me; one global atomic per cell and CTA
  uint64_t* table = static_cast<uint64_t*>(a.table);
  for (uint32_t w = tid; w < L * (uint32_t)n_acc; w += kSplitThreads) {
    const uint32_t j = w / L, s = w % L;
    const uint64_t g = ((uint64_t)s << a.lgC) + me;
    if (g >= a.cap) continue;
    const int op = sig_op<SIG>(a.plan, (int)j); const bool f = sig_f64<SIG>(a.plan, (int)j);
    const uint64_t v = smem_read(smem, L, (int)j, s, op, f);
    if (v == acc_identity(op) && !(op == EIGER_SUM && f)) continue;
    atomic_merge(table + g * (uint32_t)n_acc + j, op, f, v);
  }
}

template <int KK, int SIG>
int launch_one(const SplitLaunch& L, cudaStream_t s) {
  SplitArgs a{};
  a.key = L.key; a.plan = L.plan; a.n = L.n; a.cap = L.cap; a.local_slots = L.local_slots; a.lgC = L.lgC; a.spec = L.spec;
  a.table = L.table; a.call = L.call;
  auto kern = split_direct_kernel<KK, SIG>;
  const size_t smem = (size_t)L.plan.n_acc * 8 * L.local_slots + (size_t)(kSplitThreads / 32) * 2 * kQueue * 4;
  EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<L.blocks, kSplitThreads, smem, s>>>(a);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}
template <int KK>
int launch_sig(const SplitLaunch& L, cudaStream_t s) {
  switch (L.sig) {
    case SIG_SC: return launch_one<KK, SIG_SC>(L, s);
    case SIG_SC32: return launch_one<KK, SIG_SC32>(L, s);
    default: return launch_one<KK, SIG_GENERIC>(L, s);
  }
}

// ---- the same split for keys that are not dense: per-CTA hash tables ----------------------------
// Owner of key u = top lgC bits of a multiplicative hash of u (independent of the table's bucket
// hash); every CTA of a group scans all keys of the group's tiles, queues the rows it owns and runs
// them through its own shared-memory hash table (hashagg.cuh: Front) with full warps.  At the end the
// tables are merged into the global table like EIGER_SMEM's; a key lives in one CTA per group.
template <class U> __device__ __forceinline__ uint32_t split_owner(U u, int lgC) {
  return (uint32_t)(((uint32_t)u ^ (uint32_t)((uint64_t)u >> 32)) * 0x85EBCA77u) >> (32 - lgC);
}

template <int KK, int SIG>
__global__ void __launch_bounds__(kSplitThreads, 1)
split_hash_kernel(const __grid_constant__ HashAggArgs a, int lgC) {
  using F = Front<KK, SIG, 16 / (int)sizeof(typename KeyTraits<KK>::U)>;
  using U = typename F::U;
  constexpr int NV = F::NV;
  extern __shared__ __align__(16) unsigned char smem[];     // [table][queues: keys, row offsets]
  __shared__ uint32_t s_count, s_abort;
  const int n_vals = Sig<SIG>::kStatic ? NV : a.plan.n_vals;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t me = blockIdx.x & ((1u << lgC) - 1u);
  F f(a, smem, a.slots);
  U* q_key = reinterpret_cast<U*>(smem + a.table_off) + warp * kQueue;
  uint32_t* q_row = reinterpret_cast<uint32_t*>(smem + a.table_off + (size_t)(kSplitThreads / 32) * kQueue * sizeof(U)) + warp * kQueue;
  if (tid == 0) { s_count = 0; s_abort = 0; }
  f.init(tid, kSplitThreads);
  __syncthreads();
  bool missed = false;
  auto consume = [&](U u, int64_t row, bool valid) {       // all 32 lanes of the warp are here
    uint64_t raw[NV];
#pragma unroll
    for (int c = 0; c < NV; ++c) raw[c] = (valid && (Sig<SIG>::kStatic || c < n_vals)) ? global_val(a.plan, c, sig_vw<SIG>(a.plan, c), row) : 0ull;
    const uint32_t miss = f.pair(u, raw, valid, u, raw, false, &s_count);
    if (__any_sync(0xffffffffu, miss != 0)) { if (a.spec) missed = missed || miss != 0; else if (miss) f.back_row(u, raw); }
    __syncwarp();
  };
  using TK = TileKeys<KK>;
  constexpr int KR = TK::KR;
  const int64_t tile = TK::kTileRows;
  const int64_t groups = gridDim.x >> lgC;
  const int64_t n_full = a.n / tile;
  int cnt = 0;
  uint32_t trip = 0;
  auto scan_row = [&](U ur, bool okr, uint32_t off, int64_t base) {
    const bool mine = okr && split_owner<U>(ur, lgC) == me;
    const uint32_t m = __ballot_sync(0xffffffffu, mine);
    if (m) {
      if (mine) {
        const int p = cnt + __popc(m & ((1u << lane) - 1u));
        q_key[p] = ur;
        q_row[p] = off;
      }
      cnt += __popc(m);
      if (cnt >= 32) {
        __syncwarp();
        cnt -= 32;
        consume(q_key[cnt + lane], base + q_row[cnt + lane], true);
        __syncwarp();
      }
    }
  };
  auto drain = [&](int64_t base) {
    __syncwarp();
    if (cnt > 0) consume(lane < cnt ? q_key[lane] : (U)0, base + (lane < cnt ? q_row[lane] : 0u), lane < cnt);
    cnt = 0;
    __syncwarp();
  };
  {
    U cur[KR], nxt[KR];
    int64_t t = blockIdx.x >> lgC;
    if (t < n_full) TK::load(a.key, t * tile, tid, cur);
    for (; t < n_full; t += groups) {
      if (a.spec) { if (__any_sync(0xffffffffu, missed || ((trip++ & 15u) == 0u && *reinterpret_cast<volatile uint32_t*>(&a.call->abort)))) break; }
      const bool more = t + groups < n_full;
      if (more) TK::load(a.key, (t + groups) * tile, tid, nxt);
      const int64_t base = t * tile;
#pragma unroll
      for (int r = 0; r < KR; ++r) scan_row(cur[r], true, TK::row_of(r, tid), base);
      drain(base);
      if (more) {
#pragma unroll
        for (int r = 0; r < KR; ++r) cur[r] = nxt[r];
      }
    }
  }
  if (n_full * tile < a.n && (n_full % groups) == (blockIdx.x >> lgC) && !(a.spec && __any_sync(0xffffffffu, missed))) {
    const int64_t base = n_full * tile;
    for (int64_t o = tid - lane; base + o < a.n; o += kSplitThreads) {
      const int64_t i = base + o + lane;
      const bool okr = i < a.n;
      scan_row(okr ? load_u<KK>(a.key, i) : (U)0, okr, (uint32_t)(o + lane), base);
    }
    drain(base);
  }
  if (a.spec) {
    if (missed) { atomicOr(&a.call->abort, 1u); atomicOr(&s_abort, 1u); }
    __syncthreads();
    if (s_abort || *reinterpret_cast<volatile uint32_t*>(&a.call->abort)) return;
  } else {
    __syncthreads();
  }
  f.flush_merge(tid, kSplitThreads);
}

template <int KK, int SIG>
int launch_hash_one(const HashAggLaunch& L, int lgC, cudaStream_t s) {
  using U = typename KeyTraits<KK>::U;
  HashAggArgs a{};
  a.key = L.key; a.plan = L.plan; a.n = L.n;
  a.slots = L.slots; a.limit = L.limit; a.spec = L.spec; a.max_probes = 16; a.n_hot = 0;
  a.table = L.table; a.cap = L.cap; a.stride = L.stride; a.call = L.call;
  a.table_off = (uint32_t)((L.table_smem_bytes + 127) & ~(size_t)127);       // the queues follow the table
  const size_t smem = (size_t)a.table_off + (size_t)(kSplitThreads / 32) * kQueue * (sizeof(U) + 4);
  auto kern = split_hash_kernel<KK, SIG>;
  EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<L.blocks, kSplitThreads, smem, s>>>(a, lgC);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}
template <int KK>
int launch_hash_sig(const HashAggLaunch& L, int lgC, cudaStream_t s) {
  switch (L.sig) {
    case SIG_SC: return launch_hash_one<KK, SIG_SC>(L, lgC, s);
    case SIG_SC32: return launch_hash_one<KK, SIG_SC32>(L, lgC, s);
    default: return launch_hash_one<KK, SIG_GENERIC>(L, lgC, s);
  }
}

}  // namespace

size_t split_direct_smem(int n_acc, uint32_t local_slots) { return (size_t)n_acc * 8 * local_slots + (size_t)(kSplitThreads / 32) * 2 * kQueue * 4; }

int launch_split_direct(const SplitLaunch& L, cudaStream_t s) {
  switch (L.key_kind) {
    case KK_I32: return launch_sig<KK_I32>(L, s);
    case KK_I64: return launch_sig<KK_I64>(L, s);
    case KK_GEN32: return launch_sig<KK_GEN32>(L, s);
    case KK_GEN: return launch_sig<KK_GEN>(L, s);
    default: return EIGER_ERR_ARG;
  }
}

// queue bytes that follow the per-CTA table of the split hash kernel
size_t split_hash_queue_bytes(int key_kind) { return (size_t)(kSplitThreads / 32) * kQueue * ((key_kind == KK_I32 ? 4 : 8) + 4) + 128; }

int launch_split_hash(const HashAggLaunch& L, int lgC, cudaStream_t s) {
  switch (L.key_kind) {
    case KK_I32: return launch_hash_sig<KK_I32>(L, lgC, s);
    case KK_I64: return launch_hash_sig<KK_I64>(L, lgC, s);
    case KK_GEN: return launch_hash_sig<KK_GEN>(L, lgC, s);
    default: return EIGER_ERR_ARG;
  }
}

}  // namespace eiger
