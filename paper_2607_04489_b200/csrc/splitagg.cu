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

#include "internal.h"
#include "rows.cuh"

namespace eiger {
namespace {

constexpr int kSplitThreads = 1024;
constexpr int kQueue = 64;                       // queue entries per warp (flushed 32 at a time)

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

  // tiles of 4 x 1024 rows; group g = blockIdx.x >> lgC of gridDim.x >> lgC groups walks tiles g, g + groups, ..
  constexpr int kRows = 4;
  const int64_t tile = (int64_t)kRows * kSplitThreads;
  const int64_t groups = gridDim.x >> a.lgC;
  const int64_t n_tiles = (a.n + tile - 1) / tile;
  int cnt = 0;                                   // entries waiting in this warp's queue (warp-uniform)
  bool bad = false;
  for (int64_t t = blockIdx.x >> a.lgC; t < n_tiles; t += groups) {
    const int64_t base = t * tile;
    U u[kRows];
    bool ok[kRows];
    if (base + tile <= a.n) {
      // rows base + 2 * tid, + 1 and base + 2048 + 2 * tid, + 1: two 8- or 16-byte key loads per thread
      load_u2<KK>(a.key, base + 2 * tid, *reinterpret_cast<U(*)[2]>(&u[0]));
      load_u2<KK>(a.key, base + 2 * kSplitThreads + 2 * tid, *reinterpret_cast<U(*)[2]>(&u[2]));
#pragma unroll
      for (int r = 0; r < kRows; ++r) ok[r] = true;
    } else {
#pragma unroll
      for (int r = 0; r < kRows; ++r) {
        const int64_t i = base + (r >> 1) * 2 * kSplitThreads + 2 * tid + (r & 1);
        ok[r] = i < a.n;
        u[r] = ok[r] ? load_u<KK>(a.key, i) : (U)0;
      }
    }
#pragma unroll
    for (int r = 0; r < kRows; ++r) {
      const uint64_t uu = (uint64_t)u[r];
      if (ok[r] && uu >= a.cap) { bad = true; ok[r] = false; }            // outside the planned range (speculative / caller's statistics)
      const bool mine = ok[r] && ((uint32_t)uu & (C - 1)) == me;
      const uint32_t m = __ballot_sync(0xffffffffu, mine);
      if (m) {
        if (mine) {
          const int p = cnt + __popc(m & ((1u << lane) - 1u));
          q_slot[p] = (uint32_t)(uu >> a.lgC);
          q_row[p] = (uint32_t)((r >> 1) * 2 * kSplitThreads + 2 * tid + (r & 1));
        }
        cnt += __popc(m);
        if (cnt >= 32) {
          __syncwarp();
          cnt -= 32;
          consume(q_slot[cnt + lane], base + q_row[cnt + lane]);
          __syncwarp();
        }
      }
    }
    // the queue is drained at the end of every tile (row offsets are relative to the tile)
    __syncwarp();
    if (lane < cnt) consume(q_slot[lane], base + q_row[lane]);
    cnt = 0;
    __syncwarp();
    if (a.spec && __any_sync(0xffffffffu, bad)) break;
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

}  // namespace eiger
