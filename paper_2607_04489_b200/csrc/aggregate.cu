// Steps A5, A6a and A7: table init, the direct-index aggregation kernel (slot = key - min;
// one kernel template over what a CTA keeps in shared memory in FRONT of the global array)
// and compaction of either table kind.
//
//   EIGER_DIRECT    FRONT_PRIV (per-thread private cells, no atomics; tiny ranges),
//                   FRONT_SDIRECT (per-CTA shared-memory array, replicated per warp group) or
//                   FRONT_NONE (global atomics only; ranges beyond shared memory)
//   The hash variants (EIGER_SMEM / EIGER_GLOBAL / EIGER_PARTITION) live in hashagg.cu.
//
// GROUP BY semantics: §3.3; range test PAPER.md:219 §4.3; emit groups =
// HT.retrieveAll PAPER.md:184.
#include <algorithm>

#include "internal.h"
#include "rows.cuh"

namespace eiger {
namespace {

constexpr int kAggThreads = 256;
constexpr int kAggThreadsWide = 1024;

struct AggArgs {
  KeyDesc key;
  AggPlan plan;
  int64_t n;
  uint32_t front_slots, front_limit, front_replicas, stride;
  int32_t spec;
  void* table;
  uint64_t cap;
  CallDev* call;
  // FRONT_DICT: key -> dense id dictionary built from the key sample (image in global memory)
  const uint2* dict; uint32_t dict_slots, dict_shift;
  // dict_compact: the large dictionary (up to ~8300 keys; SUM + COUNT plans only).  Shared memory then holds
  // [SUM planes: 8 x slots][COUNT plane: 4 x slots][dictionary keys: 4 x dict_slots][dictionary ids: 2 x dict_slots],
  // one replica - 12 instead of 16 bytes per id and 6 instead of 8 per dictionary entry, which is what lets 2^13
  // keys fit one CTA
  uint32_t dict_compact;
  // several passes over the input, each with the dictionary of ONE slice of the keys (slice = the dict_pass_lg hash bits
  // below the slot bits): rows of other slices are skipped.  dict_pass_lg = 0: a single pass owns every key.
  uint32_t dict_pass_lg, dict_pass;
};

constexpr uint32_t kDictMul = 0x9E3779B1u;
// kernel-side front kind of the large dictionary (AggArgs::dict_compact): its own instantiation, so that the small
// dictionary's kernel carries none of its branches (they cost 3-4 % at 2^8 / 2^12 keys when tested at run time)
constexpr int FRONT_DICTC = 100;
constexpr int FRONT_DICTP = 101;        // the large dictionary, one of several passes (rows of other key slices are skipped)
constexpr int FRONT_DICTG = 102;        // the small dictionary searched two entries at a time (one replica, thousands of keys)
template <int FRONT> constexpr bool kIsDict = (FRONT == FRONT_DICT || FRONT == FRONT_DICTC || FRONT == FRONT_DICTP || FRONT == FRONT_DICTG);
template <int FRONT> constexpr bool kIsCompact = (FRONT == FRONT_DICTC || FRONT == FRONT_DICTP);
__host__ __device__ __forceinline__ uint32_t dict_slice(uint32_t u, uint32_t shift, uint32_t lg) {
  return ((u * kDictMul) >> (shift - lg)) & ((1u << lg) - 1u);
}

template <int KK, int SIG, int FRONT>
struct AggCtx {
  using U = typename KeyTraits<KK>::U;
  using S = Sig<SIG>;
  static constexpr int NV = S::kVals;
  static constexpr int NA = S::kAcc;

  const AggArgs& a;
  const int n_acc;
  unsigned char* smem;

  unsigned char* rep_base;       // FRONT_SDIRECT / FRONT_DICT: this warp's replica of the table
  const uint2* sdict;            // FRONT_DICT: the dictionary (key, id) in shared memory, after the replicas

  __device__ AggCtx(const AggArgs& args, unsigned char* sm)
      : a(args), n_acc(S::kStatic ? S::kAcc : args.plan.n_acc), smem(sm) {
    const uint32_t rep = args.front_replicas > 1 ? (threadIdx.x >> 5) % args.front_replicas : 0u;
    rep_base = sm + (size_t)rep * args.front_slots * 8 * (uint32_t)n_acc;
    sdict = reinterpret_cast<const uint2*>(sm + (size_t)args.front_replicas * args.front_slots * 8 * (uint32_t)n_acc);
    skey = reinterpret_cast<const uint32_t*>(sm + (size_t)args.front_slots * 12);
    sid = reinterpret_cast<const uint16_t*>(skey + args.dict_slots);
  }
  const uint32_t* skey;          // FRONT_DICT, dict_compact: dictionary keys, then 16-bit ids
  const uint16_t* sid;

  // dense id of rebased key u, ~0u when the dictionary does not hold it (empty entries carry id ~0u)
  __device__ __forceinline__ uint32_t dict_id(uint32_t u) const {
    uint32_t h = (u * kDictMul) >> a.dict_shift, id = ~0u;
    bool done = false;
    if constexpr (kIsCompact<FRONT>) {
      // groups of four keys (one LDS.128): the build kernel probes linearly from the start of the key's home group, so
      // the key sits in the first group that holds it or an empty position.  (One key per probe made this loop 77 %
      // of the kernel's instructions at load 0.5: the warp iterates as long as its unluckiest lane.)
      h &= ~3u;
      while (!done) {
        const uint4 k = *reinterpret_cast<const uint4*>(skey + h);
        const int pos = k.x == u ? 0 : (k.y == u ? 1 : (k.z == u ? 2 : (k.w == u ? 3 : -1)));
        if (pos >= 0) { id = sid[h + (uint32_t)pos]; done = true; }
        else if (k.x == kEmpty32 || k.y == kEmpty32 || k.z == kEmpty32 || k.w == kEmpty32) done = true;
        else h = (h + 4u) & (a.dict_slots - 1u);
      }
    } else if constexpr (FRONT == FRONT_DICTG) {
      // (key, id) entries, two per LDS.128: pays from a few thousand keys (2^12: aggregate 0.78 -> 0.72 ms), costs at
      // 2^4 / 2^8 keys (0.48 -> 0.57, 0.55 -> 0.65 ms), where the one-entry loop below almost never iterates
      h &= ~1u;
      while (!done) {
        const uint4 e = *reinterpret_cast<const uint4*>(sdict + h);
        if (e.x == u) { id = e.y; done = true; }
        else if (e.z == u) { id = e.w; done = true; }
        else if (e.x == kEmpty32 || e.z == kEmpty32) done = true;
        else h = (h + 2u) & (a.dict_slots - 1u);
      }
    } else {
      while (!done) {
        const uint2 e = sdict[h];
        if (e.x == u) { id = e.y; done = true; }
        else if (e.x == kEmpty32) done = true;
        else h = (h + 1u) & (a.dict_slots - 1u);
      }
    }
    return id;
  }

  __device__ void front_init() {
    const int tid = threadIdx.x, T = blockDim.x;
    if constexpr (FRONT == FRONT_PRIV) {
      uint64_t* acc = reinterpret_cast<uint64_t*>(smem);
      for (uint32_t c = 0; c < a.front_slots * (uint32_t)n_acc; ++c)
        acc[(size_t)c * T + tid] = acc_identity(sig_op<SIG>(a.plan, (int)(c % (uint32_t)n_acc)));
    } else if constexpr (FRONT == FRONT_SDIRECT || kIsDict<FRONT>) {
      constexpr bool compact = kIsCompact<FRONT>;
      if constexpr (compact) {
        uint32_t* w = reinterpret_cast<uint32_t*>(smem);
        for (uint32_t i = tid; i < 3u * a.front_slots; i += T) w[i] = 0u;        // SUM low, SUM high, COUNT
        uint32_t* k = const_cast<uint32_t*>(skey); uint16_t* d = const_cast<uint16_t*>(sid);
        for (uint32_t i = tid; i < a.dict_slots; i += T) { const uint2 e = a.dict[i]; k[i] = e.x; d[i] = (uint16_t)e.y; }
      } else {
      for (uint32_t rep = 0; rep < a.front_replicas; ++rep)
        for (int j = 0; j < n_acc; ++j)
          smem_init_plane(smem + (size_t)rep * a.front_slots * 8 * (uint32_t)n_acc, a.front_slots, j, sig_op<SIG>(a.plan, j), sig_f64<SIG>(a.plan, j), tid, T);
      if constexpr (kIsDict<FRONT>) {
        uint2* d = const_cast<uint2*>(sdict);
        for (uint32_t i = tid; i < a.dict_slots; i += T) d[i] = a.dict[i];
      }
      }
    }
    if constexpr (FRONT != FRONT_NONE) __syncthreads();
  }

  __device__ __forceinline__ void back_row(U u, const uint64_t (&raw)[NV]) {
    uint64_t* cells = static_cast<uint64_t*>(a.table) + (uint64_t)u * (uint32_t)n_acc;
#pragma unroll
    for (int j = 0; j < NA; ++j) {
      if (!S::kStatic && j >= n_acc) break;
      const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
      atomic_merge(cells + j, op, f, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
    }
  }

  __device__ __forceinline__ void row(U u, const uint64_t (&raw)[NV]) {
    if constexpr (FRONT == FRONT_DICTP) { if (dict_slice((uint32_t)u, a.dict_shift, a.dict_pass_lg) != a.dict_pass) return; }
    if constexpr (kIsDict<FRONT>) {
      // the dictionary names the keys of the sample: a key it does not hold discards the pass
      const uint32_t id = dict_id((uint32_t)u);
      if (id >= a.front_slots) { if (*reinterpret_cast<volatile uint32_t*>(&a.call->abort) == 0u) atomicOr(&a.call->abort, 1u); return; }
      u = (U)id;
    }
    // speculative run planned from a sample: the range is checked exactly here
    if (!kIsDict<FRONT> && a.spec && (uint64_t)u >= a.cap) { if (*reinterpret_cast<volatile uint32_t*>(&a.call->abort) == 0u) atomicOr(&a.call->abort, 1u); return; }
    if constexpr (FRONT == FRONT_PRIV) {
      uint64_t* acc = reinterpret_cast<uint64_t*>(smem) + (size_t)u * (uint32_t)n_acc * blockDim.x + threadIdx.x;
#pragma unroll
      for (int j = 0; j < NA; ++j) {
        if (!S::kStatic && j >= n_acc) break;
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        uint64_t* c = acc + (size_t)j * blockDim.x;
        *c = combine(op, f, *c, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
      }
    } else if constexpr (FRONT == FRONT_SDIRECT || kIsDict<FRONT>) {
      unsigned char* base = rep_base;
#pragma unroll
      for (int j = 0; j < NA; ++j) {
        if (!S::kStatic && j >= n_acc) break;
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        smem_merge(base, a.front_slots, j, (uint32_t)u, op, f, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
      }
    } else {
      back_row(u, raw);
    }
  }

  // SUM(int64) + COUNT into the shared-memory array, R rows at a time: all returning adds first,
  // then the counts, then the carries, so that a row's carry does not wait alone for its atomic
  // (ncu: short_scoreboard was 28 % of the stall samples with one row at a time)
  template <int R>
  __device__ __forceinline__ void rows_sc(const U (&uk)[R], const uint64_t (&raw)[R][NV]) {
    static_assert((SIG == SIG_SC || SIG == SIG_SC32) && (FRONT == FRONT_SDIRECT || kIsDict<FRONT>), "SUM + COUNT signature only");
    uint32_t* lo = reinterpret_cast<uint32_t*>(rep_base);
    uint32_t* cnt = reinterpret_cast<uint32_t*>(rep_base + (size_t)8 * a.front_slots);
    U u[R];
    if constexpr (kIsDict<FRONT>) {
      // all look-ups first (R independent shared-memory loads in flight), then the misses are settled
      bool bad = false;
      if constexpr (FRONT == FRONT_DICTP) {
        // rows of the other slices are left out one by one (a predicate per row, no early exit: most trips hold both kinds)
        bool own[R];
#pragma unroll
        for (int r = 0; r < R; ++r) own[r] = dict_slice((uint32_t)uk[r], a.dict_shift, a.dict_pass_lg) == a.dict_pass;
#pragma unroll
        for (int r = 0; r < R; ++r) { u[r] = own[r] ? (U)dict_id((uint32_t)uk[r]) : (U)0; bad = bad || (uint32_t)u[r] >= a.front_slots; }
        if (bad) { if (*reinterpret_cast<volatile uint32_t*>(&a.call->abort) == 0u) atomicOr(&a.call->abort, 1u); return; }
        uint32_t old[R];
#pragma unroll
        for (int r = 0; r < R; ++r) if (own[r]) old[r] = atomicAdd(lo + (uint32_t)u[r], (uint32_t)raw[r][0]);
#pragma unroll
        for (int r = 0; r < R; ++r) if (own[r]) atomicAdd(cnt + (uint32_t)u[r], 1u);
#pragma unroll
        for (int r = 0; r < R; ++r) {
          if (!own[r]) continue;
          const uint32_t vl = (uint32_t)raw[r][0];
          const uint32_t h = (uint32_t)(raw[r][0] >> 32) + ((uint32_t)(old[r] + vl) < vl ? 1u : 0u);
          if (h) atomicAdd(lo + a.front_slots + (uint32_t)u[r], h);
        }
        return;
      }
#pragma unroll
      for (int r = 0; r < R; ++r) { u[r] = (U)dict_id((uint32_t)uk[r]); bad = bad || (uint32_t)u[r] >= a.front_slots; }
      if (bad) { if (*reinterpret_cast<volatile uint32_t*>(&a.call->abort) == 0u) atomicOr(&a.call->abort, 1u); return; }
    } else {
#pragma unroll
      for (int r = 0; r < R; ++r) u[r] = uk[r];
    }
    if (!kIsDict<FRONT> && a.spec) {
      // speculative run planned from a sample: one key outside the planned range discards the whole
      // pass anyway, so the trip is skipped as a whole (one branch per R rows, not one per atomic)
      bool bad = false;
#pragma unroll
      for (int r = 0; r < R; ++r) bad = bad || (uint64_t)u[r] >= a.cap;
      if (bad) { if (*reinterpret_cast<volatile uint32_t*>(&a.call->abort) == 0u) atomicOr(&a.call->abort, 1u); return; }
    }
    uint32_t old[R];
#pragma unroll
    for (int r = 0; r < R; ++r) old[r] = atomicAdd(lo + (uint32_t)u[r], (uint32_t)raw[r][0]);
#pragma unroll
    for (int r = 0; r < R; ++r) atomicAdd(cnt + (uint32_t)u[r], 1u);
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const uint32_t vl = (uint32_t)raw[r][0];
      const uint32_t h = (uint32_t)(raw[r][0] >> 32) + ((uint32_t)(old[r] + vl) < vl ? 1u : 0u);
      if (h) atomicAdd(lo + a.front_slots + (uint32_t)u[r], h);
    }
  }

  // merge one partial accumulator vector (already in partial form) into the back table
  __device__ __forceinline__ void back_merge(uint64_t u, int j, uint64_t part, uint64_t* cells) {
    const int op = sig_op<SIG>(a.plan, j);
    if (part == acc_identity(op) && !(op == EIGER_SUM && sig_f64<SIG>(a.plan, j))) return;
    atomic_merge(cells + j, op, sig_f64<SIG>(a.plan, j), part);
  }

  __device__ void front_flush() {
    if constexpr (FRONT == FRONT_NONE) return;
    __syncthreads();
    const int tid = threadIdx.x, T = blockDim.x;
    if constexpr (FRONT == FRONT_PRIV) {
      // each warp reduces the T private copies of one (slot, accumulator) cell at a time
      const uint64_t* acc = reinterpret_cast<const uint64_t*>(smem);
      const int lane = tid & 31, warp = tid >> 5, nw = T >> 5;
      for (uint32_t c = warp; c < a.front_slots * (uint32_t)n_acc; c += nw) {
        const int j = (int)(c % (uint32_t)n_acc);
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        uint64_t v = acc_identity(op);
        for (int t = lane; t < T; t += 32) v = combine(op, f, v, acc[(size_t)c * T + t]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = combine(op, f, v, __shfl_xor_sync(0xffffffffu, v, o));
        if (lane == 0) back_merge(c / (uint32_t)n_acc, j, v, static_cast<uint64_t*>(a.table) + (uint64_t)(c / (uint32_t)n_acc) * (uint32_t)n_acc);
      }
    } else if constexpr (FRONT == FRONT_SDIRECT || kIsDict<FRONT>) {
      // the CTA's replicas are combined first: one global atomic per cell and CTA (with 8 replicas of
      // a 256-slot table the flush of ~900 CTAs otherwise queues millions of atomics on 512 addresses)
      const uint32_t per = a.front_slots * (uint32_t)n_acc;
      for (uint32_t w = tid; w < per; w += T) {
        const uint32_t j = w / a.front_slots, u = w % a.front_slots;
        const int op = sig_op<SIG>(a.plan, (int)j); const bool f = sig_f64<SIG>(a.plan, (int)j);
        uint64_t v;
        const bool compact_count = kIsCompact<FRONT> && op == EIGER_COUNT;
        if (compact_count) v = reinterpret_cast<const uint32_t*>(smem + (size_t)8 * a.front_slots)[u];    // 4-byte COUNT plane
        else v = smem_read(smem, a.front_slots, (int)j, u, op, f);
        for (uint32_t rep = 1; rep < a.front_replicas; ++rep)
          v = combine(op, f, v, smem_read(smem + (size_t)rep * a.front_slots * 8 * (uint32_t)n_acc, a.front_slots, (int)j, u, op, f));
        back_merge(u, (int)j, v, static_cast<uint64_t*>(a.table) + (uint64_t)u * (uint32_t)n_acc);
      }
    }
  }
};

// THREADS = 256, or 1024 for shared-memory arrays of which fewer than three fit an SM (a 256-thread
// CTA per SM leaves 8 warps to hide the loads: measured 0.93 ms instead of 0.5 ms per 2^28 rows)
template <int KK, int SIG, int FRONT, int THREADS>
__global__ void __launch_bounds__(THREADS)
aggregate_kernel(const __grid_constant__ AggArgs a) {
  constexpr int kAggThreads = THREADS;
  extern __shared__ __align__(16) unsigned char smem[];
  using Ctx = AggCtx<KK, SIG, FRONT>;
  using U = typename Ctx::U;
  constexpr int NV = Ctx::NV;
  constexpr int UNR = !Sig<SIG>::kStatic ? 1 : (NV >= 4 ? 2 : 4);
  Ctx ctx(a, smem);
  ctx.front_init();

  const int tid = threadIdx.x;
  const int n_vals = Sig<SIG>::kStatic ? NV : a.plan.n_vals;
  constexpr int64_t kStep = 2 * kAggThreads, kTile = kStep * UNR;
  const int64_t n_tiles = a.n / kTile;
  [[maybe_unused]] uint32_t trip = 0;
  for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    // speculative run: somebody met a key outside the sampled range -> the result is discarded, stop
    // (only the global-atomics flavour polls: in the shared-memory flavours the poll cost 10 % of
    // a pass that is over in a fraction of a millisecond anyway)
    if constexpr (FRONT == FRONT_NONE) {
      if (a.spec && (trip++ & 15u) == 0u && __any_sync(0xffffffffu, *reinterpret_cast<volatile uint32_t*>(&a.call->abort) != 0u)) break;
    }
    const int64_t r0 = t * kTile + 2 * tid;
    U u[UNR][2];
    uint64_t raw[UNR][2][NV];
#pragma unroll
    for (int s = 0; s < UNR; ++s) {
      load_u2<KK>(a.key, r0 + s * kStep, u[s]);
#pragma unroll
      for (int c = 0; c < NV; ++c) {
        if (!Sig<SIG>::kStatic && c >= n_vals) { raw[s][0][c] = 0; raw[s][1][c] = 0; continue; }
        global_val2(a.plan, c, sig_vw<SIG>(a.plan, c), r0 + s * kStep, raw[s][0][c], raw[s][1][c]);
      }
    }
    if constexpr ((SIG == SIG_SC || SIG == SIG_SC32) && (FRONT == FRONT_SDIRECT || kIsDict<FRONT>)) {
      U uu[2 * UNR]; uint64_t rr[2 * UNR][NV];
#pragma unroll
      for (int s = 0; s < UNR; ++s) { uu[2 * s] = u[s][0]; uu[2 * s + 1] = u[s][1]; rr[2 * s][0] = raw[s][0][0]; rr[2 * s + 1][0] = raw[s][1][0]; }
      ctx.template rows_sc<2 * UNR>(uu, rr);
    } else {
#pragma unroll
      for (int s = 0; s < UNR; ++s) { ctx.row(u[s][0], raw[s][0]); ctx.row(u[s][1], raw[s][1]); }
    }
  }
  // ragged tail: row at a time, spread over the whole grid
  for (int64_t i = n_tiles * kTile + (int64_t)blockIdx.x * kAggThreads + tid; i < a.n; i += (int64_t)gridDim.x * kAggThreads) {
    uint64_t raw[NV];
#pragma unroll
    for (int c = 0; c < NV; ++c) raw[c] = (Sig<SIG>::kStatic || c < n_vals) ? global_val(a.plan, c, sig_vw<SIG>(a.plan, c), i) : 0ull;
    ctx.row(load_u<KK>(a.key, i), raw);
  }
  ctx.front_flush();
}

// ---- dictionary of the sampled keys (FRONT_DICT) ----------------------------------------------------
// One thread per sampled row (the same evenly spaced rows the sample statistics were taken from):
// the rebased fused key u is inserted into an open-addressing image (u, dense id) in global memory;
// the first thread to claim a key draws its id.  This is the paper's dictionary encoding
// (Algorithm 1, steps 1-2: insert-and-find, one leader per key) applied to the
// sample: keys that are sparse in a wide range get dense codes, and the aggregation pass then
// indexes a direct array with the code.  id >= cap (more keys than planned): the pass gives up.
__global__ void __launch_bounds__(256)
dict_build_kernel(const __grid_constant__ KeyDesc key, int64_t n, int64_t samples, uint2* __restrict__ img, uint32_t slots, uint32_t shift,
                  uint32_t cap, uint32_t* __restrict__ dict_keys, uint32_t* __restrict__ dict_n, CallDev* call, uint32_t pass_lg, uint32_t group) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= samples) return;
  const int64_t i = (int64_t)(((unsigned __int128)t * (unsigned __int128)n) / (unsigned __int128)samples);
  const uint64_t u64 = load_u<KK_GEN>(key, i);
  if (u64 >= 0xFFFFFFFFull) return;                           // outside the planned ranges: the aggregation pass will notice
  const uint32_t u = (uint32_t)u64;
  uint32_t h = ((u * kDictMul) >> shift) & ~(group - 1u);      // group = 4: the large dictionaries are searched four keys at a time
  // several passes: slice p of the keys has its own image, its own ids 0 .. cap - 1 and its own part of dict_keys
  const uint32_t p = pass_lg ? dict_slice(u, shift, pass_lg) : 0u;
  img += (size_t)p * slots; dict_keys += (size_t)p * cap; dict_n += p;
  uint32_t* w = reinterpret_cast<uint32_t*>(img);
  for (uint32_t probes = 0; probes < slots; ++probes) {
    const uint32_t old = atomicCAS(w + 2 * (size_t)h, kEmpty32, u);
    if (old == kEmpty32) {
      const uint32_t id = atomicAdd(dict_n, 1u);
      if (id < cap) { dict_keys[id] = u; __threadfence(); w[2 * (size_t)h + 1] = id; }
      else atomicOr(&call->abort, 1u);
      return;
    }
    if (old == u) return;
    h = (h + 1u) & (slots - 1u);
  }
  atomicOr(&call->abort, 1u);
}

// ---- table init (step A5) ----------------------------------------------------------------
__global__ void table_init_kernel(uint64_t* table, uint64_t n_words, uint32_t words_per_slot, int hash, AggPlan plan) {
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  for (uint64_t w = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_words; w += stride) {
    const uint32_t pos = (uint32_t)(w % words_per_slot);
    uint64_t v;
    if (hash) v = pos == 0 ? kEmpty64 : (pos <= (uint32_t)plan.n_acc ? acc_identity(plan.op[pos - 1]) : 0ull);
    else v = acc_identity(plan.op[pos]);
    table[w] = v;
  }
}

// ---- compaction (step A7) ------------------------------------------------------------------
struct CompactArgs {
  KeyDesc key;
  AggPlan plan;
  const unsigned char* table;
  uint64_t cap; uint32_t stride; int back;
  void* out_keys[kMaxKeyCols]; uint64_t* out_aggs[kMaxAggs]; int n_out;
  int64_t out_capacity;
  uint64_t R;               // several key columns: fused keys are below R; anything else is a row outside the planned ranges
  const uint32_t* dict_keys; // FRONT_DICT: slot = dense id, key = dict_keys[id]
  CallDev* call;
};

__global__ void __launch_bounds__(256) compact_kernel(const __grid_constant__ CompactArgs c) {
  const uint64_t n_slots = c.cap + (c.back == BACK_HASH ? 1 : 0);
  const uint64_t gstride = (uint64_t)gridDim.x * blockDim.x;
  const int lane = threadIdx.x & 31;
  const uint64_t first = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  // warp-uniform trip count so the ballots below are full-warp
  for (uint64_t base = first - lane; base < n_slots; base += gstride) {
    const uint64_t s = base + lane;
    bool occ = false;
    const uint64_t* slot = nullptr;
    uint64_t u = 0;
    if (s < n_slots) {
      slot = reinterpret_cast<const uint64_t*>(c.table + s * c.stride);
      if (c.back == BACK_HASH) {
        const uint64_t k = slot[0];
        if (s == c.cap) { occ = (k == 0ull); u = kEmpty64; }
        else { occ = (k != kEmpty64); u = k; }
        slot += 1;
      } else {
        occ = slot[c.plan.cnt_acc] != 0ull;
        u = c.dict_keys ? (uint64_t)c.dict_keys[s] : s;
      }
    }
    // several key columns: a row with a column outside its planned range was fused to the marker
    // (rows.cuh: fuse_cols) and sits in the side slot / beyond the fused domain: the caller's
    // statistics do not bound the keys
    if (occ && c.key.ncols > 1 && c.back == BACK_HASH && (s == c.cap || u >= c.R)) { atomicOr(&c.call->abort, 1u); occ = false; }
    const uint32_t m = __ballot_sync(0xffffffffu, occ);
    if (m == 0) continue;
    unsigned long long start = 0;
    if (lane == 0) start = atomicAdd(&c.call->n_groups, (unsigned long long)__popc(m));
    start = __shfl_sync(0xffffffffu, start, 0);
    if (!occ) continue;
    const uint64_t g = start + __popc(m & ((1u << lane) - 1u));
    if ((int64_t)g >= c.out_capacity) continue;
    // un-fuse and un-rebase (PAPER.md:219-221 in reverse)
    uint64_t part[kMaxKeyCols];
    unfuse_key(c.key, u, part);
    for (int k = 0; k < c.key.ncols; ++k) {
      const uint64_t v = part[k] + c.key.base[k];
      switch (c.key.dtype[k]) {
        case EIGER_I8: static_cast<int8_t*>(c.out_keys[k])[g] = (int8_t)v; break;
        case EIGER_I32: static_cast<int32_t*>(c.out_keys[k])[g] = (int32_t)v; break;
        default: static_cast<int64_t*>(c.out_keys[k])[g] = (int64_t)v; break;
      }
    }
    for (int j = 0; j < c.n_out; ++j) c.out_aggs[j][g] = acc_finalize(c.plan.op[j], c.plan.f64[j] != 0, slot[j]);
  }
}

// ---- dispatch --------------------------------------------------------------------------------
template <int KK, int SIG, int FRONT, int THREADS = kAggThreads>
int launch_one(const AggLaunch& L, cudaStream_t s) {
  auto kern = aggregate_kernel<KK, SIG, FRONT, THREADS>;
  if (L.smem_bytes > 32 * 1024) EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem_bytes));
  AggArgs a;
  a.key = L.key; a.plan = L.plan; a.n = L.n;
  a.front_slots = L.front_slots; a.front_limit = L.front_limit; a.front_replicas = L.front_replicas; a.spec = L.spec;
  a.stride = L.stride; a.table = L.table; a.cap = L.cap; a.call = L.call;
  a.dict = static_cast<const uint2*>(L.dict); a.dict_slots = L.dict_slots; a.dict_shift = L.dict_shift;
  a.dict_compact = L.dict_compact; a.dict_pass_lg = L.dict_pass_lg; a.dict_pass = L.dict_pass;
  kern<<<L.blocks, THREADS, L.smem_bytes, s>>>(a);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

template <int KK, int SIG>
int launch_fb(const AggLaunch& L, cudaStream_t s) {
  if (L.back != BACK_DIRECT) return EIGER_ERR_ARG;
  switch (L.front) {
    case FRONT_NONE: return launch_one<KK, SIG, FRONT_NONE>(L, s);
    case FRONT_PRIV: return launch_one<KK, SIG, FRONT_PRIV>(L, s);
    case FRONT_SDIRECT: return L.threads == kAggThreadsWide ? launch_one<KK, SIG, FRONT_SDIRECT, kAggThreadsWide>(L, s)
                                                            : launch_one<KK, SIG, FRONT_SDIRECT>(L, s);
    case FRONT_DICT:
      if constexpr (sizeof(typename KeyTraits<KK>::U) == 4 && (SIG == SIG_SC || SIG == SIG_SC32)) {
        if (L.dict_compact && L.dict_pass_lg > 0) return launch_one<KK, SIG, FRONT_DICTP, kAggThreadsWide>(L, s);
        if (L.dict_compact) return launch_one<KK, SIG, FRONT_DICTC, kAggThreadsWide>(L, s);
        if (L.dict_group == 2) return launch_one<KK, SIG, FRONT_DICTG, kAggThreadsWide>(L, s);
      }
      if (L.dict_compact) return EIGER_ERR_ARG;
      if constexpr (sizeof(typename KeyTraits<KK>::U) == 4) return launch_one<KK, SIG, FRONT_DICT, kAggThreadsWide>(L, s);
      else return EIGER_ERR_ARG;
    default: return EIGER_ERR_ARG;
  }
}

template <int KK>
int launch_sig(const AggLaunch& L, cudaStream_t s) {
  switch (L.sig) {
    case SIG_GENERIC: case SIG_G1: return launch_fb<KK, SIG_GENERIC>(L, s);      // (SIG_G1 has its own kernels in hashagg.cuh only)
    case SIG_SC: return launch_fb<KK, SIG_SC>(L, s);
    case SIG_A4I: return launch_fb<KK, SIG_A4I>(L, s);
    case SIG_A4F: return launch_fb<KK, SIG_A4F>(L, s);
    case SIG_S4C: return launch_fb<KK, SIG_S4C>(L, s);
    case SIG_SC32: return launch_fb<KK, SIG_SC32>(L, s);
    default: return EIGER_ERR_ARG;
  }
}

}  // namespace

bool aggregate_supported(int key_kind, int sig, int front, int back) {
  (void)sig;
  return back == BACK_DIRECT && key_kind != KK_U64PRE && key_kind != KK_U32PRE &&
         (front == FRONT_NONE || front == FRONT_PRIV || front == FRONT_SDIRECT || front == FRONT_DICT);
}

int launch_aggregate(const AggLaunch& L, cudaStream_t s) {
  if (L.threads != kAggThreads && !(L.threads == kAggThreadsWide && (L.front == FRONT_SDIRECT || L.front == FRONT_DICT))) return EIGER_ERR_ARG;
  switch (L.key_kind) {
    case KK_I32: return launch_sig<KK_I32>(L, s);
    case KK_I64: return launch_sig<KK_I64>(L, s);
    case KK_I8I8: return launch_sig<KK_I8I8>(L, s);
    case KK_GEN: return launch_sig<KK_GEN>(L, s);
    case KK_GEN32: return launch_sig<KK_GEN32>(L, s);
    default: return EIGER_ERR_ARG;
  }
}

int launch_dict_build(const AggLaunch& L, int64_t samples, uint32_t* dict_keys, uint32_t* dict_n, cudaStream_t s) {
  // (L.dict_pass_lg > 0: 2^dict_pass_lg images / id ranges / counters, one per key slice)
  EIGER_CUDA(cudaMemsetAsync(L.dict, 0xFF, ((size_t)L.dict_slots * 8) << L.dict_pass_lg, s));
  EIGER_CUDA(cudaMemsetAsync(dict_n, 0, (size_t)4 << L.dict_pass_lg, s));
  KeyDesc k = L.key;
  k.flags &= ~kKey32;      // 64-bit fusion here (one thread per sampled row: speed is irrelevant), the marker stays ~0ull
  dict_build_kernel<<<(unsigned)((samples + 255) / 256), 256, 0, s>>>(k, L.n, samples, static_cast<uint2*>(L.dict), L.dict_slots, L.dict_shift,
                                                                       L.front_slots, dict_keys, dict_n, L.call, L.dict_pass_lg, L.dict_compact ? 4u : (L.dict_group == 2 ? 2u : 1u));
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

int launch_table_init(const AggLaunch& L, cudaStream_t s) {
  const bool hash = L.back == BACK_HASH;
  const uint64_t slots = L.cap + (hash ? 1 : 0);
  const uint32_t wps = L.stride / 8;
  const uint64_t n_words = slots * wps;
  bool all_zero = !hash;
  for (int j = 0; j < L.plan.n_acc; ++j) all_zero = all_zero && (L.plan.op[j] == EIGER_SUM || L.plan.op[j] == EIGER_COUNT);
  if (all_zero) {
    EIGER_CUDA(cudaMemsetAsync(L.table, 0, n_words * 8, s));
    return EIGER_OK;
  }
  const int blocks = (int)std::max<uint64_t>(1, std::min<uint64_t>((n_words + 255) / 256, 148ull * 16));
  table_init_kernel<<<blocks, 256, 0, s>>>(static_cast<uint64_t*>(L.table), n_words, wps, hash ? 1 : 0, L.plan);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

int launch_compact(const CompactLaunch& c, int sm_count, cudaStream_t s) {
  CompactArgs a;
  a.key = c.key; a.plan = c.plan; a.table = static_cast<const unsigned char*>(c.table);
  a.cap = c.cap; a.stride = c.stride; a.back = c.back;
  for (int k = 0; k < kMaxKeyCols; ++k) a.out_keys[k] = c.out_keys[k];
  for (int j = 0; j < kMaxAggs; ++j) a.out_aggs[j] = static_cast<uint64_t*>(c.out_aggs[j]);
  a.n_out = c.n_out_aggs; a.out_capacity = c.out_capacity; a.call = c.call; a.R = c.R; a.dict_keys = c.dict_keys;
  const uint64_t n_slots = c.cap + 1;
  const int blocks = (int)std::max<uint64_t>(1, std::min<uint64_t>((n_slots + 255) / 256, (uint64_t)sm_count * 8));
  compact_kernel<<<blocks, 256, 0, s>>>(a);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

}  // namespace eiger
