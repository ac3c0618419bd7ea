// Steps A5-A7: table init, the aggregation kernels (all four variants are one kernel
// template over a FRONT — what a CTA keeps in shared memory — and a BACK — the table in
// global memory / L2), and compaction.
//
//   EIGER_DIRECT    BACK_DIRECT (slot = u) with FRONT_PRIV (per-thread private cells, no
//                   atomics; tiny ranges), FRONT_SDIRECT (per-CTA shared-memory array) or
//                   FRONT_NONE (global atomics only; ranges beyond shared memory)
//   EIGER_SMEM      FRONT_SHASH (per-CTA open addressing in shared memory) + BACK_HASH
//   EIGER_GLOBAL    FRONT_NONE or a small FRONT_SHASH hot-key cache + BACK_HASH
//   EIGER_PARTITION partition.cu reorders the rows, then BACK_HASH over KK_U64PRE keys
//
// GROUP BY semantics: §3.3; hash group-by "perform well when the hash table is
// cache-resident" PAPER.md:23; emit groups = HT.retrieveAll PAPER.md:184.
#include <algorithm>

#include "internal.h"

namespace eiger {
namespace {

constexpr int kAggThreads = 256;
constexpr int kFrontProbes = 8;
constexpr int kBackProbes = 4096;

template <int KK> struct KeyTraits;
template <> struct KeyTraits<KK_I32> { using U = uint32_t; };
template <> struct KeyTraits<KK_I8I8> { using U = uint32_t; };
template <> struct KeyTraits<KK_I64> { using U = uint64_t; };
template <> struct KeyTraits<KK_GEN> { using U = uint64_t; };
template <> struct KeyTraits<KK_U64PRE> { using U = uint64_t; };

template <class U> __device__ __forceinline__ U empty_of();
template <> __device__ __forceinline__ uint32_t empty_of<uint32_t>() { return kEmpty32; }
template <> __device__ __forceinline__ uint64_t empty_of<uint64_t>() { return kEmpty64; }

// ---- key loading ---------------------------------------------------------------------
template <int KK>
__device__ __forceinline__ typename KeyTraits<KK>::U load_u(const KeyDesc& k, int64_t i) {
  using U = typename KeyTraits<KK>::U;
  if constexpr (KK == KK_I32) {
    return (U)(ldg_stream_4((const int32_t*)k.ptr[0] + i) - (uint32_t)k.base[0]);
  } else if constexpr (KK == KK_I64) {
    return ldg_stream_u64((const int64_t*)k.ptr[0] + i) - k.base[0];
  } else if constexpr (KK == KK_U64PRE) {
    return ldg_stream_u64((const uint64_t*)k.ptr[0] + i);
  } else if constexpr (KK == KK_I8I8) {
    const uint32_t a = (uint32_t)(int32_t)(int8_t)ldg_stream_1((const int8_t*)k.ptr[0] + i) - (uint32_t)k.base[0];
    const uint32_t b = (uint32_t)(int32_t)(int8_t)ldg_stream_1((const int8_t*)k.ptr[1] + i) - (uint32_t)k.base[1];
    return a * (uint32_t)k.mul + b;
  } else {
    uint64_t u = sext_load(k.ptr[0], k.dtype[0], i) - k.base[0];
    if (k.ncols == 2) u = u * k.mul + (sext_load(k.ptr[1], k.dtype[1], i) - k.base[1]);
    return u;
  }
}
// two consecutive rows starting at an even row index (vector loads)
template <int KK>
__device__ __forceinline__ void load_u2(const KeyDesc& k, int64_t i, typename KeyTraits<KK>::U (&u)[2]) {
  if constexpr (KK == KK_I32) {
    const uint2 v = ldg_stream_8((const int32_t*)k.ptr[0] + i);
    u[0] = v.x - (uint32_t)k.base[0]; u[1] = v.y - (uint32_t)k.base[0];
  } else if constexpr (KK == KK_I64 || KK == KK_U64PRE) {
    const uint4 v = ldg_stream_16((const uint64_t*)k.ptr[0] + i);
    const uint64_t b = KK == KK_I64 ? k.base[0] : 0ull;
    u[0] = (((uint64_t)v.y << 32) | v.x) - b; u[1] = (((uint64_t)v.w << 32) | v.z) - b;
  } else if constexpr (KK == KK_I8I8) {
    const uint32_t a = ldg_stream_2((const int8_t*)k.ptr[0] + i), b = ldg_stream_2((const int8_t*)k.ptr[1] + i);
    const uint32_t b0 = (uint32_t)k.base[0], b1 = (uint32_t)k.base[1], m = (uint32_t)k.mul;
    u[0] = ((uint32_t)(int32_t)(int8_t)(a & 0xFF) - b0) * m + ((uint32_t)(int32_t)(int8_t)(b & 0xFF) - b1);
    u[1] = ((uint32_t)(int32_t)(int8_t)(a >> 8) - b0) * m + ((uint32_t)(int32_t)(int8_t)(b >> 8) - b1);
  } else {
    u[0] = load_u<KK>(k, i); u[1] = load_u<KK>(k, i + 1);
  }
}

// ---- the global hash table (BACK_HASH) -------------------------------------------------
// Slot s lives at table + s * stride: [u64 key][acc 0]..[acc n-1][pad]; key = ~0 means empty.
// Slot `cap` is the side slot of the one key whose rebased value equals the empty marker
// (R18).  Returns the slot's accumulator cells, or nullptr when probing gave up.
__device__ __forceinline__ uint64_t* back_hash_cells(void* table, uint64_t cap, uint32_t stride,
                                                     uint64_t u, CallDev* call) {
  if (u == kEmpty64) {
    uint64_t* kp = reinterpret_cast<uint64_t*>(static_cast<char*>(table) + cap * stride);
    if (__ldcg(kp) != 0ull) atomicExch(reinterpret_cast<unsigned long long*>(kp), 0ull);  // mark used
    return kp + 1;
  }
  uint64_t slot = __umul64hi(table_hash64(u), cap);
  for (int probe = 0; probe < kBackProbes; ++probe) {
    uint64_t* kp = reinterpret_cast<uint64_t*>(static_cast<char*>(table) + slot * stride);
    const uint64_t k = __ldcg(kp);
    if (k == u) return kp + 1;
    if (k == kEmpty64) {
      const uint64_t old = atomicCAS(reinterpret_cast<unsigned long long*>(kp), kEmpty64, u);
      if (old == kEmpty64 || old == u) return kp + 1;
    }
    slot = slot + 1 == cap ? 0 : slot + 1;
  }
  atomicOr(&call->overflow, 1u);
  return nullptr;
}

// ---- shared-memory accumulators ------------------------------------------------------------
// B200 shared memory has native 32-bit atomics (ATOMS.ADD / ATOMS.MAX, ~2 T/s chip-wide,
// measured) but 64-bit ones are CAS loops (~0.1-0.3 T/s).  Integer SUM and COUNT cells are
// therefore kept as two 32-bit planes, lo[S] then hi[S], and added with an explicit carry:
// the final (hi:lo) equals the wrapping 64-bit sum whatever the interleaving, because every
// wrap of lo is seen by exactly one atomicAdd's return value.  MIN / MAX and fp64 SUM keep
// 64-bit cells; MIN / MAX look before they leap, so the CAS loop only runs on a new record.
__device__ __forceinline__ bool add_type(int op, bool f64) { return op == EIGER_COUNT || (op == EIGER_SUM && !f64); }
__device__ __forceinline__ void smem_add64(uint32_t* lo, uint32_t* hi, uint64_t v) {
  const uint32_t vl = (uint32_t)v;
  const uint32_t old = atomicAdd(lo, vl);
  const uint32_t h = (uint32_t)(v >> 32) + ((uint32_t)(old + vl) < vl ? 1u : 0u);
  if (h) atomicAdd(hi, h);
}
// accumulator j of a table of S slots that starts at base occupies 8 * S bytes
__device__ __forceinline__ void smem_merge(unsigned char* base, uint32_t S, int j, uint32_t s, int op, bool f64, uint64_t part) {
  unsigned char* plane = base + (size_t)j * 8 * S;
  if (add_type(op, f64)) {
    uint32_t* lo = reinterpret_cast<uint32_t*>(plane) + s;
    smem_add64(lo, lo + S, part);
  } else if (op == EIGER_SUM) {
    atomicAdd(reinterpret_cast<double*>(plane) + s, __longlong_as_double((long long)part));
  } else {
    long long* cell = reinterpret_cast<long long*>(plane) + s;
    const long long cur = *reinterpret_cast<volatile long long*>(cell);
    if (op == EIGER_MIN) { if ((long long)part < cur) atomicMin(cell, (long long)part); }
    else { if ((long long)part > cur) atomicMax(cell, (long long)part); }
  }
}
__device__ __forceinline__ uint64_t smem_read(const unsigned char* base, uint32_t S, int j, uint32_t s, int op, bool f64) {
  const unsigned char* plane = base + (size_t)j * 8 * S;
  if (add_type(op, f64)) {
    const uint32_t* lo = reinterpret_cast<const uint32_t*>(plane) + s;
    return ((uint64_t)lo[S] << 32) | lo[0];
  }
  return reinterpret_cast<const uint64_t*>(plane)[s];
}
__device__ __forceinline__ void smem_init_plane(unsigned char* base, uint32_t S, int j, int op, bool f64, int tid, int T) {
  uint64_t* plane = reinterpret_cast<uint64_t*>(base + (size_t)j * 8 * S);
  const uint64_t v = add_type(op, f64) ? 0ull : acc_identity(op);
  for (uint32_t c = tid; c < S; c += T) plane[c] = v;
}

struct AggArgs {
  KeyDesc key;
  AggPlan plan;
  int64_t n;
  uint32_t front_slots, front_limit, front_replicas, stride;
  void* table;
  uint64_t cap;
  CallDev* call;
};

template <int SIG> __device__ __forceinline__ int sig_op(const AggPlan& p, int j) { if constexpr (Sig<SIG>::kStatic) return Sig<SIG>::op(j); else return p.op[j]; }
template <int SIG> __device__ __forceinline__ int sig_col(const AggPlan& p, int j) { if constexpr (Sig<SIG>::kStatic) return Sig<SIG>::col(j); else return p.col[j]; }
template <int SIG> __device__ __forceinline__ bool sig_f64(const AggPlan& p, int j) { if constexpr (Sig<SIG>::kStatic) return Sig<SIG>::f64(j); else return p.f64[j] != 0; }

template <int KK, int SIG, int FRONT, int BACK>
struct AggCtx {
  using U = typename KeyTraits<KK>::U;
  using S = Sig<SIG>;
  static constexpr int NV = S::kVals;
  static constexpr int NA = S::kAcc;

  const AggArgs& a;
  const int n_acc;
  unsigned char* smem;
  // FRONT_SHASH views
  U* skeys; uint64_t* sacc; uint32_t* scount;

  __device__ AggCtx(const AggArgs& args, unsigned char* sm)
      : a(args), n_acc(S::kStatic ? S::kAcc : args.plan.n_acc), smem(sm) {
    if constexpr (FRONT == FRONT_SHASH) {
      sacc = reinterpret_cast<uint64_t*>(smem);
      skeys = reinterpret_cast<U*>(sacc + (size_t)n_acc * a.front_slots);
      scount = reinterpret_cast<uint32_t*>(skeys + a.front_slots);
    }
  }

  __device__ void front_init() {
    const int tid = threadIdx.x, T = blockDim.x;
    if constexpr (FRONT == FRONT_PRIV) {
      uint64_t* acc = reinterpret_cast<uint64_t*>(smem);
      for (uint32_t c = 0; c < a.front_slots * (uint32_t)n_acc; ++c)
        acc[(size_t)c * T + tid] = acc_identity(sig_op<SIG>(a.plan, (int)(c % (uint32_t)n_acc)));
    } else if constexpr (FRONT == FRONT_SDIRECT) {
      for (uint32_t rep = 0; rep < a.front_replicas; ++rep)
        for (int j = 0; j < n_acc; ++j)
          smem_init_plane(smem + (size_t)rep * a.front_slots * 8 * (uint32_t)n_acc, a.front_slots, j, sig_op<SIG>(a.plan, j), sig_f64<SIG>(a.plan, j), tid, T);
    } else if constexpr (FRONT == FRONT_SHASH) {
      for (uint32_t c = tid; c < a.front_slots; c += T) skeys[c] = empty_of<U>();
      for (int j = 0; j < n_acc; ++j)
        smem_init_plane(reinterpret_cast<unsigned char*>(sacc), a.front_slots, j, sig_op<SIG>(a.plan, j), sig_f64<SIG>(a.plan, j), tid, T);
      if (tid == 0) *scount = 0;
    }
    if constexpr (FRONT != FRONT_NONE) __syncthreads();
  }

  __device__ __forceinline__ int shash_find(U u) {
    const uint32_t mask = a.front_slots - 1;
    uint32_t h;
    if constexpr (sizeof(U) == 4) h = table_hash32((uint32_t)u) & mask;
    else { if (u == kEmpty64) return -1; h = (uint32_t)(table_hash64((uint64_t)u) >> 20) & mask; }
#pragma unroll 1
    for (int probe = 0; probe < kFrontProbes; ++probe) {
      const U k = *reinterpret_cast<volatile U*>(skeys + h);
      if (k == u) return (int)h;
      if (k == empty_of<U>()) {
        if (*reinterpret_cast<volatile uint32_t*>(scount) >= a.front_limit) return -1;
        U old;
        if constexpr (sizeof(U) == 4) old = atomicCAS(skeys + h, kEmpty32, u);
        else old = (U)atomicCAS(reinterpret_cast<unsigned long long*>(skeys + h), (unsigned long long)kEmpty64, (unsigned long long)u);
        if (old == empty_of<U>()) { atomicAdd(scount, 1u); return (int)h; }
        if (old == u) return (int)h;
      }
      h = (h + 1) & mask;
    }
    return -1;
  }

  __device__ __forceinline__ void back_row(U u, const uint64_t (&raw)[NV]) {
    uint64_t* cells;
    if constexpr (BACK == BACK_DIRECT) cells = static_cast<uint64_t*>(a.table) + (uint64_t)u * (uint32_t)n_acc;
    else { cells = back_hash_cells(a.table, a.cap, a.stride, (uint64_t)u, a.call); if (!cells) return; }
#pragma unroll
    for (int j = 0; j < NA; ++j) {
      if (!S::kStatic && j >= n_acc) break;
      const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
      atomic_merge(cells + j, op, f, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
    }
  }

  __device__ __forceinline__ void row(U u, const uint64_t (&raw)[NV]) {
    if constexpr (FRONT == FRONT_PRIV) {
      uint64_t* acc = reinterpret_cast<uint64_t*>(smem) + (size_t)u * (uint32_t)n_acc * blockDim.x + threadIdx.x;
#pragma unroll
      for (int j = 0; j < NA; ++j) {
        if (!S::kStatic && j >= n_acc) break;
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        uint64_t* c = acc + (size_t)j * blockDim.x;
        *c = combine(op, f, *c, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
      }
    } else if constexpr (FRONT == FRONT_SDIRECT) {
      const uint32_t rep = a.front_replicas > 1 ? (threadIdx.x >> 5) % a.front_replicas : 0u;
      unsigned char* base = smem + (size_t)rep * a.front_slots * 8 * (uint32_t)n_acc;
#pragma unroll
      for (int j = 0; j < NA; ++j) {
        if (!S::kStatic && j >= n_acc) break;
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        smem_merge(base, a.front_slots, j, (uint32_t)u, op, f, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
      }
    } else if constexpr (FRONT == FRONT_SHASH) {
      const int h = shash_find(u);
      if (h < 0) { back_row(u, raw); return; }
#pragma unroll
      for (int j = 0; j < NA; ++j) {
        if (!S::kStatic && j >= n_acc) break;
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        smem_merge(reinterpret_cast<unsigned char*>(sacc), a.front_slots, j, (uint32_t)h, op, f, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
      }
    } else {
      back_row(u, raw);
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
    } else if constexpr (FRONT == FRONT_SDIRECT) {
      const uint32_t per = a.front_slots * (uint32_t)n_acc, tot = per * a.front_replicas;
      for (uint32_t c = tid; c < tot; c += T) {
        const uint32_t rep = c / per, w = c % per, j = w / a.front_slots, u = w % a.front_slots;
        const uint64_t v = smem_read(smem + (size_t)rep * a.front_slots * 8 * (uint32_t)n_acc, a.front_slots, (int)j, u,
                                     sig_op<SIG>(a.plan, (int)j), sig_f64<SIG>(a.plan, (int)j));
        back_merge(u, (int)j, v, static_cast<uint64_t*>(a.table) + (uint64_t)u * (uint32_t)n_acc);
      }
    } else if constexpr (FRONT == FRONT_SHASH) {
      for (uint32_t h = tid; h < a.front_slots; h += T) {
        const U k = skeys[h];
        if (k == empty_of<U>()) continue;
        uint64_t* cells = back_hash_cells(a.table, a.cap, a.stride, (uint64_t)k, a.call);
        if (!cells) continue;
        for (int j = 0; j < n_acc; ++j)
          back_merge((uint64_t)k, j, smem_read(reinterpret_cast<const unsigned char*>(sacc), a.front_slots, j, h, sig_op<SIG>(a.plan, j), sig_f64<SIG>(a.plan, j)), cells);
      }
    }
  }
};

template <int KK, int SIG, int FRONT, int BACK>
__global__ void __launch_bounds__(kAggThreads)
aggregate_kernel(const __grid_constant__ AggArgs a) {
  extern __shared__ __align__(16) unsigned char smem[];
  using Ctx = AggCtx<KK, SIG, FRONT, BACK>;
  using U = typename Ctx::U;
  constexpr int NV = Ctx::NV;
  constexpr int UNR = !Sig<SIG>::kStatic ? 1 : (NV >= 4 ? 2 : 4);
  Ctx ctx(a, smem);
  ctx.front_init();

  const int tid = threadIdx.x;
  const int n_vals = Sig<SIG>::kStatic ? NV : a.plan.n_vals;
  constexpr int64_t kStep = 2 * kAggThreads, kTile = kStep * UNR;
  const int64_t n_tiles = a.n / kTile;
  for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    const int64_t r0 = t * kTile + 2 * tid;
    U u[UNR][2];
    uint64_t raw[UNR][2][NV];
#pragma unroll
    for (int s = 0; s < UNR; ++s) {
      load_u2<KK>(a.key, r0 + s * kStep, u[s]);
#pragma unroll
      for (int c = 0; c < NV; ++c) {
        if (!Sig<SIG>::kStatic && c >= n_vals) { raw[s][0][c] = 0; raw[s][1][c] = 0; continue; }
        const uint4 v = ldg_stream_16(static_cast<const uint64_t*>(a.plan.vals[c]) + r0 + s * kStep);
        raw[s][0][c] = ((uint64_t)v.y << 32) | v.x; raw[s][1][c] = ((uint64_t)v.w << 32) | v.z;
      }
    }
#pragma unroll
    for (int s = 0; s < UNR; ++s) { ctx.row(u[s][0], raw[s][0]); ctx.row(u[s][1], raw[s][1]); }
  }
  // ragged tail: row at a time, spread over the whole grid
  for (int64_t i = n_tiles * kTile + (int64_t)blockIdx.x * kAggThreads + tid; i < a.n; i += (int64_t)gridDim.x * kAggThreads) {
    uint64_t raw[NV];
#pragma unroll
    for (int c = 0; c < NV; ++c) raw[c] = (Sig<SIG>::kStatic || c < n_vals) ? ldg_stream_u64(static_cast<const uint64_t*>(a.plan.vals[c]) + i) : 0ull;
    ctx.row(load_u<KK>(a.key, i), raw);
  }
  ctx.front_flush();
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
  void* out_keys[2]; uint64_t* out_aggs[kMaxAggs]; int n_out;
  int64_t out_capacity;
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
        u = s;
      }
    }
    const uint32_t m = __ballot_sync(0xffffffffu, occ);
    if (m == 0) continue;
    unsigned long long start = 0;
    if (lane == 0) start = atomicAdd(&c.call->n_groups, (unsigned long long)__popc(m));
    start = __shfl_sync(0xffffffffu, start, 0);
    if (!occ) continue;
    const uint64_t g = start + __popc(m & ((1u << lane) - 1u));
    if ((int64_t)g >= c.out_capacity) continue;
    // un-fuse and un-rebase (PAPER.md:219-221 in reverse)
    uint64_t part[2];
    if (c.key.ncols == 2) { part[0] = u / c.key.mul; part[1] = u % c.key.mul; } else { part[0] = u; part[1] = 0; }
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
template <int KK, int SIG, int FRONT, int BACK>
int launch_one(const AggLaunch& L, cudaStream_t s) {
  auto kern = aggregate_kernel<KK, SIG, FRONT, BACK>;
  if (L.smem_bytes > 48 * 1024) EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem_bytes));
  AggArgs a;
  a.key = L.key; a.plan = L.plan; a.n = L.n;
  a.front_slots = L.front_slots; a.front_limit = L.front_limit; a.front_replicas = L.front_replicas;
  a.stride = L.stride; a.table = L.table; a.cap = L.cap; a.call = L.call;
  kern<<<L.blocks, kAggThreads, L.smem_bytes, s>>>(a);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

template <int KK, int SIG>
int launch_fb(const AggLaunch& L, cudaStream_t s) {
  if (L.back == BACK_DIRECT) {
    if constexpr (KK == KK_U64PRE) return EIGER_ERR_ARG;
    else switch (L.front) {
      case FRONT_NONE: return launch_one<KK, SIG, FRONT_NONE, BACK_DIRECT>(L, s);
      case FRONT_PRIV: return launch_one<KK, SIG, FRONT_PRIV, BACK_DIRECT>(L, s);
      case FRONT_SDIRECT: return launch_one<KK, SIG, FRONT_SDIRECT, BACK_DIRECT>(L, s);
      default: return EIGER_ERR_ARG;
    }
  } else {
    if constexpr (KK == KK_I8I8) return EIGER_ERR_ARG;
    else switch (L.front) {
      case FRONT_NONE: return launch_one<KK, SIG, FRONT_NONE, BACK_HASH>(L, s);
      case FRONT_SHASH: return launch_one<KK, SIG, FRONT_SHASH, BACK_HASH>(L, s);
      default: return EIGER_ERR_ARG;
    }
  }
}

template <int KK>
int launch_sig(const AggLaunch& L, cudaStream_t s) {
  switch (L.sig) {
    case SIG_GENERIC: return launch_fb<KK, SIG_GENERIC>(L, s);
    case SIG_SC: return launch_fb<KK, SIG_SC>(L, s);
    case SIG_A4I: return launch_fb<KK, SIG_A4I>(L, s);
    case SIG_A4F: return launch_fb<KK, SIG_A4F>(L, s);
    case SIG_S4C: return launch_fb<KK, SIG_S4C>(L, s);
    default: return EIGER_ERR_ARG;
  }
}

}  // namespace

bool aggregate_supported(int key_kind, int sig, int front, int back) {
  (void)sig;
  if (back == BACK_DIRECT) return key_kind != KK_U64PRE && front != FRONT_SHASH;
  return key_kind != KK_I8I8 && (front == FRONT_NONE || front == FRONT_SHASH);
}

int launch_aggregate(const AggLaunch& L, cudaStream_t s) {
  if (L.threads != kAggThreads) return EIGER_ERR_ARG;
  switch (L.key_kind) {
    case KK_I32: return launch_sig<KK_I32>(L, s);
    case KK_I64: return launch_sig<KK_I64>(L, s);
    case KK_I8I8: return launch_sig<KK_I8I8>(L, s);
    case KK_GEN: return launch_sig<KK_GEN>(L, s);
    case KK_U64PRE: return launch_sig<KK_U64PRE>(L, s);
    default: return EIGER_ERR_ARG;
  }
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
  a.out_keys[0] = c.out_keys[0]; a.out_keys[1] = c.out_keys[1];
  for (int j = 0; j < kMaxAggs; ++j) a.out_aggs[j] = static_cast<uint64_t*>(c.out_aggs[j]);
  a.n_out = c.n_out_aggs; a.out_capacity = c.out_capacity; a.call = c.call;
  const uint64_t n_slots = c.cap + 1;
  const int blocks = (int)std::max<uint64_t>(1, std::min<uint64_t>((n_slots + 255) / 256, (uint64_t)sm_count * 8));
  compact_kernel<<<blocks, 256, 0, s>>>(a);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

}  // namespace eiger
