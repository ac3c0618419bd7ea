// Step A6b / A6c / second half of A6d: hash aggregation with a per-CTA open-addressing table
// in shared memory in front of the global table.
//
//   whole-input mode  (EIGER_SMEM, EIGER_GLOBAL): every CTA streams its share of the rows into
//       its own shared-memory table; rows whose key finds no room there go straight to the
//       global table (L2 atomics); at the end each CTA merges its occupied slots into the
//       global table, which compaction (A7) then reads.
//   partition mode    (EIGER_PARTITION): the rows were reordered by partition.cu so that each
//       partition holds a disjoint set of keys; one CTA owns a partition, aggregates it in
//       shared memory and EMITS its groups straight into the output columns (A7 fused; no
//       global table, no init, no compaction pass).  Keys that do not fit go to the global
//       table as before and are appended by the compaction kernel.
//
// Shared memory is where this hardware aggregates fast: three native 32-bit ATOMS per row
// sustain ~880 G rows/s chip-wide (measured), L2 atomics ~190 G/s in total.
// PAPER.md:79 §3.3 (hash group-by, partitioned hash group-by); PAPER.md:23 ("perform well when
// the hash table is cache-resident"); PAPER.md:184 (retrieveAll).
#include <algorithm>

#include "internal.h"
#include "rows.cuh"

namespace eiger {
namespace {

constexpr int kMaxThreads = 1024;

struct HashAggArgs {
  KeyDesc key;
  AggPlan plan;
  int64_t n;
  const unsigned long long* part_off;   // partition mode: [n_parts + 1] row offsets
  int32_t n_parts;
  uint32_t slots;        // shared-memory slots per CTA (any number >= 64)
  uint32_t limit;        // stop inserting new keys beyond this many
  int32_t spec;          // speculative: a full table raises call->abort and everybody stops
  void* table; uint64_t cap; uint32_t stride;   // global table
  CallDev* call;
  void* out_keys[2]; uint64_t* out_aggs[kMaxAggs]; int32_t n_out; int64_t out_capacity;
};

template <int KK> struct IsPre { static constexpr bool v = (KK == KK_U32PRE || KK == KK_U64PRE); };

// plane width of accumulator (op, f64) in the shared-memory table: COUNT keeps 32 bits (a CTA
// never sees 2^32 rows of one key: api.cu guards n), everything else 64
__device__ __forceinline__ uint32_t plane_width(int op) { return op == EIGER_COUNT ? 4u : 8u; }

template <int KK, int SIG>
struct Front {
  using U = typename KeyTraits<KK>::U;
  using S = Sig<SIG>;
  static constexpr int NV = S::kVals;
  static constexpr int NA = S::kAcc;

  const HashAggArgs& a;
  unsigned char* smem;
  const int n_acc;
  const uint32_t Sn;      // slots in use (<= a.slots)
  U* skeys;

  __device__ Front(const HashAggArgs& args, unsigned char* sm, uint32_t slots_used)
      : a(args), smem(sm), n_acc(S::kStatic ? S::kAcc : args.plan.n_acc), Sn(slots_used) {
    uint32_t w = 0;
#pragma unroll
    for (int j = 0; j < NA; ++j) { if (!S::kStatic && j >= n_acc) break; w += plane_width(sig_op<SIG>(a.plan, j)); }
    skeys = reinterpret_cast<U*>(smem + (size_t)w * a.slots);   // planes are laid out for a.slots
  }

  __device__ void init(int tid, int T) {
    uint32_t off = 0;
#pragma unroll
    for (int j = 0; j < NA; ++j) {
      if (!S::kStatic && j >= n_acc) break;
      const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
      if (op == EIGER_COUNT) {
        uint32_t* p = reinterpret_cast<uint32_t*>(smem + (size_t)off * a.slots);
        for (uint32_t c = tid; c < Sn; c += T) p[c] = 0u;
      } else if (add_type(op, f)) {
        uint32_t* p = reinterpret_cast<uint32_t*>(smem + (size_t)off * a.slots);
        for (uint32_t c = tid; c < Sn; c += T) { p[c] = 0u; p[c + a.slots] = 0u; }
      } else {
        uint64_t* p = reinterpret_cast<uint64_t*>(smem + (size_t)off * a.slots);
        const uint64_t v = op == EIGER_SUM ? 0ull : acc_identity(op);
        for (uint32_t c = tid; c < Sn; c += T) p[c] = v;
      }
      off += plane_width(op);
    }
    for (uint32_t c = tid; c < Sn; c += T) skeys[c] = empty_of<U>();
  }

  __device__ __forceinline__ uint32_t home(U u) const {
    if constexpr (sizeof(U) == 4) return __umulhi(table_hash32b((uint32_t)u), Sn);
    else return __umulhi((uint32_t)table_hash64((uint64_t)u), Sn);   // low word: the top bits chose the partition
  }

  // find-or-insert in the shared-memory table; single exit.  Returns the slot or -1.
  __device__ __forceinline__ int find(U u, uint32_t* s_count) {
    int res = -1;
    bool done = false;
    if constexpr (sizeof(U) == 8) { if (u == kEmpty64) done = true; }
    uint32_t h = home(u);
    int probes = 0;
    while (!done) {
      U k = *reinterpret_cast<volatile U*>(skeys + h);
      if (k == empty_of<U>()) {
        if (*reinterpret_cast<volatile uint32_t*>(s_count) >= a.limit) { done = true; }
        else {
          if constexpr (sizeof(U) == 4) k = atomicCAS(skeys + h, kEmpty32, u);
          else k = (U)atomicCAS(reinterpret_cast<unsigned long long*>(skeys + h), (unsigned long long)kEmpty64, (unsigned long long)u);
          if (k == empty_of<U>()) { atomicAdd(s_count, 1u); k = u; }
        }
      }
      if (!done) {
        if (k == u) { res = (int)h; done = true; }
        else { h = h + 1 == Sn ? 0 : h + 1; if (++probes >= 64) done = true; }
      }
    }
    return res;
  }

  __device__ __forceinline__ void update(uint32_t h, const uint64_t (&raw)[NV]) {
    uint32_t off = 0;
#pragma unroll
    for (int j = 0; j < NA; ++j) {
      if (!S::kStatic && j >= n_acc) break;
      const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
      unsigned char* plane = smem + (size_t)off * a.slots;
      if (op == EIGER_COUNT) {
        atomicAdd(reinterpret_cast<uint32_t*>(plane) + h, 1u);
      } else {
        const uint64_t part = row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]);
        if (add_type(op, f)) {
          uint32_t* lo = reinterpret_cast<uint32_t*>(plane) + h;
          smem_add64(lo, lo + a.slots, part);
        } else if (op == EIGER_SUM) {
          atomicAdd(reinterpret_cast<double*>(plane) + h, __longlong_as_double((long long)part));
        } else {
          long long* cell = reinterpret_cast<long long*>(plane) + h;
          const long long cur = *reinterpret_cast<volatile long long*>(cell);
          if (op == EIGER_MIN) { if ((long long)part < cur) atomicMin(cell, (long long)part); }
          else { if ((long long)part > cur) atomicMax(cell, (long long)part); }
        }
      }
      off += plane_width(op);
    }
  }

  // accumulator j of slot h in partial form (64 bits)
  __device__ __forceinline__ uint64_t read(uint32_t h, int j, uint32_t off) const {
    const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
    const unsigned char* plane = smem + (size_t)off * a.slots;
    if (op == EIGER_COUNT) return (uint64_t)(reinterpret_cast<const uint32_t*>(plane)[h]);
    if (add_type(op, f)) { const uint32_t* lo = reinterpret_cast<const uint32_t*>(plane) + h; return ((uint64_t)lo[a.slots] << 32) | lo[0]; }
    return reinterpret_cast<const uint64_t*>(plane)[h];
  }

  __device__ __forceinline__ void back_row(U u, const uint64_t (&raw)[NV]) {
    uint64_t* cells = back_find_or_insert(a.table, a.cap, a.stride, (uint64_t)u, a.call);
    if (cells) {
#pragma unroll
      for (int j = 0; j < NA; ++j) {
        if (!S::kStatic && j >= n_acc) break;
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        atomic_merge(cells + j, op, f, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
      }
    }
  }

  __device__ __forceinline__ void row(U u, const uint64_t (&raw)[NV], uint32_t* s_count, bool& missed) {
    const int h = find(u, s_count);
    if (h >= 0) update((uint32_t)h, raw);
    else if (a.spec) missed = true;
    else back_row(u, raw);
  }

  // merge every occupied slot into the global table
  __device__ void flush_merge(int tid, int T) {
    for (uint32_t h = tid; h < Sn; h += T) {
      const U k = skeys[h];
      if (k == empty_of<U>()) continue;
      uint64_t* cells = back_find_or_insert(a.table, a.cap, a.stride, (uint64_t)k, a.call);
      if (!cells) continue;
      uint32_t off = 0;
      for (int j = 0; j < n_acc; ++j) {
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        const uint64_t v = read(h, j, off);
        off += plane_width(op);
        if (v == acc_identity(op) && !(op == EIGER_SUM && f)) continue;
        atomic_merge(cells + j, op, f, v);
      }
    }
  }

  // write every occupied slot as one output group (the CTA owns these keys exclusively)
  __device__ void flush_emit(int tid, int T, uint32_t n_keys, unsigned long long* s_base, uint32_t* s_cursor) {
    if (tid == 0) { *s_base = n_keys ? atomicAdd(&a.call->n_groups, (unsigned long long)n_keys) : 0ull; *s_cursor = 0u; }
    __syncthreads();
    const unsigned long long base = *s_base;
    const int lane = tid & 31;
    for (uint32_t h0 = tid - lane; h0 < Sn; h0 += T) {      // warp-uniform trip count
      const uint32_t h = h0 + lane;
      const U k = h < Sn ? skeys[h] : empty_of<U>();
      const bool occ = k != empty_of<U>();
      const uint32_t m = __ballot_sync(0xffffffffu, occ);
      if (m == 0) continue;
      uint32_t start = 0;
      if (lane == 0) start = atomicAdd(s_cursor, (uint32_t)__popc(m));
      start = __shfl_sync(0xffffffffu, start, 0);
      if (!occ) continue;
      const uint64_t g = base + start + __popc(m & ((1u << lane) - 1u));
      if ((int64_t)g >= a.out_capacity) continue;
      store_group_key(a.key, a.out_keys, (uint64_t)k, g);
      uint32_t off = 0;
      for (int j = 0; j < a.n_out; ++j) {
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        a.out_aggs[j][g] = acc_finalize(op, f, read(h, j, off));
        off += plane_width(op);
      }
    }
  }
};

template <int KK, int SIG>
__global__ void __launch_bounds__(kMaxThreads, 1)
hash_agg_kernel(const __grid_constant__ HashAggArgs a) {
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ uint32_t s_count, s_cursor, s_abort;
  __shared__ unsigned long long s_base;
  using F = Front<KK, SIG>;
  using U = typename F::U;
  constexpr int NV = F::NV;
  const int tid = threadIdx.x, T = blockDim.x;
  const int n_vals = Sig<SIG>::kStatic ? NV : a.plan.n_vals;

  if constexpr (!IsPre<KK>::v) {
    // ---- whole-input mode: tiles of 2 * T * UNR rows, grid-strided ----
    constexpr int UNR = !Sig<SIG>::kStatic ? 1 : 2;
    F f(a, smem, a.slots);
    if (tid == 0) { s_count = 0; s_abort = 0; }
    f.init(tid, T);
    __syncthreads();
    const int64_t step = 2 * (int64_t)T, tile = step * UNR;
    const int64_t n_tiles = a.n / tile;
    bool missed = false;
    for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
      if (a.spec) { if (missed || *reinterpret_cast<volatile uint32_t*>(&a.call->abort)) break; }
      const int64_t r0 = t * tile + 2 * tid;
      U u[UNR][2];
      uint64_t raw[UNR][2][NV];
#pragma unroll
      for (int s = 0; s < UNR; ++s) {
        load_u2<KK>(a.key, r0 + s * step, u[s]);
#pragma unroll
        for (int c = 0; c < NV; ++c) {
          if (!Sig<SIG>::kStatic && c >= n_vals) { raw[s][0][c] = 0; raw[s][1][c] = 0; continue; }
          const uint4 v = ldg_stream_16(static_cast<const uint64_t*>(a.plan.vals[c]) + r0 + s * step);
          raw[s][0][c] = ((uint64_t)v.y << 32) | v.x; raw[s][1][c] = ((uint64_t)v.w << 32) | v.z;
        }
      }
#pragma unroll
      for (int s = 0; s < UNR; ++s) { f.row(u[s][0], raw[s][0], &s_count, missed); f.row(u[s][1], raw[s][1], &s_count, missed); }
    }
    if (!(a.spec && missed)) {
      for (int64_t i = n_tiles * tile + (int64_t)blockIdx.x * T + tid; i < a.n; i += (int64_t)gridDim.x * T) {
        uint64_t raw[NV];
#pragma unroll
        for (int c = 0; c < NV; ++c) raw[c] = (Sig<SIG>::kStatic || c < n_vals) ? ldg_stream_u64(static_cast<const uint64_t*>(a.plan.vals[c]) + i) : 0ull;
        f.row(load_u<KK>(a.key, i), raw, &s_count, missed);
      }
    }
    if (a.spec) {
      if (missed) { atomicOr(&a.call->abort, 1u); atomicOr(&s_abort, 1u); }
      __syncthreads();
      if (s_abort || *reinterpret_cast<volatile uint32_t*>(&a.call->abort)) return;   // result is discarded
    } else {
      __syncthreads();
    }
    f.flush_merge(tid, T);
  } else {
    // ---- partition mode: this CTA owns partitions blockIdx.x, + gridDim.x, ... ----
    for (int p = blockIdx.x; p < a.n_parts; p += gridDim.x) {
      const int64_t r0 = (int64_t)a.part_off[p], r1 = (int64_t)a.part_off[p + 1];
      if (r1 <= r0) continue;
      // a table no larger than the partition needs: 2 slots per row is always enough
      const uint64_t want = 2ull * (uint64_t)(r1 - r0) + 64;
      const uint32_t Sn = (uint32_t)(want < a.slots ? want : a.slots);
      F f(a, smem, Sn);
      __syncthreads();                       // the previous partition's emit is over
      if (tid == 0) s_count = 0;
      f.init(tid, T);
      __syncthreads();
      bool missed = false;
      constexpr int UNR = 4;
      int64_t i = r0 + tid;
      for (; i + (int64_t)(UNR - 1) * T < r1; i += (int64_t)UNR * T) {
        U u[UNR];
        uint64_t raw[UNR][NV];
#pragma unroll
        for (int s = 0; s < UNR; ++s) {
          u[s] = load_u<KK>(a.key, i + (int64_t)s * T);
#pragma unroll
          for (int c = 0; c < NV; ++c) raw[s][c] = (Sig<SIG>::kStatic || c < n_vals) ? ldg_stream_u64(static_cast<const uint64_t*>(a.plan.vals[c]) + i + (int64_t)s * T) : 0ull;
        }
#pragma unroll
        for (int s = 0; s < UNR; ++s) f.row(u[s], raw[s], &s_count, missed);
      }
      for (; i < r1; i += T) {
        uint64_t raw[NV];
#pragma unroll
        for (int c = 0; c < NV; ++c) raw[c] = (Sig<SIG>::kStatic || c < n_vals) ? ldg_stream_u64(static_cast<const uint64_t*>(a.plan.vals[c]) + i) : 0ull;
        f.row(load_u<KK>(a.key, i), raw, &s_count, missed);
      }
      __syncthreads();
      f.flush_emit(tid, T, s_count, &s_base, &s_cursor);
    }
  }
}

template <int KK, int SIG>
int launch_one(const HashAggLaunch& L, cudaStream_t s) {
  auto kern = hash_agg_kernel<KK, SIG>;
  if (L.smem_bytes > 48 * 1024) EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem_bytes));
  HashAggArgs a;
  a.key = L.key; a.plan = L.plan; a.n = L.n; a.part_off = L.part_off; a.n_parts = L.n_parts;
  a.slots = L.slots; a.limit = L.limit; a.spec = L.spec;
  a.table = L.table; a.cap = L.cap; a.stride = L.stride; a.call = L.call;
  a.out_keys[0] = L.out_keys[0]; a.out_keys[1] = L.out_keys[1];
  for (int j = 0; j < kMaxAggs; ++j) a.out_aggs[j] = static_cast<uint64_t*>(L.out_aggs[j]);
  a.n_out = L.n_out_aggs; a.out_capacity = L.out_capacity;
  kern<<<L.blocks, L.threads, L.smem_bytes, s>>>(a);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

template <int KK>
int launch_sig(const HashAggLaunch& L, cudaStream_t s) {
  switch (L.sig) {
    case SIG_GENERIC: return launch_one<KK, SIG_GENERIC>(L, s);
    case SIG_SC: return launch_one<KK, SIG_SC>(L, s);
    case SIG_A4I: return launch_one<KK, SIG_A4I>(L, s);
    case SIG_A4F: return launch_one<KK, SIG_A4F>(L, s);
    case SIG_S4C: return launch_one<KK, SIG_S4C>(L, s);
    default: return EIGER_ERR_ARG;
  }
}

}  // namespace

size_t hash_agg_slot_bytes(const AggPlan& p, int key_kind) {
  size_t w = (key_kind == KK_I32 || key_kind == KK_U32PRE) ? 4 : 8;
  for (int j = 0; j < p.n_acc; ++j) w += p.op[j] == EIGER_COUNT ? 4 : 8;
  return w;
}

int launch_hash_agg(const HashAggLaunch& L, cudaStream_t s) {
  if (L.threads < 32 || L.threads > kMaxThreads || (L.threads & 31) || L.slots < 64) return EIGER_ERR_ARG;
  switch (L.key_kind) {
    case KK_I32: return launch_sig<KK_I32>(L, s);
    case KK_I64: return launch_sig<KK_I64>(L, s);
    case KK_GEN: return launch_sig<KK_GEN>(L, s);
    case KK_U32PRE: return launch_sig<KK_U32PRE>(L, s);
    case KK_U64PRE: return launch_sig<KK_U64PRE>(L, s);
    default: return EIGER_ERR_ARG;
  }
}

}  // namespace eiger
