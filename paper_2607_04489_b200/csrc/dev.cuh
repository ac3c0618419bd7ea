// Device-side building blocks shared by the kernels of libeiger (sm_100a).
// Nothing here is shared with oracle/: the sketch hash and the estimator are
// restated independently on each side.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/eiger.h"

namespace eiger {

constexpr int kMaxAggs = 8;            // user aggregates per call
constexpr int kMaxAcc = 9;             // + one hidden COUNT for the direct table's presence test
constexpr int kMaxVals = 8;
constexpr int kMaxKeyCols = 4;         // key columns fused into one 64-bit key
constexpr int kMaxHot = 8;              // heavy-hitter keys handled outside the hash table
constexpr int kHllP = 14;              // DESIGN.md R1
constexpr int kHllM = 1 << kHllP;
constexpr int kHllQ = 64 - kHllP;      // rho in [1, kHllQ + 1]
constexpr uint64_t kEmpty64 = ~0ull;
constexpr uint32_t kEmpty32 = ~0u;

// How the key column(s) are read.  u = rebased, fused key (frame of reference +
// positional packing): u = (..((k0 - min0) * rng1 + (k1 - min1)) * rng2 + ..),
// rng_c = max_c - min_c + 1 (mixed radix: no bits lost to rounding ranges up to powers of two).
// KK_GEN32: the generic fused key when its domain fits 32 bits, as a 32-bit value (source kind of
// the partition pass: 4-byte partitioned keys, 4-byte table slots).
enum KeyKind : int { KK_I32 = 0, KK_I64 = 1, KK_I8I8 = 2, KK_GEN = 3, KK_U64PRE = 4, KK_U32PRE = 5, KK_GEN32 = 6 };

constexpr int kKeyAll32 = 1;   // every key column is EIGER_I32: 8-byte vector loads, 32-bit rebasing
constexpr int kKey32 = 2;      // the fused domain fits 32 bits: 32-bit multiplies
struct KeyDesc {
  const void* ptr[kMaxKeyCols];
  int32_t dtype[kMaxKeyCols];
  int32_t ncols;
  int32_t flags;      // kKeyAll32 | kKey32 (generic path only)
  uint64_t base[kMaxKeyCols];   // min of each column, sign-extended, as two's complement bits
  uint64_t rng[kMaxKeyCols];    // range of each column; 1 for unused columns
  uint64_t mul;       // range of column 1 (1 for a single column): the two-column fast paths
};

// Aggregate signatures with compile-time plans (the shapes of BASELINE.json's configs);
// everything else runs the generic, plan-driven path.
enum SigKind : int {
  SIG_GENERIC = 0,
  SIG_SC = 1,    // SUM(int64 c0), COUNT                        (C4, C5)
  SIG_A4I = 2,   // SUM, COUNT, MIN, MAX of int64 c0            (C1)
  SIG_A4F = 3,   // SUM, COUNT, MIN, MAX of fp64  c0            (C3)
  SIG_S4C = 4,   // SUM(int64 c0..c3), COUNT                    (C2)
  SIG_SC32 = 5,  // SUM(int32 c0), COUNT: the paper's 4-byte payloads
  SIG_G1 = 6     // any plan of at most 4 accumulators over at most ONE value column, ops read from the plan at run time:
                 // the generic path with 1 instead of 8 value registers per row in flight (hash kernels only)
};

struct AggPlan {
  const void* vals[kMaxVals];
  int32_t n_vals;
  int32_t n_acc;            // accumulators per group (user aggregates [+ hidden COUNT])
  uint8_t op[12];
  uint8_t f64[12];
  uint8_t col[12];
  uint8_t vw[kMaxVals];     // bytes per element of value column c: 8, or 4 for EIGER_I32 (sign-extended into the 64-bit accumulators)
  int32_t cnt_acc;          // index of an accumulator that counts rows (presence test)
};

template <int SIG> struct Sig;
template <> struct Sig<SIG_GENERIC> {
  static constexpr bool kStatic = false;
  static constexpr int kAcc = kMaxAcc, kVals = kMaxVals;
  __device__ static constexpr int op(int) { return 0; }
  __device__ static constexpr int col(int) { return 0; }
  __device__ static constexpr bool f64(int) { return false; }
  __device__ static constexpr int vwidth(int) { return 8; }
};
template <> struct Sig<SIG_G1> {
  static constexpr bool kStatic = false;
  static constexpr int kAcc = 4, kVals = 1;
  __device__ static constexpr int op(int) { return 0; }
  __device__ static constexpr int col(int) { return 0; }
  __device__ static constexpr bool f64(int) { return false; }
  __device__ static constexpr int vwidth(int) { return 8; }
};
template <> struct Sig<SIG_SC> {
  static constexpr bool kStatic = true;
  static constexpr int kAcc = 2, kVals = 1;
  __device__ static constexpr int op(int j) { return j == 0 ? EIGER_SUM : EIGER_COUNT; }
  __device__ static constexpr int col(int) { return 0; }
  __device__ static constexpr bool f64(int) { return false; }
  __device__ static constexpr int vwidth(int) { return 8; }
};
template <> struct Sig<SIG_A4I> {
  static constexpr bool kStatic = true;
  static constexpr int kAcc = 4, kVals = 1;
  __device__ static constexpr int op(int j) { return j; }
  __device__ static constexpr int col(int) { return 0; }
  __device__ static constexpr bool f64(int) { return false; }
  __device__ static constexpr int vwidth(int) { return 8; }
};
template <> struct Sig<SIG_A4F> {
  static constexpr bool kStatic = true;
  static constexpr int kAcc = 4, kVals = 1;
  __device__ static constexpr int op(int j) { return j; }
  __device__ static constexpr int col(int) { return 0; }
  __device__ static constexpr bool f64(int j) { return j != 1; }
  __device__ static constexpr int vwidth(int) { return 8; }
};
template <> struct Sig<SIG_SC32> {
  static constexpr bool kStatic = true;
  static constexpr int kAcc = 2, kVals = 1;
  __device__ static constexpr int op(int j) { return j == 0 ? EIGER_SUM : EIGER_COUNT; }
  __device__ static constexpr int col(int) { return 0; }
  __device__ static constexpr bool f64(int) { return false; }
  __device__ static constexpr int vwidth(int) { return 4; }
};
template <> struct Sig<SIG_S4C> {
  static constexpr bool kStatic = true;
  static constexpr int kAcc = 5, kVals = 4;
  __device__ static constexpr int op(int j) { return j < 4 ? EIGER_SUM : EIGER_COUNT; }
  __device__ static constexpr int col(int j) { return j < 4 ? j : 0; }
  __device__ static constexpr bool f64(int) { return false; }
  __device__ static constexpr int vwidth(int) { return 8; }
};

// ---- streamed loads: read once, keep out of L1, first to leave L2 ----------------
// EIGER_STREAM_L2_HINT (default 1): the loads carry an L2 evict_first policy, so that what the kernels
// keep L2-resident next to the stream (the global hash table, the global direct array) is not pushed
// out by rows that are read exactly once (hash tables "perform well when ... cache-resident").
#ifndef EIGER_STREAM_L2_HINT
#define EIGER_STREAM_L2_HINT 1
#endif
#if EIGER_STREAM_L2_HINT
// not volatile: a pure value, computed once per thread wherever the compiler hoists it
__device__ __forceinline__ uint64_t stream_policy() {
  uint64_t p;
  asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
#define EIGER_LDG_HINT ".L2::cache_hint"
#define EIGER_LDG_POL(n) ", %" #n
#define EIGER_LDG_POL_ARG , "l"(stream_policy())
#else
#define EIGER_LDG_HINT ""
#define EIGER_LDG_POL(n) ""
#define EIGER_LDG_POL_ARG
#endif
__device__ __forceinline__ uint4 ldg_stream_16(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate" EIGER_LDG_HINT ".v4.u32 {%0,%1,%2,%3}, [%4]" EIGER_LDG_POL(5) ";"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p) EIGER_LDG_POL_ARG);
  return r;
}
__device__ __forceinline__ uint2 ldg_stream_8(const void* p) {
  uint2 r;
  asm volatile("ld.global.nc.L1::no_allocate" EIGER_LDG_HINT ".v2.u32 {%0,%1}, [%2]" EIGER_LDG_POL(3) ";"
               : "=r"(r.x), "=r"(r.y) : "l"(p) EIGER_LDG_POL_ARG);
  return r;
}
__device__ __forceinline__ uint32_t ldg_stream_4(const void* p) {
  uint32_t r;
  asm volatile("ld.global.nc.L1::no_allocate" EIGER_LDG_HINT ".u32 %0, [%1]" EIGER_LDG_POL(2) ";" : "=r"(r) : "l"(p) EIGER_LDG_POL_ARG);
  return r;
}
__device__ __forceinline__ uint32_t ldg_stream_2(const void* p) {
  uint16_t r;
  asm volatile("ld.global.nc.L1::no_allocate" EIGER_LDG_HINT ".u16 %0, [%1]" EIGER_LDG_POL(2) ";" : "=h"(r) : "l"(p) EIGER_LDG_POL_ARG);
  return r;
}
__device__ __forceinline__ uint32_t ldg_stream_1(const void* p) {
  uint32_t r;
  asm volatile("ld.global.nc.L1::no_allocate" EIGER_LDG_HINT ".u8 %0, [%1]" EIGER_LDG_POL(2) ";" : "=r"(r) : "l"(p) EIGER_LDG_POL_ARG);
  return r;
}
__device__ __forceinline__ uint64_t ldg_stream_u64(const void* p) {
  uint64_t r;
  asm volatile("ld.global.nc.L1::no_allocate" EIGER_LDG_HINT ".u64 %0, [%1]" EIGER_LDG_POL(2) ";" : "=l"(r) : "l"(p) EIGER_LDG_POL_ARG);
  return r;
}

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

__device__ __forceinline__ uint64_t sext_load(const void* base, int dtype, int64_t i) {
  switch (dtype) {
    case EIGER_I8: return (uint64_t)(int64_t)(int8_t)ldg_stream_1((const int8_t*)base + i);
    case EIGER_I32: return (uint64_t)(int64_t)(int32_t)ldg_stream_4((const int32_t*)base + i);
    default: return ldg_stream_u64((const int64_t*)base + i);
  }
}

// ---- hashes ------------------------------------------------------------------------
// Sketch hash (R2): splitmix64 output function of the sign-extended key.
__device__ __forceinline__ uint64_t hll_hash64(uint64_t x) {
  uint64_t z = x + 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
// Table hashes: free choice, results do not depend on them (R11).
__device__ __forceinline__ uint64_t table_hash64(uint64_t u) {
  uint64_t h = (u ^ (u >> 32)) * 0x9FB21C651E98DF25ull;
  h = (h ^ (h >> 29)) * 0xD6E8FEB86659FD93ull;
  return h ^ (h >> 32);
}
__device__ __forceinline__ uint32_t table_hash32(uint32_t u) {
  uint32_t h = u * 0x9E3779B1u;
  h = (h ^ (h >> 15)) * 0x85EBCA77u;
  return h ^ (h >> 13);
}
// a second, independent 32-bit hash: table_hash32's top bits choose the partition, this one
// the slot inside the partition's shared-memory table
__device__ __forceinline__ uint32_t table_hash32b(uint32_t u) {
  uint32_t h = (u ^ (u >> 16)) * 0x7FEB352Du;
  h = (h ^ (h >> 15)) * 0x846CA68Bu;
  return h ^ (h >> 16);
}

// partition id of a rebased key: the top bits of the table hash (32-bit keys hash in 32 bits,
// 64-bit keys in 64); shift = key bits - log2(fan-out), so that the ids of a smaller fan-out are
// the ids of a larger one shifted right (histograms fold)
template <class U> __device__ __forceinline__ uint32_t part_id(U u, int shift, uint32_t mask);
template <> __device__ __forceinline__ uint32_t part_id<uint32_t>(uint32_t u, int shift, uint32_t mask) {
  return (table_hash32(u) >> shift) & mask;
}
template <> __device__ __forceinline__ uint32_t part_id<uint64_t>(uint64_t u, int shift, uint32_t mask) {
  return (uint32_t)(table_hash64(u) >> shift) & mask;
}
constexpr int kPreBits = 10;             // fan-out of the histogram taken together with the slice sketch
constexpr int kPreFan = 1 << kPreBits;

// ---- accumulator algebra -------------------------------------------------------------
// fp64 MIN/MAX run on an order-preserving int64 image of the double (an involution).
__device__ __forceinline__ int64_t f64_order(uint64_t bits) {
  const int64_t b = (int64_t)bits;
  return b ^ ((b >> 63) & 0x7FFFFFFFFFFFFFFFll);
}
__device__ __forceinline__ uint64_t acc_identity(int op) {
  return op == EIGER_MIN ? (uint64_t)INT64_MAX : op == EIGER_MAX ? (uint64_t)INT64_MIN : 0ull;
}
// What one row contributes to accumulator (op, f64): the "partial" form that merges with
// add (SUM, COUNT) or min/max on int64 (MIN, MAX; doubles in f64_order space).
__device__ __forceinline__ uint64_t row_partial(int op, bool f64, uint64_t raw) {
  if (op == EIGER_COUNT) return 1ull;
  if (f64 && op != EIGER_SUM) return (uint64_t)f64_order(raw);
  return raw;
}
__device__ __forceinline__ uint64_t combine(int op, bool f64, uint64_t a, uint64_t b) {
  if (op == EIGER_SUM && f64) return (uint64_t)__double_as_longlong(__longlong_as_double((int64_t)a) + __longlong_as_double((int64_t)b));
  if (op == EIGER_SUM || op == EIGER_COUNT) return a + b;
  if (op == EIGER_MIN) return (uint64_t)min((int64_t)a, (int64_t)b);
  return (uint64_t)max((int64_t)a, (int64_t)b);
}
// Atomic merge of a partial into an accumulator cell (shared or global address).
__device__ __forceinline__ void atomic_merge(uint64_t* cell, int op, bool f64, uint64_t part) {
  if (op == EIGER_SUM && f64) atomicAdd(reinterpret_cast<double*>(cell), __longlong_as_double((int64_t)part));
  else if (op == EIGER_SUM || op == EIGER_COUNT) atomicAdd(reinterpret_cast<unsigned long long*>(cell), (unsigned long long)part);
  else if (op == EIGER_MIN) atomicMin(reinterpret_cast<long long*>(cell), (long long)part);
  else atomicMax(reinterpret_cast<long long*>(cell), (long long)part);
}
__device__ __forceinline__ uint64_t acc_finalize(int op, bool f64, uint64_t acc) {
  if (f64 && (op == EIGER_MIN || op == EIGER_MAX)) return (uint64_t)f64_order(acc);
  return acc;
}

}  // namespace eiger
