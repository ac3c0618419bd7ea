// Row access shared by the aggregation and partition kernels: how the key column(s) become
// the rebased, fused key u (step A0: frame of reference + positional packing,
// PAPER.md:219-221 §4.3), the shared-memory accumulator planes, and the global hash table.
#pragma once
#include "dev.cuh"

namespace eiger {

template <int KK> struct KeyTraits;
template <> struct KeyTraits<KK_I32> { using U = uint32_t; };
template <> struct KeyTraits<KK_I8I8> { using U = uint32_t; };
template <> struct KeyTraits<KK_I64> { using U = uint64_t; };
template <> struct KeyTraits<KK_GEN> { using U = uint64_t; };
template <> struct KeyTraits<KK_U64PRE> { using U = uint64_t; };
template <> struct KeyTraits<KK_U32PRE> { using U = uint32_t; };
template <> struct KeyTraits<KK_GEN32> { using U = uint32_t; };

template <class U> __device__ __forceinline__ U empty_of();
template <> __device__ __forceinline__ uint32_t empty_of<uint32_t>() { return kEmpty32; }
template <> __device__ __forceinline__ uint64_t empty_of<uint64_t>() { return kEmpty64; }

// ---- key loading ---------------------------------------------------------------------
// Generic fusion of up to kMaxKeyCols rebased column values d[c] (0 for unused columns, whose
// range is 1).  All columns are loaded before the multiply chain starts (independent loads in
// flight together); a value outside its column's planned range gives ~0, which no valid fused
// key equals (the product of the ranges fits 64 bits): speculative runs plan from a sample and
// must notice such rows instead of aliasing them onto another group.
__device__ __forceinline__ uint64_t fuse_cols(const KeyDesc& k, const uint64_t (&d)[kMaxKeyCols]) {
  bool ok = true;
#pragma unroll
  for (int c = 0; c < kMaxKeyCols; ++c) ok = ok && d[c] < k.rng[c];
  uint64_t u;
  if (k.flags & kKey32) {
    uint32_t w = (uint32_t)d[0];
#pragma unroll
    for (int c = 1; c < kMaxKeyCols; ++c) w = w * (uint32_t)k.rng[c] + (uint32_t)d[c];
    u = w;
  } else {
    u = d[0];
#pragma unroll
    for (int c = 1; c < kMaxKeyCols; ++c) u = u * k.rng[c] + d[c];
  }
  return ok ? u : ~0ull;
}
// All-int32 key columns with a fused domain below 2^32, two consecutive rows: rebasing, range
// checks and packing in 32-bit arithmetic, NC columns known at compile time (one code copy per
// column count: no work for absent columns, every load in one basic block).  ~0u = some column
// outside its planned range (no valid fused key: the domain is below 2^32).
template <int NC>
__device__ __forceinline__ void fuse32_pair(const KeyDesc& k, int64_t i, uint32_t (&w)[2]) {
  uint2 v[NC];
#pragma unroll
  for (int c = 0; c < NC; ++c) v[c] = ldg_stream_8((const int32_t*)k.ptr[c] + i);
  uint32_t w0 = 0, w1 = 0;
  bool ok0 = true, ok1 = true;
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    const uint32_t b = (uint32_t)k.base[c], r = (uint32_t)k.rng[c];
    const uint32_t e0 = v[c].x - b, e1 = v[c].y - b;
    ok0 = ok0 && e0 < r; ok1 = ok1 && e1 < r;
    w0 = w0 * r + e0; w1 = w1 * r + e1;         // c = 0: 0 * r + e
  }
  w[0] = ok0 ? w0 : ~0u; w[1] = ok1 ? w1 : ~0u;
}
__device__ __forceinline__ void fuse32_pair_any(const KeyDesc& k, int64_t i, uint32_t (&w)[2]) {
  switch (k.ncols) {
    case 1: fuse32_pair<1>(k, i, w); break;
    case 2: fuse32_pair<2>(k, i, w); break;
    case 3: fuse32_pair<3>(k, i, w); break;
    default: fuse32_pair<4>(k, i, w); break;
  }
}

template <int KK>
__device__ __forceinline__ typename KeyTraits<KK>::U load_u(const KeyDesc& k, int64_t i) {
  using U = typename KeyTraits<KK>::U;
  if constexpr (KK == KK_I32) {
    return (U)(ldg_stream_4((const int32_t*)k.ptr[0] + i) - (uint32_t)k.base[0]);
  } else if constexpr (KK == KK_I64) {
    return ldg_stream_u64((const int64_t*)k.ptr[0] + i) - k.base[0];
  } else if constexpr (KK == KK_U64PRE) {
    return ldg_stream_u64((const uint64_t*)k.ptr[0] + i);
  } else if constexpr (KK == KK_U32PRE) {
    return ldg_stream_4((const uint32_t*)k.ptr[0] + i);
  } else if constexpr (KK == KK_GEN32) {
    return (uint32_t)load_u<KK_GEN>(k, i);      // ~0 (out of range) stays ~0
  } else if constexpr (KK == KK_I8I8) {
    const uint32_t a = (uint32_t)(int32_t)(int8_t)ldg_stream_1((const int8_t*)k.ptr[0] + i) - (uint32_t)k.base[0];
    const uint32_t b = (uint32_t)(int32_t)(int8_t)ldg_stream_1((const int8_t*)k.ptr[1] + i) - (uint32_t)k.base[1];
    return b < (uint32_t)k.mul ? a * (uint32_t)k.mul + b : ~0u;    // ~0: outside the planned range (speculative runs)
  } else {
    uint64_t d[kMaxKeyCols];
    if (k.flags & kKeyAll32) {
      // branch-free: unused columns point at column 0 (host side) and are masked out, so that the
      // (volatile) loads of all columns sit in one basic block and go out back to back
      uint32_t v[kMaxKeyCols];
#pragma unroll
      for (int c = 0; c < kMaxKeyCols; ++c) v[c] = ldg_stream_4((const int32_t*)k.ptr[c] + i);
#pragma unroll
      for (int c = 0; c < kMaxKeyCols; ++c) d[c] = c < k.ncols ? (uint64_t)(uint32_t)(v[c] - (uint32_t)k.base[c]) : 0ull;
    } else {
#pragma unroll
      for (int c = 0; c < kMaxKeyCols; ++c) d[c] = c < k.ncols ? sext_load(k.ptr[c], k.dtype[c], i) - k.base[c] : 0ull;
    }
    return fuse_cols(k, d);
  }
}
// two consecutive rows starting at an even row index (vector loads)
template <int KK>
__device__ __forceinline__ void load_u2(const KeyDesc& k, int64_t i, typename KeyTraits<KK>::U (&u)[2]) {
  if constexpr (KK == KK_I32 || KK == KK_U32PRE) {
    const uint2 v = ldg_stream_8((const int32_t*)k.ptr[0] + i);
    const uint32_t b = KK == KK_I32 ? (uint32_t)k.base[0] : 0u;
    u[0] = v.x - b; u[1] = v.y - b;
  } else if constexpr (KK == KK_I64 || KK == KK_U64PRE) {
    const uint4 v = ldg_stream_16((const uint64_t*)k.ptr[0] + i);
    const uint64_t b = KK == KK_I64 ? k.base[0] : 0ull;
    u[0] = (((uint64_t)v.y << 32) | v.x) - b; u[1] = (((uint64_t)v.w << 32) | v.z) - b;
  } else if constexpr (KK == KK_GEN32) {
    if (k.flags & kKeyAll32) { fuse32_pair_any(k, i, u); }
    else {
      uint64_t w[2];
      load_u2<KK_GEN>(k, i, w);
      u[0] = (uint32_t)w[0]; u[1] = (uint32_t)w[1];
    }
  } else if constexpr (KK == KK_I8I8) {
    const uint32_t a = ldg_stream_2((const int8_t*)k.ptr[0] + i), b = ldg_stream_2((const int8_t*)k.ptr[1] + i);
    const uint32_t b0 = (uint32_t)k.base[0], b1 = (uint32_t)k.base[1], m = (uint32_t)k.mul;
    const uint32_t lo0 = (uint32_t)(int32_t)(int8_t)(b & 0xFF) - b1, lo1 = (uint32_t)(int32_t)(int8_t)(b >> 8) - b1;
    u[0] = lo0 < m ? ((uint32_t)(int32_t)(int8_t)(a & 0xFF) - b0) * m + lo0 : ~0u;   // ~0: outside the planned range
    u[1] = lo1 < m ? ((uint32_t)(int32_t)(int8_t)(a >> 8) - b0) * m + lo1 : ~0u;
  } else {
    uint64_t d0[kMaxKeyCols], d1[kMaxKeyCols];
    if ((k.flags & (kKeyAll32 | kKey32)) == (kKeyAll32 | kKey32)) {
      uint32_t w[2];
      fuse32_pair_any(k, i, w);
      u[0] = w[0] == ~0u ? ~0ull : (uint64_t)w[0]; u[1] = w[1] == ~0u ? ~0ull : (uint64_t)w[1];
      return;
    }
    if (k.flags & kKeyAll32) {
      // branch-free per column (see load_u): one code copy per column count
      uint2 v[kMaxKeyCols];
      if (k.ncols <= 2) {
#pragma unroll
        for (int c = 0; c < 2; ++c) v[c] = ldg_stream_8((const int32_t*)k.ptr[c] + i);
        v[2] = v[0]; v[3] = v[0];
      } else if (k.ncols == 3) {
#pragma unroll
        for (int c = 0; c < 3; ++c) v[c] = ldg_stream_8((const int32_t*)k.ptr[c] + i);
        v[3] = v[0];
      } else {
#pragma unroll
        for (int c = 0; c < kMaxKeyCols; ++c) v[c] = ldg_stream_8((const int32_t*)k.ptr[c] + i);
      }
#pragma unroll
      for (int c = 0; c < kMaxKeyCols; ++c) {
        d0[c] = c < k.ncols ? (uint64_t)(uint32_t)(v[c].x - (uint32_t)k.base[c]) : 0ull;
        d1[c] = c < k.ncols ? (uint64_t)(uint32_t)(v[c].y - (uint32_t)k.base[c]) : 0ull;
      }
    } else {
#pragma unroll
      for (int c = 0; c < kMaxKeyCols; ++c) {
        if (c < k.ncols) { d0[c] = sext_load(k.ptr[c], k.dtype[c], i) - k.base[c]; d1[c] = sext_load(k.ptr[c], k.dtype[c], i + 1) - k.base[c]; }
        else { d0[c] = 0ull; d1[c] = 0ull; }
      }
    }
    u[0] = fuse_cols(k, d0); u[1] = fuse_cols(k, d1);
  }
}

// un-fuse and un-rebase group key u into the caller's key columns at row g
__device__ __forceinline__ void unfuse_key(const KeyDesc& key, uint64_t u, uint64_t (&part)[kMaxKeyCols]) {
  for (int k = key.ncols - 1; k > 0; --k) { part[k] = u % key.rng[k]; u /= key.rng[k]; }
  part[0] = u;
}
__device__ __forceinline__ void store_group_key(const KeyDesc& key, void* const* out_keys, uint64_t u, uint64_t g) {
  uint64_t part[kMaxKeyCols];
  unfuse_key(key, u, part);
  for (int k = 0; k < key.ncols; ++k) {
    const uint64_t v = part[k] + key.base[k];
    switch (key.dtype[k]) {
      case EIGER_I8: static_cast<int8_t*>(out_keys[k])[g] = (int8_t)v; break;
      case EIGER_I32: static_cast<int32_t*>(out_keys[k])[g] = (int32_t)v; break;
      default: static_cast<int64_t*>(out_keys[k])[g] = (int64_t)v; break;
    }
  }
}

// value column c straight from global memory: one row, or two consecutive rows starting at an
// even row index.  w = bytes per element: 8, or 4 for int32 payloads (sign-extended)
__device__ __forceinline__ uint64_t global_val(const AggPlan& p, int c, int w, int64_t i) {
  if (w == 8) return ldg_stream_u64(static_cast<const uint64_t*>(p.vals[c]) + i);
  return (uint64_t)(int64_t)(int32_t)ldg_stream_4(static_cast<const int32_t*>(p.vals[c]) + i);
}
__device__ __forceinline__ void global_val2(const AggPlan& p, int c, int w, int64_t i, uint64_t& a, uint64_t& b) {
  if (w == 8) {
    const uint4 v = ldg_stream_16(static_cast<const uint64_t*>(p.vals[c]) + i);
    a = ((uint64_t)v.y << 32) | v.x; b = ((uint64_t)v.w << 32) | v.z;
  } else {
    const uint2 v = ldg_stream_8(static_cast<const int32_t*>(p.vals[c]) + i);
    a = (uint64_t)(int64_t)(int32_t)v.x; b = (uint64_t)(int64_t)(int32_t)v.y;
  }
}
template <int SIG> __device__ __forceinline__ int sig_vw(const AggPlan& p, int c) { if constexpr (Sig<SIG>::kStatic) return Sig<SIG>::vwidth(c); else return p.vw[c]; }

template <int SIG> __device__ __forceinline__ int sig_op(const AggPlan& p, int j) { if constexpr (Sig<SIG>::kStatic) return Sig<SIG>::op(j); else return p.op[j]; }
template <int SIG> __device__ __forceinline__ int sig_col(const AggPlan& p, int j) { if constexpr (Sig<SIG>::kStatic) return Sig<SIG>::col(j); else return p.col[j]; }
template <int SIG> __device__ __forceinline__ bool sig_f64(const AggPlan& p, int j) { if constexpr (Sig<SIG>::kStatic) return Sig<SIG>::f64(j); else return p.f64[j] != 0; }

// ---- shared-memory accumulators ------------------------------------------------------------
// B200 shared memory has native 32-bit atomics (ATOMS.ADD / ATOMS.MAX; 3 per row sustain
// ~880 G rows/s chip-wide, measured) but 64-bit ones are CAS loops (~0.05-0.4 T/s).  Integer
// SUM and COUNT cells are therefore kept as two 32-bit planes, lo[S] then hi[S], and added
// with an explicit carry: the final (hi:lo) equals the wrapping 64-bit sum whatever the
// interleaving, because every wrap of lo is seen by exactly one atomicAdd's return value.
// MIN / MAX and fp64 SUM keep 64-bit cells; MIN / MAX look before they leap, so the CAS loop
// only runs on a new record.
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
  if (op == EIGER_COUNT) {
    // a CTA never sees 2^32 rows (that many rows per CTA do not fit the device's memory): no carry,
    // hence no returning atomic
    atomicAdd(reinterpret_cast<uint32_t*>(plane) + s, (uint32_t)part);
  } else if (add_type(op, f64)) {
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

// ---- the global hash table -------------------------------------------------------------
// Slot s lives at table + s * stride: [u64 key][acc 0]..[acc n-1][pad]; key = ~0 means empty.
// Slot `cap` is the side slot of the one key whose rebased value equals the empty marker
// (R18).  Find-or-insert with a single exit so that the lanes of a warp stay
// converged (an early-return version ran 15x slower: every lane took its own copy of the
// tail).  Returns the slot's accumulator cells, or nullptr when probing gave up.
constexpr int kBackProbes = 4096;
__device__ __forceinline__ uint64_t* back_find_or_insert(void* table, uint64_t cap, uint32_t stride,
                                                         uint64_t u, CallDev* call) {
  uint64_t* cells = nullptr;
  uint64_t slot = __umul64hi(table_hash64(u), cap);
  int probes = 0;
  bool done = false;
  if (u == kEmpty64) { slot = cap; }
  while (!done) {
    unsigned long long* kp = reinterpret_cast<unsigned long long*>(static_cast<char*>(table) + slot * stride);
    if (slot == cap) {            // side slot: key word 0 = used
      if (__ldcg(kp) != 0ull) atomicExch(kp, 0ull);
      cells = reinterpret_cast<uint64_t*>(kp) + 1; done = true;
    } else {
      unsigned long long k = __ldcg(kp);
      if (k == kEmpty64) { k = atomicCAS(kp, kEmpty64, (unsigned long long)u); if (k == kEmpty64) k = u; }
      if (k == u) { cells = reinterpret_cast<uint64_t*>(kp) + 1; done = true; }
      else {
        slot = slot + 1 == cap ? 0 : slot + 1;
        if (++probes >= kBackProbes) { atomicOr(&call->overflow, 1u); done = true; }
      }
    }
  }
  return cells;
}

}  // namespace eiger
