// Steps A1-A3: the fused single-pass profile kernel — exact min/max and HyperLogLog
// registers of one key column — and the register-histogram / estimator that follow.
// PAPER.md:30 §1, §4 ("close to the memory bandwidth"), §4.1
// (HLL++ [14] before the group-by), §4.3 (range first).  Readings R1-R6.
#include <algorithm>
#include <cmath>
#include <type_traits>

#include "internal.h"
#include "rows.cuh"

namespace eiger {
namespace {

constexpr int kProfThreads = 512;
constexpr int kProfUnroll = 4;     // 16-byte vectors in flight per thread

__global__ void profile_reset_kernel(ProfileDev* out, int with_regs) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < kMaxKeyCols) { out->min[t] = INT64_MAX; out->max[t] = INT64_MIN; }
  if (t < 64) out->hist[t] = 0;
  if (t == 0) { out->pair_eq = 0; out->pair_n = 0; out->oor = 0; }
  if (with_regs) for (int i = t; i < kHllM; i += gridDim.x * blockDim.x) out->regs[i] = 0;
  if (with_regs) for (int i = t; i < kPreFan; i += gridDim.x * blockDim.x) out->part_hist[i] = 0;
}

// One sketch update against the CTA's registers in shared memory: one word per register and
// one native ATOMS.MAX per key (B200 shared memory does ~2 T 32-bit atomics/s, measured, so
// the unconditional atomic is cheaper than a look-before-you-leap branch plus a CAS loop).
__device__ __forceinline__ void hll_update(uint32_t* sregs, uint64_t x) {
  // hll_hash64 with its last step (z ^= z >> 31) written out on 32-bit halves: idx and rho need
  // the high word of w = z << p only, except for the one key in 2^32 whose top 32 bits of w are
  // zero.  Same registers bit for bit; 19 instead of 25 ALU-pipe instructions per key (the full
  // profile is ALU-bound: ncu 79 % ALU pipe on 4-byte keys).
  uint64_t z = x + 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  const uint32_t zh = (uint32_t)(z >> 32), zl = (uint32_t)z;
  const uint32_t fh = zh ^ (zh >> 31);
  const uint32_t fl = zl ^ __funnelshift_r(zl, zh, 31);
  const uint32_t idx = fh >> (32 - kHllP);
  const uint32_t wh = __funnelshift_l(fl, fh, kHllP);
  uint32_t rho;
  if (wh != 0u) {
    rho = (uint32_t)__clz((int)wh) + 1u;
  } else {
    const uint32_t wl = fl << kHllP;
    rho = (uint32_t)min(32 + __clz((int)wl), kHllQ) + 1u;
  }
  atomicMax(sregs + idx, rho);
}

template <int DT> struct Elem;
template <> struct Elem<EIGER_I8> { static constexpr int kPerVec = 16; };
template <> struct Elem<EIGER_I32> { static constexpr int kPerVec = 4; };
template <> struct Elem<EIGER_I64> { static constexpr int kPerVec = 2; };

template <int DT> struct MinMaxT { using T = int; };
template <> struct MinMaxT<EIGER_I64> { using T = long long; };

template <int DT, bool HLL>
__device__ __forceinline__ void consume_vec(const uint4 v, typename MinMaxT<DT>::T& lo, typename MinMaxT<DT>::T& hi, uint32_t* sregs) {
  if constexpr (DT == EIGER_I64) {
    const long long a = (long long)(((uint64_t)v.y << 32) | v.x), b = (long long)(((uint64_t)v.w << 32) | v.z);
    lo = min(lo, min(a, b)); hi = max(hi, max(a, b));
    if constexpr (HLL) { hll_update(sregs, (uint64_t)a); hll_update(sregs, (uint64_t)b); }
  } else if constexpr (DT == EIGER_I32) {
    const int a = (int)v.x, b = (int)v.y, c = (int)v.z, d = (int)v.w;
    const int l = min(min(a, b), min(c, d)), h = max(max(a, b), max(c, d));
    lo = min(lo, l); hi = max(hi, h);
    if constexpr (HLL) {
      hll_update(sregs, (uint64_t)(long long)a); hll_update(sregs, (uint64_t)(long long)b);
      hll_update(sregs, (uint64_t)(long long)c); hll_update(sregs, (uint64_t)(long long)d);
    }
  } else {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
    // per-byte sign extension + 32-bit min/max: ~3 ALU instructions per key, far below the
    // issue budget of a 1-byte-per-key stream (the SIMD-in-word intrinsics are emulated)
    int l = INT32_MAX, h = INT32_MIN;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int b0 = (int)(int8_t)(w[k]), b1 = (int)(int8_t)(w[k] >> 8), b2 = (int)(int8_t)(w[k] >> 16), b3 = (int)w[k] >> 24;
      l = min(min(l, b0), min(min(b1, b2), b3));
      h = max(max(h, b0), max(max(b1, b2), b3));
    }
    lo = min(lo, l); hi = max(hi, h);
    if constexpr (HLL) {
#pragma unroll
      for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int b = 0; b < 4; ++b) hll_update(sregs, (uint64_t)(long long)(int8_t)(w[k] >> (8 * b)));
    }
  }
}

template <int DT, bool HLL>
__global__ void __launch_bounds__(kProfThreads)
profile_kernel(const void* __restrict__ keys, int64_t n, ProfileDev* __restrict__ out, int which) {
  extern __shared__ uint32_t sregs[];   // kHllM words when HLL
  __shared__ long long s_lo[kProfThreads / 32], s_hi[kProfThreads / 32];
  const int tid = threadIdx.x;
  if constexpr (HLL) {
    for (int i = tid; i < kHllM; i += kProfThreads) sregs[i] = 0;
    __syncthreads();
  }
  using MM = typename MinMaxT<DT>::T;     // 32-bit min/max for 1- and 4-byte keys, widened once at the end
  MM lo_t = DT == EIGER_I64 ? (MM)INT64_MAX : (MM)INT32_MAX, hi_t = DT == EIGER_I64 ? (MM)INT64_MIN : (MM)INT32_MIN;
  constexpr int EPV = Elem<DT>::kPerVec;
  const int64_t nvec = n / EPV;
  const uint4* vp = static_cast<const uint4*>(keys);
  const int64_t stride = (int64_t)gridDim.x * kProfThreads;
  int64_t v = (int64_t)blockIdx.x * kProfThreads + tid;
  for (; v + (kProfUnroll - 1) * stride < nvec; v += kProfUnroll * stride) {
    uint4 r[kProfUnroll];
#pragma unroll
    for (int k = 0; k < kProfUnroll; ++k) r[k] = ldg_stream_16(vp + v + k * stride);
#pragma unroll
    for (int k = 0; k < kProfUnroll; ++k) consume_vec<DT, HLL>(r[k], lo_t, hi_t, sregs);
  }
  for (; v < nvec; v += stride) consume_vec<DT, HLL>(ldg_stream_16(vp + v), lo_t, hi_t, sregs);
  long long lo = lo_t > hi_t ? INT64_MAX : (long long)lo_t, hi = lo_t > hi_t ? INT64_MIN : (long long)hi_t;
  // ragged tail: fewer than EPV elements, taken by the first threads of CTA 0
  if (blockIdx.x == 0 && tid < (int)(n - nvec * EPV)) {
    const uint64_t x = sext_load(keys, DT, nvec * EPV + tid);
    lo = min(lo, (long long)x); hi = max(hi, (long long)x);
    if constexpr (HLL) hll_update(sregs, x);
  }
  // CTA-level merge: shuffles for the 64-bit min/max, one global atomic pair per CTA
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
  }
  if ((tid & 31) == 0) { s_lo[tid >> 5] = lo; s_hi[tid >> 5] = hi; }
  __syncthreads();
  if (tid < 32) {
    lo = tid < kProfThreads / 32 ? s_lo[tid] : INT64_MAX;
    hi = tid < kProfThreads / 32 ? s_hi[tid] : INT64_MIN;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
      hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if (tid == 0) {
      if (lo != INT64_MAX) atomicMin(&out->min[which], lo);
      if (hi != INT64_MIN) atomicMax(&out->max[which], hi);
    }
  }
  if constexpr (HLL) {
    // one CTA-level merge of the sketch: only non-zero registers touch global memory
    __syncthreads();
    for (int i = tid; i < kHllM; i += kProfThreads) {
      const uint32_t r = sregs[i];
      if (r) atomicMax(&out->regs[i], r);
    }
  }
}

// Keys-only pass that replaces the full profile when the sample has already settled the variant
// (PARTITION): exact min/max, the level-1 partition histogram at fan-out kPreFan of
// u = key - base, and the sketch of the keys of partitions [0, sel) only.  Partitions are cut by
// a hash of the key, so the keys of `sel` of them are a uniform sample of the column's DISTINCT
// keys whatever their frequencies (distinct sampling): NDV ~ slice NDV * kPreFan / sel with
// relative error 1 / sqrt(slice NDV), and only sel / kPreFan of the keys pay the 64-bit sketch hash.
template <int DT>
__global__ void __launch_bounds__(kProfThreads)
part_hist_hll_kernel(const void* __restrict__ keys, int64_t n, uint64_t base, uint32_t sel, ProfileDev* __restrict__ out) {
  using U = typename std::conditional<DT == EIGER_I32, uint32_t, uint64_t>::type;
  using S = typename std::conditional<DT == EIGER_I32, int, long long>::type;
  extern __shared__ uint32_t sregs[];   // kHllM sketch words, kPreFan counters, one 64-key queue per warp
  uint32_t* s_hist = sregs + kHllM;
  __shared__ long long s_lo[kProfThreads / 32], s_hi[kProfThreads / 32];
  const int tid = threadIdx.x, lane = tid & 31;
  S* wq = reinterpret_cast<S*>(s_hist + kPreFan) + (tid >> 5) * 64;
  for (int i = tid; i < kHllM + kPreFan; i += kProfThreads) sregs[i] = 0;
  __syncthreads();
  constexpr int EPV = Elem<DT>::kPerVec;
  constexpr int kShift = 8 * (int)sizeof(U) - kPreBits;
  S lo = DT == EIGER_I32 ? (S)INT32_MAX : (S)INT64_MAX, hi = DT == EIGER_I32 ? (S)INT32_MIN : (S)INT64_MIN;
  int cnt = 0;        // keys waiting in this warp's queue (warp-uniform)
  // The keys of the slice are a minority spread over all lanes: they are queued per warp and
  // sketched 32 at a time by a full warp, so the 64-bit sketch hash costs sel / kPreFan of a key's
  // issue slots instead of a divergent branch that almost every warp would take.
  auto one = [&](S k) {                  // all 32 lanes of the warp are here
    lo = min(lo, k); hi = max(hi, k);
    const uint32_t q = part_id<U>((U)k - (U)base, kShift, kPreFan - 1);
    atomicAdd(s_hist + q, 1u);
    const bool in = q < sel;
    const uint32_t m = __ballot_sync(0xffffffffu, in);
    if (m) {
      if (in) wq[cnt + __popc(m & ((1u << lane) - 1u))] = k;
      cnt += __popc(m);
      if (cnt >= 32) {
        __syncwarp();
        cnt -= 32;
        hll_update(sregs, (uint64_t)(long long)wq[cnt + lane]);
        __syncwarp();
      }
    }
  };
  auto one_tail = [&](S k) {             // any subset of lanes
    lo = min(lo, k); hi = max(hi, k);
    const uint32_t q = part_id<U>((U)k - (U)base, kShift, kPreFan - 1);
    atomicAdd(s_hist + q, 1u);
    if (q < sel) hll_update(sregs, (uint64_t)(long long)k);
  };
  const int64_t nvec = n / EPV;
  const uint4* vp = static_cast<const uint4*>(keys);
  const int64_t stride = (int64_t)gridDim.x * kProfThreads;
  int64_t v = (int64_t)blockIdx.x * kProfThreads + tid;
  // warp-uniform bound: the whole warp's last vector of the trip is inside the column
  for (; v - lane + 31 + (kProfUnroll - 1) * stride < nvec; v += kProfUnroll * stride) {
    uint4 r[kProfUnroll];
#pragma unroll
    for (int k = 0; k < kProfUnroll; ++k) r[k] = ldg_stream_16(vp + v + k * stride);
#pragma unroll
    for (int k = 0; k < kProfUnroll; ++k) {
      if constexpr (DT == EIGER_I32) { one((int)r[k].x); one((int)r[k].y); one((int)r[k].z); one((int)r[k].w); }
      else { one((long long)(((uint64_t)r[k].y << 32) | r[k].x)); one((long long)(((uint64_t)r[k].w << 32) | r[k].z)); }
    }
  }
  for (; v < nvec; v += stride) {
    const uint4 r = ldg_stream_16(vp + v);
    if constexpr (DT == EIGER_I32) { one_tail((int)r.x); one_tail((int)r.y); one_tail((int)r.z); one_tail((int)r.w); }
    else { one_tail((long long)(((uint64_t)r.y << 32) | r.x)); one_tail((long long)(((uint64_t)r.w << 32) | r.z)); }
  }
  if (blockIdx.x == 0 && tid < (int)(n - nvec * EPV)) one_tail((S)sext_load(keys, DT, nvec * EPV + tid));
  __syncwarp();
  if (lane < cnt) hll_update(sregs, (uint64_t)(long long)wq[lane]);
  long long lo64 = (long long)lo, hi64 = (long long)hi;
  if (DT == EIGER_I32) { if (lo > hi) { lo64 = INT64_MAX; hi64 = INT64_MIN; } }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo64 = min(lo64, __shfl_xor_sync(0xffffffffu, lo64, o));
    hi64 = max(hi64, __shfl_xor_sync(0xffffffffu, hi64, o));
  }
  if (lane == 0) { s_lo[tid >> 5] = lo64; s_hi[tid >> 5] = hi64; }
  __syncthreads();
  if (tid == 0) {
    for (int w = 1; w < kProfThreads / 32; ++w) { lo64 = min(lo64, s_lo[w]); hi64 = max(hi64, s_hi[w]); }
    if (lo64 != INT64_MAX) atomicMin(&out->min[0], lo64);
    if (hi64 != INT64_MIN) atomicMax(&out->max[0], hi64);
  }
  for (int i = tid; i < kHllM; i += kProfThreads) { const uint32_t r = sregs[i]; if (r) atomicMax(&out->regs[i], r); }
  for (int i = tid; i < kPreFan; i += kProfThreads) { const uint32_t c = s_hist[i]; if (c) atomicAdd(&out->part_hist[i], c); }
}

// Statistics of an evenly spaced SAMPLE of the column (step A1/A2 on `samples` keys): what the
// speculative single pass of EIGER_AUTO is planned from.  The sample can only under-estimate the
// range and the NDV; the speculative kernels check both exactly and give up if it did.
__global__ void __launch_bounds__(256)
profile_sample_kernel(const void* __restrict__ keys, int dtype, int64_t n, int64_t samples, ProfileDev* __restrict__ out,
                      int which, int with_hll, int last) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  long long lo = INT64_MAX, hi = INT64_MIN;
  uint64_t x = 0;
  if (t < samples) {
    const int64_t i = (int64_t)(((unsigned __int128)t * (unsigned __int128)n) / (unsigned __int128)samples);
    x = sext_load(keys, dtype, i);
    lo = hi = (long long)x;
    if (with_hll) {
      const uint64_t z = hll_hash64(x);
      const uint32_t idx = (uint32_t)(z >> (64 - kHllP));
      const uint32_t rho = (uint32_t)min(__clzll((long long)(z << kHllP)), kHllQ) + 1u;
      if (out->regs[idx] < rho) atomicMax(&out->regs[idx], rho);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
  }
  if ((threadIdx.x & 31) == 0 && lo != INT64_MAX) { atomicMin(&out->min[which], lo); atomicMax(&out->max[which], hi); }
  // skew test: how often two neighbouring sample keys are equal estimates sum p_i^2 (1 / NDV when
  // uniform, ~0.02 for C3's Zipf); the selector keeps hot-key inputs away from the partitioner
  const uint64_t nb = __shfl_down_sync(0xffffffffu, x, 1);
  const bool cmp = (threadIdx.x & 31) < 31 && t + 1 < samples;
  const uint32_t eq = __ballot_sync(0xffffffffu, cmp && nb == x), nn = __ballot_sync(0xffffffffu, cmp);
  // several key columns (one launch per column, in stream order): two neighbouring sample ROWS are equal when
  // they agree in every column - each launch ANDs its column's verdicts into a bit mask, the last one counts
  if ((threadIdx.x & 31) == 0 && nn) {
    const int64_t w = t >> 5;
    uint32_t all = eq;
    if (w < kPairWords) {
      if (which > 0) all &= out->pair_mask[w];
      if (!last) out->pair_mask[w] = all;
    } else if (which > 0 || !last) all = 0u;             // beyond the mask (more than 2^18 samples): a single column's pairs only
    if (last && (w < kPairWords || which == 0)) { atomicAdd(&out->pair_eq, (uint32_t)__popc(all)); atomicAdd(&out->pair_n, (uint32_t)__popc(nn)); }
  }
}

// Heavy hitters of 4096 evenly spaced keys: a shared-memory count table (8192 slots), then the
// slots above 0.4 % of the sample are ranked by one thread.  A heuristic input of the selector:
// results never depend on it.
constexpr int kHotSamples = 4096, kHotSlots = 8192, kHotCand = 64;
constexpr long long kHotEmpty = INT64_MIN + 1;     // a key with this value is simply never reported
__global__ void __launch_bounds__(1024)
hot_keys_kernel(const void* __restrict__ keys, int dtype, int64_t n, ProfileDev* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char hot_smem[];       // 96 KB: keys, then counts
  unsigned long long* s_k = reinterpret_cast<unsigned long long*>(hot_smem);
  uint32_t* s_c = reinterpret_cast<uint32_t*>(hot_smem + sizeof(unsigned long long) * kHotSlots);
  __shared__ long long s_ck[kHotCand];
  __shared__ uint32_t s_cc[kHotCand], s_n;
  const int tid = threadIdx.x;
  for (int i = tid; i < kHotSlots; i += 1024) { s_k[i] = (unsigned long long)kHotEmpty; s_c[i] = 0; }
  if (tid == 0) s_n = 0;
  __syncthreads();
  const int64_t samples = n < kHotSamples ? n : kHotSamples;
  for (int64_t t = tid; t < samples; t += 1024) {
    const int64_t i = (int64_t)(((unsigned __int128)t * (unsigned __int128)n) / (unsigned __int128)samples);
    const unsigned long long x = sext_load(keys, dtype, i);
    if ((long long)x == kHotEmpty) continue;
    uint32_t slot = (uint32_t)(table_hash64(x) >> 51);       // 13 bits
    bool done = false;
    while (!done) {
      const unsigned long long prev = atomicCAS(&s_k[slot], (unsigned long long)kHotEmpty, x);
      if (prev == (unsigned long long)kHotEmpty || prev == x) { atomicAdd(&s_c[slot], 1u); done = true; }
      else slot = (slot + 1) & (kHotSlots - 1);
    }
  }
  __syncthreads();
  const uint32_t thr = (uint32_t)(samples / 256 > 4 ? samples / 256 : 4);      // 0.4 % of the sample
  for (int i = tid; i < kHotSlots; i += 1024) {
    if (s_c[i] >= thr) { const uint32_t pos = atomicAdd(&s_n, 1u); if (pos < kHotCand) { s_ck[pos] = (long long)s_k[i]; s_cc[pos] = s_c[i]; } }
  }
  __syncthreads();
  if (tid == 0) {
    const int nc = (int)(s_n < kHotCand ? s_n : kHotCand);
    int taken = 0;
    for (; taken < kMaxHot && taken < nc; ++taken) {          // selection of the kMaxHot largest counts
      int best = taken;
      for (int c = taken + 1; c < nc; ++c) if (s_cc[c] > s_cc[best]) best = c;
      const long long k = s_ck[best]; const uint32_t c = s_cc[best];
      s_ck[best] = s_ck[taken]; s_cc[best] = s_cc[taken]; s_ck[taken] = k; s_cc[taken] = c;
      out->hot_key[taken] = k; out->hot_cnt[taken] = c;
    }
    out->hot_n = (uint32_t)taken; out->hot_samples = (uint32_t)samples;
  }
}

__global__ void hll_hist_kernel(ProfileDev* out) {
  __shared__ uint32_t h[64];
  if (threadIdx.x < 64) h[threadIdx.x] = 0;
  __syncthreads();
  for (int i = threadIdx.x; i < kHllM; i += blockDim.x) atomicAdd(&h[out->regs[i] & 63u], 1u);
  __syncthreads();
  if (threadIdx.x < 64) out->hist[threadIdx.x] = h[threadIdx.x];
}

__global__ void regs_to_bytes_kernel(const ProfileDev* in, uint8_t* out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < kHllM) out[i] = (uint8_t)in->regs[i];
}

// Sketch of the FUSED key of a multi-column key (smart key fusion: where the range
// cannot settle it, "calculate the HLL++ sketch on the key and find the number of distinct
// values"): the same registers as profile_kernel's, over u = the rebased, packed key (rows.cuh:
// fuse_cols) taken as a 64-bit value.  The product of the column ranges bounds the group count
// only loosely (5000 distinct triples can span a 2^61 domain); this estimate sizes the tables.
__global__ void __launch_bounds__(kProfThreads)
fused_hll_kernel(const __grid_constant__ KeyDesc k, int64_t n, ProfileDev* __restrict__ out) {
  extern __shared__ uint32_t sregs[];   // kHllM words
  const int tid = threadIdx.x;
  for (int i = tid; i < kHllM; i += kProfThreads) sregs[i] = 0;
  __syncthreads();
  const int64_t pairs = n / 2, stride = (int64_t)gridDim.x * kProfThreads;
  int64_t p = (int64_t)blockIdx.x * kProfThreads + tid;
  for (; p + 3 * stride < pairs; p += 4 * stride) {
    uint64_t a[4][2];
#pragma unroll
    for (int j = 0; j < 4; ++j) load_u2<KK_GEN>(k, 2 * (p + j * stride), a[j]);
#pragma unroll
    for (int j = 0; j < 4; ++j) { hll_update(sregs, a[j][0]); hll_update(sregs, a[j][1]); }
  }
  for (; p < pairs; p += stride) {
    uint64_t a[2];
    load_u2<KK_GEN>(k, 2 * p, a);
    hll_update(sregs, a[0]); hll_update(sregs, a[1]);
  }
  if ((n & 1) && blockIdx.x == 0 && tid == 0) hll_update(sregs, load_u<KK_GEN>(k, n - 1));
  __syncthreads();
  for (int i = tid; i < kHllM; i += kProfThreads) {
    const uint32_t r = sregs[i];
    if (r) atomicMax(&out->regs[i], r);
  }
}

// The slice-sketch pass for SEVERAL key columns: one pass over the key columns fuses
// them with the sample's ranges (rows.cuh; a value outside its column's range makes the fused key ~0, which
// raises out->oor: the caller then falls back to the full profile), takes the level-1 partition histogram of
// the fused key at fan-out kPreFan and sketches the fused keys of partitions [0, sel).
template <int KK>
__global__ void __launch_bounds__(kProfThreads)
fused_part_hist_hll_kernel(const __grid_constant__ KeyDesc k, int64_t n, uint32_t sel, ProfileDev* __restrict__ out) {
  using U = typename KeyTraits<KK>::U;
  extern __shared__ uint32_t sregs[];   // kHllM sketch words, kPreFan counters, one 64-key queue per warp
  uint32_t* s_hist = sregs + kHllM;
  const int tid = threadIdx.x, lane = tid & 31;
  uint64_t* wq = reinterpret_cast<uint64_t*>(s_hist + kPreFan) + (tid >> 5) * 64;
  for (int i = tid; i < kHllM + kPreFan; i += kProfThreads) sregs[i] = 0;
  __syncthreads();
  constexpr int kShift = 8 * (int)sizeof(U) - kPreBits;
  int cnt = 0;
  bool bad = false;
  auto one = [&](U u) {                  // all 32 lanes of the warp are here
    bad = bad || u == empty_of<U>();
    const uint32_t q = part_id<U>(u, kShift, kPreFan - 1);
    atomicAdd(s_hist + q, 1u);
    const bool in = q < sel;
    const uint32_t m = __ballot_sync(0xffffffffu, in);
    if (m) {
      if (in) wq[cnt + __popc(m & ((1u << lane) - 1u))] = (uint64_t)u;
      cnt += __popc(m);
      if (cnt >= 32) {
        __syncwarp();
        cnt -= 32;
        hll_update(sregs, wq[cnt + lane]);
        __syncwarp();
      }
    }
  };
  auto one_tail = [&](U u) {             // any subset of lanes
    bad = bad || u == empty_of<U>();
    const uint32_t q = part_id<U>(u, kShift, kPreFan - 1);
    atomicAdd(s_hist + q, 1u);
    if (q < sel) hll_update(sregs, (uint64_t)u);
  };
  const int64_t pairs = n / 2, stride = (int64_t)gridDim.x * kProfThreads;
  int64_t p = (int64_t)blockIdx.x * kProfThreads + tid;
  // warp-uniform bound: the whole warp's last pair of the trip is inside the columns
  for (; p - lane + 31 + 3 * stride < pairs; p += 4 * stride) {
    U a[4][2];
#pragma unroll
    for (int j = 0; j < 4; ++j) load_u2<KK>(k, 2 * (p + j * stride), a[j]);
#pragma unroll
    for (int j = 0; j < 4; ++j) { one(a[j][0]); one(a[j][1]); }
  }
  for (; p < pairs; p += stride) {
    U a[2];
    load_u2<KK>(k, 2 * p, a);
    one_tail(a[0]); one_tail(a[1]);
  }
  if ((n & 1) && blockIdx.x == 0 && tid == 0) one_tail(load_u<KK>(k, n - 1));
  __syncwarp();
  if (lane < cnt) hll_update(sregs, wq[lane]);
  if (bad) atomicOr(&out->oor, 1u);
  __syncthreads();
  for (int i = tid; i < kHllM; i += kProfThreads) { const uint32_t r = sregs[i]; if (r) atomicMax(&out->regs[i], r); }
  for (int i = tid; i < kPreFan; i += kProfThreads) { const uint32_t c = s_hist[i]; if (c) atomicAdd(&out->part_hist[i], c); }
}

template <int DT>
int launch_profile_dt(Runtime* rt, const void* keys, int64_t n, int which, int with_hll, cudaStream_t s) {
  const int64_t nvec = n / Elem<DT>::kPerVec;
  const int64_t want = (nvec + (int64_t)kProfThreads * kProfUnroll - 1) / ((int64_t)kProfThreads * kProfUnroll);
  // persistent grid: two CTAs (32 warps) per SM, or fewer when the column is short
  const int blocks = (int)std::max<int64_t>(1, std::min<int64_t>(want, 2LL * rt->sm_count));
  if (with_hll) {
    auto kern = profile_kernel<DT, true>;
    EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kHllM * 4));
    kern<<<blocks, kProfThreads, kHllM * 4, s>>>(keys, n, rt->prof, which);
  } else {
    profile_kernel<DT, false><<<blocks, kProfThreads, 0, s>>>(keys, n, rt->prof, which);
  }
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

}  // namespace

int launch_profile(Runtime* rt, const void* keys, int dtype, int64_t n, int which, int with_hll,
                   bool reset, cudaStream_t s) {
  if (reset) {
    profile_reset_kernel<<<16, 1024, 0, s>>>(rt->prof, 1);
    count_launch();
    EIGER_CUDA(cudaGetLastError());
  }
  if (n == 0) return EIGER_OK;
  switch (dtype) {
    case EIGER_I8: return launch_profile_dt<EIGER_I8>(rt, keys, n, which, with_hll, s);
    case EIGER_I32: return launch_profile_dt<EIGER_I32>(rt, keys, n, which, with_hll, s);
    case EIGER_I64: return launch_profile_dt<EIGER_I64>(rt, keys, n, which, with_hll, s);
    default: return EIGER_ERR_ARG;
  }
}

int launch_fused_hll(Runtime* rt, const KeyDesc& key, int64_t n, cudaStream_t s) {
  EIGER_CUDA(cudaMemsetAsync(rt->prof->regs, 0, sizeof(uint32_t) * kHllM, s));
  if (n == 0) return EIGER_OK;
  const int64_t want = (n / 2 + (int64_t)kProfThreads * 4 - 1) / ((int64_t)kProfThreads * 4);
  const int blocks = (int)std::max<int64_t>(1, std::min<int64_t>(want, 2LL * rt->sm_count));
  auto kern = fused_hll_kernel;
  EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kHllM * 4));
  kern<<<blocks, kProfThreads, kHllM * 4, s>>>(key, n, rt->prof);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

int launch_fused_part_hist_hll(Runtime* rt, const KeyDesc& key, int key_kind, int64_t n, uint32_t sel, cudaStream_t s) {
  if (key_kind != KK_GEN && key_kind != KK_GEN32) return EIGER_ERR_ARG;
  profile_reset_kernel<<<16, 1024, 0, s>>>(rt->prof, 1);
  count_launch();
  const int64_t want = (n / 2 + (int64_t)kProfThreads * 4 - 1) / ((int64_t)kProfThreads * 4);
  const int blocks = (int)std::max<int64_t>(1, std::min<int64_t>(want, 2LL * rt->sm_count));
  const int smem = (kHllM + kPreFan) * 4 + (kProfThreads / 32) * 64 * 8;
  if (key_kind == KK_GEN32) {
    auto kern = fused_part_hist_hll_kernel<KK_GEN32>;
    EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    kern<<<blocks, kProfThreads, smem, s>>>(key, n, sel, rt->prof);
  } else {
    auto kern = fused_part_hist_hll_kernel<KK_GEN>;
    EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    kern<<<blocks, kProfThreads, smem, s>>>(key, n, sel, rt->prof);
  }
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

int launch_part_hist_hll(Runtime* rt, const void* keys, int dtype, int64_t n, uint64_t base, uint32_t sel, cudaStream_t s) {
  if (dtype != EIGER_I32 && dtype != EIGER_I64) return EIGER_ERR_ARG;
  profile_reset_kernel<<<16, 1024, 0, s>>>(rt->prof, 1);
  count_launch();
  const int epv = dtype == EIGER_I32 ? 4 : 2;
  const int64_t nvec = n / epv;
  const int64_t want = (nvec + (int64_t)kProfThreads * kProfUnroll - 1) / ((int64_t)kProfThreads * kProfUnroll);
  const int blocks = (int)std::max<int64_t>(1, std::min<int64_t>(want, 2LL * rt->sm_count));
  const int smem = (kHllM + kPreFan) * 4 + (kProfThreads / 32) * 64 * 8;
  if (dtype == EIGER_I32) {
    auto kern = part_hist_hll_kernel<EIGER_I32>;
    EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    kern<<<blocks, kProfThreads, smem, s>>>(keys, n, base, sel, rt->prof);
  } else {
    auto kern = part_hist_hll_kernel<EIGER_I64>;
    EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    kern<<<blocks, kProfThreads, smem, s>>>(keys, n, base, sel, rt->prof);
  }
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

int launch_profile_sample(Runtime* rt, const void* keys, int dtype, int64_t n, int64_t samples, int which, int with_hll,
                          bool reset, cudaStream_t s, bool last) {
  if (reset) {
    profile_reset_kernel<<<16, 1024, 0, s>>>(rt->prof, 1);
    count_launch();
  }
  if (n > 0 && samples > 0) {
    profile_sample_kernel<<<(unsigned)((samples + 255) / 256), 256, 0, s>>>(keys, dtype, n, samples, rt->prof, which, with_hll, last ? 1 : 0);
    count_launch();
  }
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

int launch_hot_keys(Runtime* rt, const void* keys, int dtype, int64_t n, cudaStream_t s) {
  if (n <= 0) return EIGER_ERR_ARG;
  constexpr int smem = kHotSlots * 12;
  EIGER_CUDA(cudaFuncSetAttribute(hot_keys_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  hot_keys_kernel<<<1, 1024, smem, s>>>(keys, dtype, n, rt->prof);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

int launch_hll_hist(Runtime* rt, cudaStream_t s) {
  hll_hist_kernel<<<1, 1024, 0, s>>>(rt->prof);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

int launch_regs_to_bytes(Runtime* rt, uint8_t* out, cudaStream_t s) {
  regs_to_bytes_kernel<<<kHllM / 256, 256, 0, s>>>(rt->prof, out);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

// Step A3 (R5): table-free estimator from the register-value histogram.
//   z = m tau(1 - C[q+1]/m); for k = q..1: z = (z + C[k]) / 2; z += m sigma(C[0]/m);
//   est = m^2 / (2 ln 2 z)
static double hll_sigma(double x) {
  if (x == 1.0) return INFINITY;
  double y = 1.0, z = x, prev;
  do { x *= x; prev = z; z += x * y; y += y; } while (prev != z);
  return z;
}
static double hll_tau(double x) {
  if (x == 0.0 || x == 1.0) return 0.0;
  double y = 1.0, z = 1.0 - x, prev;
  do { x = std::sqrt(x); prev = z; y *= 0.5; const double d = 1.0 - x; z -= d * d * y; } while (prev != z);
  return z / 3.0;
}
double hll_estimate_from_hist(const uint32_t* hist) {
  const double m = (double)kHllM;
  double z = m * hll_tau(1.0 - (double)hist[kHllQ + 1] / m);
  for (int k = kHllQ; k >= 1; --k) z = 0.5 * (z + (double)hist[k]);
  z += m * hll_sigma((double)hist[0] / m);
  return m * m / (2.0 * std::log(2.0) * z);
}

}  // namespace eiger
