// Step A6d, first half: radix partition of the rows by the top bits of the table hash
// ("applies a hash function to the keys before partitioning to ensure more even partition
// sizes", §3.3; best for g > 2^20).  Keys leave this pass
// already rebased and fused (KK_U64PRE); value columns travel with their keys (the paper's
// GFTR).  Because the global table's slot is mulhi(hash, cap), rows of one
// partition land in one contiguous slice of the table, which is what keeps the following
// BACK_HASH pass inside L2.
#include <algorithm>

#include "internal.h"

namespace eiger {
namespace {

constexpr int kPartThreads = 256;
constexpr int kPartRows = 8;              // rows per thread per tile
constexpr int kMaxPartBits = 12;

template <int KK> struct PK;
template <> struct PK<KK_I32> { using U = uint32_t; };
template <> struct PK<KK_I64> { using U = uint64_t; };
template <> struct PK<KK_GEN> { using U = uint64_t; };

template <int KK>
__device__ __forceinline__ uint64_t part_load_u(const KeyDesc& k, int64_t i) {
  if constexpr (KK == KK_I32) return (uint64_t)(uint32_t)(ldg_stream_4((const int32_t*)k.ptr[0] + i) - (uint32_t)k.base[0]);
  else if constexpr (KK == KK_I64) return ldg_stream_u64((const int64_t*)k.ptr[0] + i) - k.base[0];
  else {
    uint64_t u = sext_load(k.ptr[0], k.dtype[0], i) - k.base[0];
    if (k.ncols == 2) u = u * k.mul + (sext_load(k.ptr[1], k.dtype[1], i) - k.base[1]);
    return u;
  }
}

template <int KK>
__global__ void __launch_bounds__(kPartThreads)
partition_hist_kernel(const __grid_constant__ KeyDesc key, int64_t n, int bits, uint32_t* __restrict__ hist) {
  __shared__ uint32_t s_hist[1 << kMaxPartBits];
  const int P = 1 << bits;
  for (int p = threadIdx.x; p < P; p += kPartThreads) s_hist[p] = 0;
  __syncthreads();
  const int64_t stride = (int64_t)gridDim.x * kPartThreads;
  for (int64_t i = (int64_t)blockIdx.x * kPartThreads + threadIdx.x; i < n; i += stride) {
    const uint64_t u = part_load_u<KK>(key, i);
    atomicAdd(&s_hist[(uint32_t)(table_hash64(u) >> (64 - bits))], 1u);
  }
  __syncthreads();
  for (int p = threadIdx.x; p < P; p += kPartThreads) if (s_hist[p]) atomicAdd(&hist[p], s_hist[p]);
}

// exclusive prefix sum of P <= 4096 counts -> 64-bit write cursors
__global__ void partition_scan_kernel(const uint32_t* __restrict__ hist, unsigned long long* __restrict__ cursor, int P) {
  __shared__ unsigned long long s_part[1024];
  const int per = (P + 1023) / 1024;
  unsigned long long local = 0;
  for (int k = 0; k < per; ++k) { const int p = threadIdx.x * per + k; if (p < P) local += hist[p]; }
  s_part[threadIdx.x] = local;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {
    const unsigned long long v = threadIdx.x >= o ? s_part[threadIdx.x - o] : 0ull;
    __syncthreads();
    s_part[threadIdx.x] += v;
    __syncthreads();
  }
  unsigned long long run = s_part[threadIdx.x] - local;
  for (int k = 0; k < per; ++k) { const int p = threadIdx.x * per + k; if (p < P) { cursor[p] = run; run += hist[p]; } }
}

struct ScatterArgs {
  KeyDesc key;
  const uint64_t* vals[kMaxVals];
  uint64_t* out_vals[kMaxVals];
  uint64_t* out_u;
  unsigned long long* cursor;
  int64_t n;
  int n_vals, bits;
};

template <int KK>
__global__ void __launch_bounds__(kPartThreads)
partition_scatter_kernel(const __grid_constant__ ScatterArgs a) {
  __shared__ uint32_t s_cnt[1 << kMaxPartBits];
  __shared__ unsigned long long s_base[1 << kMaxPartBits];
  const int P = 1 << a.bits, tid = threadIdx.x;
  constexpr int64_t kTile = (int64_t)kPartThreads * kPartRows;
  const int64_t n_tiles = (a.n + kTile - 1) / kTile;
  for (int p = tid; p < P; p += kPartThreads) s_cnt[p] = 0;
  __syncthreads();
  for (int64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
    uint64_t u[kPartRows];
    uint32_t part[kPartRows], rank[kPartRows];
#pragma unroll
    for (int r = 0; r < kPartRows; ++r) {
      const int64_t i = t * kTile + (int64_t)r * kPartThreads + tid;
      if (i < a.n) {
        u[r] = part_load_u<KK>(a.key, i);
        part[r] = (uint32_t)(table_hash64(u[r]) >> (64 - a.bits));
        rank[r] = atomicAdd(&s_cnt[part[r]], 1u);
      }
    }
    __syncthreads();
    for (int p = tid; p < P; p += kPartThreads) {
      const uint32_t c = s_cnt[p];
      if (c) s_base[p] = atomicAdd(&a.cursor[p], (unsigned long long)c);
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kPartRows; ++r) {
      const int64_t i = t * kTile + (int64_t)r * kPartThreads + tid;
      if (i < a.n) {
        const unsigned long long dst = s_base[part[r]] + rank[r];
        a.out_u[dst] = u[r];
        for (int c = 0; c < a.n_vals; ++c) a.out_vals[c][dst] = ldg_stream_u64(a.vals[c] + i);
      }
    }
    __syncthreads();
    for (int p = tid; p < P; p += kPartThreads) s_cnt[p] = 0;
    __syncthreads();
  }
}

template <int KK>
int launch_kk(const PartitionLaunch& L, int sm_count, cudaStream_t s) {
  const int P = 1 << L.bits;
  EIGER_CUDA(cudaMemsetAsync(L.hist, 0, sizeof(uint32_t) * P, s));
  const int64_t want = (L.n + kPartThreads * 16 - 1) / (kPartThreads * 16);
  const int blocks = (int)std::max<int64_t>(1, std::min<int64_t>(want, (int64_t)sm_count * 6));
  partition_hist_kernel<KK><<<blocks, kPartThreads, 0, s>>>(L.key, L.n, L.bits, L.hist);
  count_launch();
  partition_scan_kernel<<<1, 1024, 0, s>>>(L.hist, L.cursor, P);
  count_launch();
  ScatterArgs a;
  a.key = L.key; a.out_u = L.out_u; a.cursor = L.cursor; a.n = L.n; a.n_vals = L.plan.n_vals; a.bits = L.bits;
  for (int c = 0; c < kMaxVals; ++c) { a.vals[c] = static_cast<const uint64_t*>(L.plan.vals[c]); a.out_vals[c] = L.out_vals[c]; }
  const int64_t tiles = (L.n + kPartThreads * kPartRows - 1) / (kPartThreads * kPartRows);
  const int sblocks = (int)std::max<int64_t>(1, std::min<int64_t>(tiles, (int64_t)sm_count * 4));
  partition_scatter_kernel<KK><<<sblocks, kPartThreads, 0, s>>>(a);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

}  // namespace

int launch_partition(const PartitionLaunch& L, int sm_count, cudaStream_t s) {
  if (L.bits < 1 || L.bits > kMaxPartBits) return EIGER_ERR_ARG;
  switch (L.key_kind) {
    case KK_I32: return launch_kk<KK_I32>(L, sm_count, s);
    case KK_I64: return launch_kk<KK_I64>(L, sm_count, s);
    case KK_GEN: case KK_I8I8: return launch_kk<KK_GEN>(L, sm_count, s);
    default: return EIGER_ERR_ARG;
  }
}

}  // namespace eiger
