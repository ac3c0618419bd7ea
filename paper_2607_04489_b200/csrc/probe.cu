// Machine probes: the measured rates the selector's thresholds and the kernel designs rest on
// (DESIGN.md section 5 "machine facts").  The paper's crossovers are "platform-dependent"
// (PAPER.md:304-306); these micro-kernels measure, on the GPU the library runs on, how fast the
// building blocks of each variant are: streamed reads (ld.global vs cp.async.bulk + mbarrier),
// shared-memory and L2 atomics, distributed-shared-memory atomics / stores / bulk copies inside a
// thread-block cluster, and small bulk stores (the write-combining scatter).
// One entry point, eiger_probe(name, param, &result); `python -m paper_2607_04489_b200.probe`
// prints all of them.  Nothing on the hot path calls this file.
#include <algorithm>
#include <cstdio>
#include <cstring>

#include "internal.h"
#include "ring.cuh"

namespace eiger {
namespace {

__device__ __forceinline__ uint32_t xorshift(uint32_t& s) { s ^= s << 13; s ^= s >> 17; s ^= s << 5; return s; }

// ---- 1. streamed read: plain 16-byte loads, summed --------------------------------------------
__global__ void __launch_bounds__(1024) read_ldg_kernel(const uint4* __restrict__ p, int64_t nvec, unsigned long long* out) {
  uint32_t acc = 0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (; i + 3 * stride < nvec; i += 4 * stride) {
    uint4 v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = ldg_stream_16(p + i + k * stride);
#pragma unroll
    for (int k = 0; k < 4; ++k) acc += v[k].x ^ v[k].y ^ v[k].z ^ v[k].w;
  }
  for (; i < nvec; i += stride) { const uint4 v = ldg_stream_16(p + i); acc += v.x ^ v.y ^ v.z ^ v.w; }
  if (acc == 0x12345u) atomicAdd(out, 1ull);
}

// ---- 2. streamed read through cp.async.bulk into a shared-memory ring -------------------------
// One producer thread, `STAGES` stages of `chunk` bytes; all other threads consume from shared memory.
template <int STAGES>
__global__ void __launch_bounds__(1024) read_bulk_kernel(const unsigned char* __restrict__ p, int64_t bytes, int chunk, unsigned long long* out) {
  extern __shared__ __align__(128) unsigned char ring[];
  __shared__ __align__(8) uint64_t full[STAGES], empty[STAGES];
  const int tid = threadIdx.x, T = blockDim.x;
  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], T / 32); }
    mbar_fence_init();
  }
  __syncthreads();
  const int64_t n_chunks = bytes / chunk;
  uint32_t acc = 0;
  int64_t k = 0;
  // every thread walks the same chunk sequence; thread 0 additionally keeps the ring full
  int64_t issued = 0;
  auto issue = [&](int64_t c) {   // thread 0 only: c-th chunk of this CTA
    const int s = (int)(c % STAGES);
    if (c >= STAGES) mbar_wait(&empty[s], (uint32_t)((c / STAGES - 1) & 1));
    mbar_expect_tx(&full[s], (uint32_t)chunk);
    bulk_g2s(ring + (size_t)s * chunk, p + ((int64_t)blockIdx.x + c * gridDim.x) * chunk, (uint32_t)chunk, &full[s]);
  };
  const int64_t mine = (n_chunks - blockIdx.x + gridDim.x - 1) / gridDim.x;
  if (tid == 0) for (; issued < mine && issued < STAGES; ++issued) issue(issued);
  for (k = 0; k < mine; ++k) {
    const int s = (int)(k % STAGES);
    mbar_wait(&full[s], (uint32_t)((k / STAGES) & 1));
    const uint4* v = reinterpret_cast<const uint4*>(ring + (size_t)s * chunk);
    for (int i = tid; i < chunk / 16; i += T) { const uint4 x = v[i]; acc += x.x ^ x.y ^ x.z ^ x.w; }
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(&empty[s]);
    if (tid == 0 && issued < mine) { issue(issued); ++issued; }
  }
  if (acc == 0x12345u) atomicAdd(out, 1ull);
}

// ---- 3. shared-memory / distributed-shared-memory atomics ----------------------------------------
// mode 0: red.add.u32 x3 per "row" (count, sum-lo, rare carry replaced by a third add);
// mode 1: atom.add.u32 (returning) + red.add.u32 per row, carry computed from the return value;
// mode 2: ld + atom.cas per row (key look-up / claim); mode 3: st.v2.u32 per row (row exchange);
// owner CTA of a row = random rank of the cluster (cluster size 1 = plain shared memory).
template <int MODE>
__global__ void __launch_bounds__(1024) dsmem_kernel(int slots, int rows_per_thread, unsigned long long* out) {
  extern __shared__ __align__(16) uint32_t tab[];
  const int tid = threadIdx.x, T = blockDim.x;
  for (int i = tid; i < slots * 4; i += T) tab[i] = 0;
  const uint32_t C = cluster_size(), me = cluster_rank();
  cluster_sync_all();
  uint32_t rng = (blockIdx.x * 1024u + tid) * 2654435761u + 12345u;
  const uint32_t base = smem_u32(tab);
  uint32_t sink = 0;
  const uint32_t P = (uint32_t)slots * 4u;      // bytes per plane
  for (int r = 0; r < rows_per_thread; r += 4) {
    uint32_t addr[4], val[4], old[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t x = xorshift(rng);
      const uint32_t slot = __umulhi(x, (uint32_t)slots);
      const uint32_t owner = C > 1 ? (x & (C - 1)) : me;
      addr[k] = mapa(base + slot * (MODE == 3 ? 8u : 4u), owner);        // planes lo | cnt | hi | key of `slots` words each (mode 3: 8-byte rows)
      val[k] = x >> 3;
    }
    if constexpr (MODE == 0) {
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        asm volatile("red.shared::cluster.add.u32 [%0], %1;" :: "r"(addr[k]), "r"(val[k]) : "memory");
        asm volatile("red.shared::cluster.add.u32 [%0], %1;" :: "r"(addr[k] + P), "r"(1u) : "memory");
      }
    } else if constexpr (MODE == 1) {
#pragma unroll
      for (int k = 0; k < 4; ++k) asm volatile("atom.shared::cluster.add.u32 %0, [%1], %2;" : "=r"(old[k]) : "r"(addr[k]), "r"(val[k]) : "memory");
#pragma unroll
      for (int k = 0; k < 4; ++k) asm volatile("red.shared::cluster.add.u32 [%0], %1;" :: "r"(addr[k] + P), "r"(1u) : "memory");
#pragma unroll
      for (int k = 0; k < 4; ++k) if ((uint32_t)(old[k] + val[k]) < val[k]) asm volatile("red.shared::cluster.add.u32 [%0], %1;" :: "r"(addr[k] + 2 * P), "r"(1u) : "memory");
    } else if constexpr (MODE == 2) {
#pragma unroll
      for (int k = 0; k < 4; ++k) asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(old[k]) : "r"(addr[k] + 3 * P) : "memory");
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (old[k] == 0u) asm volatile("atom.shared::cluster.cas.b32 %0, [%1], %2, %3;" : "=r"(old[k]) : "r"(addr[k] + 3 * P), "r"(0u), "r"(val[k] | 1u) : "memory");
        sink += old[k];
      }
    } else {
#pragma unroll
      for (int k = 0; k < 4; ++k) asm volatile("st.shared::cluster.v2.u32 [%0], {%1, %2};" :: "r"(addr[k]), "r"(val[k]), "r"(sink) : "memory");
    }
  }
  cluster_sync_all();
  if (sink == 0x12345u || tab[tid % (slots * 4)] == 0xdeadbeefu) atomicAdd(out, 1ull);
}

// ---- 4. bulk copies shared -> remote shared inside a cluster ---------------------------------------
// every CTA sends `chunk`-byte blocks round-robin to the other CTAs of its cluster; the receiver's
// mbarrier counts the bytes.  One elected thread per CTA issues (that is how TMA is driven).
__global__ void __launch_bounds__(128) dsmem_bulk_kernel(int chunk, int rounds, unsigned long long* out) {
  extern __shared__ __align__(128) unsigned char buf[];       // [send chunk][recv: C chunks]
  __shared__ __align__(8) uint64_t bar;
  const uint32_t C = cluster_size(), me = cluster_rank();
  const int tid = threadIdx.x;
  if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
  for (int i = tid; i < chunk / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(buf)[i] = i;
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  cluster_sync_all();
  for (int r = 0; r < rounds; ++r) {
    if (tid == 0) {
      // expect what the C - 1 peers will send me this round, then send my block to every peer
      mbar_expect_tx(&bar, (uint32_t)chunk * (C - 1));
      for (uint32_t d = 1; d < C; ++d) {
        const uint32_t peer = (me + d) % C;
        const uint32_t dst = mapa(smem_u32(buf + (size_t)chunk * (1 + me)), peer);
        const uint32_t rbar = mapa(smem_u32(&bar), peer);
        asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     :: "r"(dst), "r"(smem_u32(buf)), "r"((uint32_t)chunk), "r"(rbar) : "memory");
      }
      mbar_wait(&bar, (uint32_t)(r & 1));
    }
    // the next round overwrites the receive area: everyone has to be done reading (nobody reads here)
    cluster_sync_all();
  }
  if (buf[chunk + tid] == 0xee && tid == 127) atomicAdd(out, 1ull);
}

// ---- 5. small stores to random aligned destinations: bulk (TMA) vs one warp-wide store ------------
// mode 0: cp.async.bulk shared -> global, `chunk` bytes per copy, one issuing lane per warp;
// mode 1: the warp writes the same chunk with 16-byte (chunk >= 512), 8-byte or 4-byte stores.
template <int MODE>
__global__ void __launch_bounds__(512) small_store_kernel(unsigned char* dst, int64_t dst_chunks, int chunk, int per_warp, unsigned long long* out) {
  extern __shared__ __align__(128) unsigned char stage[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int i = tid; i < (int)(blockDim.x / 32) * chunk / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(stage)[i] = i;
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncthreads();
  uint32_t rng = (blockIdx.x * 512u + (tid & ~31)) * 2654435761u + 777u;
  unsigned char* mine = stage + (size_t)warp * chunk;
  for (int k = 0; k < per_warp; ++k) {
    const uint64_t c = ((uint64_t)xorshift(rng) * (uint64_t)dst_chunks) >> 32;
    unsigned char* d = dst + c * (uint64_t)chunk;
    if constexpr (MODE == 0) {
      if (lane == 0) {
        bulk_s2g(d, mine, (uint32_t)chunk);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        if ((k & 7) == 7) asm volatile("cp.async.bulk.wait_group.read 4;" ::: "memory");
      }
    } else {
      if (chunk >= 512) { for (int o = lane * 16; o < chunk; o += 512) *reinterpret_cast<uint4*>(d + o) = *reinterpret_cast<const uint4*>(mine + o); }
      else if (chunk >= 256) { *reinterpret_cast<uint2*>(d + lane * 8) = *reinterpret_cast<const uint2*>(mine + lane * 8); }
      else if (lane * 4 < chunk) { *reinterpret_cast<uint32_t*>(d + lane * 4) = *reinterpret_cast<const uint32_t*>(mine + lane * 4); }
    }
  }
  if constexpr (MODE == 0) { if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
  if (stage[tid] == 0xee && out) atomicAdd(out, 1ull);
}

// ---- 6. global (L2) reductions on a table of `cells` 8-byte cells ---------------------------------
__global__ void __launch_bounds__(1024) l2_red_kernel(unsigned long long* table, uint32_t cells, int rows_per_thread) {
  uint32_t rng = (blockIdx.x * 1024u + threadIdx.x) * 2654435761u + 99u;
  for (int r = 0; r < rows_per_thread; ++r) {
    const uint32_t x = xorshift(rng);
    const uint32_t c = __umulhi(x, cells);
    atomicAdd(table + 2 * (size_t)c, (unsigned long long)(x >> 3));
    atomicAdd(table + 2 * (size_t)c + 1, 1ull);
  }
}

struct Scratch { void* p = nullptr; size_t bytes = 0; };
int reserve(Scratch& s, size_t bytes) {
  if (s.bytes >= bytes) return EIGER_OK;
  if (s.p) cudaFree(s.p);
  s.p = nullptr; s.bytes = 0;
  EIGER_CUDA(cudaMalloc(&s.p, bytes));
  s.bytes = bytes;
  return EIGER_OK;
}

template <class F>
int timed(cudaStream_t s, int reps, double* ms_out, F&& launch) {
  cudaEvent_t a, b;
  EIGER_CUDA(cudaEventCreate(&a)); EIGER_CUDA(cudaEventCreate(&b));
  int rc = launch(); if (rc) return rc;                    // warm-up
  EIGER_CUDA(cudaStreamSynchronize(s));
  float best = 1e30f;
  for (int i = 0; i < reps; ++i) {
    EIGER_CUDA(cudaEventRecord(a, s));
    rc = launch(); if (rc) return rc;
    EIGER_CUDA(cudaEventRecord(b, s));
    EIGER_CUDA(cudaEventSynchronize(b));
    float ms = 0; EIGER_CUDA(cudaEventElapsedTime(&ms, a, b));
    best = std::min(best, ms);
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  *ms_out = best;
  return EIGER_OK;
}

template <class K, class... A>
int launch_cluster(K kern, int grid, int block, size_t smem, int cluster, cudaStream_t s, A... args) {
  if (smem > 48 * 1024) EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  if (cluster > 8) EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  EIGER_CUDA(cudaLaunchKernelEx(&cfg, kern, args...));
  return EIGER_OK;
}

}  // namespace
}  // namespace eiger

using namespace eiger;

extern "C" int eiger_probe(const char* name, int64_t param, int64_t param2, double* result, void* stream) {
  if (!name || !result) return EIGER_ERR_ARG;
  Runtime* rt = runtime();
  if (!rt) return EIGER_ERR_CUDA;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  static Scratch big, cnt;
  int rc = reserve(cnt, 256); if (rc) return rc;
  unsigned long long* out = static_cast<unsigned long long*>(cnt.p);
  const int sms = rt->sm_count;
  double ms = 0;
  *result = 0;
  if (!std::strcmp(name, "read_ldg") || !std::strcmp(name, "read_bulk")) {
    // param = MiB to read (default 4096), param2 = chunk bytes of the bulk ring (default 16384); result = GB/s
    const size_t bytes = (size_t)(param > 0 ? param : 4096) << 20;
    rc = reserve(big, bytes); if (rc) return rc;
    EIGER_CUDA(cudaMemsetAsync(big.p, 1, bytes, s));
    if (!std::strcmp(name, "read_ldg")) {
      rc = timed(s, 5, &ms, [&] { read_ldg_kernel<<<sms * 2, 1024, 0, s>>>(static_cast<const uint4*>(big.p), (int64_t)(bytes / 16), out); return cudaGetLastError() == cudaSuccess ? 0 : EIGER_ERR_CUDA; });
    } else {
      const int chunk = (int)(param2 > 0 ? param2 : 16384);
      constexpr int ST = 4;
      auto kern = read_bulk_kernel<ST>;
      EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, ST * chunk));
      rc = timed(s, 5, &ms, [&] { kern<<<sms, 512, (size_t)ST * chunk, s>>>(static_cast<const unsigned char*>(big.p), (int64_t)bytes, chunk, out); return cudaGetLastError() == cudaSuccess ? 0 : EIGER_ERR_CUDA; });
    }
    if (rc) return rc;
    *result = (double)bytes / (ms * 1e-3) / 1e9;
    return EIGER_OK;
  }
  if (!std::strncmp(name, "dsmem_", 6) && std::strcmp(name, "dsmem_bulk")) {
    // param = cluster size (1, 2, 4, 8, 16), param2 = slots per CTA (16 bytes each, default 8192); result = G rows/s
    const int C = (int)(param > 0 ? param : 1);
    const int slots = (int)(param2 > 0 ? param2 : 8192);
    const int grid = sms / C * C, rows = 4096;
    const size_t smem = (size_t)slots * 16;
    auto run = [&](auto kern) { return timed(s, 5, &ms, [&] { return launch_cluster(kern, grid, 1024, smem, C, s, slots, rows, out); }); };
    if (!std::strcmp(name, "dsmem_red")) rc = run(dsmem_kernel<0>);
    else if (!std::strcmp(name, "dsmem_atom")) rc = run(dsmem_kernel<1>);
    else if (!std::strcmp(name, "dsmem_cas")) rc = run(dsmem_kernel<2>);
    else if (!std::strcmp(name, "dsmem_st")) rc = run(dsmem_kernel<3>);
    else return EIGER_ERR_ARG;
    if (rc) return rc;
    *result = (double)grid * 1024.0 * rows / (ms * 1e-3) / 1e9;
    return EIGER_OK;
  }
  if (!std::strcmp(name, "dsmem_bulk")) {
    // param = cluster size, param2 = chunk bytes (default 4096); result = GB/s received chip-wide
    const int C = (int)(param > 1 ? param : 2);
    const int chunk = (int)(param2 > 0 ? param2 : 4096);
    const int grid = sms / C * C, rounds = 2000;
    const size_t smem = (size_t)chunk * (1 + C);
    rc = timed(s, 3, &ms, [&] { return launch_cluster(dsmem_bulk_kernel, grid, 128, smem, C, s, chunk, rounds, out); });
    if (rc) return rc;
    *result = (double)grid * (C - 1) * (double)chunk * rounds / (ms * 1e-3) / 1e9;
    return EIGER_OK;
  }
  if (!std::strcmp(name, "store_bulk") || !std::strcmp(name, "store_warp")) {
    // param = chunk bytes (128 .. 4096), param2 = MiB of destination (default 4096); result = GB/s written
    const int chunk = (int)(param > 0 ? param : 256);
    const size_t bytes = (size_t)(param2 > 0 ? param2 : 4096) << 20;
    rc = reserve(big, bytes); if (rc) return rc;
    const int per_warp = 4096, grid = sms * 2;
    const size_t smem = (size_t)16 * chunk;
    auto run = [&](auto kern) {
      if (smem > 48 * 1024) { cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); }
      return timed(s, 3, &ms, [&] { kern<<<grid, 512, smem, s>>>(static_cast<unsigned char*>(big.p), (int64_t)(bytes / chunk), chunk, per_warp, out); return cudaGetLastError() == cudaSuccess ? 0 : EIGER_ERR_CUDA; });
    };
    rc = !std::strcmp(name, "store_bulk") ? run(small_store_kernel<0>) : run(small_store_kernel<1>);
    if (rc) return rc;
    *result = (double)grid * 16.0 * per_warp * chunk / (ms * 1e-3) / 1e9;
    return EIGER_OK;
  }
  if (!std::strcmp(name, "l2_red")) {
    // param = log2 cells (16 bytes each); result = G rows/s (two 64-bit RED per row)
    const uint32_t cells = 1u << (int)(param > 0 ? param : 16);
    rc = reserve(big, (size_t)cells * 16); if (rc) return rc;
    EIGER_CUDA(cudaMemsetAsync(big.p, 0, (size_t)cells * 16, s));
    const int rows = 1024;
    rc = timed(s, 3, &ms, [&] { l2_red_kernel<<<sms * 2, 1024, 0, s>>>(static_cast<unsigned long long*>(big.p), cells, rows); return cudaGetLastError() == cudaSuccess ? 0 : EIGER_ERR_CUDA; });
    if (rc) return rc;
    *result = (double)sms * 2 * 1024.0 * rows / (ms * 1e-3) / 1e9;
    return EIGER_OK;
  }
  if (!std::strcmp(name, "release")) {
    if (big.p) cudaFree(big.p);
    big = Scratch{};
    return EIGER_OK;
  }
  return EIGER_ERR_ARG;
}
