// Order-preserving dictionary encoding of one key column, PAPER.md:171-211 (Algorithm 1) and
// PAPER.md:219-223 (smart key fusion: "If NDV is below a certain threshold, we will use dictionary
// encoding"; "it must preserve the order of the keys in the encoded values").
//
// The paper's five steps, on this library's own building blocks (api.cu: eiger_dict_encode):
//   (1) insert-and-find + (2) retrieveAll  = a COUNT group-by of the column: its hash table is the
//       paper's HT, its emitted keys are uniqueKeys (any variant; EIGER_AUTO picks it);
//   (3) argsort(uniqueKeys)                 = the radix sort of EIGER_SORT over the unique keys;
//   (4) scatter of the ranks                = dict_fill_kernel: key -> rank into a global
//       open-addressing table (rows.cuh: back_find_or_insert);
//   (5) gather                              = dict_gather_kernel: every row looks its key up.
// The paper materialises a per-row leader id (groupIdLoc, 8 bytes per row) in step 1 and gathers
// through it in step 5; here step 5 probes the table with the key itself, which costs the same
// random access per row and saves writing and re-reading 8 n bytes.
#include <algorithm>

#include "internal.h"
#include "rows.cuh"

namespace eiger {
namespace {

struct DictArgs {
  const void* keys; int32_t dtype; int64_t n;
  void* table; uint64_t cap;                    // [cap + 1] slots of 16 bytes: [u64 key][u64 rank]
  CallDev* call;
};

// rank r of the sorted unique keys -> table[key] = r
__global__ void __launch_bounds__(256) dict_fill_kernel(const __grid_constant__ DictArgs a) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  const int lane = threadIdx.x & 31;
  for (int64_t r0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x - lane; r0 < a.n; r0 += stride) {   // warp-uniform trips
    const int64_t r = r0 + lane;
    if (r < a.n) {
      const uint64_t u = sext_load(a.keys, a.dtype, r);
      uint64_t* cell = back_find_or_insert(a.table, a.cap, 16u, u, a.call);
      if (cell) *cell = (uint64_t)r;
    }
    __syncwarp();
  }
}

// codes[i] = table[keys[i]]; every key is in the table (step 1 saw all of them)
__global__ void __launch_bounds__(256) dict_gather_kernel(const __grid_constant__ DictArgs a, int32_t* __restrict__ codes) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  const int lane = threadIdx.x & 31;
  for (int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x - lane; i0 < a.n; i0 += stride) {
    const int64_t i = i0 + lane;
    if (i < a.n) {
      const uint64_t u = sext_load(a.keys, a.dtype, i);
      uint64_t slot = u == kEmpty64 ? a.cap : __umul64hi(table_hash64(u), a.cap);
      int32_t code = -1;
      bool done = false;
      int probes = 0;
      while (!done) {
        const unsigned long long* kp = reinterpret_cast<const unsigned long long*>(static_cast<const char*>(a.table) + slot * 16u);
        if (slot == a.cap) { code = (int32_t)kp[1]; done = true; }
        else {
          const unsigned long long k = __ldg(kp);
          if (k == u) { code = (int32_t)__ldg(kp + 1); done = true; }
          else if (k == kEmpty64 || ++probes >= kBackProbes) { atomicOr(&a.call->overflow, 1u); done = true; }
          else slot = slot + 1 == a.cap ? 0 : slot + 1;
        }
      }
      codes[i] = code;
    }
    __syncwarp();
  }
}

}  // namespace

int launch_dict_fill(const void* sorted_keys, int dtype, int64_t ndv, void* table, uint64_t cap, CallDev* call, int sm_count, cudaStream_t s) {
  DictArgs a{sorted_keys, dtype, ndv, table, cap, call};
  const int blocks = (int)std::max<int64_t>(1, std::min<int64_t>((ndv + 255) / 256, (int64_t)sm_count * 8));
  dict_fill_kernel<<<blocks, 256, 0, s>>>(a);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}
int launch_dict_gather(const void* keys, int dtype, int64_t n, const void* table, uint64_t cap, int32_t* codes, CallDev* call, int sm_count, cudaStream_t s) {
  DictArgs a{keys, dtype, n, const_cast<void*>(table), cap, call};
  const int blocks = (int)std::max<int64_t>(1, std::min<int64_t>((n + 255) / 256, (int64_t)sm_count * 16));
  dict_gather_kernel<<<blocks, 256, 0, s>>>(a, codes);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

}  // namespace eiger
