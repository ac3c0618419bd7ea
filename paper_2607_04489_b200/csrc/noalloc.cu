// eiger_groupby_direct_static: the direct-index variant ("array-based" group-by
// when the key range is small) for callers that must not allocate - code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc.  The accumulator array that the ordinary
// path carves from a workspace or from the library's arena lives here in a file-scope __device__
// array of a fixed, modest size (kStaticMaxSlots slots: 1 MiB + a 256-byte header per GPU that
// loads the library, held until the process exits).  Nothing in this file calls cudaMalloc, cudaFree,
// runtime() or any other allocating routine.
//
// Every call on a device shares the one array and finds the previous call's contents in it: the
// header and the slots a call will use are cleared at its start, on the caller's stream.  Calls that
// overlap on the GPU (different streams, different host threads) therefore race on the array.
#include <mutex>

#include "internal.h"

namespace eiger {
namespace {

constexpr uint32_t kStaticMaxSlots = EIGER_STATIC_MAX_SLOTS;
constexpr uint32_t kHeaderWords = 32;     // 256 bytes: [0] groups emitted, [1] rows outside [key_min, key_max]
constexpr int kMaxDevices = 64;

// In host code this name is a host-side stand-in for the device array, not a device address:
// static_scratch() asks the runtime for the address on the current device and kernels get THAT.
static __device__ __align__(256) unsigned long long g_static_scratch[kHeaderWords + 2ull * kStaticMaxSlots];

std::mutex g_static_mu;
unsigned long long* g_static_ptr[kMaxDevices] = {};

// the array's device address on the current device, looked up once per device
int static_scratch(unsigned long long** out) {
  int dev = -1;
  EIGER_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return EIGER_ERR_ARG;
  std::lock_guard<std::mutex> lk(g_static_mu);
  if (!g_static_ptr[dev]) {
    unsigned long long* p = nullptr;
    EIGER_CUDA(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_scratch));
    g_static_ptr[dev] = p;
  }
  *out = g_static_ptr[dev];
  return EIGER_OK;
}

template <class K>
__global__ void __launch_bounds__(256)
static_direct_kernel(const K* __restrict__ keys, const long long* __restrict__ vals, long long n, long long key_min,
                     unsigned long long range, unsigned long long* __restrict__ scratch) {
  unsigned long long* sum = scratch + kHeaderWords;
  unsigned long long* cnt = sum + range;
  bool bad = false;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const unsigned long long u = (unsigned long long)(long long)keys[i] - (unsigned long long)key_min;   // wraps
    if (u < range) {
      atomicAdd(sum + u, (unsigned long long)vals[i]);      // result unused: a reduction at the L2
      atomicAdd(cnt + u, 1ull);
    } else {
      bad = true;
    }
  }
  if (bad) scratch[1] = 1ull;
}

template <class K>
__global__ void __launch_bounds__(256)
static_emit_kernel(unsigned long long range, long long key_min, unsigned long long* __restrict__ scratch,
                   K* __restrict__ out_keys, long long* __restrict__ out_sum, long long* __restrict__ out_count,
                   unsigned long long capacity) {
  const unsigned long long* sum = scratch + kHeaderWords;
  const unsigned long long* cnt = sum + range;
  const int lane = threadIdx.x & 31;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  const unsigned long long first = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  for (unsigned long long u0 = first - lane; u0 < range; u0 += stride) {       // warp-uniform trip count
    const unsigned long long u = u0 + lane;
    const unsigned long long c = u < range ? cnt[u] : 0ull;
    const uint32_t m = __ballot_sync(0xffffffffu, c != 0ull);
    if (!m) continue;
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(scratch, (unsigned long long)__popc(m));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (c != 0ull) {
      const unsigned long long pos = base + __popc(m & ((1u << lane) - 1u));
      if (pos < capacity) {
        out_keys[pos] = (K)(long long)((unsigned long long)key_min + u);
        out_sum[pos] = (long long)sum[u];
        out_count[pos] = (long long)c;
      }
    }
  }
}

template <class K>
int run_static(const void* keys, int64_t n, int64_t key_min, uint64_t range, const int64_t* vals, void* out_keys,
               int64_t* out_sum, int64_t* out_count, int64_t out_capacity, unsigned long long* scratch, cudaStream_t s) {
  int dev = 0, sms = 0;
  EIGER_CUDA(cudaGetDevice(&dev));
  EIGER_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const long long want = (n + 255) / 256;
  const int gx = (int)(want < (long long)sms * 8 ? want : (long long)sms * 8);
  static_direct_kernel<K><<<gx, 256, 0, s>>>(static_cast<const K*>(keys), reinterpret_cast<const long long*>(vals),
                                             (long long)n, (long long)key_min, range, scratch);
  const int ge = (int)((range + 255) / 256 < (uint64_t)sms * 4 ? (range + 255) / 256 : (uint64_t)sms * 4);
  static_emit_kernel<K><<<ge, 256, 0, s>>>(range, (long long)key_min, scratch, static_cast<K*>(out_keys),
                                           reinterpret_cast<long long*>(out_sum), reinterpret_cast<long long*>(out_count),
                                           (unsigned long long)out_capacity);
  count_launch(2);
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

}  // namespace
}  // namespace eiger

extern "C" {

int64_t eiger_static_max_slots(void) { return (int64_t)eiger::kStaticMaxSlots; }

int eiger_groupby_direct_static(const void* keys, int32_t key_dtype, int64_t n, int64_t key_min, int64_t key_max,
                                const int64_t* vals, void* out_keys, int64_t* out_sum, int64_t* out_count,
                                int64_t out_capacity, int64_t* n_groups, void* stream) {
  using namespace eiger;
  if (!n_groups) return EIGER_ERR_ARG;
  *n_groups = 0;
  if (n < 0 || out_capacity < 0 || key_max < key_min) return EIGER_ERR_ARG;
  if (key_dtype != EIGER_I8 && key_dtype != EIGER_I32 && key_dtype != EIGER_I64) return EIGER_ERR_ARG;
  const uint64_t span = (uint64_t)key_max - (uint64_t)key_min;             // range - 1; cannot wrap: key_max >= key_min
  if (span >= (uint64_t)kStaticMaxSlots) return EIGER_ERR_STATIC_LIMIT;
  const uint64_t range = span + 1;
  if (n == 0) return EIGER_OK;
  if (!keys || !vals || (out_capacity > 0 && (!out_keys || !out_sum || !out_count))) return EIGER_ERR_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(stream);

  unsigned long long* scratch = nullptr;
  if (int rc = static_scratch(&scratch)) return rc;
  // the array keeps the last call's contents: the header and this call's slots start at zero
  EIGER_CUDA(cudaMemsetAsync(scratch, 0, (kHeaderWords + 2 * range) * sizeof(unsigned long long), s));
  int rc = EIGER_OK;
  switch (key_dtype) {
    case EIGER_I8:  rc = run_static<int8_t>(keys, n, key_min, range, vals, out_keys, out_sum, out_count, out_capacity, scratch, s); break;
    case EIGER_I32: rc = run_static<int32_t>(keys, n, key_min, range, vals, out_keys, out_sum, out_count, out_capacity, scratch, s); break;
    default:        rc = run_static<int64_t>(keys, n, key_min, range, vals, out_keys, out_sum, out_count, out_capacity, scratch, s); break;
  }
  if (rc) return rc;
  unsigned long long back[2] = {0, 0};                                     // groups, rows out of range
  EIGER_CUDA(cudaMemcpyAsync(back, scratch, sizeof(back), cudaMemcpyDeviceToHost, s));
  EIGER_CUDA(cudaStreamSynchronize(s));
  if (back[1]) return EIGER_ERR_STATS;
  *n_groups = (int64_t)back[0];
  return (int64_t)back[0] > out_capacity ? EIGER_ERR_OUT_CAPACITY : EIGER_OK;
}

}  // extern "C"
