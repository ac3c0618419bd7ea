// Host-side declarations shared by the translation units of libeiger.
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

#include "dev.cuh"

namespace eiger {

constexpr int kPairWords = 8192;     // 2^18 samples
// Device block owned by the library (allocated once): profile outputs and call counters.
struct ProfileDev {
  long long min[kMaxKeyCols];
  long long max[kMaxKeyCols];
  uint32_t hist[64];        // register-value histogram C[0 .. kHllQ + 1]
  uint32_t pair_eq, pair_n; // sample pass: adjacent sample keys that are equal / compared (skew test)
  uint32_t oor, oor_pad;    // fused slice-sketch pass: some row had a key column outside the planned range
  uint32_t regs[kHllM];     // sketch registers, one per word (global atomicMax)
  uint32_t part_hist[kPreFan];   // rows per level-1 partition at fan-out kPreFan (slice-sketch pass)
  long long hot_key[kMaxHot];    // heavy hitters of a key sample (hot_keys pass), most frequent first
  uint32_t hot_cnt[kMaxHot];     // their sample counts
  uint32_t hot_n, hot_samples;
  uint32_t pair_mask[kPairWords];   // sample pass over several key columns: neighbouring sample rows equal in every column so far
};
struct CallDev {
  unsigned long long n_groups;   // compaction claim counter
  uint32_t overflow;             // a hash table ran out of probes
  uint32_t abort;                // speculative pass: some CTA's shared-memory table filled up
  unsigned long long spill_chunks;   // EIGER_GLOBAL with a spill buffer: chunks reserved so far (may exceed the buffer)
};

struct Runtime {
  int device = -1;
  int sm_count = 0;
  size_t smem_optin = 0;
  size_t l2_bytes = 0;
  ProfileDev* prof = nullptr;    // device
  CallDev* call = nullptr;       // device
  void* pinned = nullptr;        // host staging for small read-backs (64 KB)
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
};
Runtime* runtime();              // lazily initialised for the current device; nullptr on failure
void count_launch(int k = 1);
int cuda_fail(cudaError_t e, const char* what);   // records the message, returns EIGER_ERR_CUDA
#define EIGER_CUDA(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) return ::eiger::cuda_fail(e__, #expr); } while (0)

// ---- profile.cu ------------------------------------------------------------------------
// Fused min/max (+ sketch registers) over one key column into rt->prof, slot `which` of
// min/max.  with_hll = 0 skips the sketch (range-first order).
int launch_profile(Runtime* rt, const void* keys, int dtype, int64_t n, int which, int with_hll,
                   bool reset, cudaStream_t s);
int launch_profile_sample(Runtime* rt, const void* keys, int dtype, int64_t n, int64_t samples, int which, int with_hll,
                          bool reset, cudaStream_t s, bool last = true);   // last: the final column of a multi-column key (counts the equal neighbour rows)
// Keys-only pass of EIGER_AUTO when the sample already settles PARTITION: exact min/max, the
// partition histogram at fan-out kPreFan of u = key - base, and the sketch of the keys whose
// partition id is below `sel` (a slice of the hash space: NDV = slice NDV * kPreFan / sel).
int launch_part_hist_hll(Runtime* rt, const void* keys, int dtype, int64_t n, uint64_t base, uint32_t sel, cudaStream_t s);
// The same for several key columns: histogram and slice sketch of the FUSED key (key.base / rng / mul / flags from
// the sample's ranges; key_kind KK_GEN or KK_GEN32); rt->prof->oor != 0 afterwards: a row lay outside those ranges.
int launch_fused_part_hist_hll(Runtime* rt, const KeyDesc& key, int key_kind, int64_t n, uint32_t sel, cudaStream_t s);
// Heavy hitters of an evenly spaced key sample (single CTA): keys that own more than ~0.5 % of
// the sample, at most kMaxHot, into rt->prof->hot_*.  EIGER_AUTO runs it when the sample's
// collision rate says the keys are skewed; the whole-input hash kernel then reduces those keys'
// rows inside the warp instead of hammering one shared-memory slot with atomics.
int launch_hot_keys(Runtime* rt, const void* keys, int dtype, int64_t n, cudaStream_t s);
// Sketch registers of the fused key of a multi-column key (key.base / rng / flags filled in) into
// rt->prof->regs; launch_hll_hist then gives the histogram the estimator reads.
int launch_fused_hll(Runtime* rt, const KeyDesc& key, int64_t n, cudaStream_t s);
int launch_hll_hist(Runtime* rt, cudaStream_t s);
int launch_regs_to_bytes(Runtime* rt, uint8_t* out, cudaStream_t s);
double hll_estimate_from_hist(const uint32_t* hist);

// ---- aggregate.cu ----------------------------------------------------------------------
enum FrontKind : int { FRONT_NONE = 0, FRONT_PRIV = 1, FRONT_SDIRECT = 2, FRONT_SHASH = 3, FRONT_DICT = 4, FRONT_SPLIT = 5 };
enum BackKind : int { BACK_DIRECT = 0, BACK_HASH = 1 };

struct AggLaunch {
  KeyDesc key;
  AggPlan plan;
  int64_t n;
  int key_kind, sig, front, back;
  // front
  int spec;                 // speculative: a key outside [0, cap) raises call->abort instead of being aggregated
  uint32_t front_slots;     // SDIRECT: R; PRIV: R
  uint32_t front_limit;     // SHASH: stop inserting new keys beyond this many
  uint32_t front_replicas;  // SDIRECT: table copies per CTA
  // back
  void* table;              // DIRECT: [cap][n_acc] cells; HASH: [cap] slots of `stride` bytes
  uint64_t cap;
  uint32_t stride;          // HASH: bytes per slot (power of two); DIRECT: 8 * n_acc
  CallDev* call;
  // FRONT_DICT: dictionary image (key, dense id) of dict_slots entries (a power of two), slot = (u * mul) >> dict_shift
  void* dict; uint32_t dict_slots, dict_shift;
  uint32_t dict_compact;    // FRONT_DICT: the large-dictionary shared-memory layout (aggregate.cu: AggArgs)
  uint32_t dict_group;      // FRONT_DICT, small layout: 2 = entries are placed and searched in pairs (SUM + COUNT plans, one replica)
  uint32_t dict_pass_lg, dict_pass;   // FRONT_DICT, several passes: this launch aggregates key slice dict_pass of 2^dict_pass_lg
  // launch shape
  int threads, blocks;
  size_t smem_bytes;
};
int launch_dict_build(const AggLaunch& a, int64_t samples, uint32_t* dict_keys, uint32_t* dict_n, cudaStream_t s);
int launch_table_init(const AggLaunch& a, cudaStream_t s);
int launch_aggregate(const AggLaunch& a, cudaStream_t s);
bool aggregate_supported(int key_kind, int sig, int front, int back);

struct CompactLaunch {
  KeyDesc key;              // for un-fusing / un-rebasing
  AggPlan plan;
  int back;
  const void* table; uint64_t cap; uint32_t stride;
  void* out_keys[kMaxKeyCols]; void* out_aggs[kMaxAggs]; int n_out_aggs;
  int64_t out_capacity;
  uint64_t R;               // fused key range (several key columns)
  const uint32_t* dict_keys; // FRONT_DICT: key of dense id
  CallDev* call;
};
int launch_compact(const CompactLaunch& c, int sm_count, cudaStream_t s);

// ---- hashagg.cu -------------------------------------------------------------------------
struct HashAggLaunch {
  KeyDesc key;              // whole-input mode: the caller's columns; partition mode: ptr[0] = partitioned keys
  AggPlan plan;             // value column pointers (partition mode: the partitioned copies)
  int64_t n;
  int key_kind, sig;
  const unsigned long long* part_off;   // partition mode only: [n_parts + 1]
  const unsigned long long* item_off;   // partition mode only: [n_parts + 1] work items per partition
  const uint32_t* item_part;            // partition mode only: [items] partition of each work item
  int n_parts;
  uint32_t slots, limit;    // shared-memory table of each CTA
  int max_probes;           // 0 = default (16 buckets); 1 = home bucket only (hot-key cache in front of the global table)
  int bucket_keys;          // 0 = 16-byte buckets; 2 = 8-byte buckets of 32-bit keys (nearly empty tables)
  int spec;                 // speculative run (EIGER_AUTO without statistics)
  uint64_t hot[kMaxHot]; int n_hot;   // whole-input mode: rebased heavy-hitter keys reduced inside the warp
  void* table; uint64_t cap; uint32_t stride;   // global table (BACK_HASH layout)
  CallDev* call;
  void* out_keys[kMaxKeyCols]; void* out_aggs[kMaxAggs]; int n_out_aggs; int64_t out_capacity;   // partition mode emits
  int threads, blocks;
  int ring;                 // rows arrive through the shared-memory ring (ring.cuh) instead of per-thread loads
  int stages;               // shared-memory ring stages; 0 = default
  bool hot_reserved;        // room for the heavy-hitter cells is part of the layout (EIGER_GLOBAL)
  size_t table_smem_bytes;  // shared-memory table of one CTA
  size_t queue_bytes;       // whole-input mode: per-warp miss queues behind the table (0 = misses go to the global table lane by lane)
  // whole-input mode, EIGER_GLOBAL: the rows the front cannot hold are appended to a spill buffer (rebased 64-bit
  // keys + raw 64-bit values, chunks of 2^spill_lg rows reserved per CTA; the tail of a CTA's last chunk is padded
  // with the empty marker) instead of going to the global table row by row; they are partitioned and aggregated
  // per partition afterwards.  spill_keys = nullptr: off.
  uint64_t* spill_keys; uint64_t* spill_vals[kMaxVals]; uint64_t spill_cap_chunks; int spill_lg;
  // partition mode over a spill buffer: rows whose key is the empty marker are padding; every item merges into the
  // global table (its keys may also sit there, put by the fronts of the first pass)
  int skip_empty, force_merge;
};
int launch_hash_agg(const HashAggLaunch& L, cudaStream_t s);
size_t hash_agg_slot_bytes(const AggPlan& p, int key_kind);   // shared-memory bytes per slot
// Dynamic shared memory of the hash aggregation kernel: [ring: stages x stage_bytes][heavy-hitter cells][table].
// A stage holds 2 x threads rows column by column (each column 128-byte aligned).
struct HashAggSmem {
  uint32_t koff[kMaxKeyCols], voff[kMaxVals];
  uint8_t kw[kMaxKeyCols], vw[kMaxVals];
  int n_src;                // key columns in the ring (1 in partition mode: the pre-fused key)
  int stages; uint32_t stage_bytes, hot_off, table_off;
};
HashAggSmem hash_agg_smem_layout(const KeyDesc& key, const AggPlan& plan, int key_kind, int threads, bool hot, int stages);
constexpr int kDefaultStages = 3;

// ---- partition.cu ----------------------------------------------------------------------
struct PartitionLaunch {
  KeyDesc key;
  AggPlan plan;             // value column pointers
  int64_t n;
  int key_kind;             // KK_I32 (keys stay 32-bit), KK_I64 or KK_GEN
  int bits1, bits2;         // fan-out 2^bits1 x 2^bits2 from the top bits of the table hash; bits2 = 0: one level
  // workspace carved by the caller
  uint32_t* hist;           // [2^(bits1 + bits2)]
  unsigned long long* off1; // [2^bits1 + 1]
  unsigned long long* cur1; // [2^bits1]
  unsigned long long* off2; // [2^(bits1 + bits2) + 1]   (two levels)
  unsigned long long* cur2; // [2^(bits1 + bits2)]
  void* keysA; void* valsA[kMaxVals];   // level-1 output, n rows each (value columns keep their width)
  void* keysB; void* valsB[kMaxVals];   // level-2 output
  unsigned long long* item_off;   // [2^(bits1 + bits2) + 1] work items of the aggregation pass
  uint32_t* item_part;            // [2 * 2^(bits1 + bits2) + 2] partition of each work item
  int64_t chunk_rows;       // partitions above 2 * chunk_rows rows are cut into items of chunk_rows
  const uint32_t* pre_hist; // level-1 histogram already taken at fan-out kPreFan with this key base (or nullptr)
  // results
  const void* out_keys; void* const* out_vals; const unsigned long long* out_off; int n_parts;
};
int launch_partition(PartitionLaunch& p, int sm_count, size_t smem_optin, cudaStream_t s);
int partition_max_bits_per_level();

// ---- splitagg.cu ------------------------------------------------------------------------
// Direct-index array split over 2^lgC co-operating CTAs (slot u belongs to CTA u mod 2^lgC of its group).
struct SplitLaunch {
  KeyDesc key; AggPlan plan; int64_t n;
  int key_kind, sig, lgC, spec;
  uint64_t cap; uint32_t local_slots;
  void* table; CallDev* call;
  int blocks;
};
int launch_split_direct(const SplitLaunch& L, cudaStream_t s);
size_t split_direct_smem(int n_acc, uint32_t local_slots);
// The same split with per-CTA hash tables (scattered keys): key owner = hash bits; L.table_smem_bytes = the table
int launch_split_hash(const HashAggLaunch& L, int lgC, cudaStream_t s);
size_t split_hash_queue_bytes(int key_kind);

// ---- dictenc.cu -------------------------------------------------------------------------
int launch_dict_fill(const void* sorted_keys, int dtype, int64_t ndv, void* table, uint64_t cap, CallDev* call, int sm_count, cudaStream_t s);
int launch_dict_gather(const void* keys, int dtype, int64_t n, const void* table, uint64_t cap, int32_t* codes, CallDev* call, int sm_count, cudaStream_t s);

// ---- sortagg.cu -------------------------------------------------------------------------
// EIGER_SORT: LSD radix sort of the rows on the `bits` significant bits of the rebased fused key,
// then a segmented reduce that emits the groups in key order.
struct SortLaunch {
  KeyDesc key;
  AggPlan plan;
  int64_t n;
  int key_kind, sig, bits;
  void* keysA; void* valsA[kMaxVals];      // ping
  void* keysB; void* valsB[kMaxVals];      // pong (two or more passes)
  uint32_t* tile_hist;                     // [n / 1024 + 2][256]
  unsigned long long* digit_base;          // [512]
  void* out_keys[kMaxKeyCols]; void* out_aggs[kMaxAggs]; int n_out_aggs; int64_t out_capacity;
  CallDev* call;
};
int launch_sort_groupby(SortLaunch& L, int sm_count, size_t smem_optin, cudaStream_t s);

}  // namespace eiger
