/* eiger.h — C ABI of the B200-native adaptive GROUP BY library (libeiger.so).
 *
 * One hot path of Eiger (arxiv/paper_2607_04489): runtime-adaptive GROUP BY
 * aggregation (SUM / COUNT / MIN / MAX over integer keys) whose kernel variant
 * and hash-table size are chosen from statistics gathered on the key column at
 * run time — an exact min/max range pass and a HyperLogLog NDV sketch
 * (§1 "Runtime adaptive execution"; §4.1; PAPER.md:79
 * §3.3; §4.3 for the range-first order).
 *
 * Conventions (all entry points):
 *   - Columnar input, one contiguous region per column, 64-bit row counts
 *     (§3.1).  No null masks (the paper never mentions any).
 *   - Unless a parameter says HOST, data pointers are DEVICE pointers owned by
 *     the caller and must be 16-byte aligned (any cudaMalloc / torch allocation
 *     is).  The library never frees or keeps them.
 *   - Work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream).  Host-visible outputs (eiger_stats, *n_groups,
 *     *chosen) are valid when the call returns: the library synchronises the
 *     stream where it has to read a statistic or a count back.
 *   - Scratch memory comes from the caller's `workspace` (device memory, sized
 *     by eiger_groupby_workspace_bytes).  The library itself holds one small
 *     per-process device block (sketch registers, counters) and one pinned host
 *     block, allocated on first use and released by eiger_shutdown().
 *   - Every function returns 0 (EIGER_OK) or a negative eiger_status.  Nothing
 *     throws, nothing aborts; there is no CPU fallback of any step.
 */
#ifndef EIGER_H_
#define EIGER_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { EIGER_I8 = 0, EIGER_I32 = 1, EIGER_I64 = 2, EIGER_F64 = 3 } eiger_dtype;
typedef enum { EIGER_SUM = 0, EIGER_COUNT = 1, EIGER_MIN = 2, EIGER_MAX = 3 } eiger_op;
typedef enum {
  EIGER_AUTO = 0,      /* profile, then pick one of the four below            */
  EIGER_DIRECT = 1,    /* direct-index array, slot = key - min                */
  EIGER_SMEM = 2,      /* per-CTA shared-memory open addressing, merged       */
  EIGER_GLOBAL = 3,    /* one global open-addressing table (L2-resident)      */
  EIGER_PARTITION = 4, /* radix partition by hash bits, then aggregate        */
  EIGER_SORT = 5       /* radix sort on the key bits, then segmented reduce;  */
                       /* groups come out in ascending key order              */
} eiger_variant;

typedef enum {
  EIGER_OK = 0,
  EIGER_ERR_ARG = -1,          /* null pointer, bad dtype/op, n < 0, misaligned column      */
  EIGER_ERR_WORKSPACE = -2,    /* workspace too small; see eiger_groupby_workspace_bytes     */
  EIGER_ERR_OUT_CAPACITY = -3, /* more groups than out_capacity; *n_groups holds the count   */
  EIGER_ERR_INFEASIBLE = -4,   /* the forced variant cannot run on this input                */
  EIGER_ERR_CUDA = -5,         /* a CUDA runtime call failed; eiger_last_cuda_error() says   */
  EIGER_ERR_TABLE_OVERFLOW = -6, /* NDV estimate too low and no room in workspace to retry  */
  EIGER_ERR_STATS = -7,        /* a key lies outside the caller's eiger_stats [min, max]     */
  EIGER_ERR_STATIC_LIMIT = -8  /* eiger_groupby_direct_static: key range > EIGER_STATIC_MAX_SLOTS */
} eiger_status;

typedef struct { const void* data; int32_t dtype; int32_t reserved; } eiger_col; /* length n */
typedef struct { int32_t op; int32_t val_col; } eiger_agg;   /* COUNT ignores val_col        */

/* HOST struct filled by eiger_groupby / eiger_groupby_host when a pointer to it is passed: what the call did. */
typedef struct {
  int32_t variant;              /* the variant that ran (also returned through `chosen`)                        */
  int32_t attempts;             /* 1 + re-runs after a table overflow (NDV under-estimated, R10)       */
  int32_t partition_levels;     /* EIGER_PARTITION: 1 or 2 radix levels; else 0                                  */
  int32_t partition_prehist;    /* EIGER_PARTITION: 1 when the level-1 histogram came from the statistics pass   */
  int32_t partition_key_bytes;  /* EIGER_PARTITION: bytes per key (4 or 8) of the partitioned copy               */
  int32_t sort_passes;          /* EIGER_SORT: 8-bit radix passes                                                 */
  double ndv_est;               /* the NDV estimate the tables were sized with (after clamping to min(n, range)) */
  int64_t kernel_launches;      /* kernels this call launched                                                     */
  int64_t spill_rows;           /* EIGER_GLOBAL: rows (padding included) that went through the spill buffer; else 0 */
  int32_t dict_ids;             /* EIGER_SMEM through the dictionary front: ids each dictionary (one per pass) was planned for; else 0 */
  int32_t reserved;
} eiger_call_info;

/* HOST struct.  n = 0 gives min = INT64_MAX, max = INT64_MIN, ndv_est = 0. */
typedef struct { int64_t min, max; double ndv_est; int64_t n; } eiger_stats;

/* eiger_profile — statistics of one integer key column in a single fused pass
 * (steps A1-A3 of DESIGN.md): exact min and max, and the
 * HyperLogLog estimate of the number of distinct values (p = 14, hash = splitmix64
 * output function of the sign-extended key, table-free estimator; R1-R5),
 * clamped to [0, min(n, max - min + 1)].
 *   keys  DEVICE, n elements of `dtype` (EIGER_I8 / I32 / I64)
 *   out   HOST
 * Errors: EIGER_ERR_ARG, EIGER_ERR_CUDA. */
int eiger_profile(const void* keys, int32_t dtype, int64_t n, eiger_stats* out, void* stream);

/* eiger_profile_keys — the statistics pass exactly as EIGER_AUTO runs it inside eiger_groupby
 * when no statistics are supplied: one read-back for all key columns; min/max of each; the
 * sketch only where the range test cannot decide ("range first"): 1-byte keys and
 * multi-column keys get ndv_est = min(n, max - min + 1) per column without a sketch, unless
 * those ranges multiply to more than 2^22 (beyond a direct-index array): then one more pass
 * sketches the FUSED key (the HLL++ branch of smart key fusion), out[0].ndv_est
 * holds the estimate for the whole key and out[k >= 1].ndv_est = 1 (eiger_groupby multiplies
 * the columns' estimates).
 *   keys[n_key_cols] DEVICE columns; out[n_key_cols] HOST. */
int eiger_profile_keys(const eiger_col* keys, int32_t n_key_cols, int64_t n, eiger_stats* out, void* stream);

/* eiger_hll_registers — test hook: the raw sketch registers of a key column.
 *   regs_out  DEVICE, 16384 bytes, register j in byte j (values 0 .. 51).
 * The register array is an exact function of the key set (R3). */
int eiger_hll_registers(const void* keys, int32_t dtype, int64_t n, uint8_t* regs_out, void* stream);

/* eiger_hll_estimate_host — step A3 alone: estimate from 16384 HOST registers. */
double eiger_hll_estimate_host(const uint8_t* regs);

/* eiger_groupby — GROUP BY keys, aggregating value columns (steps A0, A4-A7;
 * PAPER.md:79 §3.3, §4.1, PAPER.md:184 retrieveAll).
 *   keys[n_key_cols]   1 to 4 integer key columns (EIGER_I8 / I32 / I64, any mix).  Several
 *                      columns are fused on the fly into one 64-bit key by frame of reference +
 *                      positional packing (smart key fusion without the dictionary step,
 *                      PAPER.md:215-221 §4.3): u = (..((k0 - min0) * r1 + (k1 - min1)) * r2 + ..),
 *                      r_c = max_c - min_c + 1, and un-fused on output.  The product of the
 *                      column ranges must fit 64 bits, else EIGER_ERR_INFEASIBLE (the paper
 *                      dictionary-encodes such keys first; not built).
 *   vals[n_vals]       value columns, EIGER_I64 or EIGER_F64, n_vals <= 8
 *   aggs[n_aggs]       n_aggs <= 8; result type: SUM/MIN/MAX of I64 -> int64 (SUM wraps modulo
 *                      2^64), of F64 -> double; COUNT -> int64 row count
 *   stats              HOST, n_key_cols entries from eiger_profile (min / max MUST bound every key of
 *                      their column; ndv_est may be off, R10).  A key outside them is detected where
 *                      it would matter - direct-index arrays and fused multi-column keys run with a
 *                      range check - and fails the call with EIGER_ERR_STATS; single-column hash
 *                      variants rebase modulo 2^32 / 2^64 and are indifferent to it.  Or NULL: the library then
 *                      gathers the statistics inside this call (that is what EIGER_AUTO timing
 *                      includes).  A forced variant runs the full profile.  EIGER_AUTO on
 *                      n >= 2^22 rows first profiles an evenly spaced sample of 2^16 keys; if
 *                      that settles DIRECT or SMEM, one speculative pass aggregates and verifies
 *                      the plan exactly (a key outside the sampled range or a full table discards
 *                      it); if it settles PARTITION (single I32 / I64 key, no hot keys), one
 *                      keys-only pass takes min/max, the level-1 partition histogram and the
 *                      sketch of a hash-space slice of the keys (NDV = slice NDV * 1024 / slice
 *                      partitions); otherwise, or when verification fails, the full profile
 *                      (A1-A3) runs.  Results never depend on which of these ran.
 *   out_keys[k]        DEVICE array of out_capacity elements of key column k's dtype
 *   out_aggs[j]        DEVICE array of out_capacity 8-byte elements
 *   n_groups           HOST; number of groups written (order of groups unspecified)
 *   force              EIGER_AUTO or a variant to run regardless of the statistics
 *   chosen             HOST, may be NULL; the variant that ran
 *   workspace          DEVICE scratch of workspace_bytes (eiger_groupby_workspace_bytes), or NULL: the library
 *                      then uses its own arena, grown on demand (cudaMalloc, a stream synchronisation when
 *                      it grows) and kept until eiger_shutdown().  With NULL a table overflow after an NDV
 *                      under-estimate (R10) is always retried inside the call
 *   info               HOST, may be NULL: what the call did (eiger_call_info)
 * Errors: EIGER_ERR_ARG; EIGER_ERR_WORKSPACE; EIGER_ERR_OUT_CAPACITY (a safe capacity is
 * min(n, range)); EIGER_ERR_INFEASIBLE (e.g. EIGER_DIRECT on a 2^40 range);
 * EIGER_ERR_TABLE_OVERFLOW (the sketch under-estimated and the workspace has no room for the
 * larger table: call again with stats->ndv_est raised, e.g. to min(n, range)); EIGER_ERR_STATS;
 * EIGER_ERR_CUDA.
 * fp64 MIN/MAX order -0.0 below +0.0; NaN inputs are not supported. */
int eiger_groupby(const eiger_col* keys, int32_t n_key_cols, int64_t n,
                  const eiger_col* vals, int32_t n_vals,
                  const eiger_agg* aggs, int32_t n_aggs,
                  const eiger_stats* stats,
                  void* const* out_keys, void* const* out_aggs, int64_t out_capacity,
                  int64_t* n_groups, int32_t force, int32_t* chosen,
                  void* workspace, size_t workspace_bytes, void* stream, eiger_call_info* info);

/* Workspace needed by eiger_groupby for the same arguments (data pointers inside keys / vals
 * are ignored and may be NULL).  stats may be NULL: worst case over the variants `force`
 * allows, with the group count bounded by n only.  Returns 0 on bad arguments. */
size_t eiger_groupby_workspace_bytes(const eiger_col* keys, int32_t n_key_cols, int64_t n,
                                     const eiger_col* vals, int32_t n_vals,
                                     const eiger_agg* aggs, int32_t n_aggs,
                                     const eiger_stats* stats, int32_t force);

/* The variant EIGER_AUTO picks for these statistics (step A4), without running anything;
 * negative eiger_status on bad arguments. */
int32_t eiger_select_variant(const eiger_col* keys, int32_t n_key_cols, int64_t n,
                             const eiger_col* vals, int32_t n_vals,
                             const eiger_agg* aggs, int32_t n_aggs, const eiger_stats* stats);

/* eiger_groupby_host — the same operation end to end from HOST buffers (pinned or pageable):
 * copies the columns to the device, profiles, aggregates and copies the groups back.
 * keys/vals/out_keys/out_aggs are HOST pointers here.  Device memory comes from library arenas
 * that grow on demand and are kept between calls (eiger_shutdown releases them).  Inside, the
 * statistics are gathered exactly as eiger_groupby does with stats = NULL (sample, speculative single
 * pass or profile).
 * h2d_bytes / d2h_bytes (HOST, may be NULL) receive the bytes copied in each direction. */
int eiger_groupby_host(const eiger_col* keys, int32_t n_key_cols, int64_t n,
                       const eiger_col* vals, int32_t n_vals,
                       const eiger_agg* aggs, int32_t n_aggs,
                       void* const* out_keys, void* const* out_aggs, int64_t out_capacity,
                       int64_t* n_groups, int32_t force, int32_t* chosen,
                       int64_t* h2d_bytes, int64_t* d2h_bytes, void* stream, eiger_call_info* info);

/* eiger_dict_encode — order-preserving dictionary encoding of one integer column (PAPER.md:171-211
 * Algorithm 1; "If NDV is below a certain threshold, we will use dictionary encoding";
 * PAPER.md:223 "it must preserve the order of the keys in the encoded values"):
 *   codes_out[i] = number of distinct values of the column that are smaller than keys[i],
 *   dict_out[c]  = the value with code c (the distinct values in ascending order), *ndv of them.
 * Steps as in the paper: hash insert-and-find + retrieveAll (a COUNT group-by, EIGER_AUTO), argsort of
 * the unique keys (the radix sort of EIGER_SORT), scatter of the ranks into a look-up table, gather.
 *   keys       DEVICE, n elements of dtype (EIGER_I8 / I32 / I64), 16-byte aligned
 *   codes_out  DEVICE, n int32
 *   dict_out   DEVICE, dict_capacity elements of dtype
 *   ndv        HOST; set even when EIGER_ERR_OUT_CAPACITY says dict_capacity was too small
 *   workspace  DEVICE, eiger_dict_encode_workspace_bytes(dtype, n, dict_capacity) bytes, 256-byte aligned
 * Errors: EIGER_ERR_ARG, EIGER_ERR_WORKSPACE, EIGER_ERR_OUT_CAPACITY, EIGER_ERR_CUDA. */
int eiger_dict_encode(const void* keys, int32_t dtype, int64_t n, int32_t* codes_out, void* dict_out, int64_t dict_capacity,
                      int64_t* ndv, void* workspace, size_t workspace_bytes, void* stream);
size_t eiger_dict_encode_workspace_bytes(int32_t dtype, int64_t n, int64_t dict_capacity);

/* eiger_groupby_direct_static — SUM + COUNT of one int64 value column per key, direct-index variant
 * (the array-based group-by for a small key range), for callers that cannot
 * allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
 * This entry point calls no cudaMalloc / cudaFree and no allocating library routine, and does not
 * touch the library's arena or runtime state.  Its accumulator array is a file-scope __device__ array
 * of EIGER_STATIC_MAX_SLOTS slots (1 MiB + 256 bytes on every GPU that loads the library, held until
 * the process exits).
 *   keys        DEVICE, n elements of key_dtype (EIGER_I8 / I32 / I64)
 *   key_min, key_max   bounds of the keys, inclusive; key_max - key_min + 1 <= EIGER_STATIC_MAX_SLOTS,
 *               else EIGER_ERR_STATIC_LIMIT (nothing is launched).  A key outside the bounds is not
 *               aggregated and fails the call with EIGER_ERR_STATS.
 *   vals        DEVICE, n int64; SUM wraps modulo 2^64 like eiger_groupby's
 *   out_keys    DEVICE, out_capacity elements of key_dtype; out_sum, out_count DEVICE, out_capacity
 *               int64 each; group order unspecified (as eiger_groupby).  Owned by the caller.
 *   n_groups    HOST; set to the group count even when EIGER_ERR_OUT_CAPACITY says out_capacity was
 *               too small (the first out_capacity positions are then filled)
 *   stream      cudaStream_t (NULL = the default stream); the call returns after the stream has drained
 * The array is shared by every call on a device and keeps the last call's contents; each call clears
 * the part it uses on `stream` first.  Calls that overlap on the GPU (two streams, two host threads)
 * RACE on it: serialise them.  Not usable from several processes' worth of concurrency either way -
 * each process has its own copy.
 * Errors: EIGER_ERR_ARG, EIGER_ERR_STATIC_LIMIT, EIGER_ERR_STATS, EIGER_ERR_OUT_CAPACITY, EIGER_ERR_CUDA. */
#define EIGER_STATIC_MAX_SLOTS 65536
int eiger_groupby_direct_static(const void* keys, int32_t key_dtype, int64_t n, int64_t key_min, int64_t key_max,
                                const int64_t* vals, void* out_keys, int64_t* out_sum, int64_t* out_count,
                                int64_t out_capacity, int64_t* n_groups, void* stream);
int64_t eiger_static_max_slots(void);

/* Number of kernels this library has launched in this process (bench.py's gpu_launches). */
int64_t eiger_launch_count(void);

/* Per-kernel device time, measured with CUDA events on the caller's stream inside the calls
 * above while enabled (eiger_set_kernel_timing(1)); off by default.  `which`: 0 = aggregation
 * kernel (the dominant one), 1 = profile kernel, 2 = partition kernels, 3 = table init,
 * 4 = compaction, 5 = aggregation of the spill buffer's partitions (EIGER_GLOBAL).  Returns the milliseconds accumulated since the last call with reset != 0;
 * *launches (may be NULL) receives how many launches that covers. */
void eiger_set_kernel_timing(int32_t enabled);

/* The EIGER_* environment variables that override the selector's thresholds are
 * read once per process; call this after changing them (crossover sweeps, tests). */
void eiger_reload_tunables(void);
double eiger_kernel_time_ms(int32_t which, int32_t reset, int64_t* launches);

/* eiger_probe — machine probes: measures one building-block rate on the current device, the
 * numbers the selector's thresholds rest on (the paper's crossovers are "platform-dependent",
 * PAPER.md:304-306).  Not on the hot path.  `name`:
 *   "read_ldg"  / "read_bulk"   streamed read of param MiB (default 4096) with 16-byte loads / with
 *                               cp.async.bulk into a 4-stage shared-memory ring of param2-byte chunks -> GB/s
 *   "dsmem_red" / "dsmem_atom" / "dsmem_cas" / "dsmem_st"
 *                               rows/s of random updates of a table spread over the shared memory of a
 *                               thread-block cluster of param CTAs (1 = plain shared memory), param2 slots
 *                               per CTA: 2 non-returning adds / 1 returning add + 1 add + carry /
 *                               look-up + compare-and-swap / one 8-byte store per row -> G rows/s
 *   "dsmem_bulk"                cp.async.bulk shared -> remote shared, cluster of param CTAs, param2 bytes -> GB/s
 *   "store_bulk" / "store_warp" param-byte chunks to random aligned places in param2 MiB: cp.async.bulk
 *                               from shared memory / one warp-wide store -> GB/s
 *   "l2_red"                    two 64-bit global reductions per row on 2^param 16-byte cells -> G rows/s
 *   "release"                   frees the probe's scratch memory
 * result HOST.  Errors: EIGER_ERR_ARG (unknown name), EIGER_ERR_CUDA. */
int eiger_probe(const char* name, int64_t param, int64_t param2, double* result, void* stream);

const char* eiger_strerror(int code);
const char* eiger_last_cuda_error(void);
const char* eiger_variant_name(int32_t variant);
void eiger_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* EIGER_H_ */
