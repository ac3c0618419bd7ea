// The C ABI of libeiger (include/eiger.h): runtime state, step A4 (select + size) and the
// host-side orchestration of profile -> init -> aggregate -> compact.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstddef>
#include <cstring>
#include <mutex>

#include "internal.h"

namespace eiger {

namespace {
std::mutex g_mu;
Runtime g_rt;
std::atomic<int64_t> g_launches{0};
char g_cuda_err[512] = "";
bool g_timing = false;
constexpr int kTimeSlots = 6;
double g_time_ms[kTimeSlots] = {0, 0, 0, 0, 0, 0};
int64_t g_time_n[kTimeSlots] = {0, 0, 0, 0, 0, 0};

// event pairs recorded during one call, resolved after the call's final synchronise
struct Pending { cudaEvent_t a, b; int slot; };
Pending g_pending[16];
int g_n_pending = 0;
cudaEvent_t g_pool[32];
int g_pool_n = 0, g_pool_used = 0;

cudaEvent_t take_event() {
  if (g_pool_used == g_pool_n) {
    if (g_pool_n == 32) return nullptr;
    if (cudaEventCreate(&g_pool[g_pool_n]) != cudaSuccess) return nullptr;
    ++g_pool_n;
  }
  return g_pool[g_pool_used++];
}
struct Timed {
  cudaStream_t s; int slot; cudaEvent_t a = nullptr, b = nullptr;
  Timed(cudaStream_t st, int sl) : s(st), slot(sl) {
    if (g_timing && g_n_pending < 16) { a = take_event(); b = take_event(); if (a && b) cudaEventRecord(a, s); }
  }
  ~Timed() {
    if (a && b) { cudaEventRecord(b, s); g_pending[g_n_pending++] = Pending{a, b, slot}; }
  }
};
void resolve_timing() {
  for (int i = 0; i < g_n_pending; ++i) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, g_pending[i].a, g_pending[i].b) == cudaSuccess) {
      g_time_ms[g_pending[i].slot] += ms; g_time_n[g_pending[i].slot] += 1;
    }
  }
  g_n_pending = 0; g_pool_used = 0;
}

constexpr double kSigma = 0.008125;             // 1.04 / sqrt(2^14)
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline bool is_key_dtype(int d) { return d == EIGER_I8 || d == EIGER_I32 || d == EIGER_I64; }
inline int dtype_size(int d) { return d == EIGER_I8 ? 1 : d == EIGER_I32 ? 4 : 8; }

// Tunables of step A4; EIGER_* environment variables override them
// for the crossover sweeps.  Re-read on every call so that a sweep can change them in-process.
struct Tunables {
  size_t priv_smem;                   // FRONT_PRIV: private cells of one CTA
  int priv_max_range;                 // ... and only for this many keys (measured: 4 keys 0.46 vs 0.59 ms for the shared array, 8 keys 0.55 vs 0.48, 16 keys 0.52 vs 0.46; C2's 6 x 5 cells 2.89 vs 2.94)
  size_t sdirect_bytes = 160 * 1024;  // FRONT_SDIRECT: largest per-CTA direct array
  size_t sdirect_replica_budget;
  int sdirect_max_replicas, sdirect_wide;
  size_t smem_total;                  // dynamic shared memory of one hash-aggregation CTA: ring + table (1 CTA per SM)
  int stages;                         // stages of the shared-memory ring the rows stream through (ring.cuh)
  int ring;                           // bit 0: whole-input hash kernels, bit 1: per-partition aggregation take their rows from the ring
  size_t smem_table_bytes;            // EIGER_SMEM / EIGER_GLOBAL: shared-memory table of one CTA; 0 = what the ring leaves of smem_total
  int smem_threads;
  size_t part_table_bytes;            // EIGER_PARTITION: the same for the per-partition tables
  int part_threads;
  int part_min_bits;                  // at least this many partitions (parallelism of the emit pass)
  size_t direct_l2_bytes;             // AUTO takes DIRECT with global atomics up to this table size
  size_t global_l2_bytes;             // AUTO takes GLOBAL up to this table size
  double load;                        // target load factor of every hash table
  double smem_fill;                   // AUTO takes EIGER_SMEM while ndv <= smem_fill * slots
  int global_front;                   // hot-key shared-memory table in front of the global table
  int global_front_probes;            // buckets that table looks at per key (1: set-associative cache)
  int spec;                           // EIGER_AUTO without statistics tries one speculative pass first
  int global_always;                  // take EIGER_GLOBAL whenever its table fits L2 (not only for skewed keys)
  double skew_collision;              // sample collision rate above which the keys count as skewed
  int64_t spec_samples, spec_min_rows;
  double narrow_load;                 // 32-bit keys: 8-byte buckets while keys per table <= narrow_load x slots
  int hot;                            // skewed inputs: heavy hitters are reduced inside the warp (hashagg.cu)
  double hot_min_share;               // a key is hot from this share of the sample
  int slice;                          // EIGER_AUTO sizes PARTITION from a hash-space slice sketch instead of the full profile
  double slice_min_keys;              // distinct keys wanted in the slice (relative error 1 / sqrt of it)
  double fused_sketch_min_range;      // multi-column keys: sketch the fused key when the ranges multiply to more than this
  int part_full_table;                // EIGER_PARTITION reserves the full-size global table when partitions may be cut (round-1 behaviour)
  int split_max;                      // direct-index array split over up to this many CTAs (splitagg.cu); 0 = off
  int sig_g1;                         // plans of <= 4 accumulators over <= 1 value column take the light generic hash kernels (SIG_G1)
  int slice_fused;                    // the slice-sketch pass also for several key columns (fused key)
  int miss_queue;                     // EIGER_GLOBAL queues the front's misses per warp (hashagg.cuh)
  int global_spill;                   // EIGER_GLOBAL: the front's misses go to a spill buffer that is partitioned and aggregated afterwards
  double spill_frac;                  // ... with room for this share of the rows (what does not fit takes the global table)
  double spill_min_rows;              // ... for inputs of at least this many rows
  double spill_lg;                    // ... reserved by the CTAs in chunks of at least 2^spill_lg rows
  int split_hash;                     // EIGER_SMEM may split its hash tables over up to 16 CTAs (experiment, off)
  size_t split_bytes;                 // ... each holding at most this much of it in shared memory
  int pack_stride;                    // global hash table slots of 40 / 48 bytes are not padded to 64
  int dict;                           // EIGER_AUTO: scattered keys the sample names completely get a dictionary + direct array (FRONT_DICT)
  double dict_max_keys;               // ... while the sample holds at most this many distinct keys
  int dict_pairs;                     // small dictionaries with one replica are searched two entries at a time
  int dict_max_pass_lg;               // ... or 2^this many times that, in as many passes over the input (one key slice each)
  double dict_big_max_keys;           // ... or, for SUM + COUNT plans, this many in the compact layout (dictionary from 4x the sample); 0 = off
  Tunables() {
    auto env = [](const char* k, double dflt) { const char* v = std::getenv(k); return v ? std::atof(v) : dflt; };
    priv_smem = (size_t)env("EIGER_PRIV_KB", 96) << 10;
    fused_sketch_min_range = env("EIGER_FUSED_SKETCH_MIN_RANGE", 4194304.0);   // beyond any direct-index array AUTO would take
    priv_max_range = (int)env("EIGER_PRIV_MAX_RANGE", 6);
    smem_total = (size_t)env("EIGER_SMEM_TOTAL_KB", 225) << 10;
    stages = (int)env("EIGER_STAGES", kDefaultStages);
    ring = (int)env("EIGER_RING", 0);
    smem_table_bytes = (size_t)env("EIGER_SMEM_KB", 0) << 10;
    sdirect_replica_budget = (size_t)env("EIGER_SDIRECT_REPLICA_KB", 64) << 10;
    sdirect_max_replicas = (int)env("EIGER_SDIRECT_MAX_REPLICAS", 8);
    sdirect_wide = (int)env("EIGER_SDIRECT_WIDE", 1);
    smem_threads = (int)env("EIGER_SMEM_THREADS", 1024);
    part_table_bytes = (size_t)env("EIGER_PART_KB", 0) << 10;
    part_threads = (int)env("EIGER_PART_THREADS", 1024);
    part_min_bits = (int)env("EIGER_PART_MIN_BITS", 7);
    direct_l2_bytes = (size_t)env("EIGER_DIRECT_L2_MB", 48) << 20;
    global_l2_bytes = (size_t)env("EIGER_GLOBAL_L2_MB", 192) << 20;
    global_front = (int)env("EIGER_GLOBAL_FRONT", 1);
    global_front_probes = (int)env("EIGER_GLOBAL_FRONT_PROBES", 1);
    load = env("EIGER_LOAD", 0.5);
    smem_fill = env("EIGER_SMEM_FILL", 0.67);          // scattered 2^13 keys (load 0.66): 2.7 ms in one CTA's table, 3.6 ms partitioned
    spec = (int)env("EIGER_SPEC", 1);
    global_always = (int)env("EIGER_GLOBAL_ALWAYS", 0);
    skew_collision = env("EIGER_SKEW_COLLISION", 1e-3);
    spec_samples = (int64_t)env("EIGER_SPEC_SAMPLES", 1 << 16);
    spec_min_rows = (int64_t)env("EIGER_SPEC_MIN_ROWS", 1 << 22);
    narrow_load = env("EIGER_NARROW_LOAD", 0.10);
    hot = (int)env("EIGER_HOT", 1);
    hot_min_share = env("EIGER_HOT_MIN_SHARE", 0.02);
    slice = (int)env("EIGER_SLICE", 1);
    slice_min_keys = env("EIGER_SLICE_MIN_KEYS", 2048);
    dict = (int)env("EIGER_DICT", 1);
    pack_stride = (int)env("EIGER_PACK_STRIDE", 1);
    split_max = (int)env("EIGER_SPLIT_MAX", 4);        // measured (C5 dense, ms): C = 2 / 4 / 8 / 16 -> 1.26 / 1.86 / 3.11 / 5.15 against 2.8-3.3 for global RED
    slice_fused = (int)env("EIGER_SLICE_FUSED", 1);
    sig_g1 = (int)env("EIGER_SIG_G1", 1);
    miss_queue = (int)env("EIGER_MISS_QUEUE", 0);     // measured on C3: 5.25 ms with the queues (and a 32 KB smaller front) against 4.84 ms without
    global_spill = (int)env("EIGER_GLOBAL_SPILL", 0);  // measured on C3: 7.8 ms with the spill buffer against 5.5 ms without
    spill_frac = env("EIGER_SPILL_FRAC", 0.5);
    spill_min_rows = env("EIGER_SPILL_MIN_ROWS", 4194304);
    spill_lg = env("EIGER_SPILL_LG", 9);
    split_hash = (int)env("EIGER_SPLIT_HASH", 0);      // the hash flavour loses everywhere (scattered 2^13 / 2^14: 3.1 / 6.4 ms against 2.7 / 3.4)
    split_bytes = (size_t)env("EIGER_SPLIT_KB", 192) << 10;
    part_full_table = (int)env("EIGER_PART_FULL_TABLE", 0);
    dict_big_max_keys = env("EIGER_DICT_BIG_MAX_KEYS", 8600);
    dict_pairs = (int)env("EIGER_DICT_PAIRS", 1);
    dict_max_pass_lg = (int)env("EIGER_DICT_MAX_PASS_LG", 1);   // measured (C5 scattered, ms per call): 2 passes at 2^14 keys 2.78 against 3.54 partitioned; 4 passes at 2^15 4.52 against 3.47
    dict_max_keys = env("EIGER_DICT_MAX_KEYS", 4600);   // measured: scattered 2^12 keys 0.90 ms through the dictionary, 1.25 ms through the hash table
  }
};
// read once per process (about 30 getenv calls used to run several times per eiger_groupby: 15 us of a
// 0.6 ms call); eiger_reload_tunables() re-reads them (the crossover sweeps and the tests change them in-process)
Tunables g_tun;
std::atomic<bool> g_tun_dirty{false};
const Tunables& tun() {
  if (g_tun_dirty.exchange(false)) g_tun = Tunables();
  return g_tun;
}

struct QueryPlan {
  int variant = 0, key_kind = 0, sig = 0, front = 0, back = 0;
  KeyDesc key{};
  AggPlan plan{};
  int n_user_aggs = 0;
  int val_src[kMaxVals];        // plan value slot -> caller's value column
  uint64_t R = 0;               // fused key range; 0 = 2^64 (or not representable)
  double ndv = 0;
  // direct
  uint32_t front_slots = 0, front_limit = 0, front_replicas = 1;
  // hash variants
  uint32_t slots = 0, limit = 0;
  int threads = 0;
  int bits1 = 0, bits2 = 0;
  size_t smem_bytes = 0;        // direct variants: the CTA's array; hash variants: the CTA's table
  size_t smem_dyn = 0;          // hash variants: ring + table
  int stages = 0;
  size_t queue_bytes = 0;
  bool ring = false;
  bool hot_reserved = false;
  uint64_t cap = 0, cap_bound = 0, cap_hot = 0;
  uint32_t stride = 0;
  size_t table_bytes = 0, part_bytes = 0, total_bytes = 0;
  const uint32_t* pre_hist = nullptr;   // PARTITION: level-1 histogram taken with key.base at fan-out kPreFan
  int sort_bits = 0, sort_passes = 0;   // SORT: significant bits of the rebased fused key, 8-bit passes
  uint32_t dict_slots = 0, dict_shift = 0;   // FRONT_DICT: dictionary image entries (power of two)
  uint32_t dict_compact = 0;                 // FRONT_DICT: the large-dictionary layout (SUM + COUNT plans, up to ~8300 keys)
  uint32_t dict_pass_lg = 0;                 // FRONT_DICT: 2^dict_pass_lg passes, each with the dictionary of one slice of the keys
  int split_lg = 0;                          // FRONT_SPLIT: log2 of the CTAs that share the array
  // GLOBAL with a spill buffer: capacity in rows (0 = none; a multiple of the chunk), chunk = 2^spill_lg rows, and
  // the plan of the partition + per-partition aggregation that follows
  uint64_t spill_rows = 0; int spill_lg = 0;
  int sp_bits1 = 0, sp_bits2 = 0, sp_threads = 0;
  uint32_t sp_slots = 0, sp_limit = 0;
  size_t sp_smem_bytes = 0, sp_smem_dyn = 0;
};

uint64_t range_of(const eiger_stats& s) {   // max - min + 1, 0 when it is 2^64
  return (uint64_t)s.max - (uint64_t)s.min + 1ull;
}

int detect_sig(const AggPlan& p, int n_user);
// the per-warp miss queue exists in the kernels with a compile-time plan of at most two value columns
inline bool Sig_static_or_small(const AggPlan& p, int na) { const int sg = detect_sig(p, na); return sg == SIG_SC || sg == SIG_A4I || sg == SIG_A4F || sg == SIG_SC32; }

int detect_sig(const AggPlan& p, int n_user) {
  auto is = [&](int j, int op, int col, int f) { return p.op[j] == op && (op == EIGER_COUNT || (p.col[j] == col && p.f64[j] == f)); };
  const int fallback = (p.n_vals <= 1 && p.n_acc <= 4 && tun().sig_g1) ? SIG_G1 : SIG_GENERIC;
  if (p.n_acc != n_user) return fallback;
  bool any32 = false;
  for (int c = 0; c < p.n_vals; ++c) any32 = any32 || p.vw[c] == 4;
  if (any32) return (n_user == 2 && p.n_vals == 1 && is(0, EIGER_SUM, 0, 0) && is(1, EIGER_COUNT, 0, 0)) ? SIG_SC32 : fallback;
  if (n_user == 2 && is(0, EIGER_SUM, 0, 0) && is(1, EIGER_COUNT, 0, 0)) return SIG_SC;
  if (n_user == 4 && is(1, EIGER_COUNT, 0, 0)) {
    if (is(0, EIGER_SUM, 0, 0) && is(2, EIGER_MIN, 0, 0) && is(3, EIGER_MAX, 0, 0)) return SIG_A4I;
    if (is(0, EIGER_SUM, 0, 1) && is(2, EIGER_MIN, 0, 1) && is(3, EIGER_MAX, 0, 1)) return SIG_A4F;
  }
  if (n_user == 5 && p.n_vals == 4 && is(0, EIGER_SUM, 0, 0) && is(1, EIGER_SUM, 1, 0) && is(2, EIGER_SUM, 2, 0) &&
      is(3, EIGER_SUM, 3, 0) && is(4, EIGER_COUNT, 0, 0)) return SIG_S4C;
  return fallback;
}

// Step A4: choose the variant and size everything (readings R8-R10).
int plan_query(const Runtime* rt, const eiger_col* keys, int nk, int64_t n, const eiger_col* vals, int nv,
               const eiger_agg* aggs, int na, const eiger_stats* st, int force, QueryPlan* q, bool skewed = false) {
  if (!keys || nk < 1 || nk > kMaxKeyCols || n < 0 || nv < 0 || nv > kMaxVals || na < 1 || na > kMaxAggs || !aggs) return EIGER_ERR_ARG;
  if (nv > 0 && !vals) return EIGER_ERR_ARG;
  if (force < EIGER_AUTO || force > EIGER_SORT) return EIGER_ERR_ARG;
  for (int k = 0; k < nk; ++k) if (!is_key_dtype(keys[k].dtype)) return EIGER_ERR_ARG;
  for (int c = 0; c < nv; ++c) if (vals[c].dtype != EIGER_I64 && vals[c].dtype != EIGER_F64 && vals[c].dtype != EIGER_I32) return EIGER_ERR_ARG;

  // aggregates -> accumulator plan over the value columns that are actually used
  AggPlan& p = q->plan;
  std::memset(&p, 0, sizeof(p));
  int slot_of[kMaxVals];
  for (int c = 0; c < kMaxVals; ++c) slot_of[c] = -1;
  bool has_count = false;
  p.cnt_acc = -1;
  for (int j = 0; j < na; ++j) {
    const int op = aggs[j].op;
    if (op < EIGER_SUM || op > EIGER_MAX) return EIGER_ERR_ARG;
    p.op[j] = (uint8_t)op;
    if (op == EIGER_COUNT) { if (!has_count) p.cnt_acc = j; has_count = true; continue; }
    const int c = aggs[j].val_col;
    if (c < 0 || c >= nv) return EIGER_ERR_ARG;
    if (slot_of[c] < 0) {
      slot_of[c] = p.n_vals; q->val_src[p.n_vals] = c; p.vals[p.n_vals] = vals[c].data;
      p.vw[p.n_vals] = vals[c].dtype == EIGER_I32 ? 4 : 8;      // int32 payloads are widened on the fly
      ++p.n_vals;
    }
    p.col[j] = (uint8_t)slot_of[c];
    p.f64[j] = vals[c].dtype == EIGER_F64;
  }
  p.n_acc = na;
  q->n_user_aggs = na;

  // keys: ranges and fusion (A0)
  KeyDesc& kd = q->key;
  std::memset(&kd, 0, sizeof(kd));
  kd.ncols = nk; kd.mul = 1;
  bool have_stats = st != nullptr;
  uint64_t Rk[kMaxKeyCols] = {0, 0, 0, 0};
  for (int k = 0; k < nk; ++k) {
    kd.ptr[k] = keys[k].data; kd.dtype[k] = keys[k].dtype;
    if (have_stats) { kd.base[k] = (uint64_t)st[k].min; Rk[k] = n > 0 ? range_of(st[k]) : 1; }
    else {  // bound by the type
      const int bits = 8 * dtype_size(keys[k].dtype);
      kd.base[k] = bits == 64 ? (uint64_t)INT64_MIN : (uint64_t)(-(1ll << (bits - 1)));
      Rk[k] = bits == 64 ? 0 : (1ull << bits);
    }
  }
  uint64_t R = Rk[0];
  for (int k = nk; k < kMaxKeyCols; ++k) { kd.ptr[k] = kd.ptr[0]; kd.dtype[k] = kd.dtype[0]; }   // loadable, masked out (rows.cuh)
  for (int k = 0; k < kMaxKeyCols; ++k) kd.rng[k] = k < nk ? Rk[k] : 1;     // rng[0] = 0 (full 64-bit range) only on the single-column paths
  if (nk >= 2) {
    unsigned __int128 prod = 1;
    bool fits = true;
    for (int k = 0; k < nk && fits; ++k) {
      if (Rk[k] == 0) { fits = false; break; }
      prod *= Rk[k];
      if (prod >> 64) fits = false;                  // fused key must fit 64 bits
    }
    // without statistics (workspace sizing before the profile) the type ranges of several int32 /
    // int64 columns always multiply past 2^64: size for "range unknown", the group count bounded by n
    if (!fits && have_stats) return EIGER_ERR_INFEASIBLE;
    R = fits ? (uint64_t)prod : 0; kd.mul = Rk[1];
  }
  {
    bool all32 = true;
    for (int k = 0; k < nk; ++k) all32 = all32 && keys[k].dtype == EIGER_I32;
    kd.flags = (all32 ? kKeyAll32 : 0) | (R != 0 && R <= 0xFFFFFFFFull ? kKey32 : 0);
  }
  q->R = R;
  // group-count bound and estimate
  double bound = (double)n;
  if (R != 0) bound = std::min(bound, (double)R);
  double ndv = bound;
  if (have_stats) {
    double e = st[0].ndv_est;
    for (int k = 1; k < nk; ++k) e *= st[k].ndv_est;
    ndv = std::min(bound, std::max(e, 1.0));
  }
  q->ndv = ndv;
  q->cap_bound = (uint64_t)std::max(1.0, std::ceil(bound / tun().load)) + 64;

  const Tunables& T = tun();
  const int n_acc_direct = na + (has_count ? 0 : 1);
  const bool direct_ok = R != 0 && R <= (1ull << 33);
  const unsigned __int128 direct_bytes = (unsigned __int128)R * 8 * n_acc_direct;

  // hash variants: key kind, shared-memory slot size, global slot stride
  // a single int32 column is hashed as 32-bit keys whatever its range: u = key - min (mod 2^32) is a
  // bijection, and the one key that may land on the empty marker is kept in the global table
  const int hk = (nk == 1 && keys[0].dtype == EIGER_I32) ? KK_I32
                 : (nk == 1 && keys[0].dtype == EIGER_I64) ? KK_I64 : KK_GEN;
  // partition source kind: a fused key whose domain fits 32 bits is partitioned and aggregated as 32-bit keys
  const int hkp = (hk == KK_GEN && (kd.flags & kKey32)) ? KK_GEN32 : hk;
  const size_t slot_bytes = hash_agg_slot_bytes(p, hk), part_slot_bytes = hash_agg_slot_bytes(p, hkp);
  // the table gets what the ring (and, for EIGER_GLOBAL, the heavy-hitter cells) leaves of the CTA's shared memory
  const int pre_kind = (hkp == KK_I32 || hkp == KK_GEN32) ? KK_U32PRE : KK_U64PRE;
  auto table_bytes_for = [&](int kind, int threads, bool hot, size_t fixed) {
    if (fixed) return fixed;
    const bool pre = kind == KK_U32PRE || kind == KK_U64PRE;
    if (!(T.ring & (pre ? 2 : 1))) return pre ? (size_t)200 << 10 : ((size_t)200 << 10);     // per-thread loads: the table is the whole allocation (heavy-hitter cells are static)
    const HashAggSmem lay = hash_agg_smem_layout(kd, p, kind, threads, hot, T.stages);
    return T.smem_total > lay.table_off + 4096 ? T.smem_total - lay.table_off : (size_t)4096;
  };
  const bool want_hot = force == EIGER_GLOBAL || (force == EIGER_AUTO && skewed);
  // EIGER_GLOBAL: the rows the front cannot hold are queued per warp (64 entries of key + values) and sent to
  // the global table 32 at a time; the queues take their room from the front table
  const size_t miss_queue = (want_hot && T.miss_queue && !(T.ring & 1) && Sig_static_or_small(p, na)) ? (size_t)(T.smem_threads / 32) * 64 * 8 * (1 + p.n_vals) + 128 : 0;
  const size_t smem_tab = table_bytes_for(hk, T.smem_threads, want_hot, T.smem_table_bytes) - (T.smem_table_bytes ? 0 : miss_queue);
  const size_t part_tab = table_bytes_for(pre_kind, T.part_threads, false, T.part_table_bytes);
  const uint32_t smem_slots = (uint32_t)std::max<size_t>(64, (smem_tab - 64) / slot_bytes) & ~7u;   // planes stay 8-byte aligned
  const uint32_t part_slots = (uint32_t)std::max<size_t>(64, (part_tab - 64) / part_slot_bytes) & ~7u;
  // slot = [key][accumulators]: rounded up to a power of two (a slot then never straddles a 32-byte
  // sector more than its size requires), except where that wastes a quarter of the table or more:
  // C3's four aggregates need 40 bytes; 64-byte slots make its table 132 MB (past the 126 MB L2), packed
  // 40-byte slots 84 MB - and a 40-byte slot at a multiple of 8 covers two sectors either way
  const uint32_t hash_stride = [&] {
    uint32_t s = 16; while (s < 8u * (1 + na)) s *= 2;
    const uint32_t packed = 8u * (1 + na);
    return (T.pack_stride && packed > 32 && 4 * packed <= 3 * s) ? packed : s;
  }();
  auto hash_cap = [&](double g) { return (uint64_t)std::max(1024.0, std::ceil(g * (1.0 + 4 * kSigma) * 1.02 / T.load)); };

  // EIGER_SMEM split over 2^lg CTAs: the smallest group whose tables hold the keys at the target load; 0 = one CTA
  // holds them all (or no group is large enough: the plain variant then overflows into the global table)
  const uint32_t split_slots = (uint32_t)std::max<size_t>(64, (((size_t)200 << 10) - split_hash_queue_bytes(hk) - 64) / slot_bytes) & ~7u;
  auto split_lg_for = [&](double g) -> int {
    const double fill = hk == KK_I32 ? T.smem_fill : 0.6 * T.smem_fill;
    if (g * (1.0 + 4 * kSigma) <= fill * smem_slots || !T.split_hash) return 0;
    for (int lg = 1; (1 << lg) <= 16; ++lg)
      if (g * (1.0 + 4 * kSigma) <= 0.9 * fill * (double)split_slots * (double)(1 << lg)) return lg;
    return 0;
  };
  int variant = force;
  if (variant == EIGER_AUTO) {
    if (direct_ok && (direct_bytes * 256 <= T.priv_smem || direct_bytes <= T.sdirect_bytes ||
                      (!skewed && direct_bytes <= T.direct_l2_bytes && (double)R <= 16.0 * (double)std::max<int64_t>(n, 1)))) variant = EIGER_DIRECT;   // hot keys serialise global atomics
    else if (ndv * (1.0 + 4 * kSigma) <= (hk == KK_I32 ? T.smem_fill : 0.6 * T.smem_fill) * smem_slots) variant = EIGER_SMEM;   // 2-key buckets fill up sooner
    // ... or the tables of up to 16 co-operating CTAs, each owning a hash slice of the keys (splitagg.cu)
    else if (!skewed && split_lg_for(ndv) > 0) variant = EIGER_SMEM;
    // uniform keys: partition + shared-memory aggregation beats L2 atomics at every size measured
    // (C5 sweep); a few hot keys in front of a long tail (sample collision rate) is where the global
    // table with its hot-key front wins (C3), while its table still fits L2
    else if ((skewed || T.global_always) && (unsigned __int128)hash_cap(ndv) * hash_stride <= T.global_l2_bytes) variant = EIGER_GLOBAL;
    else variant = EIGER_PARTITION;
  }
  q->variant = variant;

  if (variant == EIGER_DIRECT) {
    if (!direct_ok) return EIGER_ERR_INFEASIBLE;
    if (!has_count) { p.op[na] = EIGER_COUNT; p.cnt_acc = na; p.n_acc = na + 1; }
    q->back = BACK_DIRECT;
    q->key_kind = (nk == 1 && keys[0].dtype == EIGER_I32 && R <= 0xFFFFFFFFull) ? KK_I32
                  : (nk == 1 && keys[0].dtype == EIGER_I64) ? KK_I64
                  : (nk == 2 && keys[0].dtype == EIGER_I8 && keys[1].dtype == EIGER_I8) ? KK_I8I8
                  : (kd.flags & kKey32) ? KK_GEN32 : KK_GEN;      // fused domain below 2^32: 32-bit slots indices
    q->cap = R; q->stride = 8u * p.n_acc;
    q->table_bytes = align_up((size_t)R * q->stride, 256);
    if (direct_bytes * 256 <= T.priv_smem && R <= (uint64_t)T.priv_max_range) {
      q->front = FRONT_PRIV; q->front_slots = (uint32_t)R; q->smem_bytes = (size_t)direct_bytes * 256;
    } else if (direct_bytes <= T.sdirect_bytes) {
      q->front = FRONT_SDIRECT; q->front_slots = (uint32_t)R;
      q->front_replicas = (uint32_t)std::max<size_t>(1, std::min<size_t>((size_t)T.sdirect_max_replicas, T.sdirect_replica_budget / (size_t)direct_bytes));
      q->smem_bytes = (size_t)direct_bytes * q->front_replicas;
    } else {
      q->front = FRONT_NONE;
      // between one CTA's shared memory and the L2-atomics regime: the array split over 2 .. 16 CTAs that
      // walk the same tiles (splitagg.cu); the smallest group whose share fits
      if (q->key_kind != KK_I8I8 && !skewed) {
        for (int lg = 1; (1 << lg) <= T.split_max; ++lg) {
          const uint64_t local = (R + (1ull << lg) - 1) >> lg;
          if ((unsigned __int128)local * 8 * p.n_acc <= T.split_bytes) {
            q->front = FRONT_SPLIT; q->split_lg = lg; q->front_slots = (uint32_t)local;
            q->smem_bytes = split_direct_smem(p.n_acc, (uint32_t)local);
            break;
          }
        }
      }
    }
    q->sig = detect_sig(p, na);
    if (q->front != FRONT_SPLIT && !aggregate_supported(q->key_kind, q->sig, q->front, q->back)) return EIGER_ERR_INFEASIBLE;
  } else if (variant == EIGER_SORT) {
    // sort-based group-by: LSD radix sort on the bits the key range needs, then
    // a segmented reduce.  No table: the workspace holds one or two copies of the rows.
    if (n >= (1ll << 32)) return EIGER_ERR_INFEASIBLE;       // 32-bit tile offsets
    q->back = BACK_HASH; q->stride = hash_stride; q->cap = 0; q->table_bytes = 0;
    q->key_kind = hkp;
    q->sig = detect_sig(p, na);
    int bits = 64;
    if (R != 0) { bits = 0; while (bits < 64 && (R - 1) >> bits) ++bits; }
    if (hkp == KK_I32 && bits > 32) bits = 32;
    q->sort_bits = bits; q->sort_passes = std::max(1, (bits + 7) / 8);
    const size_t kb = (bits <= 32) ? 4 : 8;
    size_t copy = align_up((size_t)n * kb, 256);
    for (int c = 0; c < p.n_vals; ++c) copy += align_up((size_t)n * 8, 256);
    q->part_bytes = copy * (q->sort_passes >= 2 ? 2 : 1) + align_up(((size_t)n / 1024 + 2) * 256 * 4, 256) + align_up(512 * 8, 256);
  } else {
    q->back = BACK_HASH;
    q->stride = hash_stride;
    q->key_kind = hk;
    q->sig = detect_sig(p, na);
    if (variant == EIGER_PARTITION) {
      if (n >= (1ll << 32)) return EIGER_ERR_INFEASIBLE;     // 32-bit per-partition counts
      q->key_kind = hkp;
      q->threads = T.part_threads; q->slots = part_slots; q->limit = (uint32_t)(0.85 * part_slots);
      const double per = std::max(1.0, T.load * part_slots);
      const double need = ndv * (1.0 + 4 * kSigma) / per;
      int bits = T.part_min_bits;
      while (bits < 20 && (double)(1u << bits) < need) ++bits;
      const int mb = partition_max_bits_per_level();
      if (bits <= mb) { q->bits1 = bits; q->bits2 = 0; } else { q->bits1 = (bits + 1) / 2; q->bits2 = bits - q->bits1; }
      // the global table only takes what overflows a partition's shared-memory table
      // the global table only takes what overflows a partition's shared-memory table, and the keys
      // of hot partitions that are cut into several work items (possible once n / P >= 32768)
      q->cap = std::min(q->cap_bound, (uint64_t)std::max(4096.0, ndv / 64.0));
      q->cap_hot = std::min(q->cap_bound, hash_cap(ndv));
      const size_t P1 = (size_t)1 << q->bits1, P = (size_t)1 << (q->bits1 + q->bits2);
      // (round 1 reserved the full-size table whenever the average partition held >= 32768 rows, because a
      // partition of more than twice the average is cut into items that merge through it: for uniform keys
      // nothing is ever cut and the unused 1 GB table cost 0.45 ms of init + compaction per call at
      // NDV 2^24.  A skewed input that does cut partitions now overflows the small table once and is
      // re-run with 4x the capacity, R10; EIGER_AUTO keeps skewed inputs away from this variant anyway)
      if (T.part_full_table && n / (int64_t)P >= 32768) q->cap = q->cap_hot;
      const size_t kb = (hkp == KK_I32 || hkp == KK_GEN32) ? 4 : 8;
      const size_t col = align_up((size_t)n * 8, 256), kcol = align_up((size_t)n * kb, 256);
      q->part_bytes = align_up(P * 4, 256) + align_up((P + 1) * 8, 256) + align_up((2 * P + 2) * 4, 256) + align_up((P1 + 1) * 8, 256) + align_up(P1 * 8, 256) +
                      (kcol + (size_t)p.n_vals * col);
      if (q->bits2 > 0) q->part_bytes += align_up((P + 1) * 8, 256) + align_up(P * 8, 256) + (kcol + (size_t)p.n_vals * col);
    } else {
      q->threads = T.smem_threads;
      const bool front = variant == EIGER_SMEM || T.global_front;
      q->slots = front ? smem_slots : 64;
      q->limit = front ? (uint32_t)((variant == EIGER_SMEM ? 0.75 : 0.5) * smem_slots) : 0;
      q->cap = std::min(hash_cap(ndv), q->cap_bound);
      if (variant == EIGER_SMEM && !skewed && (q->split_lg = split_lg_for(ndv)) > 0) {
        q->slots = split_slots; q->limit = (uint32_t)(0.75 * split_slots); q->threads = 1024;
      }
      // EIGER_GLOBAL: the rows the front cannot hold (C3: 28 % of them) cost a look-up and one L2 reduction per
      // accumulator each.  They are appended to a spill buffer instead, partitioned by hash and aggregated per
      // partition in shared memory like EIGER_PARTITION's rows; the partitions merge into the global table.
      // 64-bit rebased keys below the empty marker only (the marker pads the buffer), 8-byte value columns.
      bool all8 = true;
      for (int c = 0; c < p.n_vals; ++c) all8 = all8 && p.vw[c] != 4;
      if (variant == EIGER_GLOBAL && T.global_spill && T.global_front && hk != KK_I32 && R != 0 && all8 && !(T.ring & 1) &&
          (double)n >= T.spill_min_rows && n < (1ll << 32)) {
        const int sms = rt ? std::max(1, rt->sm_count) : 148;
        int lg = (int)T.spill_lg;
        while (((uint64_t)n / (uint64_t)sms) >> lg >= 1000) ++lg;        // a CTA reserves at most 1024 chunks (hashagg.cuh)
        const uint64_t chunk = 1ull << lg;
        q->spill_lg = lg;
        q->spill_rows = std::max<uint64_t>(chunk, ((uint64_t)((double)n * std::min(1.0, T.spill_frac)) + chunk - 1) / chunk * chunk);
        const size_t sp_slot_bytes = hash_agg_slot_bytes(p, KK_U64PRE);
        const size_t sp_tab = table_bytes_for(KK_U64PRE, T.part_threads, false, T.part_table_bytes);
        q->sp_slots = (uint32_t)std::max<size_t>(64, (sp_tab - 64) / sp_slot_bytes) & ~7u;
        q->sp_limit = (uint32_t)(0.85 * q->sp_slots); q->sp_threads = T.part_threads;
        const double per = std::max(1.0, T.load * q->sp_slots);
        const double need = ndv * (1.0 + 4 * kSigma) / per;
        int bits = T.part_min_bits;
        while (bits < 20 && (double)(1u << bits) < need) ++bits;
        const int mb = partition_max_bits_per_level();
        if (bits <= mb) { q->sp_bits1 = bits; q->sp_bits2 = 0; } else { q->sp_bits1 = (bits + 1) / 2; q->sp_bits2 = bits - q->sp_bits1; }
        q->sp_smem_bytes = align_up((size_t)q->sp_slots * sp_slot_bytes + 64, 16);
        q->sp_smem_dyn = q->sp_smem_bytes;                                  // this pass always loads its rows per thread
        const size_t P1 = (size_t)1 << q->sp_bits1, P = (size_t)1 << (q->sp_bits1 + q->sp_bits2);
        const size_t col = align_up((size_t)q->spill_rows * 8, 256);
        const size_t copy = (1 + (size_t)p.n_vals) * col;
        q->part_bytes = copy + align_up(P * 4, 256) + align_up((P + 1) * 8, 256) + align_up((2 * P + 2) * 4, 256) + align_up((P1 + 1) * 8, 256) +
                        align_up(P1 * 8, 256) + copy;
        if (q->sp_bits2 > 0) q->part_bytes += align_up((P + 1) * 8, 256) + align_up(P * 8, 256) + copy;
      }
    }
    q->smem_bytes = align_up((size_t)q->slots * (variant == EIGER_PARTITION ? part_slot_bytes : slot_bytes) + 64, 16);
    q->stages = T.stages; q->hot_reserved = variant != EIGER_PARTITION && want_hot;
    q->queue_bytes = variant == EIGER_GLOBAL ? miss_queue : 0;
    q->ring = (T.ring & (variant == EIGER_PARTITION ? 2 : 1)) != 0;
    q->smem_dyn = q->smem_bytes + (q->ring ? hash_agg_smem_layout(kd, p, variant == EIGER_PARTITION ? pre_kind : hk, q->threads, q->hot_reserved, T.stages).table_off : 0);
    q->table_bytes = align_up((size_t)(q->cap + 1) * q->stride, 256);
  }
  q->total_bytes = q->table_bytes + q->part_bytes + 256;
  return EIGER_OK;
}

// Turns the EIGER_SMEM plan of a key sample into the dictionary plan (FRONT_DICT): the sample's keys
// get dense ids (dictionary encoding; "if NDV is below a certain
// threshold, we will use dictionary encoding") and the aggregation indexes a per-CTA direct array with
// the id - the batched accumulate of FRONT_SDIRECT instead of the hash table's find-or-insert.
// Only for rebased keys of 32 bits; false when the shape does not fit.
bool make_dict_plan(QueryPlan* q, const eiger_col* keys, int nk, int na, double sample_ndv, const Tunables& T) {
  if (!T.dict || sample_ndv > std::max(T.dict_max_keys, T.dict_big_max_keys * (double)(1 << std::max(0, T.dict_max_pass_lg)))) return false;
  int kk;
  if (nk == 1 && keys[0].dtype == EIGER_I32) kk = KK_I32;
  else if (q->key.flags & kKey32) kk = KK_GEN32;
  else return false;
  AggPlan& p = q->plan;
  bool has_count = false;
  for (int j = 0; j < na; ++j) has_count = has_count || p.op[j] == EIGER_COUNT;
  if (!has_count) { if (na >= kMaxAcc) return false; p.op[na] = EIGER_COUNT; p.cnt_acc = na; p.n_acc = na + 1; }
  // ids: an eighth more than the sample shows (keys the sample missed abort the pass anyway)
  // more keys than one large dictionary holds: 2 or 4 passes, each with the dictionary of one hash slice of the keys
  int pass_lg = 0;
  if (sample_ndv > T.dict_max_keys) {
    if (T.dict_big_max_keys <= 0) return false;
    while (pass_lg < T.dict_max_pass_lg && sample_ndv > T.dict_big_max_keys * (double)(1 << pass_lg)) ++pass_lg;
    if (sample_ndv > T.dict_big_max_keys * (double)(1 << pass_lg)) return false;
  }
  // ids (per pass): an eighth more than the estimate, and four standard deviations of a slice's share on top
  const double per_pass = sample_ndv / (double)(1 << pass_lg);
  const uint32_t cap = (uint32_t)(((size_t)(1.125 * per_pass + (pass_lg ? 4.0 * std::sqrt(per_pass) : 0.0)) + 64 + 63) / 64 * 64);
  if (sample_ndv > T.dict_max_keys) {
    // the large dictionary: 12 bytes per id (SUM 8 + COUNT 4), 6 per dictionary entry (key 4 + id 2), one replica,
    // 16384 entries (load <= 0.57): 2^13 scattered keys in one CTA's shared memory.  SUM + COUNT plans only.
    const int sg = detect_sig(p, na);
    const uint32_t slots = 16384;
    if ((sg != SIG_SC && sg != SIG_SC32) || p.n_acc != 2 || cap > 65535u || 100 * (size_t)cap > 63 * (size_t)slots ||
        (size_t)cap * 12 + (size_t)slots * 6 > (220u << 10)) return false;
    q->back = BACK_DIRECT; q->front = FRONT_DICT; q->key_kind = kk;
    const size_t P = (size_t)1 << pass_lg;
    q->front_slots = cap; q->front_replicas = 1; q->cap = (uint64_t)cap * P; q->stride = 8u * p.n_acc;
    q->dict_slots = slots; q->dict_shift = 32 - 14; q->dict_compact = 1; q->dict_pass_lg = (uint32_t)pass_lg;
    q->smem_bytes = (size_t)cap * 12 + (size_t)slots * 6;
    q->sig = sg;
    q->variant = EIGER_SMEM;                 // (the sample's plan may have said PARTITION: the dictionary passes replace it)
    q->table_bytes = align_up((size_t)q->cap * q->stride, 256);
    q->part_bytes = align_up(P * slots * 8, 256) + align_up((size_t)q->cap * 4, 256) + 256;
    q->total_bytes = q->table_bytes + q->part_bytes + 256;
    return aggregate_supported(kk, q->sig, FRONT_DICT, BACK_DIRECT);
  }
  const size_t cell = (size_t)cap * 8 * p.n_acc;
  if (cell > (96u << 10)) return false;
  uint32_t slots = 4096;
  while (slots < 16384 && slots < 8 * cap) slots *= 2;
  if (cell + (size_t)slots * 8 > (220u << 10) || slots < 2 * cap) return false;
  int shift = 32; for (uint32_t x = slots; x > 1; x >>= 1) --shift;
  const uint32_t reps = (uint32_t)std::max<size_t>(1, std::min<size_t>(8, std::min<size_t>((64u << 10) / cell, ((220u << 10) - (size_t)slots * 8) / cell)));
  q->back = BACK_DIRECT; q->front = FRONT_DICT; q->key_kind = kk;
  q->front_slots = cap; q->front_replicas = reps; q->cap = cap; q->stride = 8u * p.n_acc;
  q->dict_slots = slots; q->dict_shift = (uint32_t)shift;
  q->smem_bytes = cell * reps + (size_t)slots * 8;
  q->sig = detect_sig(p, na);
  q->table_bytes = align_up((size_t)cap * q->stride, 256);
  q->part_bytes = align_up((size_t)slots * 8, 256) + align_up((size_t)cap * 4, 256) + 256;
  q->total_bytes = q->table_bytes + q->part_bytes + 256;
  return aggregate_supported(kk, q->sig, FRONT_DICT, BACK_DIRECT);
}

// Profiles nk key columns with one read-back: min/max of each, and (single column only) the
// sketch.  with_hll = 0 is the range-first shortcut: ndv_est = min(n, range).
// samples > 0: statistics of an evenly spaced sample of that many keys (plan of the speculative pass).
int do_profile(Runtime* rt, const eiger_col* cols, int nk, int64_t n, int with_hll, eiger_stats* out, cudaStream_t s,
               int64_t samples = 0, double* collision = nullptr) {
  if (nk > 1) with_hll = 0;
  {
    Timed t(s, 1);
    for (int k = 0; k < nk; ++k) {
      int rc = samples > 0 ? launch_profile_sample(rt, cols[k].data, cols[k].dtype, n, samples, k, with_hll, k == 0, s, k == nk - 1)
                           : launch_profile(rt, cols[k].data, cols[k].dtype, n, k, with_hll, k == 0, s);
      if (rc) return rc;
    }
    if (with_hll) { int rc = launch_hll_hist(rt, s); if (rc) return rc; }
  }
  struct Back { long long mn[kMaxKeyCols], mx[kMaxKeyCols]; uint32_t hist[64]; uint32_t pair_eq, pair_n; };
  Back* b = static_cast<Back*>(rt->pinned);
  EIGER_CUDA(cudaMemcpyAsync(b, rt->prof, sizeof(Back), cudaMemcpyDeviceToHost, s));
  EIGER_CUDA(cudaStreamSynchronize(s));
  resolve_timing();
  if (collision) *collision = b->pair_n ? (double)b->pair_eq / (double)b->pair_n : 0.0;
  for (int k = 0; k < nk; ++k) {
    out[k].min = b->mn[k]; out[k].max = b->mx[k]; out[k].n = n;
    if (n == 0) { out[k].ndv_est = 0.0; continue; }
    const double range = (double)((uint64_t)b->mx[k] - (uint64_t)b->mn[k]) + 1.0;
    double est = with_hll ? hll_estimate_from_hist(b->hist) : range;
    est = std::min(est, std::min((double)(samples > 0 ? std::min(n, samples) : n), range));
    out[k].ndv_est = std::max(est, 0.0);
  }
  // several key columns whose ranges multiply to more than a direct-index array can hold: the
  // product says little about the number of groups, so sketch the FUSED key (the
  // "otherwise HLL++" branch of smart key fusion).  out[0].ndv_est then carries the estimate for
  // the whole key and the other columns 1 (the planner multiplies the columns' estimates).
  if (nk > 1 && samples == 0 && n > 0) {
    KeyDesc kd;
    std::memset(&kd, 0, sizeof(kd));
    kd.ncols = nk; kd.mul = 1;
    unsigned __int128 prod = 1;
    bool fits = true, all32 = true;
    for (int k = 0; k < kMaxKeyCols; ++k) {
      kd.rng[k] = 1;
      if (k >= nk) { kd.ptr[k] = cols[0].data; kd.dtype[k] = cols[0].dtype; continue; }
      kd.ptr[k] = cols[k].data; kd.dtype[k] = cols[k].dtype; kd.base[k] = (uint64_t)out[k].min;
      kd.rng[k] = range_of(out[k]);
      all32 = all32 && cols[k].dtype == EIGER_I32;
      if (kd.rng[k] == 0) fits = false;
      if (fits) { prod *= kd.rng[k]; if (prod >> 64) fits = false; }
    }
    if (fits && prod > (unsigned __int128)tun().fused_sketch_min_range) {
      kd.flags = (all32 ? kKeyAll32 : 0) | (prod <= 0xFFFFFFFFull ? kKey32 : 0);
      { Timed t(s, 1);
        int rc = launch_fused_hll(rt, kd, n, s); if (rc) return rc;
        rc = launch_hll_hist(rt, s); if (rc) return rc; }
      EIGER_CUDA(cudaMemcpyAsync(b, rt->prof, sizeof(Back), cudaMemcpyDeviceToHost, s));
      EIGER_CUDA(cudaStreamSynchronize(s));
      resolve_timing();
      const double est = std::min(hll_estimate_from_hist(b->hist), std::min((double)n, (double)prod));
      out[0].ndv_est = std::max(est, 1.0);
      for (int k = 1; k < nk; ++k) out[k].ndv_est = 1.0;
    }
  }
  return EIGER_OK;
}

// device arenas owned by the library: g_arena holds the columns of eiger_groupby_host, g_ws the scratch of
// calls that pass workspace = NULL; both grow on demand and live until eiger_shutdown
struct Arena { char* base = nullptr; size_t size = 0; } g_arena, g_ws, g_enc;
int g_chain_depth = 0;
int ws_reserve(size_t bytes) {
  if (bytes <= g_ws.size) return EIGER_OK;
  if (g_ws.base) { cudaFree(g_ws.base); g_ws.base = nullptr; g_ws.size = 0; }
  EIGER_CUDA(cudaMalloc(reinterpret_cast<void**>(&g_ws.base), bytes));
  g_ws.size = bytes;
  return EIGER_OK;
}

int dict_encode_impl(Runtime* rt, const void* keys, int32_t dtype, int64_t n, int32_t* codes_out, void* dict_out, int64_t dict_capacity,
                     int64_t* ndv, void* workspace, size_t workspace_bytes, cudaStream_t s);
size_t dict_encode_ws_bytes(int32_t dtype, int64_t n, int64_t dict_capacity);
int groupby_through_dictionaries(Runtime* rt, const eiger_col* keys, int nk, int64_t n, const eiger_col* vals, int nv,
                                 const eiger_agg* aggs, int na, const eiger_stats* st, void* const* out_keys, void* const* out_aggs,
                                 int64_t out_capacity, int64_t* n_groups, int force, int32_t* chosen, cudaStream_t s, eiger_call_info* info);

int run_groupby(Runtime* rt, const eiger_col* keys, int nk, int64_t n, const eiger_col* vals, int nv,
                const eiger_agg* aggs, int na, const eiger_stats* stats_in,
                void* const* out_keys, void* const* out_aggs, int64_t out_capacity,
                int64_t* n_groups, int force, int32_t* chosen, void* workspace, size_t workspace_bytes,
                cudaStream_t s, eiger_call_info* info = nullptr) {
  if (!n_groups || !out_keys || !out_aggs || out_capacity < 0) return EIGER_ERR_ARG;
  *n_groups = 0;
  if (!keys || nk < 1 || nk > kMaxKeyCols || n < 0) return EIGER_ERR_ARG;
  for (int k = 0; k < nk; ++k) {
    if (!is_key_dtype(keys[k].dtype)) return EIGER_ERR_ARG;
    if (n > 0 && (!keys[k].data || ((uintptr_t)keys[k].data & 15))) return EIGER_ERR_ARG;
    if (!out_keys[k] && out_capacity > 0) return EIGER_ERR_ARG;
  }
  for (int c = 0; c < nv; ++c) if (n > 0 && vals && (!vals[c].data || ((uintptr_t)vals[c].data & 15))) return EIGER_ERR_ARG;
  if (n == 0) {   // legal: no groups; nothing is launched
    if (force < EIGER_AUTO || force > EIGER_SORT) return EIGER_ERR_ARG;
    if (chosen) *chosen = force;
    return EIGER_OK;
  }
  if ((uintptr_t)workspace & 255) return EIGER_ERR_ARG;
  eiger_call_info local_info;
  if (!info) info = &local_info;
  std::memset(info, 0, sizeof(*info));
  const int64_t launches0 = g_launches.load();
  struct LaunchCount { eiger_call_info* i; int64_t l0; ~LaunchCount() { i->kernel_launches = g_launches.load() - l0; } } launch_count{info, launches0};
  // workspace = NULL: the library's own arena, grown to what the plan at hand needs
  const bool own_ws = workspace == nullptr;
  if (own_ws) { if (!g_ws.base) { const int rc0 = ws_reserve((size_t)64 << 20); if (rc0) return rc0; } workspace = g_ws.base; workspace_bytes = g_ws.size; }
  for (int j = 0; j < na; ++j) if (!out_aggs[j] && out_capacity > 0) return EIGER_ERR_ARG;
  char* ws = static_cast<char*>(workspace);
  auto have_room = [&](size_t bytes) -> bool {             // may grow the library's arena (never the caller's workspace)
    if (bytes <= workspace_bytes) return true;
    if (!own_ws) return false;
    if (cudaStreamSynchronize(s) != cudaSuccess) return false;
    if (ws_reserve(bytes + bytes / 8) != EIGER_OK) return false;
    workspace = g_ws.base; workspace_bytes = g_ws.size; ws = g_ws.base;
    return true;
  };
  struct Back { unsigned long long n_groups; uint32_t overflow; uint32_t abort; };
  Back* hb = reinterpret_cast<Back*>(static_cast<char*>(rt->pinned) + 1024);
  int rc = EIGER_OK;

  // runs plan q; spec != 0: a speculative run that may give up (*aborted) and leaves no result then
  const int T_front_probes = tun().global_front_probes;
  int hot_n = 0;                 // heavy hitters of the key sample (skewed inputs only)
  long long hot_key[kMaxHot];
  // checked != 0: the statistics are the caller's: a key outside them must not corrupt memory
  // (direct arrays are indexed with key - min) or alias onto another group (fused keys); the kernels
  // run with the range check of the speculative pass and the call fails with EIGER_ERR_STATS
  const int checked = stats_in != nullptr;
  auto execute = [&](QueryPlan& q, const eiger_stats* st, int spec, bool* aborted) -> int {
  if (!have_room(q.total_bytes) || !workspace) return EIGER_ERR_WORKSPACE;
  info->dict_ids = q.front == FRONT_DICT ? (int32_t)q.front_slots : 0;
  info->variant = q.variant; info->ndv_est = q.ndv; info->sort_passes = q.variant == EIGER_SORT ? q.sort_passes : 0;
  const int src_kind = q.key_kind;
  for (int attempt = 0;; ++attempt) {
    info->attempts += 1;
    // workspace: [table][partition scratch]
    void* table = ws;
    char* pws = ws + q.table_bytes;
    EIGER_CUDA(cudaMemsetAsync(rt->call, 0, sizeof(CallDev), s));
    AggLaunch L{};
    L.key = q.key; L.plan = q.plan; L.n = n;
    L.key_kind = q.key_kind; L.sig = q.sig; L.front = q.front; L.back = q.back;
    L.front_slots = q.front_slots; L.front_limit = q.front_limit; L.front_replicas = q.front_replicas;
    L.table = table; L.cap = q.cap; L.stride = q.stride; L.call = rt->call;
    L.threads = 256; L.smem_bytes = q.smem_bytes; L.spec = spec | checked;
    if (q.variant == EIGER_SORT) {
      SortLaunch S{};
      S.key = q.key; S.plan = q.plan; S.n = n; S.key_kind = q.key_kind; S.sig = q.sig; S.bits = q.sort_bits;
      const size_t kb = (q.sort_bits <= 32) ? 4 : 8;
      const size_t col = align_up((size_t)n * 8, 256), kcol = align_up((size_t)n * kb, 256);
      auto take = [&](size_t bytes) { char* r = pws; pws += align_up(bytes, 256); return r; };
      S.tile_hist = reinterpret_cast<uint32_t*>(take(((size_t)n / 1024 + 2) * 256 * 4));
      S.digit_base = reinterpret_cast<unsigned long long*>(take(512 * 8));
      S.keysA = take(kcol);
      for (int c = 0; c < q.plan.n_vals; ++c) S.valsA[c] = take(col);
      if (q.sort_passes >= 2) { S.keysB = take(kcol); for (int c = 0; c < q.plan.n_vals; ++c) S.valsB[c] = take(col); }
      for (int k = 0; k < kMaxKeyCols; ++k) S.out_keys[k] = k < nk ? out_keys[k] : nullptr;
      for (int j = 0; j < na; ++j) S.out_aggs[j] = out_aggs[j];
      S.n_out_aggs = na; S.out_capacity = out_capacity; S.call = rt->call;
      { Timed t(s, 0); rc = launch_sort_groupby(S, rt->sm_count, rt->smem_optin, s); if (rc) return rc; }
      EIGER_CUDA(cudaMemcpyAsync(hb, rt->call, sizeof(Back), cudaMemcpyDeviceToHost, s));
      EIGER_CUDA(cudaStreamSynchronize(s));
      resolve_timing();
      *n_groups = (int64_t)hb->n_groups;
      if ((int64_t)hb->n_groups > out_capacity) return EIGER_ERR_OUT_CAPACITY;
      return EIGER_OK;
    }
    { Timed t(s, 3); rc = launch_table_init(L, s); if (rc) return rc; }

    uint32_t* dict_keys = nullptr;
    uint32_t* dict_counts = nullptr;
    if (q.front == FRONT_DICT) {
      // workspace after the table: dictionary image, id -> key, id counter
      auto take = [&](size_t bytes) { char* r = pws; pws += align_up(bytes, 256); return r; };
      L.dict = take(((size_t)q.dict_slots * 8) << q.dict_pass_lg); L.dict_slots = q.dict_slots; L.dict_shift = q.dict_shift;
      L.dict_compact = q.dict_compact; L.dict_pass_lg = q.dict_pass_lg;
      // small dictionaries at a load of 0.25 and more are placed and searched in pairs of entries (measured, 2^28 rows: 4096
      // keys 0.78 -> 0.72 ms; at 2048 keys / load 0.14 the pairs cost 6 %, at 2^4 / 2^8 keys 20 %)
      L.dict_group = (!q.dict_compact && q.front_replicas == 1 && 4 * (uint64_t)q.front_slots >= q.dict_slots &&
                      (q.sig == SIG_SC || q.sig == SIG_SC32) && tun().dict_pairs) ? 2u : 1u;
      dict_keys = reinterpret_cast<uint32_t*>(take((size_t)q.cap * 4));
      uint32_t* dict_n = reinterpret_cast<uint32_t*>(take(256));
      dict_counts = dict_n;
      // the large dictionaries are built from 4x the sample per pass (every key must be in it: 32 samples per key)
      const int64_t build_rows = std::min<int64_t>(n, tun().spec_samples * (q.dict_compact ? ((int64_t)4 << q.dict_pass_lg) : 1));
      { Timed t(s, 1); rc = launch_dict_build(L, build_rows, dict_keys, dict_n, s); if (rc) return rc; }
    }
    if (q.variant == EIGER_DIRECT || q.front == FRONT_DICT) {
      // persistent grid: as many CTAs as fit, never more than there are tiles
      const size_t per_cta = std::max<size_t>(q.smem_bytes, 1024);
      int occ = (int)std::min<size_t>(8, std::max<size_t>(1, (rt->smem_optin + 1024) / (per_cta + 1024)));
      if (q.front == FRONT_NONE) occ = 8;
      // shared-memory arrays: one 1024-thread CTA per SM.  Measured per 2^28 rows (C5 dense): 256-thread
      // CTAs reach 0.53 ms only while three of them fit the 196 KB carve-out (65.5 KB arrays), 0.61 ms
      // at 69.6 KB and 0.93 ms at 128 KB (one CTA = 8 warps per SM); the wide CTA runs 0.51-0.53 ms
      // at every size from 2^5 to 2^13 slots
      if (q.front == FRONT_DICT || (q.front == FRONT_SDIRECT && (tun().sdirect_wide || 3 * (per_cta + 1024) > (196u << 10)))) { L.threads = 1024; occ = 1; }
      const int64_t tiles = std::max<int64_t>(1, (n + 1023) / 1024);
      L.blocks = (int)std::min<int64_t>((int64_t)rt->sm_count * occ, tiles);
      if (q.front == FRONT_SPLIT) {
        SplitLaunch SL{};
        SL.key = q.key; SL.plan = q.plan; SL.n = n; SL.key_kind = q.key_kind; SL.sig = q.sig; SL.lgC = q.split_lg; SL.spec = spec | checked;
        SL.cap = q.cap; SL.local_slots = q.front_slots; SL.table = table; SL.call = rt->call;
        const int C = 1 << q.split_lg;
        const int64_t want = std::min<int64_t>(rt->sm_count / C, (n + 4095) / 4096);
        SL.blocks = (int)std::max<int64_t>(1, want) * C;
        { Timed t(s, 0); rc = launch_split_direct(SL, s); if (rc) return rc; }
      } else if (q.front == FRONT_DICT && q.dict_pass_lg > 0) {
        // one pass per key slice: its dictionary image, its part of the id table
        const char* img0 = static_cast<const char*>(L.dict);
        for (uint32_t pi = 0; pi < (1u << q.dict_pass_lg); ++pi) {
          AggLaunch Lp = L;
          Lp.dict = const_cast<char*>(img0) + (size_t)pi * q.dict_slots * 8;
          Lp.table = static_cast<char*>(table) + (size_t)pi * q.front_slots * q.stride;
          Lp.cap = q.front_slots; Lp.dict_pass = pi;
          { Timed t(s, 0); rc = launch_aggregate(Lp, s); if (rc) return rc; }
        }
      } else
      { Timed t(s, 0); rc = launch_aggregate(L, s); if (rc) return rc; }
    } else {
      HashAggLaunch H{};
      H.key = q.key; H.plan = q.plan; H.n = n; H.key_kind = src_kind; H.sig = q.sig;
      H.slots = q.slots; H.limit = q.limit; H.spec = spec;
      // EIGER_SMEM at loads up to 0.67: a chain of 16 full buckets turns up about once per million inserts - one
      // such row discards a speculative pass (scattered 2^13 keys did), so the chain may be as long as 64 buckets
      H.max_probes = q.variant == EIGER_GLOBAL ? T_front_probes : (q.variant == EIGER_SMEM ? 64 : 0);
      H.n_hot = (!spec && nk == 1 && q.variant != EIGER_PARTITION && (q.hot_reserved || !q.ring)) ? hot_n : 0;
      for (int i = 0; i < H.n_hot; ++i) H.hot[i] = (uint64_t)hot_key[i] - q.key.base[0];
      if (H.n_hot && src_kind == KK_I32) for (int i = 0; i < H.n_hot; ++i) H.hot[i] &= 0xFFFFFFFFull;
      H.table = table; H.cap = q.cap; H.stride = q.stride; H.call = rt->call;
      for (int k = 0; k < kMaxKeyCols; ++k) H.out_keys[k] = k < nk ? out_keys[k] : nullptr;
      for (int j = 0; j < na; ++j) H.out_aggs[j] = out_aggs[j];
      H.n_out_aggs = na; H.out_capacity = out_capacity;
      H.threads = q.threads; H.table_smem_bytes = q.smem_bytes; H.stages = q.stages; H.hot_reserved = q.hot_reserved; H.ring = q.ring ? 1 : 0; H.queue_bytes = spec ? 0 : q.queue_bytes;
      {   // 32-bit keys in a nearly empty shared-memory table: 8-byte buckets (hashagg.cuh: BK)
        const double per_table = q.variant == EIGER_PARTITION ? q.ndv / (double)((size_t)1 << (q.bits1 + q.bits2)) : q.ndv;
        H.bucket_keys = ((src_kind == KK_I32 || src_kind == KK_GEN32) && q.variant != EIGER_GLOBAL && per_table <= tun().narrow_load * q.slots) ? 2 : 0;
      }
      if (q.variant == EIGER_PARTITION) {
        PartitionLaunch P{};
        P.key = q.key; P.plan = q.plan; P.n = n; P.key_kind = src_kind; P.bits1 = q.bits1; P.bits2 = q.bits2;
        const size_t P1 = (size_t)1 << q.bits1, PP = (size_t)1 << (q.bits1 + q.bits2);
        const size_t kb = (src_kind == KK_I32 || src_kind == KK_GEN32) ? 4 : 8;
        const size_t col = align_up((size_t)n * 8, 256), kcol = align_up((size_t)n * kb, 256);
        auto take = [&](size_t bytes) { char* r = pws; pws += align_up(bytes, 256); return r; };
        P.hist = reinterpret_cast<uint32_t*>(take(PP * 4));
        P.item_off = reinterpret_cast<unsigned long long*>(take((PP + 1) * 8));
        P.item_part = reinterpret_cast<uint32_t*>(take((2 * PP + 2) * 4));
        P.chunk_rows = std::max<int64_t>(32768, n / (int64_t)PP);
        P.pre_hist = q.pre_hist;
        P.off1 = reinterpret_cast<unsigned long long*>(take((P1 + 1) * 8));
        P.cur1 = reinterpret_cast<unsigned long long*>(take(P1 * 8));
        P.keysA = take(kcol);
        for (int c = 0; c < q.plan.n_vals; ++c) P.valsA[c] = take(col);
        if (q.bits2 > 0) {
          P.off2 = reinterpret_cast<unsigned long long*>(take((PP + 1) * 8));
          P.cur2 = reinterpret_cast<unsigned long long*>(take(PP * 8));
          P.keysB = take(kcol);
          for (int c = 0; c < q.plan.n_vals; ++c) P.valsB[c] = take(col);
        }
        { Timed t(s, 2); rc = launch_partition(P, rt->sm_count, rt->smem_optin, s); if (rc) return rc; }
        info->partition_levels = q.bits2 > 0 ? 2 : 1;
        info->partition_prehist = q.pre_hist ? 1 : 0;
        info->partition_key_bytes = (int)kb;
        // the aggregation pass reads the partitioned copy, one CTA per partition at a time
        H.key.ptr[0] = P.out_keys;
        for (int c = 0; c < q.plan.n_vals; ++c) H.plan.vals[c] = P.out_vals[c];
        H.key_kind = (src_kind == KK_I32 || src_kind == KK_GEN32) ? KK_U32PRE : KK_U64PRE;
        H.part_off = P.out_off; H.item_off = P.item_off; H.item_part = P.item_part; H.n_parts = P.n_parts;
        const int occ = (int)std::max<size_t>(1, std::min<size_t>((size_t)(2048 / q.threads), (rt->smem_optin + 1024) / (q.smem_dyn + 1024)));
        H.blocks = (int)std::min<int64_t>((int64_t)rt->sm_count * occ, (int64_t)P.n_parts + n / P.chunk_rows);
      } else {
        const int64_t tiles = std::max<int64_t>(1, n / (4 * (int64_t)q.threads));
        H.blocks = (int)std::min<int64_t>(rt->sm_count, tiles);
      }
      // EIGER_GLOBAL with a spill buffer: [keys][value columns] of q.spill_rows rows each, then the partition scratch
      const bool spilling = q.variant == EIGER_GLOBAL && q.spill_rows > 0 && !spec && !q.ring;
      const size_t sp_col = align_up((size_t)q.spill_rows * 8, 256);
      if (spilling) {
        H.spill_keys = reinterpret_cast<uint64_t*>(pws); pws += sp_col;
        for (int c = 0; c < q.plan.n_vals; ++c) { H.spill_vals[c] = reinterpret_cast<uint64_t*>(pws); pws += sp_col; }
        H.spill_lg = q.spill_lg; H.spill_cap_chunks = q.spill_rows >> q.spill_lg;
      }
      if (q.variant == EIGER_SMEM && q.split_lg > 0) {
        const int C = 1 << q.split_lg;
        H.blocks = (int)std::max<int64_t>(1, std::min<int64_t>(rt->sm_count / C, (n + 4095) / 4096)) * C;
        H.bucket_keys = 0;
        { Timed t(s, 0); rc = launch_split_hash(H, q.split_lg, s); if (rc) return rc; }
      } else
      { Timed t(s, 0); rc = launch_hash_agg(H, s); if (rc) return rc; }
      if (spilling) {
        // how much was spilled (whole chunks; the tail of every CTA's last chunk is padding)
        unsigned long long* chunks = reinterpret_cast<unsigned long long*>(static_cast<char*>(rt->pinned) + 1536);
        EIGER_CUDA(cudaMemcpyAsync(chunks, reinterpret_cast<const char*>(rt->call) + offsetof(CallDev, spill_chunks), sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
        EIGER_CUDA(cudaStreamSynchronize(s));
        const int64_t n_sp = (int64_t)(std::min<unsigned long long>(*chunks, H.spill_cap_chunks) << q.spill_lg);
        info->spill_rows = n_sp;
        if (n_sp > 0) {
          PartitionLaunch P{};
          P.key = q.key; P.key.ptr[0] = H.spill_keys; P.key.ncols = 1;
          for (int k = 1; k < kMaxKeyCols; ++k) P.key.ptr[k] = nullptr;
          P.plan = q.plan;
          for (int c = 0; c < q.plan.n_vals; ++c) { P.plan.vals[c] = H.spill_vals[c]; P.plan.vw[c] = 8; }
          P.n = n_sp; P.key_kind = KK_U64PRE; P.bits1 = q.sp_bits1; P.bits2 = q.sp_bits2;
          const size_t P1 = (size_t)1 << q.sp_bits1, PP = (size_t)1 << (q.sp_bits1 + q.sp_bits2);
          auto take = [&](size_t bytes) { char* r = pws; pws += align_up(bytes, 256); return r; };
          P.hist = reinterpret_cast<uint32_t*>(take(PP * 4));
          P.item_off = reinterpret_cast<unsigned long long*>(take((PP + 1) * 8));
          P.item_part = reinterpret_cast<uint32_t*>(take((2 * PP + 2) * 4));
          P.chunk_rows = std::max<int64_t>(32768, n_sp / (int64_t)PP);
          P.off1 = reinterpret_cast<unsigned long long*>(take((P1 + 1) * 8));
          P.cur1 = reinterpret_cast<unsigned long long*>(take(P1 * 8));
          P.keysA = take(sp_col);
          for (int c = 0; c < q.plan.n_vals; ++c) P.valsA[c] = take(sp_col);
          if (q.sp_bits2 > 0) {
            P.off2 = reinterpret_cast<unsigned long long*>(take((PP + 1) * 8));
            P.cur2 = reinterpret_cast<unsigned long long*>(take(PP * 8));
            P.keysB = take(sp_col);
            for (int c = 0; c < q.plan.n_vals; ++c) P.valsB[c] = take(sp_col);
          }
          { Timed t(s, 2); rc = launch_partition(P, rt->sm_count, rt->smem_optin, s); if (rc) return rc; }
          info->partition_levels = q.sp_bits2 > 0 ? 2 : 1;
          info->partition_key_bytes = 8;
          HashAggLaunch H2 = H;
          H2.key = P.key; H2.key.ptr[0] = P.out_keys; H2.plan = P.plan;
          for (int c = 0; c < q.plan.n_vals; ++c) H2.plan.vals[c] = P.out_vals[c];
          H2.n = n_sp; H2.key_kind = KK_U64PRE;
          H2.part_off = P.out_off; H2.item_off = P.item_off; H2.item_part = P.item_part; H2.n_parts = P.n_parts;
          H2.slots = q.sp_slots; H2.limit = q.sp_limit; H2.max_probes = 0; H2.bucket_keys = 0; H2.n_hot = 0;
          H2.threads = q.sp_threads; H2.table_smem_bytes = q.sp_smem_bytes; H2.hot_reserved = false; H2.ring = 0; H2.queue_bytes = 0;
          H2.spill_keys = nullptr; H2.skip_empty = 1; H2.force_merge = 1;
          const int occ = (int)std::max<size_t>(1, std::min<size_t>((size_t)(2048 / q.sp_threads), (rt->smem_optin + 1024) / (q.sp_smem_dyn + 1024)));
          H2.blocks = (int)std::min<int64_t>((int64_t)rt->sm_count * occ, (int64_t)P.n_parts + n_sp / P.chunk_rows);
          { Timed t(s, 5); rc = launch_hash_agg(H2, s); if (rc) return rc; }
        }
      }
    }

    CompactLaunch C{};
    C.key = q.key; C.plan = q.plan; C.back = q.back; C.table = table; C.cap = q.cap; C.stride = q.stride;
    for (int k = 0; k < kMaxKeyCols; ++k) C.out_keys[k] = k < nk ? out_keys[k] : nullptr;
    for (int j = 0; j < na; ++j) C.out_aggs[j] = out_aggs[j];
    C.n_out_aggs = na; C.out_capacity = out_capacity; C.call = rt->call; C.R = q.R; C.dict_keys = dict_keys;
    { Timed t(s, 4); rc = launch_compact(C, rt->sm_count, s); if (rc) return rc; }

    EIGER_CUDA(cudaMemcpyAsync(hb, rt->call, sizeof(Back), cudaMemcpyDeviceToHost, s));
    EIGER_CUDA(cudaStreamSynchronize(s));
    resolve_timing();
    if (dict_counts && std::getenv("EIGER_DEBUG")) {
      uint32_t dn[4] = {0, 0, 0, 0};
      cudaMemcpy(dn, dict_counts, sizeof(uint32_t) << q.dict_pass_lg, cudaMemcpyDeviceToHost);
      std::fprintf(stderr, "[eiger] dictionary: abort %u overflow %u groups %llu, ids per slice %u %u %u %u of %u\n", hb->abort, hb->overflow,
                   (unsigned long long)hb->n_groups, dn[0], dn[1], dn[2], dn[3], q.front_slots);
    }
    if (spec && (hb->abort || hb->overflow)) { *aborted = true; return EIGER_OK; }
    if (hb->abort) return EIGER_ERR_STATS;
    if (hb->overflow) {
      // the sketch under-estimated (R10): grow towards the exact bound and run again
      if (std::getenv("EIGER_DEBUG")) std::fprintf(stderr, "[eiger] table overflow (attempt %d): variant %d cap %llu slots %u limit %u bits %d+%d ndv %.0f\n", attempt, q.variant, (unsigned long long)q.cap, q.slots, q.limit, q.bits1, q.bits2, q.ndv);
      if (q.back != BACK_HASH || attempt >= 8) return EIGER_ERR_TABLE_OVERFLOW;
      if (q.cap >= q.cap_bound && q.variant != EIGER_PARTITION) return EIGER_ERR_TABLE_OVERFLOW;
      q.cap = std::min(q.cap_bound, q.cap * 4);
      q.table_bytes = align_up((size_t)(q.cap + 1) * q.stride, 256);
      if (q.variant == EIGER_PARTITION) {
        // more partitions as well: re-plan the fan-out for four times the estimate
        eiger_stats grown[kMaxKeyCols];
        for (int k = 0; k < kMaxKeyCols; ++k) { grown[k] = st[k < nk ? k : 0]; grown[k].ndv_est = 1.0; }
        grown[0].ndv_est = std::min((double)n, std::max(q.ndv, 1.0) * 4.0);
        QueryPlan q2;
        rc = plan_query(rt, keys, nk, n, vals, nv, aggs, na, grown, EIGER_PARTITION, &q2);
        if (rc) return rc;
        q2.cap = std::max(q2.cap, q.cap); q2.table_bytes = align_up((size_t)(q2.cap + 1) * q2.stride, 256);
        q2.total_bytes = q2.table_bytes + q2.part_bytes + 256;
        q2.key = q.key; q2.pre_hist = q.pre_hist;      // same key base (any base gives the same groups)
        q = q2;
      }
      q.total_bytes = q.table_bytes + q.part_bytes + 256;
      if (!have_room(q.total_bytes)) return EIGER_ERR_TABLE_OVERFLOW;
      info->ndv_est = q.ndv;
      continue;
    }
    *n_groups = (int64_t)hb->n_groups;
    if ((int64_t)hb->n_groups > out_capacity) return EIGER_ERR_OUT_CAPACITY;
    return EIGER_OK;
  }
  };

  eiger_stats local[kMaxKeyCols];
  const Tunables& T = tun();
  bool skewed = false;
  if (!stats_in && force == EIGER_AUTO && n >= T.spec_min_rows) {
    // EIGER_AUTO, no statistics: first the statistics of an evenly spaced sample (one tiny kernel).
    // When the sample says "few groups" one speculative pass aggregates AND verifies (every key
    // inside the sampled range / room in every CTA's table), so low-NDV inputs are read exactly
    // once; otherwise, or if the verification fails, the full profile (A1-A3) and the selected
    // variant run as usual.  The sample also tells hot-key inputs from uniform ones.
    double collision = 0.0;
    rc = do_profile(rt, keys, nk, n, keys[0].dtype != EIGER_I8, local, s, T.spec_samples, &collision);
    if (rc) return rc;
    // uniform keys collide at rate 1 / NDV: "skewed" means well above that (and above the floor)
    // (several key columns: `collision` compares whole sample rows, and the NDV beside it is the product of the
    // columns' sample estimates, capped by the sample size)
    double sample_ndv = 1.0;
    for (int k = 0; k < nk; ++k) sample_ndv = std::min((double)T.spec_samples, sample_ndv * std::max(local[k].ndv_est, 1.0));
    skewed = collision > T.skew_collision && collision * sample_ndv > 4.0;
    if (skewed && T.hot && nk == 1) {
      // which keys are the hot ones: the whole-input hash kernel reduces their rows inside the warp
      { Timed t(s, 1); rc = launch_hot_keys(rt, keys[0].data, keys[0].dtype, n, s); if (rc) return rc; }
      struct HBack { long long key[kMaxHot]; uint32_t cnt[kMaxHot]; uint32_t n, samples; };
      HBack* hbk = reinterpret_cast<HBack*>(static_cast<char*>(rt->pinned) + 2048);
      EIGER_CUDA(cudaMemcpyAsync(hbk, reinterpret_cast<const char*>(rt->prof) + offsetof(ProfileDev, hot_key), sizeof(HBack), cudaMemcpyDeviceToHost, s));
      EIGER_CUDA(cudaStreamSynchronize(s));
      resolve_timing();
      for (uint32_t i = 0; i < hbk->n && i < (uint32_t)kMaxHot; ++i)
        if ((double)hbk->cnt[i] >= T.hot_min_share * (double)hbk->samples) hot_key[hot_n++] = hbk->key[i];
      if (std::getenv("EIGER_DEBUG")) std::fprintf(stderr, "[eiger] heavy hitters: %d (top share %.3f)\n", hot_n, hbk->n ? (double)hbk->cnt[0] / hbk->samples : 0.0);
    }
    // every key kind notices a key outside the planned range of its column (rows.cuh: fuse_cols)
    const bool fusable = true;
    for (int k = 0; k < nk; ++k) {       // a little slack around the sampled range (clamped to the key type)
      const int bits = 8 * dtype_size(keys[k].dtype);
      const int64_t tmin = bits == 64 ? INT64_MIN : -(1ll << (bits - 1)), tmax = bits == 64 ? INT64_MAX : (1ll << (bits - 1)) - 1;
      const uint64_t R = (uint64_t)local[k].max - (uint64_t)local[k].min + 1ull;
      const int64_t margin = (R > 64 && R <= (1ull << 24)) ? (int64_t)(R / 32) : 0;   // only direct tables need the range
      // room to the type's ends in unsigned arithmetic (min - INT64_MIN overflows int64 for any min >= 0)
      const uint64_t room_lo = (uint64_t)local[k].min - (uint64_t)tmin, room_hi = (uint64_t)tmax - (uint64_t)local[k].max;
      local[k].min = room_lo >= (uint64_t)margin ? local[k].min - margin : tmin;
      local[k].max = room_hi >= (uint64_t)margin ? local[k].max + margin : tmax;
      local[k].n = n;
    }
    {
      // scattered keys that the sample names completely: dictionary + direct array, verified exactly
      // (a key the dictionary does not hold discards the pass)
      QueryPlan qd;
      double sndv = local[0].ndv_est;
      for (int k = 1; k < nk; ++k) sndv *= local[k].ndv_est;
      sndv = std::min(sndv, (double)T.spec_samples);
      // a single column whose sample is far from having seen every key twice: what that many distinct keys among s
      // samples mean for UNIFORM keys (the inversion also used below); the large dictionaries are built from a larger
      // sample, and a key they still lack only costs the discarded pass
      if (nk == 1 && sndv > T.dict_max_keys) {
        const double smp = (double)std::min<int64_t>(n, T.spec_samples), r = std::min(sndv / smp, 0.98);
        if (r > 0.05) {
          double lo = 0.02, hi = 50.0;
          for (int it = 0; it < 60; ++it) { const double x = 0.5 * (lo + hi); if ((1.0 - std::exp(-x)) / x > r) lo = x; else hi = x; }
          sndv = std::max(sndv, smp / (0.5 * (lo + hi)));
        }
      }
      if (T.spec && T.dict && !skewed && plan_query(rt, keys, nk, n, vals, nv, aggs, na, local, EIGER_AUTO, &qd, skewed) == EIGER_OK &&
          (qd.variant == EIGER_SMEM || (qd.variant == EIGER_PARTITION && nk == 1 && sndv > T.dict_max_keys)) &&
          make_dict_plan(&qd, keys, nk, na, sndv, T) && have_room(qd.total_bytes)) {
        bool aborted = false;
        rc = execute(qd, local, 1, &aborted);
        if (std::getenv("EIGER_DEBUG")) std::fprintf(stderr, "[eiger] dictionary pass (%u ids, %u dictionary slots, %u replicas): rc %d aborted %d\n", qd.front_slots, qd.dict_slots, qd.front_replicas, rc, (int)aborted);
        if (rc != EIGER_OK || !aborted) { if (chosen) *chosen = EIGER_SMEM; return rc; }
      }
    }
    // The sample's NDV is a lower bound; when the sample is far from having seen every key twice, plan the
    // speculative pass for what that many distinct keys among s samples mean for UNIFORM keys
    // (ds / s = (1 - exp(-x)) / x, x = s / D); a wrong guess only costs the discarded pass
    eiger_stats plan_stats[kMaxKeyCols];
    for (int k = 0; k < nk; ++k) plan_stats[k] = local[k];
    if (nk == 1 && !skewed) {
      const double smp = (double)std::min<int64_t>(n, T.spec_samples), ds = std::max(1.0, local[0].ndv_est);
      const double r = std::min(ds / smp, 0.98);
      if (r > 0.05) {
        double lo = 0.02, hi = 50.0;
        for (int it = 0; it < 60; ++it) { const double x = 0.5 * (lo + hi); if ((1.0 - std::exp(-x)) / x > r) lo = x; else hi = x; }
        const double range = (double)((uint64_t)local[0].max - (uint64_t)local[0].min) + 1.0;
        plan_stats[0].ndv_est = std::min(std::max(ds, smp / (0.5 * (lo + hi))), std::min((double)n, range));
      }
    }
    QueryPlan qs;
    if (std::getenv("EIGER_DEBUG")) std::fprintf(stderr, "[eiger] sample: min %lld max %lld ndv %.1f collision %.5f\n", (long long)local[0].min, (long long)local[0].max, local[0].ndv_est, collision);
    if (T.spec && fusable && plan_query(rt, keys, nk, n, vals, nv, aggs, na, plan_stats, EIGER_AUTO, &qs, skewed) == EIGER_OK &&
        ((qs.variant == EIGER_DIRECT && (qs.front != FRONT_NONE || qs.R <= (1ull << 24))) ||
         (qs.variant == EIGER_SMEM && qs.ndv * (1.0 + 4 * kSigma) <= 0.70 * qs.slots * (double)(1 << qs.split_lg))) && have_room(qs.total_bytes)) {   // tables close at 0.75 x slots: a fuller table than planned discards the pass
      bool aborted = false;
      if (std::getenv("EIGER_DEBUG")) std::fprintf(stderr, "[eiger] plan: variant %d kk %d sig %d slots %u limit %u cap %llu stride %u smem %zu front %d R %llu\n", qs.variant, qs.key_kind, qs.sig, qs.slots, qs.limit, (unsigned long long)qs.cap, qs.stride, qs.smem_bytes, qs.front, (unsigned long long)qs.R);
      rc = execute(qs, local, 1, &aborted);
      if (std::getenv("EIGER_DEBUG")) std::fprintf(stderr, "[eiger] speculative %s: rc %d aborted %d\n", eiger_variant_name(qs.variant), rc, (int)aborted);
      if (rc != EIGER_OK || !aborted) { if (chosen) *chosen = qs.variant; return rc; }
    }
  }
  if (!stats_in && force == EIGER_AUTO && n >= T.spec_min_rows && T.slice && !skewed && nk == 1 && n < (1ll << 32) &&
      (keys[0].dtype == EIGER_I32 || keys[0].dtype == EIGER_I64)) {
    // The sample's range and NDV are lower bounds of the column's, and every rule of the selector
    // is monotone in both: when even the sample's statistics select PARTITION, the full statistics
    // do too.  What is still missing is the NDV that sizes the fan-out.  Instead of a full-column
    // sketch, ONE keys-only pass takes the level-1 histogram (which the partitioner needs anyway),
    // the exact min/max, and the sketch of a hash-space slice of the keys (profile.cu).
    QueryPlan qp;
    if (plan_query(rt, keys, nk, n, vals, nv, aggs, na, local, EIGER_AUTO, &qp, skewed) == EIGER_OK && qp.variant == EIGER_PARTITION) {
      // Lower bound of the column's NDV from the sample: the sample's own NDV ds, or - when the
      // sample is far from having seen every key - half of what ds distinct keys among s samples
      // mean for UNIFORM keys, ds / s = (1 - exp(-x)) / x with x = s / D (any other distribution
      // with the same D shows fewer distinct keys, so the inversion can only fall short of D).
      const double smp = (double)std::min<int64_t>(n, T.spec_samples);
      double ds = std::max(1.0, local[0].ndv_est);
      {
        const double r = std::min(ds / smp, 0.999);
        double lo = 0.05, hi = 50.0;                       // x = s / D; D capped at 20 s (sketch noise as r -> 1)
        for (int it = 0; it < 60; ++it) { const double x = 0.5 * (lo + hi); if ((1.0 - std::exp(-x)) / x > r) lo = x; else hi = x; }
        ds = std::max(ds, 0.5 * smp / (0.5 * (lo + hi)));
      }
      uint32_t sel = kPreFan;
      while (sel > 1 && ds * (double)(sel / 2) / (double)kPreFan >= T.slice_min_keys) sel /= 2;
      const uint64_t base = (uint64_t)local[0].min;
      { Timed t(s, 1);
        rc = launch_part_hist_hll(rt, keys[0].data, keys[0].dtype, n, base, sel, s); if (rc) return rc;
        rc = launch_hll_hist(rt, s); if (rc) return rc; }
      struct PBack { long long mn[kMaxKeyCols], mx[kMaxKeyCols]; uint32_t hist[64]; uint32_t pair_eq, pair_n; };
      PBack* b = static_cast<PBack*>(rt->pinned);
      EIGER_CUDA(cudaMemcpyAsync(b, rt->prof, sizeof(PBack), cudaMemcpyDeviceToHost, s));
      EIGER_CUDA(cudaStreamSynchronize(s));
      resolve_timing();
      eiger_stats st2;
      st2.min = b->mn[0]; st2.max = b->mx[0]; st2.n = n;
      const double range = (double)((uint64_t)st2.max - (uint64_t)st2.min) + 1.0;
      const double slice = hll_estimate_from_hist(b->hist);
      // 1 / sqrt(slice NDV) sampling error on top of the sketch's own: four of those as head room
      const double est = slice * (double)kPreFan / (double)sel * (1.0 + 4.0 / std::sqrt(std::max(slice, 1.0)));
      st2.ndv_est = std::max(1.0, std::min(est, std::min((double)n, range)));
      if (std::getenv("EIGER_DEBUG")) std::fprintf(stderr, "[eiger] slice sketch: sel %u / %d, slice ndv %.1f -> ndv %.1f, min %lld max %lld\n", sel, kPreFan, slice, st2.ndv_est, (long long)st2.min, (long long)st2.max);
      QueryPlan q;
      rc = plan_query(rt, keys, nk, n, vals, nv, aggs, na, &st2, EIGER_PARTITION, &q, skewed);
      if (rc) return rc;
      q.key.base[0] = base;                 // the histogram was taken with this base
      q.pre_hist = rt->prof->part_hist;
      if (chosen) *chosen = q.variant;
      return execute(q, &st2, 0, nullptr);
    }
  }
  if (!stats_in && force == EIGER_AUTO && n >= T.spec_min_rows && T.slice && T.slice_fused && !skewed && nk >= 2 && n < (1ll << 32)) {
    // Several key columns: the full profile costs one pass per column (min/max), one over all of them (sketch of
    // the fused key) and the partitioner a third (level-1 histogram).  When the sample's ranges already send the
    // query to PARTITION, ONE pass does all of it: the columns are fused with the sample's ranges - a value
    // outside its column's range flags the pass, and the full profile below runs after all - the fused key's
    // level-1 histogram is taken, and the fused keys of a sixteenth of the hash space are sketched (distinct
    // sampling, as for one column).  The product of the per-column NDVs says little about the number of groups
    // (5000 triples can span 2^61), so the selector runs again on the verified ranges and the slice estimate and
    // may still pick another variant; the histogram is used when it stays with PARTITION.
    QueryPlan qp;
    if (plan_query(rt, keys, nk, n, vals, nv, aggs, na, local, EIGER_AUTO, &qp, skewed) == EIGER_OK && qp.variant == EIGER_PARTITION &&
        (qp.key_kind == KK_GEN || qp.key_kind == KK_GEN32)) {
      const uint32_t sel = kPreFan / 16;
      { Timed t(s, 1);
        rc = launch_fused_part_hist_hll(rt, qp.key, qp.key_kind, n, sel, s); if (rc) return rc;
        rc = launch_hll_hist(rt, s); if (rc) return rc; }
      struct PBack { long long mn[kMaxKeyCols], mx[kMaxKeyCols]; uint32_t hist[64]; uint32_t pair_eq, pair_n, oor, oor_pad; };
      PBack* b = static_cast<PBack*>(rt->pinned);
      EIGER_CUDA(cudaMemcpyAsync(b, rt->prof, sizeof(PBack), cudaMemcpyDeviceToHost, s));
      EIGER_CUDA(cudaStreamSynchronize(s));
      resolve_timing();
      if (std::getenv("EIGER_DEBUG")) std::fprintf(stderr, "[eiger] fused slice sketch: out of range %u, slice ndv %.1f\n", b->oor, hll_estimate_from_hist(b->hist));
      if (b->oor == 0u) {
        eiger_stats st2[kMaxKeyCols];
        for (int k = 0; k < nk; ++k) { st2[k] = local[k]; st2[k].ndv_est = 1.0; }
        const double slice = hll_estimate_from_hist(b->hist);
        const double est = slice * (double)kPreFan / (double)sel * (1.0 + 4.0 / std::sqrt(std::max(slice, 1.0)));
        st2[0].ndv_est = std::max(256.0, std::min(est, (double)n));       // (an empty slice says "few", not "none")
        QueryPlan q;
        rc = plan_query(rt, keys, nk, n, vals, nv, aggs, na, st2, EIGER_AUTO, &q, skewed);
        if (rc) return rc;
        if (q.variant == EIGER_PARTITION && q.key_kind == qp.key_kind) q.pre_hist = rt->prof->part_hist;   // same ranges, same fusion, same hash
        if (chosen) *chosen = q.variant;
        return execute(q, st2, 0, nullptr);
      }
    }
  }
  const eiger_stats* st = stats_in;
  if (!st) {
    // profile inside the call: fused min/max + sketch for 4/8-byte keys; 1-byte keys take the
    // range test only (HLL only when the range test fails; a 1-byte range never does)
    rc = do_profile(rt, keys, nk, n, keys[0].dtype != EIGER_I8, local, s);
    if (rc) return rc;
    st = local;
  }
  QueryPlan q;
  rc = plan_query(rt, keys, nk, n, vals, nv, aggs, na, st, force, &q, skewed);
  if (rc == EIGER_ERR_INFEASIBLE && nk >= 2 && own_ws && force != EIGER_DIRECT && g_chain_depth == 0) {
    // The ranges of the key columns multiply past 2^64: no fused key exists.  The paper's order
    // (PAPER.md:219): range test first, "otherwise ... dictionary encoding" - the widest columns are
    // dictionary-encoded (order-preserving, Algorithm 1) until the fused domain fits, the group-by
    // runs on the codes and the dictionaries decode the group keys.
    bool wide = false;
    { unsigned __int128 prod = 1; for (int k = 0; k < nk; ++k) { const uint64_t r = range_of(st[k]); if (r == 0) { wide = true; break; } prod *= r; if (prod >> 64) { wide = true; break; } } }
    if (wide) {
      ++g_chain_depth;       // the call on the code columns must not encode again (codes of codes have the same NDV)
      const int rc2 = groupby_through_dictionaries(rt, keys, nk, n, vals, nv, aggs, na, st, out_keys, out_aggs, out_capacity, n_groups, force, chosen, s, info);
      --g_chain_depth;
      return rc2;
    }
  }
  if (rc) return rc;
  if (chosen) *chosen = q.variant;
  return execute(q, st, 0, nullptr);
}

// ---- device arena for eiger_groupby_host ---------------------------------------------------
int arena_reserve(size_t bytes) {
  if (bytes <= g_arena.size) return EIGER_OK;
  if (g_arena.base) { cudaFree(g_arena.base); g_arena.base = nullptr; g_arena.size = 0; }
  EIGER_CUDA(cudaMalloc(reinterpret_cast<void**>(&g_arena.base), bytes));
  g_arena.size = bytes;
  return EIGER_OK;
}

int enc_reserve(size_t bytes) {
  if (bytes <= g_enc.size) return EIGER_OK;
  if (g_enc.base) { cudaFree(g_enc.base); g_enc.base = nullptr; g_enc.size = 0; }
  EIGER_CUDA(cudaMalloc(reinterpret_cast<void**>(&g_enc.base), bytes));
  g_enc.size = bytes;
  return EIGER_OK;
}

__global__ void dict_decode_kernel(const int32_t* __restrict__ codes, const void* __restrict__ dict, int dtype, int64_t g, void* __restrict__ out) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < g; i += stride) {
    const int64_t c = codes[i];
    switch (dtype) {
      case EIGER_I8: static_cast<int8_t*>(out)[i] = static_cast<const int8_t*>(dict)[c]; break;
      case EIGER_I32: static_cast<int32_t*>(out)[i] = static_cast<const int32_t*>(dict)[c]; break;
      default: static_cast<int64_t*>(out)[i] = static_cast<const int64_t*>(dict)[c]; break;
    }
  }
}

int groupby_through_dictionaries(Runtime* rt, const eiger_col* keys, int nk, int64_t n, const eiger_col* vals, int nv,
                                 const eiger_agg* aggs, int na, const eiger_stats* st, void* const* out_keys, void* const* out_aggs,
                                 int64_t out_capacity, int64_t* n_groups, int force, int32_t* chosen, cudaStream_t s, eiger_call_info* info) {
  // widest columns first, until the product of (code ranges, remaining column ranges) fits 63 bits
  int order[kMaxKeyCols];
  for (int k = 0; k < nk; ++k) order[k] = k;
  auto width = [&](int k) { const uint64_t r = range_of(st[k]); return r == 0 ? 65.0 : std::log2((double)r); };
  std::sort(order, order + nk, [&](int a, int b) { return width(a) > width(b); });
  const int64_t dict_cap = std::min<int64_t>(n, (int64_t)1 << 26);
  bool enc[kMaxKeyCols] = {false, false, false, false};
  double bits = 0;
  for (int k = 0; k < nk; ++k) bits += width(k);
  int n_enc = 0;
  for (int i = 0; i < nk && bits > 62.0; ++i) {
    const int k = order[i];
    enc[k] = true; ++n_enc;
    bits -= width(k) - std::min(width(k), std::log2((double)std::max<int64_t>(dict_cap, 2)));    // at best: the capacity bound; refined below
  }
  // encoded columns: codes (n x 4), dictionary (dict_cap elements), decoded-later group codes (out_capacity x 4)
  size_t need = 0;
  for (int k = 0; k < nk; ++k) if (enc[k]) need += align_up((size_t)n * 4, 256) + align_up((size_t)dict_cap * dtype_size(keys[k].dtype), 256) + align_up((size_t)std::max<int64_t>(out_capacity, 1) * 4, 256);
  int rc = enc_reserve(need + 256);
  if (rc) return rc;
  char* w = g_enc.base;
  eiger_col nkeys[kMaxKeyCols];
  void* nout[kMaxKeyCols];
  int32_t* gcodes[kMaxKeyCols] = {nullptr, nullptr, nullptr, nullptr};
  void* dicts[kMaxKeyCols] = {nullptr, nullptr, nullptr, nullptr};
  for (int k = 0; k < nk; ++k) {
    nkeys[k] = keys[k]; nout[k] = out_keys[k];
    if (!enc[k]) continue;
    int32_t* codes = reinterpret_cast<int32_t*>(w); w += align_up((size_t)n * 4, 256);
    dicts[k] = w; w += align_up((size_t)dict_cap * dtype_size(keys[k].dtype), 256);
    gcodes[k] = reinterpret_cast<int32_t*>(w); w += align_up((size_t)std::max<int64_t>(out_capacity, 1) * 4, 256);
    const size_t ws_need = dict_encode_ws_bytes(keys[k].dtype, n, dict_cap);
    rc = ws_reserve(ws_need);
    if (rc) return rc;
    int64_t ndv = 0;
    rc = dict_encode_impl(rt, keys[k].data, keys[k].dtype, n, codes, dicts[k], dict_cap, &ndv, g_ws.base, g_ws.size, s);
    if (rc == EIGER_ERR_OUT_CAPACITY) return EIGER_ERR_INFEASIBLE;       // too many distinct values for a dictionary: nothing left to try
    if (rc) return rc;
    nkeys[k].data = codes; nkeys[k].dtype = EIGER_I32; nkeys[k].reserved = 0;
    nout[k] = gcodes[k];
  }
  // the same call on the code columns (statistics gathered inside: the codes are dense, so the range test settles them)
  rc = run_groupby(rt, nkeys, nk, n, vals, nv, aggs, na, nullptr, nout, out_aggs, out_capacity, n_groups, force, chosen, nullptr, 0, s, info);
  if (rc) return rc;
  const int64_t g = std::min<int64_t>(*n_groups, out_capacity);
  for (int k = 0; k < nk; ++k) {
    if (!enc[k] || g == 0) continue;
    dict_decode_kernel<<<(int)std::min<int64_t>((g + 255) / 256, (int64_t)rt->sm_count * 8), 256, 0, s>>>(gcodes[k], dicts[k], keys[k].dtype, g, out_keys[k]);
    count_launch();
  }
  EIGER_CUDA(cudaGetLastError());
  EIGER_CUDA(cudaStreamSynchronize(s));
  if (info) info->kernel_launches += n_enc;      // the decode kernels (the encode passes are counted by their own calls)
  return EIGER_OK;
}

}  // namespace

void count_launch(int k) { g_launches.fetch_add(k, std::memory_order_relaxed); }

int cuda_fail(cudaError_t e, const char* what) {
  std::snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
  cudaGetLastError();
  return EIGER_ERR_CUDA;
}

Runtime* runtime() {
  if (g_rt.device >= 0) return &g_rt;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cuda_fail(cudaGetLastError(), "cudaGetDevice"); return nullptr; }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { cuda_fail(cudaGetLastError(), "cudaGetDeviceProperties"); return nullptr; }
  g_rt.sm_count = prop.multiProcessorCount;
  g_rt.smem_optin = prop.sharedMemPerBlockOptin;
  g_rt.l2_bytes = (size_t)prop.l2CacheSize;
  if (cudaMalloc(reinterpret_cast<void**>(&g_rt.prof), sizeof(ProfileDev)) != cudaSuccess ||
      cudaMalloc(reinterpret_cast<void**>(&g_rt.call), sizeof(CallDev)) != cudaSuccess ||
      cudaMallocHost(&g_rt.pinned, 64 * 1024) != cudaSuccess) {
    cuda_fail(cudaGetLastError(), "runtime allocation");
    return nullptr;
  }
  g_rt.device = dev;
  return &g_rt;
}

}  // namespace eiger

using namespace eiger;

extern "C" {

int eiger_profile(const void* keys, int32_t dtype, int64_t n, eiger_stats* out, void* stream) {
  if (!out || n < 0 || !is_key_dtype(dtype) || (n > 0 && (!keys || ((uintptr_t)keys & 15)))) return EIGER_ERR_ARG;
  std::lock_guard<std::mutex> lk(g_mu);
  Runtime* rt = runtime();
  if (!rt) return EIGER_ERR_CUDA;
  eiger_col c{keys, dtype, 0};
  return do_profile(rt, &c, 1, n, 1, out, static_cast<cudaStream_t>(stream));
}

int eiger_profile_keys(const eiger_col* keys, int32_t nk, int64_t n, eiger_stats* out, void* stream) {
  if (!out || !keys || nk < 1 || nk > kMaxKeyCols || n < 0) return EIGER_ERR_ARG;
  for (int k = 0; k < nk; ++k)
    if (!is_key_dtype(keys[k].dtype) || (n > 0 && (!keys[k].data || ((uintptr_t)keys[k].data & 15)))) return EIGER_ERR_ARG;
  std::lock_guard<std::mutex> lk(g_mu);
  Runtime* rt = runtime();
  if (!rt) return EIGER_ERR_CUDA;
  return do_profile(rt, keys, nk, n, keys[0].dtype != EIGER_I8, out, static_cast<cudaStream_t>(stream));
}

int eiger_hll_registers(const void* keys, int32_t dtype, int64_t n, uint8_t* regs_out, void* stream) {
  if (!regs_out || n < 0 || !is_key_dtype(dtype) || (n > 0 && (!keys || ((uintptr_t)keys & 15)))) return EIGER_ERR_ARG;
  std::lock_guard<std::mutex> lk(g_mu);
  Runtime* rt = runtime();
  if (!rt) return EIGER_ERR_CUDA;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int rc = launch_profile(rt, keys, dtype, n, 0, 1, true, s);
  if (rc) return rc;
  rc = launch_regs_to_bytes(rt, regs_out, s);
  if (rc) return rc;
  EIGER_CUDA(cudaStreamSynchronize(s));
  return EIGER_OK;
}

double eiger_hll_estimate_host(const uint8_t* regs) {
  if (!regs) return -1.0;
  uint32_t hist[64] = {0};
  for (int i = 0; i < kHllM; ++i) hist[regs[i] & 63] += 1;
  return hll_estimate_from_hist(hist);
}

int eiger_groupby(const eiger_col* keys, int32_t n_key_cols, int64_t n, const eiger_col* vals, int32_t n_vals,
                  const eiger_agg* aggs, int32_t n_aggs, const eiger_stats* stats,
                  void* const* out_keys, void* const* out_aggs, int64_t out_capacity,
                  int64_t* n_groups, int32_t force, int32_t* chosen,
                  void* workspace, size_t workspace_bytes, void* stream, eiger_call_info* info) {
  std::lock_guard<std::mutex> lk(g_mu);
  Runtime* rt = runtime();
  if (!rt) return EIGER_ERR_CUDA;
  return run_groupby(rt, keys, n_key_cols, n, vals, n_vals, aggs, n_aggs, stats, out_keys, out_aggs, out_capacity,
                     n_groups, force, chosen, workspace, workspace_bytes, static_cast<cudaStream_t>(stream), info);
}

size_t eiger_groupby_workspace_bytes(const eiger_col* keys, int32_t n_key_cols, int64_t n,
                                     const eiger_col* vals, int32_t n_vals, const eiger_agg* aggs, int32_t n_aggs,
                                     const eiger_stats* stats, int32_t force) {
  size_t worst = 0;
  const int lo = (force == EIGER_AUTO && !stats) ? EIGER_DIRECT : force;
  const int hi = (force == EIGER_AUTO && !stats) ? EIGER_PARTITION : force;
  bool any = false;
  for (int v = lo; v <= hi; ++v) {
    QueryPlan q;
    const int rc = plan_query(nullptr, keys, n_key_cols, n, vals, n_vals, aggs, n_aggs, stats, v, &q);
    if (rc == EIGER_OK) { worst = std::max(worst, q.total_bytes); any = true; }
    else if (rc != EIGER_ERR_INFEASIBLE) return 0;
  }
  return any ? std::max<size_t>(worst, 256) : 0;
}

int32_t eiger_select_variant(const eiger_col* keys, int32_t n_key_cols, int64_t n, const eiger_col* vals, int32_t n_vals,
                             const eiger_agg* aggs, int32_t n_aggs, const eiger_stats* stats) {
  QueryPlan q;
  const int rc = plan_query(nullptr, keys, n_key_cols, n, vals, n_vals, aggs, n_aggs, stats, EIGER_AUTO, &q);
  return rc ? rc : q.variant;
}

int eiger_groupby_host(const eiger_col* keys, int32_t nk, int64_t n, const eiger_col* vals, int32_t nv,
                       const eiger_agg* aggs, int32_t na, void* const* out_keys, void* const* out_aggs,
                       int64_t out_capacity, int64_t* n_groups, int32_t force, int32_t* chosen,
                       int64_t* h2d_bytes, int64_t* d2h_bytes, void* stream, eiger_call_info* info) {
  if (!keys || nk < 1 || nk > kMaxKeyCols || n < 0 || nv < 0 || nv > kMaxVals || !aggs || na < 1 || na > kMaxAggs ||
      !n_groups || !out_keys || !out_aggs || out_capacity < 0) return EIGER_ERR_ARG;
  std::lock_guard<std::mutex> lk(g_mu);
  Runtime* rt = runtime();
  if (!rt) return EIGER_ERR_CUDA;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  for (int k = 0; k < nk; ++k) if (!is_key_dtype(keys[k].dtype) || (n > 0 && !keys[k].data)) return EIGER_ERR_ARG;
  for (int c = 0; c < nv; ++c) if ((vals[c].dtype != EIGER_I64 && vals[c].dtype != EIGER_F64 && vals[c].dtype != EIGER_I32) || (n > 0 && !vals[c].data)) return EIGER_ERR_ARG;

  // arena layout: input columns | output columns; the scratch is the library's workspace arena
  size_t in_bytes = 0, out_bytes = 0;
  for (int k = 0; k < nk; ++k) { in_bytes += align_up((size_t)n * dtype_size(keys[k].dtype), 256); out_bytes += align_up((size_t)out_capacity * dtype_size(keys[k].dtype), 256); }
  for (int c = 0; c < nv; ++c) in_bytes += align_up((size_t)n * (vals[c].dtype == EIGER_I32 ? 4 : 8), 256);
  out_bytes += (size_t)na * align_up((size_t)out_capacity * 8, 256);
  int rc = arena_reserve(in_bytes + out_bytes + 512);
  if (rc) return rc;
  int64_t h2d = 0, d2h = 0;
  eiger_col dk[kMaxKeyCols], dv[kMaxVals];
  char* cur = g_arena.base;
  for (int k = 0; k < nk; ++k) {
    const size_t b = (size_t)n * dtype_size(keys[k].dtype);
    dk[k].data = cur; dk[k].dtype = keys[k].dtype; dk[k].reserved = 0;
    if (b) EIGER_CUDA(cudaMemcpyAsync(cur, keys[k].data, b, cudaMemcpyHostToDevice, s));
    h2d += (int64_t)b; cur += align_up(b, 256);
  }
  for (int c = 0; c < nv; ++c) {
    const size_t b = (size_t)n * (vals[c].dtype == EIGER_I32 ? 4 : 8);
    dv[c].data = cur; dv[c].dtype = vals[c].dtype; dv[c].reserved = 0;
    if (b) EIGER_CUDA(cudaMemcpyAsync(cur, vals[c].data, b, cudaMemcpyHostToDevice, s));
    h2d += (int64_t)b; cur += align_up(b, 256);
  }
  void* dok[kMaxKeyCols] = {nullptr, nullptr, nullptr, nullptr};
  void* doa[kMaxAggs] = {nullptr};
  for (int k = 0; k < nk; ++k) { dok[k] = cur; cur += align_up((size_t)out_capacity * dtype_size(keys[k].dtype), 256); }
  for (int j = 0; j < na; ++j) { doa[j] = cur; cur += align_up((size_t)out_capacity * 8, 256); }
  // the same call a device-resident caller makes: no statistics supplied (EIGER_AUTO samples, speculates
  // or profiles inside), scratch from the library's own arena
  rc = run_groupby(rt, dk, nk, n, dv, nv, aggs, na, nullptr, dok, doa, out_capacity, n_groups, force, chosen, nullptr, 0, s, info);
  if (rc) return rc;
  const int64_t g = *n_groups;
  for (int k = 0; k < nk; ++k) {
    const size_t b = (size_t)g * dtype_size(keys[k].dtype);
    if (b) EIGER_CUDA(cudaMemcpyAsync(out_keys[k], dok[k], b, cudaMemcpyDeviceToHost, s));
    d2h += (int64_t)b;
  }
  for (int j = 0; j < na; ++j) {
    if (g) EIGER_CUDA(cudaMemcpyAsync(out_aggs[j], doa[j], (size_t)g * 8, cudaMemcpyDeviceToHost, s));
    d2h += g * 8;
  }
  EIGER_CUDA(cudaStreamSynchronize(s));
  if (h2d_bytes) *h2d_bytes = h2d;
  if (d2h_bytes) *d2h_bytes = d2h;
  return EIGER_OK;
}

// Order-preserving dictionary encoding (Algorithm 1; dictenc.cu lists the steps).
// workspace: [unique keys g x 8][counts g x 8][counts g x 8][rank table][group-by scratch]
static size_t dict_fixed_bytes(int64_t dict_capacity) {
  const size_t g = (size_t)std::max<int64_t>(dict_capacity, 1);
  return 3 * align_up(g * 8, 256) + align_up((2 * g + 1024 + 1) * 16, 256);
}
}  // extern "C"
namespace eiger { namespace {
size_t dict_encode_ws_bytes(int32_t dtype, int64_t n, int64_t dict_capacity) {
  if (!is_key_dtype(dtype) || n < 0 || dict_capacity < 0) return 0;
  eiger_col k{nullptr, dtype, 0};
  eiger_agg a{EIGER_COUNT, 0};
  const size_t all = eiger_groupby_workspace_bytes(&k, 1, n, nullptr, 0, &a, 1, nullptr, EIGER_AUTO);
  const size_t srt = eiger_groupby_workspace_bytes(&k, 1, std::min(n, std::max<int64_t>(dict_capacity, 1)), nullptr, 0, &a, 1, nullptr, EIGER_SORT);
  return dict_fixed_bytes(dict_capacity) + std::max(all, srt) + 512;
}

int dict_encode_impl(Runtime* rt, const void* keys, int32_t dtype, int64_t n, int32_t* codes_out, void* dict_out, int64_t dict_capacity,
                     int64_t* ndv, void* workspace, size_t workspace_bytes, cudaStream_t s) {
  if (!ndv || n < 0 || dict_capacity < 0 || !is_key_dtype(dtype)) return EIGER_ERR_ARG;
  *ndv = 0;
  if (n == 0) return EIGER_OK;
  if (!keys || ((uintptr_t)keys & 15) || !codes_out || !dict_out || !workspace || ((uintptr_t)workspace & 255)) return EIGER_ERR_ARG;
  const size_t fixed = dict_fixed_bytes(dict_capacity);
  if (workspace_bytes < fixed + 256) return EIGER_ERR_WORKSPACE;
  const size_t g_cap = (size_t)std::max<int64_t>(dict_capacity, 1);
  char* w = static_cast<char*>(workspace);
  void* uniq = w; w += align_up(g_cap * 8, 256);
  void* cnt1 = w; w += align_up(g_cap * 8, 256);
  void* cnt2 = w; w += align_up(g_cap * 8, 256);
  void* table = w; w += align_up((2 * g_cap + 1024 + 1) * 16, 256);
  char* gws = w;
  const size_t gws_bytes = workspace_bytes - (size_t)(gws - static_cast<char*>(workspace));
  // (1) + (2): HT.insert_and_find over the column, retrieveAll -> the unique keys (a COUNT group-by)
  eiger_col kc{keys, dtype, 0};
  eiger_agg ag{EIGER_COUNT, 0};
  void* ok[kMaxKeyCols] = {uniq, nullptr, nullptr, nullptr};
  void* oa[kMaxAggs] = {cnt1};
  int64_t g = 0;
  int rc = run_groupby(rt, &kc, 1, n, nullptr, 0, &ag, 1, nullptr, ok, oa, dict_capacity, &g, EIGER_AUTO, nullptr, gws, gws_bytes, s);
  *ndv = g;
  if (rc) return rc;
  // (3) argsort(uniqueKeys): the unique keys in ascending order = the dictionary
  eiger_col uc{uniq, dtype, 0};
  void* ok2[kMaxKeyCols] = {dict_out, nullptr, nullptr, nullptr};
  void* oa2[kMaxAggs] = {cnt2};
  int64_t g2 = 0;
  rc = run_groupby(rt, &uc, 1, g, nullptr, 0, &ag, 1, nullptr, ok2, oa2, dict_capacity, &g2, EIGER_SORT, nullptr, gws, gws_bytes, s);
  if (rc) return rc;
  if (g2 != g) return EIGER_ERR_CUDA;
  // (4) scatter: rank of every unique key into the look-up table; (5) gather: every row fetches its rank
  const uint64_t cap = 2 * (uint64_t)g + 1024;
  AggLaunch L{};
  L.back = BACK_HASH; L.table = table; L.cap = cap; L.stride = 16; L.plan.n_acc = 1; L.plan.op[0] = EIGER_SUM;
  rc = launch_table_init(L, s); if (rc) return rc;
  EIGER_CUDA(cudaMemsetAsync(rt->call, 0, sizeof(CallDev), s));
  rc = launch_dict_fill(dict_out, dtype, g, table, cap, rt->call, rt->sm_count, s); if (rc) return rc;
  rc = launch_dict_gather(keys, dtype, n, table, cap, codes_out, rt->call, rt->sm_count, s); if (rc) return rc;
  struct Back { unsigned long long n_groups; uint32_t overflow; uint32_t abort; };
  Back* hb = reinterpret_cast<Back*>(static_cast<char*>(rt->pinned) + 1024);
  EIGER_CUDA(cudaMemcpyAsync(hb, rt->call, sizeof(Back), cudaMemcpyDeviceToHost, s));
  EIGER_CUDA(cudaStreamSynchronize(s));
  return hb->overflow ? EIGER_ERR_TABLE_OVERFLOW : EIGER_OK;
}
} }  // namespace eiger::<unnamed>
extern "C" {

size_t eiger_dict_encode_workspace_bytes(int32_t dtype, int64_t n, int64_t dict_capacity) { return dict_encode_ws_bytes(dtype, n, dict_capacity); }

int eiger_dict_encode(const void* keys, int32_t dtype, int64_t n, int32_t* codes_out, void* dict_out, int64_t dict_capacity,
                      int64_t* ndv, void* workspace, size_t workspace_bytes, void* stream) {
  std::lock_guard<std::mutex> lk(g_mu);
  Runtime* rt = runtime();
  if (!rt) return EIGER_ERR_CUDA;
  return dict_encode_impl(rt, keys, dtype, n, codes_out, dict_out, dict_capacity, ndv, workspace, workspace_bytes, static_cast<cudaStream_t>(stream));
}

int64_t eiger_launch_count(void) { return g_launches.load(); }

void eiger_reload_tunables(void) { g_tun_dirty.store(true); }

void eiger_set_kernel_timing(int32_t enabled) { std::lock_guard<std::mutex> lk(g_mu); g_timing = enabled != 0; }

double eiger_kernel_time_ms(int32_t which, int32_t reset, int64_t* launches) {
  std::lock_guard<std::mutex> lk(g_mu);
  if (which < 0 || which >= kTimeSlots) return -1.0;
  const double ms = g_time_ms[which];
  if (launches) *launches = g_time_n[which];
  if (reset) { g_time_ms[which] = 0; g_time_n[which] = 0; }
  return ms;
}

const char* eiger_strerror(int code) {
  switch (code) {
    case EIGER_OK: return "ok";
    case EIGER_ERR_ARG: return "bad argument (null pointer, bad dtype/op, negative size or misaligned column)";
    case EIGER_ERR_WORKSPACE: return "workspace too small (see eiger_groupby_workspace_bytes)";
    case EIGER_ERR_OUT_CAPACITY: return "more groups than out_capacity";
    case EIGER_ERR_INFEASIBLE: return "the forced variant cannot run on this input";
    case EIGER_ERR_CUDA: return "CUDA runtime error (see eiger_last_cuda_error)";
    case EIGER_ERR_TABLE_OVERFLOW: return "hash table overflow: NDV under-estimated and no workspace to retry";
    case EIGER_ERR_STATS: return "a key lies outside the [min, max] of the statistics supplied by the caller";
    case EIGER_ERR_STATIC_LIMIT: return "key range exceeds EIGER_STATIC_MAX_SLOTS, the size of the static scratch array of eiger_groupby_direct_static";
    default: return "unknown error";
  }
}
const char* eiger_last_cuda_error(void) { return g_cuda_err; }
const char* eiger_variant_name(int32_t v) {
  switch (v) {
    case EIGER_AUTO: return "auto"; case EIGER_DIRECT: return "direct"; case EIGER_SMEM: return "smem";
    case EIGER_GLOBAL: return "global"; case EIGER_PARTITION: return "partition"; case EIGER_SORT: return "sort"; default: return "?";
  }
}
void eiger_shutdown(void) {
  std::lock_guard<std::mutex> lk(g_mu);
  if (g_arena.base) { cudaFree(g_arena.base); g_arena = Arena{}; }
  if (g_ws.base) { cudaFree(g_ws.base); g_ws = Arena{}; }
  if (g_enc.base) { cudaFree(g_enc.base); g_enc = Arena{}; }
  if (g_rt.device >= 0) {
    cudaFree(g_rt.prof); cudaFree(g_rt.call); cudaFreeHost(g_rt.pinned);
    for (int i = 0; i < g_pool_n; ++i) cudaEventDestroy(g_pool[i]);
    g_pool_n = 0; g_pool_used = 0;
    g_rt = Runtime{};
  }
}

}  // extern "C"
