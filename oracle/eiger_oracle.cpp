// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded CPU restatement of the hot path of Eiger
// (arxiv/paper_2607_04489): GROUP BY aggregation (SUM / COUNT / MIN / MAX),
// exact NDV, min/max range statistics and the HyperLogLog sketch that the
// runtime-adaptive selector is driven by.  It shares no code with the CUDA
// path under paper_2607_04489_b200/csrc/, includes no CUDA header, and may
// only be called from tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs.
//
// Every function cites the passage of /root/reference/PAPER.md (or the reading
// listed in DESIGN.md "Readings") that it follows.  Parity status:
//   * oracle_groupby_*      pinned (brute force, closed forms, invariants;
//                           tests/test_oracle_groupby.py)
//   * oracle_exact_ndv      pinned (known-NDV generators, agrees with map size)
//   * oracle_minmax         pinned (numpy min/max, closed forms)
//   * oracle_hash64         pinned (published splitmix64 outputs for seeds 0, 1;
//                           tests/golden/hll_hash_pins.txt)
//   * oracle_hll_registers  pinned (tests/golden/hll_sketch_pins.txt, set
//                           invariants, pure-Python integer re-derivation)
//   * oracle_hll_estimate   pinned (linear-counting closed form when only small
//                           registers are set, known-NDV error bound 4 sigma,
//                           golden whole-sketch estimates)
//   * oracle_dict_encode    pinned (brute-force "number of smaller distinct values" on small
//                           inputs, order / round-trip invariants, worked example;
//                           tests/test_oracle_dict.py)
//   * parity with the PAPER'S OWN implementation: unpinned (the paper prints no
//     group-by result and no sketch value; DESIGN.md says so).
//
// Build: g++ -O2 -std=c++17 -shared -fPIC -o liboracle.so eiger_oracle.cpp
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <unordered_map>
#include <utility>
#include <vector>

namespace {

enum Op : int32_t { OP_SUM = 0, OP_COUNT = 1, OP_MIN = 2, OP_MAX = 3 };

// One accumulator per (group, aggregate).  Integer SUM wraps modulo 2^64
// (reading R13); fp64 SUM is either the sequential row-order sum
// (the plain definition) or the exact fixed-point sum (reading R14).
struct Acc {
  uint64_t isum = 0;              // integer SUM (wrapping) / COUNT
  unsigned __int128 xsum = 0;     // exact fp64 SUM of k * 2^-53 values
  double fsum = 0.0;              // sequential fp64 SUM
  int64_t imin = std::numeric_limits<int64_t>::max();
  int64_t imax = std::numeric_limits<int64_t>::min();
  double fmin = std::numeric_limits<double>::infinity();
  double fmax = -std::numeric_limits<double>::infinity();
};

// A group key is the tuple of its key columns (§4.3 "group-bys with multiple
// keys"): up to kMaxKeyCols columns, unused ones held at 0.  Equality and order are the
// tuple's (lexicographic, first column most significant).
constexpr int kMaxKeyCols = 4;
struct Key {
  int64_t v[kMaxKeyCols];
  bool operator==(const Key& o) const {
    for (int c = 0; c < kMaxKeyCols; ++c) if (v[c] != o.v[c]) return false;
    return true;
  }
  bool operator<(const Key& o) const {
    for (int c = 0; c < kMaxKeyCols; ++c) if (v[c] != o.v[c]) return v[c] < o.v[c];
    return false;
  }
};
struct KeyHash {
  size_t operator()(const Key& k) const {
    // any hash works: the result of a group-by does not depend on it
    uint64_t x = 0x632BE59BD9B4E019ull;
    for (int c = 0; c < kMaxKeyCols; ++c) { x = (x ^ (uint64_t)k.v[c]) * 0x9FB21C651E98DF25ull; x ^= x >> 29; }
    return (size_t)(x * 0xD6E8FEB86659FD93ull);
  }
};
inline Key key_at(const int64_t* const* cols, int32_t nk, int64_t i) {
  Key k;
  for (int c = 0; c < kMaxKeyCols; ++c) k.v[c] = c < nk ? cols[c][i] : 0;
  return k;
}

struct Result {
  int32_t n_aggs = 0;
  int32_t n_key_cols = 0;
  std::vector<Key> keys;                       // sorted ascending (column 0 first)
  std::vector<std::vector<uint64_t>> aggs;     // [agg][group], 8-byte bit patterns
  double seconds = 0.0;
  int32_t status = 0;
};

inline uint64_t dbits(double d) { uint64_t u; std::memcpy(&u, &d, 8); return u; }

}  // namespace

extern "C" {

// ---------------------------------------------------------------------------
// GROUP BY, the plain relational definition (§3.3 "Group-by";
// PAPER.md:302 "number of groups g", "number of aggregations").  For rows
// i = 0..n-1 with key k_i = (keys[0][i], .., keys[n_key_cols-1][i]) the output is the set of distinct
// keys; per key SUM = sum of the value column over the rows of that key,
// COUNT = number of those rows, MIN / MAX = min / max over them.
//
//   keys       : n_key_cols (1..4) pointers to int64 arrays (the Python wrapper
//                widens int8/int32 keys, which is exact)
//   vals       : n_vals pointers to 8-byte columns; val_is_f64[c] says how to
//                read column c (int64 or IEEE double)
//   ops/cols   : n_aggs aggregates; COUNT ignores its column
//   f64_sum_mode: 0 = sequential row-order double sum; 1 = exact: every fp64
//                value summed must be k*2^-53 with 0 <= k < 2^53 (the
//                generator's fp64 values, reading R14); the sum is carried in
//                a 128-bit integer and rounded to double once.  A value that
//                violates the precondition sets status = -2.
//   only/n_only: (n_key_cols pointers, n_only keys) optional restriction used for spot checks at sizes where
//                the full result does not fit the host: when n_only > 0, rows
//                whose key is not one of the n_only listed keys are skipped, so
//                the result is the plain definition for exactly those groups.
// Returns an opaque handle (free with oracle_groupby_free).
// ---------------------------------------------------------------------------
void* oracle_groupby_run(const int64_t* const* keys, int32_t n_key_cols, int64_t n,
                         const void* const* vals, const int32_t* val_is_f64, int32_t n_vals,
                         const int32_t* ops, const int32_t* cols, int32_t n_aggs,
                         int32_t f64_sum_mode,
                         const int64_t* const* only_keys, int64_t n_only) {
  Result* res = new Result();
  res->n_aggs = n_aggs;
  res->n_key_cols = n_key_cols;
  if (n_key_cols < 1 || n_key_cols > kMaxKeyCols) { res->status = -1; return res; }
  for (int j = 0; j < n_aggs; ++j) {
    if (ops[j] < 0 || ops[j] > 3 || (ops[j] != OP_COUNT && (cols[j] < 0 || cols[j] >= n_vals))) {
      res->status = -1;
      return res;
    }
  }
  std::unordered_map<Key, std::vector<Acc>, KeyHash> map;
  std::unordered_map<Key, char, KeyHash> only;
  for (int64_t i = 0; i < n_only; ++i) only.emplace(key_at(only_keys, n_key_cols, i), 1);
  auto t0 = std::chrono::steady_clock::now();
  for (int64_t i = 0; i < n; ++i) {
    const Key k = key_at(keys, n_key_cols, i);
    if (n_only > 0 && only.find(k) == only.end()) continue;
    auto it = map.find(k);
    if (it == map.end()) it = map.emplace(k, std::vector<Acc>((size_t)n_aggs)).first;
    std::vector<Acc>& acc = it->second;
    for (int j = 0; j < n_aggs; ++j) {
      Acc& a = acc[(size_t)j];
      if (ops[j] == OP_COUNT) { a.isum += 1; continue; }
      const int c = cols[j];
      if (val_is_f64[c]) {
        const double v = static_cast<const double*>(vals[c])[i];
        if (ops[j] == OP_SUM) {
          if (f64_sum_mode == 1) {
            const double s = std::ldexp(v, 53);
            if (!(v >= 0.0 && v < 1.0) || s != std::floor(s)) res->status = -2;
            else a.xsum += (unsigned __int128)(uint64_t)s;
          } else {
            a.fsum += v;
          }
        } else if (ops[j] == OP_MIN) { if (v < a.fmin) a.fmin = v; }
        else { if (v > a.fmax) a.fmax = v; }
      } else {
        const int64_t v = static_cast<const int64_t*>(vals[c])[i];
        if (ops[j] == OP_SUM) a.isum += (uint64_t)v;
        else if (ops[j] == OP_MIN) { if (v < a.imin) a.imin = v; }
        else { if (v > a.imax) a.imax = v; }
      }
    }
  }
  auto t1 = std::chrono::steady_clock::now();
  res->seconds = std::chrono::duration<double>(t1 - t0).count();

  // emit sorted by key so that callers can compare position by position
  std::vector<const std::pair<const Key, std::vector<Acc>>*> order;
  order.reserve(map.size());
  for (const auto& kv : map) order.push_back(&kv);
  std::sort(order.begin(), order.end(),
            [](auto* x, auto* y) { return x->first < y->first; });
  const size_t g = order.size();
  res->keys.resize(g);
  res->aggs.assign((size_t)n_aggs, std::vector<uint64_t>(g));
  for (size_t r = 0; r < g; ++r) {
    res->keys[r] = order[r]->first;
    for (int j = 0; j < n_aggs; ++j) {
      const Acc& a = order[r]->second[(size_t)j];
      uint64_t out;
      const bool f = ops[j] != OP_COUNT && val_is_f64[cols[j]];
      if (ops[j] == OP_COUNT) out = a.isum;
      else if (ops[j] == OP_SUM) {
        if (!f) out = a.isum;
        else if (f64_sum_mode == 1) {
          // round the exact integer k_total to double once, then scale by 2^-53 (exact)
          const unsigned __int128 x = a.xsum;
          const uint64_t hi = (uint64_t)(x >> 64), lo = (uint64_t)x;
          double d;
          if (hi == 0) d = (double)lo;              // correctly rounded uint64 -> double
          else {
            // shift right until it fits 64 bits, keeping a sticky bit: the top bit of m is then
            // set, double keeps 53 bits, so bit 0 only breaks round-to-nearest-even ties
            int sh = 0; unsigned __int128 y = x; bool sticky = false;
            while ((y >> 64) != 0) { sticky = sticky || (y & 1); y >>= 1; ++sh; }
            uint64_t m = (uint64_t)y;
            if (sticky) m |= 1;
            d = std::ldexp((double)m, sh);
          }
          out = dbits(std::ldexp(d, -53));
        } else out = dbits(a.fsum);
      } else if (ops[j] == OP_MIN) out = f ? dbits(a.fmin) : (uint64_t)a.imin;
      else out = f ? dbits(a.fmax) : (uint64_t)a.imax;
      res->aggs[(size_t)j][r] = out;
    }
  }
  return res;
}

int64_t oracle_groupby_n_groups(const void* h) { return (int64_t)static_cast<const Result*>(h)->keys.size(); }
int32_t oracle_groupby_status(const void* h) { return static_cast<const Result*>(h)->status; }
double oracle_groupby_seconds(const void* h) { return static_cast<const Result*>(h)->seconds; }

// Copies the result out: keys = n_key_cols pointers to n_groups int64 each, aggs as
// n_aggs pointers to n_groups 8-byte cells (int64 bits or double bits).
void oracle_groupby_fetch(const void* h, int64_t* const* keys, void* const* aggs) {
  const Result* r = static_cast<const Result*>(h);
  const size_t g = r->keys.size();
  for (size_t i = 0; i < g; ++i)
    for (int c = 0; c < r->n_key_cols; ++c) keys[c][i] = r->keys[i].v[c];
  for (int j = 0; j < r->n_aggs; ++j) std::memcpy(aggs[j], r->aggs[(size_t)j].data(), g * 8);
}
void oracle_groupby_free(void* h) { delete static_cast<Result*>(h); }

// ---------------------------------------------------------------------------
// Exact NDV by an independent second method: sort + unique (BASELINE.json
// north_star "an exact-NDV counter").  Must equal the group-by's n_groups.
// ---------------------------------------------------------------------------
int64_t oracle_exact_ndv(const int64_t* const* keys, int32_t n_key_cols, int64_t n) {
  if (n_key_cols < 1 || n_key_cols > kMaxKeyCols) return -1;
  std::vector<Key> v((size_t)n);
  for (int64_t i = 0; i < n; ++i) v[(size_t)i] = key_at(keys, n_key_cols, i);
  std::sort(v.begin(), v.end());
  return (int64_t)(std::unique(v.begin(), v.end()) - v.begin());
}

// ---------------------------------------------------------------------------
// min / max range statistics (§4 "min, max ... calculated extremely
// fast"; §4.3 "evaluate the range of values by finding the minimum
// and maximum").  n = 0 gives min = INT64_MAX, max = INT64_MIN.
// ---------------------------------------------------------------------------
void oracle_minmax(const int64_t* keys, int64_t n, int64_t* out_min, int64_t* out_max) {
  int64_t lo = std::numeric_limits<int64_t>::max(), hi = std::numeric_limits<int64_t>::min();
  for (int64_t i = 0; i < n; ++i) { if (keys[i] < lo) lo = keys[i]; if (keys[i] > hi) hi = keys[i]; }
  *out_min = lo; *out_max = hi;
}

// ---------------------------------------------------------------------------
// The sketch hash (reading R2): the splitmix64 output function applied
// to the key sign-extended to 64 bits:  z = x + 0x9E3779B97F4A7C15;
// z = (z ^ z>>30) * 0xBF58476D1CE4E5B9; z = (z ^ z>>27) * 0x94D049BB133111EB;
// z ^ z>>31.   The paper (§4.1, ref [14]) fixes no hash.
// ---------------------------------------------------------------------------
uint64_t oracle_hash64(int64_t key) {
  uint64_t z = (uint64_t)key + 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// ---------------------------------------------------------------------------
// HyperLogLog registers (§4.1 "HyperLogLog++ [14] (HLL++) algorithm
// to estimate this group cardinality"; steps per ref [14] as read in DESIGN.md
// R1-R4):  M[0..m) = 0, m = 2^p; per key z = hash64(key); idx = top p bits;
// w = the remaining 64-p bits, left aligned; rho = min(clz64(w), 64-p) + 1;
// M[idx] = max(M[idx], rho).
// ---------------------------------------------------------------------------
void oracle_hll_registers(const int64_t* keys, int64_t n, int32_t p, uint8_t* regs /* 2^p */) {
  const size_t m = (size_t)1 << p;
  std::memset(regs, 0, m);
  for (int64_t i = 0; i < n; ++i) {
    const uint64_t z = oracle_hash64(keys[i]);
    const size_t idx = (size_t)(z >> (64 - p));
    const uint64_t w = z << p;
    int lz = 0;
    if (w == 0) lz = 64; else { uint64_t t = w; while (!(t >> 63)) { t <<= 1; ++lz; } }
    const int rho = std::min(lz, 64 - p) + 1;
    if (regs[idx] < rho) regs[idx] = (uint8_t)rho;
  }
}

// ---------------------------------------------------------------------------
// Estimate from the register-value histogram (reading R5: HLL++'s
// empirical bias tables from ref [14] are not available, so the table-free
// improved raw estimator is used):  q = 64-p, C[k] = #{j : M[j] = k}, k=0..q+1;
//   z = m * tau(1 - C[q+1]/m);  for k = q..1: z = (z + C[k]) / 2;
//   z = z + m * sigma(C[0]/m);  est = (m^2 / (2 ln 2)) / z
//   sigma(x) = x + sum_{j>=1} x^(2^j) 2^(j-1)         (x = 1 -> infinity)
//   tau(x)   = (1 - x - sum_{j>=1} (1 - x^(2^-j))^2 2^-j) / 3
// both iterated until the value stops changing.  Empty sketch -> 0.
// ---------------------------------------------------------------------------
static double sigma_fn(double x) {
  if (x == 1.0) return std::numeric_limits<double>::infinity();
  double y = 1.0, z = x;
  for (;;) {
    x = x * x;
    const double zprev = z;
    z += x * y;
    y += y;
    if (zprev == z) return z;
  }
}
static double tau_fn(double x) {
  if (x == 0.0 || x == 1.0) return 0.0;
  double y = 1.0, z = 1.0 - x;
  for (;;) {
    x = std::sqrt(x);
    const double zprev = z;
    y *= 0.5;
    z -= (1.0 - x) * (1.0 - x) * y;
    if (zprev == z) return z / 3.0;
  }
}
double oracle_hll_estimate(const uint8_t* regs, int32_t p) {
  const int q = 64 - p;
  const size_t m = (size_t)1 << p;
  std::vector<double> C((size_t)q + 2, 0.0);
  for (size_t j = 0; j < m; ++j) C[regs[j]] += 1.0;
  const double md = (double)m;
  double z = md * tau_fn(1.0 - C[(size_t)q + 1] / md);
  for (int k = q; k >= 1; --k) z = (z + C[(size_t)k]) * 0.5;
  z += md * sigma_fn(C[0] / md);
  const double alpha_inf = 0.5 / std::log(2.0);
  return alpha_inf * md * md / z;
}


// ---------------------------------------------------------------------------
// Order-preserving dictionary encoding, PAPER.md:171-211 (Algorithm 1), followed step by step in
// the paper's order and notation (one thread = one loop iteration here):
//   (1) compute_group_id: HT.insert_and_find(key[i], i) -> the first tuple that carries a key is
//       its group leader; groupIdLoc[i] = the leader's tuple id; ndv counts the successful inserts.
//   (2) [uniqueKeys, groupIds] = HT.retrieveAll()          (ndv pairs, groupIds = leader tuple ids)
//   (3) argsortIds = argsort(uniqueKeys)
//   (4) scatter: sparseGroupIds[groupIds[argsortIds[i]]] = i
//   (5) gather:  C_out[i] = sparseGroupIds[groupIdLoc[i]]
// Output: codes[n] (C_out), dict[ndv] = the unique keys in ascending order (dict[code] = key; the
// paper keeps it implicitly as uniqueKeys[argsortIds]).  Returns ndv.
// ---------------------------------------------------------------------------
int64_t oracle_dict_encode(const int64_t* keys, int64_t n, int64_t* codes, int64_t* dict) {
  std::unordered_map<int64_t, int64_t> HT;                       // key -> leader tuple id
  std::vector<int64_t> groupIdLoc((size_t)n);
  int64_t ndv = 0;
  for (int64_t i = 0; i < n; ++i) {                               // (1)
    auto r = HT.emplace(keys[i], i);
    groupIdLoc[(size_t)i] = r.first->second;
    if (r.second) ++ndv;
  }
  std::vector<int64_t> uniqueKeys, groupIds;                      // (2)
  uniqueKeys.reserve((size_t)ndv); groupIds.reserve((size_t)ndv);
  for (const auto& kv : HT) { uniqueKeys.push_back(kv.first); groupIds.push_back(kv.second); }
  std::vector<int64_t> argsortIds((size_t)ndv);                   // (3)
  for (int64_t i = 0; i < ndv; ++i) argsortIds[(size_t)i] = i;
  std::sort(argsortIds.begin(), argsortIds.end(), [&](int64_t a, int64_t b) { return uniqueKeys[(size_t)a] < uniqueKeys[(size_t)b]; });
  std::vector<int64_t> sparseGroupIds((size_t)n, -1);             // (4)
  for (int64_t i = 0; i < ndv; ++i) sparseGroupIds[(size_t)groupIds[(size_t)argsortIds[(size_t)i]]] = i;
  for (int64_t i = 0; i < n; ++i) codes[i] = sparseGroupIds[(size_t)groupIdLoc[(size_t)i]];   // (5)
  for (int64_t i = 0; i < ndv; ++i) dict[i] = uniqueKeys[(size_t)argsortIds[(size_t)i]];
  return ndv;
}

}  // extern "C"
