// Step A6b / A6c / second half of A6d: hash aggregation with a per-CTA open-addressing table
// in shared memory in front of the global table.
//
//   whole-input mode  (EIGER_SMEM, EIGER_GLOBAL): every CTA streams its share of the rows into
//       its own shared-memory table; rows whose key finds no room there go straight to the
//       global table (L2 atomics); at the end each CTA merges its occupied slots into the
//       global table, which compaction (A7) then reads.
//   partition mode    (EIGER_PARTITION): the rows were reordered by partition.cu so that each
//       partition holds a disjoint set of keys; one CTA owns a partition, aggregates it in
//       shared memory and EMITS its groups straight into the output columns (A7 fused; no
//       global table, no init, no compaction pass).  Keys that do not fit go to the global
//       table as before and are appended by the compaction kernel.
//
// Shared memory is where this hardware aggregates fast: three native 32-bit ATOMS per row
// sustain ~880 G rows/s chip-wide (measured), L2 atomics ~190 G/s in total.
// PAPER.md:79 §3.3 (hash group-by, partitioned hash group-by); PAPER.md:23 ("perform well when
// the hash table is cache-resident"); PAPER.md:184 (retrieveAll).
// (This header holds the kernel template; hashagg_i32.cu, hashagg_i64.cu and hashagg_pre.cu
// instantiate it for their key kinds so that the three compile in parallel.)
#pragma once
#include <algorithm>
#include <cstdlib>
#include <type_traits>

#include "internal.h"
#include "ring.cuh"
#include "rows.cuh"

namespace eiger {
namespace {

constexpr int kMaxThreads = 1024;

struct HashAggArgs {
  KeyDesc key;
  AggPlan plan;
  int64_t n;
  const unsigned long long* part_off;   // partition mode: [n_parts + 1] row offsets
  const unsigned long long* item_off;   // partition mode: [n_parts + 1] work items (hot partitions are cut up)
  const uint32_t* item_part;            // partition mode: partition of each work item
  int32_t n_parts;
  uint32_t slots;        // shared-memory slots per CTA (any number >= 64)
  uint32_t limit;        // stop inserting new keys beyond this many
  int32_t max_probes;    // buckets looked at per key (1 = set-associative cache: home bucket or global table)
  int32_t spec;          // speculative: a full table raises call->abort and everybody stops
  int32_t n_hot;         // whole-input mode: heavy-hitter keys reduced inside the warp (never in spec runs)
  uint64_t hot[kMaxHot]; // their rebased values
  void* table; uint64_t cap; uint32_t stride;   // global table
  CallDev* call;
  void* out_keys[kMaxKeyCols]; uint64_t* out_aggs[kMaxAggs]; int32_t n_out; int64_t out_capacity;
  // shared-memory ring (ring.cuh) and the layout of dynamic shared memory
  int32_t stages; uint32_t stage_bytes; int32_t n_src;
  uint32_t koff[kMaxKeyCols], voff[kMaxVals];   // byte offset of each column inside a stage
  uint8_t kw[kMaxKeyCols], vw[kMaxVals];        // bytes per element
  uint32_t hot_off, table_off;
  int32_t ring_hint;             // bulk copies carry an L2 evict_first policy
  uint32_t queue_off;            // whole-input mode, per-thread loads: per-warp miss queues start here in dynamic shared memory (0 = none)
  // whole-input mode: spill buffer for the rows the front cannot hold (internal.h: HashAggLaunch); partition mode: flags
  uint64_t* sp_keys; uint64_t* sp_vals[kMaxVals]; uint64_t sp_cap_chunks; int32_t sp_lg;
  int32_t skip_empty, force_merge;
};

constexpr uint32_t kSpillChunks = 1024;    // chunks one CTA can reserve in the spill buffer

template <int KK> struct IsPre { static constexpr bool v = (KK == KK_U32PRE || KK == KK_U64PRE); };

// plane width of accumulator (op, f64) in the shared-memory table: COUNT keeps 32 bits (a CTA
// never sees 2^32 rows of one key: api.cu guards n), everything else 64
__device__ __forceinline__ uint32_t plane_width(int op) { return op == EIGER_COUNT ? 4u : 8u; }

// BK = keys per bucket: 16 bytes' worth by default; 2 for 32-bit keys in nearly empty tables
// (measured, 2^28 rows: an LDS.64 look-up beats the LDS.128 one by 5-17 % at loads up to 0.08 and
// loses 5-50 % from 0.16, where the narrower bucket overflows into probe chains)
template <int KK, int SIG, int BK>
struct Front {
  using U = typename KeyTraits<KK>::U;
  using S = Sig<SIG>;
  static constexpr int NV = S::kVals;
  static constexpr int NA = S::kAcc;

  const HashAggArgs& a;
  unsigned char* smem;
  const int n_acc;
  const uint32_t Sn;      // slots in use (<= a.slots)
  U* skeys;
  uint32_t* s_spill = nullptr;   // partition mode: set when a row of this work item went to the global table
  // rows that found no room wait in a per-warp queue (64 entries: keys, then each value column) and go to
  // the global table 32 at a time with full warps (EIGER_GLOBAL: a quarter of C3's rows take this path)
  unsigned char* q_base = nullptr;
  int q_n = 0;
  // spill buffer (EIGER_GLOBAL): rows appended by this CTA so far, and 1 + the global index of the CTA's k-th chunk
  // (0 = nobody has reserved it yet, ~0 = the buffer is full: such rows take the global table)
  uint32_t* sp_cursor = nullptr;
  uint32_t* sp_base = nullptr;
  int sync_n = 0;                // threads that take part in cta_sync(): 0 = the whole CTA; else named barrier 1 (the ring's producer warp stays out)
  __device__ __forceinline__ void cta_sync() const {
    if (sync_n) asm volatile("bar.sync 1, %0;" :: "r"(sync_n) : "memory"); else __syncthreads();
  }

  __device__ Front(const HashAggArgs& args, unsigned char* sm, uint32_t slots_used)
      : a(args), smem(sm), n_acc(S::kStatic ? S::kAcc : args.plan.n_acc), Sn(slots_used) {
    uint32_t w = 0;
#pragma unroll
    for (int j = 0; j < NA; ++j) { if (!S::kStatic && j >= n_acc) break; w += plane_width(sig_op<SIG>(a.plan, j)); }
    skeys = reinterpret_cast<U*>(smem + (size_t)w * a.slots);   // planes are laid out for a.slots
  }

  __device__ void init(int tid, int T) {
    uint32_t off = 0;
#pragma unroll
    for (int j = 0; j < NA; ++j) {
      if (!S::kStatic && j >= n_acc) break;
      const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
      if (op == EIGER_COUNT) {
        uint32_t* p = reinterpret_cast<uint32_t*>(smem + (size_t)off * a.slots);
        for (uint32_t c = tid; c < Sn; c += T) p[c] = 0u;
      } else if (add_type(op, f)) {
        uint32_t* p = reinterpret_cast<uint32_t*>(smem + (size_t)off * a.slots);
        for (uint32_t c = tid; c < Sn; c += T) { p[c] = 0u; p[c + a.slots] = 0u; }
      } else {
        uint64_t* p = reinterpret_cast<uint64_t*>(smem + (size_t)off * a.slots);
        const uint64_t v = op == EIGER_SUM ? 0ull : acc_identity(op);
        for (uint32_t c = tid; c < Sn; c += T) p[c] = v;
      }
      off += plane_width(op);
    }
    for (uint32_t c = tid; c < Sn; c += T) skeys[c] = empty_of<U>();
  }

  // Buckets of 16 bytes (4 x 32-bit keys or 2 x 64-bit keys): one LDS.128 looks at a whole bucket,
  // so that at the load factors used here almost every row resolves on its first probe and the
  // lanes of a warp do not wait for each other's probe chains.
  static constexpr uint32_t kB = BK;
  static_assert(BK * sizeof(U) == 16 || (sizeof(U) == 4 && (BK == 2 || BK == 1)), "bucket of 16 bytes, or 4 / 8 bytes of 32-bit keys");
  __device__ __forceinline__ uint32_t home_bucket(U u) const {
    if constexpr (sizeof(U) == 4) return __umulhi(table_hash32b((uint32_t)u), Sn / kB);
    else return __umulhi((uint32_t)table_hash64((uint64_t)u), Sn / kB);   // low word: the top bits chose the partition
  }
  __device__ __forceinline__ uint4 load_bucket(uint32_t b) const {
    uint4 r;
    const uint32_t addr = (uint32_t)__cvta_generic_to_shared(reinterpret_cast<const unsigned char*>(skeys) + (size_t)b * (kB * sizeof(U)));
    if constexpr (kB * sizeof(U) == 16) {
      asm volatile("ld.volatile.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr) : "memory");
    } else if constexpr (kB * sizeof(U) == 8) {
      asm volatile("ld.volatile.shared.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(addr) : "memory");
      r.z = r.w = kEmpty32;
    } else {
      asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(r.x) : "r"(addr) : "memory");
      r.y = r.z = r.w = kEmpty32;
    }
    return r;
  }
  // position of u inside bucket q, or the first empty position + kB, or 2 * kB when full of others
  __device__ __forceinline__ uint32_t scan_bucket(const uint4& q, U u) const {
    if constexpr (sizeof(U) == 4 && kB == 1) {
      if (q.x == u) return 0; if (q.x == kEmpty32) return 1; return 2;
    } else if constexpr (sizeof(U) == 4 && kB == 2) {
      if (q.x == u) return 0; if (q.y == u) return 1;
      if (q.x == kEmpty32) return 2; if (q.y == kEmpty32) return 3;
      return 4;
    } else if constexpr (sizeof(U) == 4) {
      if (q.x == u) return 0; if (q.y == u) return 1; if (q.z == u) return 2; if (q.w == u) return 3;
      if (q.x == kEmpty32) return 4; if (q.y == kEmpty32) return 5; if (q.z == kEmpty32) return 6; if (q.w == kEmpty32) return 7;
      return 8;
    } else {
      const uint64_t k0 = ((uint64_t)q.y << 32) | q.x, k1 = ((uint64_t)q.w << 32) | q.z;
      if (k0 == u) return 0; if (k1 == u) return 1;
      if (k0 == kEmpty64) return 2; if (k1 == kEmpty64) return 3;
      return 4;
    }
  }
  // find-or-insert given the first bucket's contents; single exit.  Returns the slot or -1.
  __device__ __forceinline__ int resolve(U u, uint32_t b, uint4 q, uint32_t* s_count) {
    int res = -1;
    bool done = false;
    if constexpr (sizeof(U) == 8) { if (u == kEmpty64) done = true; }
    int probes = 0;
    while (!done) {
      const uint32_t r = scan_bucket(q, u);
      if (r < kB) { res = (int)(b * kB + r); done = true; }
      else if (r < 2 * kB) {
        // not in the table (an empty position ends the chain): insert unless the table is closed
        if (*reinterpret_cast<volatile uint32_t*>(s_count) >= a.limit) { done = true; }
        else {
          const uint32_t h = b * kB + (r - kB);
          U old;
          if constexpr (sizeof(U) == 4) old = atomicCAS(skeys + h, kEmpty32, u);
          else old = (U)atomicCAS(reinterpret_cast<unsigned long long*>(skeys + h), (unsigned long long)kEmpty64, (unsigned long long)u);
          if (old == empty_of<U>()) { atomicAdd(s_count, 1u); res = (int)h; done = true; }
          else if (old == u) { res = (int)h; done = true; }
          else q = load_bucket(b);          // somebody else took it: look at the bucket again
        }
      } else {
        b = b + 1 == Sn / kB ? 0 : b + 1;
        if (++probes >= a.max_probes * (int)((16 / sizeof(U)) / kB)) done = true; else q = load_bucket(b);
      }
    }
    return res;
  }

  // Accumulator updates in two steps so that the returning atomics of several rows are in flight
  // together: issue() fires the 32-bit adds (SUM low word, COUNT) and reads MIN / MAX cells,
  // finish() propagates carries and settles new minima / maxima.
  // scalars, not an array: ptxas kept `old[NA]` in local memory (STL / LDL between issue and finish)
  struct Pending {
    uint32_t o0, o1, o2, o3, o4, o5, o6, o7, o8;
    __device__ __forceinline__ uint32_t& at(int j) {
      switch (j) { case 0: return o0; case 1: return o1; case 2: return o2; case 3: return o3; case 4: return o4;
                   case 5: return o5; case 6: return o6; case 7: return o7; default: return o8; }
    }
    __device__ __forceinline__ uint32_t get(int j) const {
      switch (j) { case 0: return o0; case 1: return o1; case 2: return o2; case 3: return o3; case 4: return o4;
                   case 5: return o5; case 6: return o6; case 7: return o7; default: return o8; }
    }
  };
  __device__ __forceinline__ void issue(uint32_t h, const uint64_t (&raw)[NV], Pending& pd) {
    uint32_t off = 0;
#pragma unroll
    for (int j = 0; j < NA; ++j) {
      if (!S::kStatic && j >= n_acc) break;
      const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
      unsigned char* plane = smem + (size_t)off * a.slots;
      if (op == EIGER_COUNT) {
        atomicAdd(reinterpret_cast<uint32_t*>(plane) + h, 1u);
      } else if (add_type(op, f)) {
        pd.at(j) = atomicAdd(reinterpret_cast<uint32_t*>(plane) + h, (uint32_t)raw[sig_col<SIG>(a.plan, j)]);
      } else if (op == EIGER_SUM) {
        atomicAdd(reinterpret_cast<double*>(plane) + h, __longlong_as_double((long long)raw[sig_col<SIG>(a.plan, j)]));
      }
      off += plane_width(op);
    }
  }
  __device__ __forceinline__ void finish(uint32_t h, const uint64_t (&raw)[NV], const Pending& pd) {
    uint32_t off = 0;
#pragma unroll
    for (int j = 0; j < NA; ++j) {
      if (!S::kStatic && j >= n_acc) break;
      const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
      unsigned char* plane = smem + (size_t)off * a.slots;
      if (op != EIGER_COUNT) {
        const uint64_t v = raw[sig_col<SIG>(a.plan, j)];
        if (add_type(op, f)) {
          const uint32_t vl = (uint32_t)v;
          const uint32_t hi = (uint32_t)(v >> 32) + ((uint32_t)(pd.get(j) + vl) < vl ? 1u : 0u);
          if (hi) atomicAdd(reinterpret_cast<uint32_t*>(plane) + a.slots + h, hi);
        } else if (op != EIGER_SUM) {
          const long long part = (long long)row_partial(op, f, v);
          long long* cell = reinterpret_cast<long long*>(plane) + h;
          const long long cur = *reinterpret_cast<volatile long long*>(cell);
          if (op == EIGER_MIN) { if (part < cur) atomicMin(cell, part); }
          else { if (part > cur) atomicMax(cell, part); }
        }
      }
      off += plane_width(op);
    }
  }

  // accumulator j of slot h in partial form (64 bits)
  __device__ __forceinline__ uint64_t read(uint32_t h, int j, uint32_t off) const {
    const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
    const unsigned char* plane = smem + (size_t)off * a.slots;
    if (op == EIGER_COUNT) return (uint64_t)(reinterpret_cast<const uint32_t*>(plane)[h]);
    if (add_type(op, f)) { const uint32_t* lo = reinterpret_cast<const uint32_t*>(plane) + h; return ((uint64_t)lo[a.slots] << 32) | lo[0]; }
    return reinterpret_cast<const uint64_t*>(plane)[h];
  }

  __device__ __forceinline__ void back_row(U u, const uint64_t (&raw)[NV]) {
    uint64_t* cells = back_find_or_insert(a.table, a.cap, a.stride, (uint64_t)u, a.call);
    if (cells) {
#pragma unroll
      for (int j = 0; j < NA; ++j) {
        if (!S::kStatic && j >= n_acc) break;
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        atomic_merge(cells + j, op, f, row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]));
      }
    }
  }

  // position of u in its home bucket b as a slot number, or -1: branch-free, so that the lanes of
  // a warp take the common case (key already in its home bucket) in lock step.  ok = row is valid
  // and u is not the empty marker (which would "match" a free position).
  __device__ __forceinline__ int match_home(const uint4& q, U u, uint32_t b, bool ok) const {
    int r = -1;
    if constexpr (sizeof(U) == 4) {
      r = q.w == u ? 3 : r; r = q.z == u ? 2 : r; r = q.y == u ? 1 : r; r = q.x == u ? 0 : r;
    } else {
      const uint64_t k0 = ((uint64_t)q.y << 32) | q.x, k1 = ((uint64_t)q.w << 32) | q.z;
      r = k1 == u ? 1 : r; r = k0 == u ? 0 : r;
    }
    return ok && r >= 0 ? (int)(b * kB) + r : -1;
  }

  // two rows at a time: both first probes in flight, then both sets of atomics.  Rows whose key is
  // not in its home bucket yet (new key, or a bucket that overflowed) take the probe loop, one
  // code copy for both rows.
  // Returns bit 0 / 1 set for a row that found no room (the caller sends those to the global table).
  __device__ __forceinline__ uint32_t pair(U u0, const uint64_t (&raw0)[NV], bool v0, U u1, const uint64_t (&raw1)[NV], bool v1,
                                           uint32_t* s_count) {
    const uint32_t b0 = home_bucket(u0), b1 = home_bucket(u1);
    const uint4 q0 = load_bucket(b0), q1 = load_bucket(b1);
    // a key whose rebased value equals the empty marker lives in the global table only
    const bool ok0 = v0 && u0 != empty_of<U>(), ok1 = v1 && u1 != empty_of<U>();
    int h0, h1;
    if constexpr (sizeof(U) == 8) {
      // measured: the branch-free first look pays for 64-bit keys (C3 -3 %, C4 -3.5 %) and costs
      // 4-8 % for 32-bit keys in whole-input mode and 10-20 % in partition mode (measured again at the end of round 2:
      // C5 2^16 / 2^20 / 2^24 aggregate 1.12 / 1.30 / 1.48 -> 1.23 / 1.54 / 1.77 ms), although ncu shows that kernel at 84 %
      // of its issue slots: the four compares and selects per row cost more than the loop they bypass
      h0 = match_home(q0, u0, b0, ok0); h1 = match_home(q1, u1, b1, ok1);
      if ((ok0 && h0 < 0) || (ok1 && h1 < 0)) {
#pragma unroll 1
        for (int k = 0; k < 2; ++k) {
          const bool need = k == 0 ? (ok0 && h0 < 0) : (ok1 && h1 < 0);
          if (need) {
            const int h = resolve(k == 0 ? u0 : u1, k == 0 ? b0 : b1, k == 0 ? q0 : q1, s_count);
            if (k == 0) h0 = h; else h1 = h;
          }
        }
      }
      __syncwarp();
    } else {
      h0 = ok0 ? resolve(u0, b0, q0, s_count) : -1;
      __syncwarp();
      h1 = ok1 ? resolve(u1, b1, q1, s_count) : -1;
      __syncwarp();
    }
    Pending p0, p1;
    if (h0 >= 0 && h1 >= 0) {
      issue((uint32_t)h0, raw0, p0);
      issue((uint32_t)h1, raw1, p1);
      finish((uint32_t)h0, raw0, p0);
      finish((uint32_t)h1, raw1, p1);
    } else {
      if (h0 >= 0) { issue((uint32_t)h0, raw0, p0); finish((uint32_t)h0, raw0, p0); }
      if (h1 >= 0) { issue((uint32_t)h1, raw1, p1); finish((uint32_t)h1, raw1, p1); }
    }
    __syncwarp();
    return (v0 && h0 < 0 ? 1u : 0u) | (v1 && h1 < 0 ? 2u : 0u);
  }

  // Heavy hitters: rows whose key is one of the sample's heavy hitters skip the
  // hash table and update the WARP'S OWN cells (shared-memory atomics that only the lanes of this
  // warp carrying the same key contend on).  A key that owns 12 % of the rows (C3) otherwise has
  // ~4 lanes of every warp and all 32 warps of the SM queue on one slot (measured: 1.4 ms of C3's
  // 5.5).  Reducing the rows with shuffles instead cost more than it saved.
  // Returns whether this lane's row was absorbed.
  __device__ __forceinline__ bool hot_absorb(U u, const uint64_t (&raw)[NV], uint64_t* cells, uint32_t* rows, int lane) {
    int mine = -1;
#pragma unroll 1
    for (int hx = 0; hx < a.n_hot; ++hx) mine = u == (U)a.hot[hx] ? hx : mine;
    if (mine >= 0) {
      // the warp's own cells: only the lanes of this warp that carry the same hot key meet here
#pragma unroll
      for (int j = 0; j < NA; ++j) {
        if (!S::kStatic && j >= n_acc) break;
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        uint64_t* c = cells + mine * NA + j;
        if (op == EIGER_COUNT) continue;      // the warp's row counter below IS the count (a 64-bit add here is a CAS loop: 28 % of C3's wavefronts)
        const uint64_t part = row_partial(op, f, raw[sig_col<SIG>(a.plan, j)]);
        if (op == EIGER_SUM) atomic_merge(c, op, f, part);
        else {
          const long long cur = *reinterpret_cast<volatile long long*>(c);
          if (op == EIGER_MIN ? (long long)part < cur : (long long)part > cur) atomic_merge(c, op, f, part);
        }
      }
      atomicAdd(rows + mine, 1u);
    }
    __syncwarp();
    (void)lane;
    return mine >= 0;
  }
  // hs = cell sets per warp (the lanes of a warp are spread over them: fewer lanes retry against each other in the
  // compare-and-swap loops of the 64-bit adds)
  __device__ void hot_init(uint64_t* cells, uint32_t* rows, int tid, int T, int hs = 1) {
    for (int i = tid; i < (T >> 5) * hs * kMaxHot * NA; i += T) {
      const int j = i % NA;
      cells[i] = (S::kStatic || j < n_acc) ? acc_identity(sig_op<SIG>(a.plan, j)) : 0ull;
    }
    for (int i = tid; i < (T >> 5) * hs * kMaxHot; i += T) rows[i] = 0u;
  }
  // every warp's hot cells into the global table
  __device__ void hot_flush(const uint64_t* cells, const uint32_t* rows, int tid, int T, int hs = 1) {
    for (int i = tid; i < (T >> 5) * hs * a.n_hot; i += T) {
      const int w = i / a.n_hot, hx = i % a.n_hot;
      if (rows[w * kMaxHot + hx] == 0u) continue;
      uint64_t* dst = back_find_or_insert(a.table, a.cap, a.stride, a.hot[hx], a.call);
      if (!dst) continue;
      for (int j = 0; j < n_acc; ++j) {
        const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
        atomic_merge(dst + j, op, f, op == EIGER_COUNT ? (uint64_t)rows[w * kMaxHot + hx] : cells[(w * kMaxHot + hx) * NA + j]);
      }
    }
  }

  // rows of one trip that found no room in shared memory: global table, one code copy per trip
  template <int R>
  __device__ __forceinline__ void spill(const U (&u)[R], const uint64_t (&raw)[R][NV], uint32_t miss, bool& missed) {
    // (miss is a copy: the spill-buffer path narrows it to the rows it could not place)
    if (__any_sync(0xffffffffu, miss != 0)) {
      if (a.spec) { missed = missed || miss != 0; }
      else {
        // A key may now live in BOTH tables: a lane that found the table closed sends its row to the
        // global table while another lane, which passed the limit check a moment earlier, inserts the
        // same key here.  The work item therefore no longer owns its keys exclusively and must merge
        // (not emit) at the end.
        if (s_spill && miss) *reinterpret_cast<volatile uint32_t*>(s_spill) = 1u;
        if constexpr (sizeof(U) == 8) if (sp_cursor) {
          // Append to the spill buffer: the warp's rows get consecutive places in the CTA's numbering (one
          // shared-memory atomic per warp and row position); the lane whose row opens a chunk reserves that chunk
          // in the buffer (one global atomic per 2^sp_lg rows) and publishes it, the others wait for it.
          const int lane = threadIdx.x & 31;
          const uint32_t cmask = (1u << a.sp_lg) - 1u;
          uint32_t fb = 0;           // rows that found the buffer full
#pragma unroll
          for (int k = 0; k < R; ++k) {
            const bool mk = (miss >> k) & 1u;
            const uint32_t m = __ballot_sync(0xffffffffu, mk);
            if (m == 0u) continue;
            uint32_t pos0 = 0;
            if (lane == 0) pos0 = atomicAdd(sp_cursor, (uint32_t)__popc(m));
            pos0 = __shfl_sync(0xffffffffu, pos0, 0);
            const uint32_t li = pos0 + __popc(m & ((1u << lane) - 1u));
            const uint32_t c = li >> a.sp_lg;
            if (mk && (li & cmask) == 0u && c < kSpillChunks) {
              const unsigned long long g = atomicAdd(&a.call->spill_chunks, 1ull);
              *reinterpret_cast<volatile uint32_t*>(sp_base + c) = g < a.sp_cap_chunks ? (uint32_t)g + 1u : ~0u;
            }
            __syncwarp();
            if (mk) {
              uint32_t g = ~0u;
              if (c < kSpillChunks) while ((g = *reinterpret_cast<volatile uint32_t*>(sp_base + c)) == 0u) {}
              if (g != ~0u) {
                const uint64_t at = ((uint64_t)(g - 1u) << a.sp_lg) | (li & cmask);
                a.sp_keys[at] = (uint64_t)u[k];
#pragma unroll
                for (int cc = 0; cc < NV; ++cc) if (S::kStatic || cc < a.plan.n_vals) a.sp_vals[cc][at] = raw[k][cc];
              } else fb |= 1u << k;
            }
          }
          miss = fb;
          if (!__any_sync(0xffffffffu, miss != 0)) return;
        }
        if constexpr (NV <= 2) if (q_base) {
          const int lane = threadIdx.x & 31;
          uint64_t* qk = reinterpret_cast<uint64_t*>(q_base);
#pragma unroll
          for (int k = 0; k < R; ++k) {
            const bool mk = (miss >> k) & 1u;
            const uint32_t m = __ballot_sync(0xffffffffu, mk);
            if (m) {
              if (mk) {
                const int p = q_n + __popc(m & ((1u << lane) - 1u));
                qk[p] = (uint64_t)u[k];
#pragma unroll
                for (int c = 0; c < NV; ++c) qk[64 * (1 + c) + p] = raw[k][c];
              }
              q_n += __popc(m);
              if (q_n >= 32) {
                __syncwarp();
                q_n -= 32;
                uint64_t rr[NV];
#pragma unroll
                for (int c = 0; c < NV; ++c) rr[c] = qk[64 * (1 + c) + q_n + lane];
                back_row((U)qk[q_n + lane], rr);
                __syncwarp();
              }
            }
          }
          return;
        }
#pragma unroll 1
        for (int k = 0; k < R; ++k) {
          U uu = u[0]; uint64_t rr[NV];
#pragma unroll
          for (int c = 0; c < NV; ++c) rr[c] = raw[0][c];
#pragma unroll
          for (int r = 1; r < R; ++r)
            if (k == r) {
              uu = u[r];
#pragma unroll
              for (int c = 0; c < NV; ++c) rr[c] = raw[r][c];
            }
          if ((miss >> k) & 1u) back_row(uu, rr);
          __syncwarp();
        }
      }
    }
  }

  // spill buffer: the unused tail of this CTA's last chunk is filled with the empty marker (a key no row of a
  // spill buffer can have: api.cu takes the buffer only when the rebased keys stay below it), so that the
  // buffer is one gapless run of whole chunks for the partition pass.  Called by all threads after a barrier.
  __device__ void spill_pad(int tid, int T) {
    if constexpr (sizeof(U) == 8) {
      if (!sp_cursor) return;
      const uint32_t total = *sp_cursor, cmask = (1u << a.sp_lg) - 1u, c = total >> a.sp_lg;
      if ((total & cmask) == 0u || c >= kSpillChunks) return;
      const uint32_t g = sp_base[c];
      if (g == 0u || g == ~0u) return;
      for (uint32_t li = (total & cmask) + tid; li <= cmask; li += T) a.sp_keys[((uint64_t)(g - 1u) << a.sp_lg) | li] = kEmpty64;
    }
  }

  // the rows still waiting in this warp's queue
  __device__ __forceinline__ void drain_queue() {
    if (!q_base) return;
    const int lane = threadIdx.x & 31;
    __syncwarp();
    if (lane < q_n) {
      const uint64_t* qk = reinterpret_cast<const uint64_t*>(q_base);
      uint64_t rr[NV];
#pragma unroll
      for (int c = 0; c < NV; ++c) rr[c] = qk[64 * (1 + c) + lane];
      back_row((U)qk[lane], rr);
    }
    q_n = 0;
    __syncwarp();
  }

  // merge every occupied slot into the global table
  __device__ void flush_merge(int tid, int T) {
    const int lane = tid & 31;
    for (uint32_t h0 = tid - lane; h0 < Sn; h0 += T) {       // warp-uniform trip count
      const uint32_t h = h0 + lane;
      const U k = h < Sn ? skeys[h] : empty_of<U>();
      if (k != empty_of<U>()) {
        uint64_t* cells = back_find_or_insert(a.table, a.cap, a.stride, (uint64_t)k, a.call);
        if (cells) {
          uint32_t off = 0;
          for (int j = 0; j < n_acc; ++j) {
            const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
            const uint64_t v = read(h, j, off);
            off += plane_width(op);
            if (v == acc_identity(op) && !(op == EIGER_SUM && f)) continue;
            atomic_merge(cells + j, op, f, v);
          }
        }
      }
      __syncwarp();
    }
  }

  // Write every occupied slot as one output group (the CTA owns these keys exclusively).
  // Two passes over the slots, no atomics: ballot counts per warp, one exclusive scan of the warp
  // totals, then every warp writes its groups in slot order (consecutive lanes -> consecutive
  // rows of the output columns).  KT = the single key column's C type (0 bytes: generic path).
  template <class KT>
  __device__ __forceinline__ void emit_rows(int tid, int T, unsigned long long base, uint32_t wbase) {
    const int lane = tid & 31;
    uint32_t run = wbase;
    for (uint32_t h0 = tid - lane; h0 < Sn; h0 += T) {      // warp-uniform trip count
      const uint32_t h = h0 + lane;
      const U k = h < Sn ? skeys[h] : empty_of<U>();
      const bool occ = k != empty_of<U>();
      const uint32_t m = __ballot_sync(0xffffffffu, occ);
      const uint64_t g = base + run + __popc(m & ((1u << lane) - 1u));
      run += __popc(m);
      if (occ && (int64_t)g < a.out_capacity) {
        if constexpr (sizeof(KT) == 1 && !std::is_same<KT, int8_t>::value) store_group_key(a.key, a.out_keys, (uint64_t)k, g);
        else static_cast<KT*>(a.out_keys[0])[g] = (KT)((uint64_t)k + a.key.base[0]);
        uint32_t off = 0;
#pragma unroll
        for (int j = 0; j < NA; ++j) {
          if (j >= a.n_out) break;
          const int op = sig_op<SIG>(a.plan, j); const bool f = sig_f64<SIG>(a.plan, j);
          a.out_aggs[j][g] = acc_finalize(op, f, read(h, j, off));
          off += plane_width(op);
        }
      }
    }
  }
  __device__ void flush_emit(int tid, int T, uint32_t n_keys, unsigned long long* s_base, uint32_t* s_wtot) {
    const int lane = tid & 31, warp = tid >> 5;
    if (tid == 0) *s_base = n_keys ? atomicAdd(&a.call->n_groups, (unsigned long long)n_keys) : 0ull;
    uint32_t cnt = 0;
    for (uint32_t h0 = tid - lane; h0 < Sn; h0 += T) {
      const uint32_t h = h0 + lane;
      cnt += __popc(__ballot_sync(0xffffffffu, h < Sn && skeys[h] != empty_of<U>()));
    }
    if (lane == 0) s_wtot[warp] = cnt;
    cta_sync();
    if (warp == 0) {       // exclusive scan of up to 32 warp totals
      const uint32_t v = lane < (T >> 5) ? s_wtot[lane] : 0u;
      uint32_t inc = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += y; }
      s_wtot[lane] = inc - v;
    }
    cta_sync();
    const unsigned long long base = *s_base;
    const uint32_t wbase = s_wtot[warp];
    if (a.key.ncols == 1) {
      switch (a.key.dtype[0]) {
        case EIGER_I8: emit_rows<int8_t>(tid, T, base, wbase); break;
        case EIGER_I32: emit_rows<int32_t>(tid, T, base, wbase); break;
        default: emit_rows<int64_t>(tid, T, base, wbase); break;
      }
    } else {
      emit_rows<uint8_t>(tid, T, base, wbase);     // several key columns: un-fuse per group
    }
  }
};

// ---- rows out of the shared-memory ring (ring.cuh) ---------------------------------------------
// A stage holds `chunk` = 2 x blockDim rows column by column: key column c at koff[c] (kw[c] bytes per
// element), value column c at voff[c] (vw[c] bytes per element: int32 values are sign-extended to the
// 64-bit accumulators, "4-byte data types (I32)").
__device__ __forceinline__ uint64_t ring_elem(const unsigned char* col, int w, int r) {
  if (w == 8) return *reinterpret_cast<const uint64_t*>(col + 8 * (size_t)r);
  if (w == 4) return (uint64_t)(int64_t)*reinterpret_cast<const int32_t*>(col + 4 * (size_t)r);
  return (uint64_t)(int64_t)*reinterpret_cast<const int8_t*>(col + r);
}
template <int KK>
__device__ __forceinline__ typename KeyTraits<KK>::U ring_key(const HashAggArgs& a, const unsigned char* st, int r) {
  using U = typename KeyTraits<KK>::U;
  if constexpr (KK == KK_I32) return *reinterpret_cast<const uint32_t*>(st + a.koff[0] + 4 * (size_t)r) - (uint32_t)a.key.base[0];
  else if constexpr (KK == KK_U32PRE) return *reinterpret_cast<const uint32_t*>(st + a.koff[0] + 4 * (size_t)r);
  else if constexpr (KK == KK_I64) return *reinterpret_cast<const uint64_t*>(st + a.koff[0] + 8 * (size_t)r) - a.key.base[0];
  else if constexpr (KK == KK_U64PRE) return *reinterpret_cast<const uint64_t*>(st + a.koff[0] + 8 * (size_t)r);
  else {
    uint64_t d[kMaxKeyCols];
#pragma unroll
    for (int c = 0; c < kMaxKeyCols; ++c) d[c] = c < a.key.ncols ? ring_elem(st + a.koff[c], a.kw[c], r) - a.key.base[c] : 0ull;
    return (U)fuse_cols(a.key, d);
  }
}
template <int SIG, int NV>
__device__ __forceinline__ void ring_vals(const HashAggArgs& a, const unsigned char* st, int r, int n_vals, uint64_t (&raw)[NV]) {
#pragma unroll
  for (int c = 0; c < NV; ++c) {
    if constexpr (Sig<SIG>::kStatic) raw[c] = ring_elem(st + a.voff[c], Sig<SIG>::vwidth(c), r);
    else raw[c] = c < n_vals ? ring_elem(st + a.voff[c], a.vw[c], r) : 0ull;
  }
}
// One elected thread keeps the ring full: rows [row0, row0 + rows) of every column go into stage
// g % stages with one bulk copy per column (row0 a multiple of 32, rows a multiple of 32: every
// copy starts 16-byte aligned and is a multiple of 16 bytes long, whatever the column width).
// `quit` (may be null): a shared flag raised by a warp that leaves the chunk loop early (speculative
// runs); the stage it would have released never becomes free, so the wait gives up.  Returns whether
// the chunk was requested.
__device__ __forceinline__ bool ring_issue(const HashAggArgs& a, unsigned char* ring, uint64_t* full, uint64_t* empty,
                                           uint32_t g, int64_t row0, uint32_t rows, uint64_t policy, const uint32_t* quit = nullptr) {
  const uint32_t s = g % (uint32_t)a.stages;
  if (g >= (uint32_t)a.stages) {
    const uint32_t par = ((g / (uint32_t)a.stages) - 1u) & 1u;
    while (!mbar_try_wait(&empty[s], par)) { if (quit && *reinterpret_cast<const volatile uint32_t*>(quit)) return false; }
  }
  unsigned char* st = ring + (size_t)s * a.stage_bytes;
  uint32_t bytes = 0;
  for (int c = 0; c < a.n_src; ++c) bytes += rows * a.kw[c];
  for (int c = 0; c < a.plan.n_vals; ++c) bytes += rows * a.vw[c];
  mbar_expect_tx(&full[s], bytes);
  if (policy) {
    for (int c = 0; c < a.n_src; ++c)
      bulk_g2s_hint(st + a.koff[c], static_cast<const unsigned char*>(a.key.ptr[c]) + row0 * a.kw[c], rows * a.kw[c], &full[s], policy);
    for (int c = 0; c < a.plan.n_vals; ++c)
      bulk_g2s_hint(st + a.voff[c], static_cast<const unsigned char*>(a.plan.vals[c]) + row0 * a.vw[c], rows * a.vw[c], &full[s], policy);
  } else {
    for (int c = 0; c < a.n_src; ++c)
      bulk_g2s(st + a.koff[c], static_cast<const unsigned char*>(a.key.ptr[c]) + row0 * a.kw[c], rows * a.kw[c], &full[s]);
    for (int c = 0; c < a.plan.n_vals; ++c)
      bulk_g2s(st + a.voff[c], static_cast<const unsigned char*>(a.plan.vals[c]) + row0 * a.vw[c], rows * a.vw[c], &full[s]);
  }
  return true;
}

template <int KK, int SIG, int BK>
__global__ void __launch_bounds__(kMaxThreads, 1)
hash_agg_kernel(const __grid_constant__ HashAggArgs a) {
  extern __shared__ __align__(128) unsigned char dyn[];     // [ring stages][heavy-hitter cells][table]
  __shared__ __align__(8) uint64_t s_full[kMaxStages], s_empty[kMaxStages];
  __shared__ uint32_t s_count, s_abort, s_spilled, s_quit;
  __shared__ uint32_t s_wtot[32];
  __shared__ unsigned long long s_base;
  using F = Front<KK, SIG, BK>;
  using U = typename F::U;
  constexpr int NV = F::NV;
  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31;
  const int n_vals = Sig<SIG>::kStatic ? NV : a.plan.n_vals;
  unsigned char* ring = dyn;
  unsigned char* smem = dyn + a.table_off;
  const uint32_t chunk = 2u * (uint32_t)T;                  // rows per stage: two per thread
  if (tid == 0) {
    for (int s = 0; s < a.stages; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], (uint32_t)(T >> 5) - (IsPre<KK>::v ? 1u : 0u)); }
    mbar_fence_init();
  }
  uint32_t g_cons = 0, g_issued = 0;                        // chunks consumed (all threads) / issued (thread 0)
  const uint64_t policy = a.ring_hint ? policy_evict_first() : 0ull;   // the rows are read once: first out of L2

  if constexpr (!IsPre<KK>::v) {
    // ---- whole-input mode: chunk c = blockIdx.x, + gridDim.x, ... of the input ----
    F f(a, smem, a.slots);
    uint64_t* s_hot = reinterpret_cast<uint64_t*>(dyn + a.hot_off);
    uint32_t* s_hot_rows = reinterpret_cast<uint32_t*>(s_hot + (kMaxThreads / 32) * kMaxHot * kMaxAcc);
    uint64_t* my_hot = s_hot + (tid >> 5) * kMaxHot * F::NA;
    uint32_t* my_hot_rows = s_hot_rows + (tid >> 5) * kMaxHot;
    if (tid == 0) { s_count = 0; s_abort = 0; s_quit = 0; }
    const int64_t n_chunks = a.n / chunk;
    const int64_t mine = n_chunks > blockIdx.x ? (n_chunks - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    __syncthreads();                                         // barriers initialised
    if (tid == 0)
      for (; g_issued < (uint32_t)a.stages && (int64_t)g_issued < mine; ++g_issued)
        ring_issue(a, ring, s_full, s_empty, g_issued, ((int64_t)blockIdx.x + (int64_t)g_issued * gridDim.x) * chunk, chunk, policy);
    f.init(tid, T);
    if (a.n_hot) f.hot_init(s_hot, s_hot_rows, tid, T);
    __syncthreads();
    bool missed = false;
    // the chunk loop, compiled twice: with and without the heavy-hitter look (runtime row-valid flags
    // and the hot-key scan cost the plain path 5-15 % at low NDV when they were merely branched over)
    auto run_chunks = [&](auto hot_c) {
      constexpr bool HOT = decltype(hot_c)::value;
      for (int64_t k = 0; k < mine; ++k, ++g_cons) {
        // speculative run: look at the global give-up flag every 16th trip only (an L2 round trip each
        // time).  A warp that leaves raises s_quit first: the producer and the warps still waiting for a
        // chunk that will now never be requested must not wait for it.
        if (a.spec) {
          if (__any_sync(0xffffffffu, missed || ((g_cons & 15u) == 0u && *reinterpret_cast<volatile uint32_t*>(&a.call->abort)))) {
            if (lane == 0) *reinterpret_cast<volatile uint32_t*>(&s_quit) = 1u;
            break;
          }
        }
        const uint32_t s = g_cons % (uint32_t)a.stages;
        {
          const uint32_t par = (g_cons / (uint32_t)a.stages) & 1u;
          bool gone = false;
          while (!mbar_try_wait(&s_full[s], par)) { if (a.spec && *reinterpret_cast<volatile uint32_t*>(&s_quit)) { gone = true; break; } }
          if (a.spec && __any_sync(0xffffffffu, gone)) break;      // warp-uniform: the lanes left the wait one by one
        }
        const unsigned char* st = ring + (size_t)s * a.stage_bytes;
        U u[2]; uint64_t raw[2][NV];
        u[0] = ring_key<KK>(a, st, tid); u[1] = ring_key<KK>(a, st, T + tid);
        ring_vals<SIG, NV>(a, st, tid, n_vals, raw[0]); ring_vals<SIG, NV>(a, st, T + tid, n_vals, raw[1]);
        __syncwarp();
        if (lane == 0) mbar_arrive(&s_empty[s]);             // this warp's rows are in registers: the stage may be refilled
        if (tid == 0 && (int64_t)g_issued < mine) {
          if (ring_issue(a, ring, s_full, s_empty, g_issued, ((int64_t)blockIdx.x + (int64_t)g_issued * gridDim.x) * chunk, chunk, policy, a.spec ? &s_quit : nullptr))
            ++g_issued;
        }
        uint32_t miss;
        if constexpr (HOT) {
          const bool ab0 = f.hot_absorb(u[0], raw[0], my_hot, my_hot_rows, lane);
          const bool ab1 = f.hot_absorb(u[1], raw[1], my_hot, my_hot_rows, lane);
          miss = f.pair(u[0], raw[0], !ab0, u[1], raw[1], !ab1, &s_count);
        } else {
          miss = f.pair(u[0], raw[0], true, u[1], raw[1], true, &s_count);
        }
        f.spill(u, raw, miss, missed);
      }
    };
    if (a.n_hot) run_chunks(std::true_type{}); else run_chunks(std::false_type{});
    // a speculative run that gave up leaves bulk copies in flight: they must land before the CTA ends
    // (every requested chunk completes its `full` phase whether or not anybody consumes it)
    if (tid == 0) for (uint32_t g = g_cons; g < g_issued; ++g) mbar_wait(&s_full[g % (uint32_t)a.stages], (g / (uint32_t)a.stages) & 1u);
    if (!(a.spec && __any_sync(0xffffffffu, missed))) {
      // ragged tail (fewer than `chunk` rows): row at a time, spread over the whole grid, warp-uniform trip count
      for (int64_t i0 = n_chunks * chunk + (int64_t)blockIdx.x * T + (tid - lane); i0 < a.n; i0 += (int64_t)gridDim.x * T) {
        const int64_t i = i0 + lane;
        uint64_t rawt[NV];
        U ut = 0;
        if (i < a.n) {
#pragma unroll
          for (int c = 0; c < NV; ++c) rawt[c] = (Sig<SIG>::kStatic || c < n_vals) ? global_val(a.plan, c, sig_vw<SIG>(a.plan, c), i) : 0ull;
          ut = load_u<KK>(a.key, i);
        }
        const uint32_t miss = f.pair(ut, rawt, i < a.n, ut, rawt, false, &s_count);
        if (__any_sync(0xffffffffu, miss != 0)) { if (a.spec) missed = missed || miss != 0; else if (miss) f.back_row(ut, rawt); }
        __syncwarp();
      }
    }
    if (a.spec) {
      if (missed) { atomicOr(&a.call->abort, 1u); atomicOr(&s_abort, 1u); }
      __syncthreads();
      if (s_abort || *reinterpret_cast<volatile uint32_t*>(&a.call->abort)) return;   // result is discarded
    } else {
      __syncthreads();
    }
    f.flush_merge(tid, T);
    if (a.n_hot) f.hot_flush(s_hot, s_hot_rows, tid, T);
  } else {
    // ---- partition mode: work items blockIdx.x, + gridDim.x, ...; an item is a whole partition
    // (this CTA then owns its keys and emits them) or a slice of a hot one (merged through the
    // global table like the whole-input mode).  Warp-specialised: the LAST warp (the hardware's
    // issue arbiter favours the highest warp id) only produces - one lane walks the CTA's items and
    // keeps the ring full, ACROSS items: while the consumers read one item's table out and
    // initialise the next one's, the next item's first rows are already landing.  The other warps
    // consume and synchronise among themselves on named barrier 1. ----
    const unsigned long long n_items = a.item_off[a.n_parts];
    const int Tc = T - 32;                                   // consumer threads
    const uint32_t cchunk = 2u * (uint32_t)Tc;               // rows per stage: two per consumer thread
    // rows [r0, r1) of item `it`
    auto item_rows = [&](unsigned long long it, int64_t& r0, int64_t& r1, bool& exclusive) {
      const int p = (int)a.item_part[it];                    // one broadcast load from the map written by part_items_kernel
      const unsigned long long n_cuts = a.item_off[p + 1] - a.item_off[p], ci = it - a.item_off[p];
      const int64_t P0 = (int64_t)a.part_off[p], P1 = (int64_t)a.part_off[p + 1];
      const int64_t per = (P1 - P0 + (int64_t)n_cuts - 1) / (int64_t)n_cuts;
      r0 = P0 + (int64_t)ci * per; r1 = r0 + per < P1 ? r0 + per : P1;
      exclusive = n_cuts == 1;
    };
    __syncthreads();                                         // barriers initialised (the last whole-CTA barrier)
    if (tid >= Tc) {
      if (lane == 0) {
        uint32_t g = 0;
        for (unsigned long long it = blockIdx.x; it < n_items; it += gridDim.x) {
          int64_t r0, r1; bool ex;
          item_rows(it, r0, r1, ex);
          const int64_t A = r0 & ~(int64_t)31;               // bulk copies start 16-byte aligned in every column
          for (int64_t row0 = A; row0 < r1; row0 += cchunk, ++g) {
            const int64_t left = ((r1 - row0) + 31) & ~(int64_t)31;
            ring_issue(a, ring, s_full, s_empty, g, row0, (uint32_t)(left < (int64_t)cchunk ? left : (int64_t)cchunk), policy);
          }
        }
      }
      return;
    }
    for (unsigned long long it = blockIdx.x; it < n_items; it += gridDim.x) {
      int64_t r0, r1; bool exclusive;
      item_rows(it, r0, r1, exclusive);
      const uint32_t lo = (uint32_t)(r0 & 31), hi = (uint32_t)(r1 - (r0 & ~(int64_t)31));   // valid rows of the item, relative to A
      const uint32_t chunks = r1 > r0 ? (hi + cchunk - 1) / cchunk : 0u;
      // a table no larger than the partition needs: 2 slots per row is always enough
      const uint64_t want = 2ull * (uint64_t)(r1 - r0) + 64;
      const uint32_t Sn = (uint32_t)(want < a.slots ? want : a.slots) & ~7u;   // whole buckets
      F f(a, smem, Sn);
      f.s_spill = &s_spilled;
      f.sync_n = Tc;
      f.cta_sync();                          // the previous item's emit is over
      if (tid == 0) { s_count = 0; s_spilled = 0; }
      f.init(tid, Tc);
      f.cta_sync();
      bool missed = false;
      for (uint32_t k = 0; k < chunks; ++k, ++g_cons) {
        const uint32_t s = g_cons % (uint32_t)a.stages;
        mbar_wait(&s_full[s], (g_cons / (uint32_t)a.stages) & 1u);
        const unsigned char* st = ring + (size_t)s * a.stage_bytes;
        const uint32_t i0 = k * cchunk + (uint32_t)tid, i1 = i0 + (uint32_t)Tc;
        const bool v0 = i0 >= lo && i0 < hi, v1 = i1 >= lo && i1 < hi;
        U u[2]; uint64_t raw[2][NV];
        u[0] = ring_key<KK>(a, st, tid); u[1] = ring_key<KK>(a, st, Tc + tid);
        ring_vals<SIG, NV>(a, st, tid, n_vals, raw[0]); ring_vals<SIG, NV>(a, st, Tc + tid, n_vals, raw[1]);
        __syncwarp();
        if (lane == 0) mbar_arrive(&s_empty[s]);             // this warp's rows are in registers: the stage may be refilled
        const uint32_t miss = f.pair(v0 ? u[0] : (U)0, raw[0], v0, v1 ? u[1] : (U)0, raw[1], v1, &s_count);
        f.spill(u, raw, miss, missed);
      }
      f.cta_sync();
      // emit only what this CTA owns exclusively: a whole partition none of whose rows was sent to
      // the global table (otherwise a key could be emitted here AND by the compaction pass)
      if (exclusive && s_spilled == 0u) f.flush_emit(tid, Tc, s_count, &s_base, s_wtot);
      else f.flush_merge(tid, Tc);
    }
  }
}

// ---- the same kernel with the rows loaded by the threads themselves (16-byte streaming loads into
// registers, the next tile's loads in flight while the current one is processed).  The kernel is bound
// by the shared-memory pipe (bucket look-ups + atomics); rows that arrive through the shared-memory
// ring cost it 6 more wavefronts per 32 rows (the bulk copy's write + the threads' reads), so the ring
// version is the slower one wherever the table work dominates (measured; EIGER_RING selects). ----
template <int KK, int SIG, int BK>
__global__ void __launch_bounds__(kMaxThreads, 1)
hash_agg_ldg_kernel(const __grid_constant__ HashAggArgs a) {
  extern __shared__ __align__(16) unsigned char smem[];
  __shared__ uint32_t s_count, s_abort, s_spilled;
  __shared__ uint32_t s_wtot[32];
  __shared__ unsigned long long s_base;
  using F = Front<KK, SIG, BK>;
  using U = typename F::U;
  constexpr int NV = F::NV;
  const int tid = threadIdx.x, T = blockDim.x;
  const int n_vals = Sig<SIG>::kStatic ? NV : a.plan.n_vals;

  if constexpr (!IsPre<KK>::v) {
    // ---- whole-input mode: tiles of 2 * T * UNR rows, grid-strided; the next tile's loads are
    // in flight while the current one is processed (one CTA per SM: there is nobody else to
    // hide HBM latency behind) ----
    constexpr int UNR = !Sig<SIG>::kStatic ? 1 : (NV >= 4 ? 1 : (sizeof(U) == 8 ? 1 : 2));   // 3 spills at the 64-register cap
    F f(a, smem, a.slots);
    if (a.queue_off && !a.spec) f.q_base = smem + a.queue_off + (size_t)(tid >> 5) * 64 * 8 * (1 + NV);
    // heavy-hitter cells: two sets per warp (lanes 0-15 / 16-31) while that fits next to the 200 KB table
    constexpr int HS = F::NA <= 4 ? 2 : 1;
    __shared__ uint64_t s_hot[(kMaxThreads / 32) * HS * kMaxHot * F::NA];
    __shared__ uint32_t s_hot_rows[(kMaxThreads / 32) * HS * kMaxHot];
    const int hot_unit = (tid >> 5) * HS + (HS == 2 ? ((tid >> 4) & 1) : 0);
    uint64_t* my_hot = s_hot + hot_unit * kMaxHot * F::NA;
    uint32_t* my_hot_rows = s_hot_rows + hot_unit * kMaxHot;
    __shared__ uint32_t s_sp_cursor;
    __shared__ uint32_t s_sp_base[sizeof(U) == 8 ? kSpillChunks : 1];
    if (tid == 0) { s_count = 0; s_abort = 0; s_sp_cursor = 0; }
    if constexpr (sizeof(U) == 8) if (a.sp_keys && !a.spec) {
      for (uint32_t c = tid; c < kSpillChunks; c += T) s_sp_base[c] = 0u;
      f.sp_cursor = &s_sp_cursor; f.sp_base = s_sp_base;
    }
    f.init(tid, T);
    if (a.n_hot) f.hot_init(s_hot, s_hot_rows, tid, T, HS);
    __syncthreads();
    const int64_t step = 2 * (int64_t)T, tile = step * UNR;
    const int64_t n_tiles = a.n / tile;
    bool missed = false;
    U u[2][2 * UNR];
    uint64_t raw[2][2 * UNR][NV];
    auto load_tile = [&](int b, int64_t t) {
      const int64_t r0 = t * tile + 2 * tid;
#pragma unroll
      for (int s = 0; s < UNR; ++s) {
        { U uu[2]; load_u2<KK>(a.key, r0 + s * step, uu); u[b][2 * s] = uu[0]; u[b][2 * s + 1] = uu[1]; }
#pragma unroll
        for (int c = 0; c < NV; ++c) {
          if (!Sig<SIG>::kStatic && c >= n_vals) { raw[b][2 * s][c] = 0; raw[b][2 * s + 1][c] = 0; continue; }
          global_val2(a.plan, c, sig_vw<SIG>(a.plan, c), r0 + s * step, raw[b][2 * s][c], raw[b][2 * s + 1][c]);
        }
      }
    };
    // the tile loop, compiled twice: with and without the heavy-hitter look (runtime row-valid flags
    // and the hot-key scan cost the plain path 5-15 % at low NDV when they were merely branched over)
    auto run_tiles = [&](auto hot_c) {
      constexpr bool HOT = decltype(hot_c)::value;
      auto process_tile = [&](int b) {
        uint32_t miss = 0;
        if constexpr (HOT) {
          bool ab[2 * UNR];
#pragma unroll
          for (int r = 0; r < 2 * UNR; ++r) ab[r] = f.hot_absorb(u[b][r], raw[b][r], my_hot, my_hot_rows, tid & 31);
#pragma unroll
          for (int s = 0; s < UNR; ++s) miss |= f.pair(u[b][2 * s], raw[b][2 * s], !ab[2 * s], u[b][2 * s + 1], raw[b][2 * s + 1], !ab[2 * s + 1], &s_count) << (2 * s);
        } else {
#pragma unroll
          for (int s = 0; s < UNR; ++s) miss |= f.pair(u[b][2 * s], raw[b][2 * s], true, u[b][2 * s + 1], raw[b][2 * s + 1], true, &s_count) << (2 * s);
        }
        f.spill(u[b], raw[b], miss, missed);
      };
      int64_t t = blockIdx.x;
      uint32_t trip = 0;
      if (t < n_tiles) load_tile(0, t);
      while (t < n_tiles) {
        // speculative run: look at the global give-up flag every 16th trip only (an L2 round trip each time)
        if (a.spec) { if (__any_sync(0xffffffffu, missed || ((trip++ & 15u) == 0u && *reinterpret_cast<volatile uint32_t*>(&a.call->abort)))) break; }
        if (t + gridDim.x < n_tiles) load_tile(1, t + gridDim.x);
        process_tile(0);
        t += gridDim.x;
        if (t >= n_tiles) break;
        if (t + gridDim.x < n_tiles) load_tile(0, t + gridDim.x);
        process_tile(1);
        t += gridDim.x;
      }
    };
    if (a.n_hot) run_tiles(std::true_type{}); else run_tiles(std::false_type{});
    if (!(a.spec && __any_sync(0xffffffffu, missed))) {
      // ragged tail: row at a time, spread over the whole grid, warp-uniform trip count
      const int lane = tid & 31;
      for (int64_t i0 = n_tiles * tile + (int64_t)blockIdx.x * T + (tid - lane); i0 < a.n; i0 += (int64_t)gridDim.x * T) {
        const int64_t i = i0 + lane;
        uint64_t rawt[NV];
        U ut = 0;
        if (i < a.n) {
#pragma unroll
          for (int c = 0; c < NV; ++c) rawt[c] = (Sig<SIG>::kStatic || c < n_vals) ? global_val(a.plan, c, sig_vw<SIG>(a.plan, c), i) : 0ull;
          ut = load_u<KK>(a.key, i);
        }
        const uint32_t miss = f.pair(ut, rawt, i < a.n, ut, rawt, false, &s_count);
        if (__any_sync(0xffffffffu, miss != 0)) { if (a.spec) missed = missed || miss != 0; else if (miss) f.back_row(ut, rawt); }
        __syncwarp();
      }
    }
    f.drain_queue();
    if (a.spec) {
      if (missed) { atomicOr(&a.call->abort, 1u); atomicOr(&s_abort, 1u); }
      __syncthreads();
      if (s_abort || *reinterpret_cast<volatile uint32_t*>(&a.call->abort)) return;   // result is discarded
    } else {
      __syncthreads();
    }
    f.spill_pad(tid, T);
    f.flush_merge(tid, T);
    if (a.n_hot) f.hot_flush(s_hot, s_hot_rows, tid, T, HS);
  } else {
    // ---- partition mode: work items blockIdx.x, + gridDim.x, ...; an item is a whole partition
    // (this CTA then owns its keys and emits them) or a slice of a hot one (merged through the
    // global table like the whole-input mode) ----
    const unsigned long long n_items = a.item_off[a.n_parts];
    for (unsigned long long it = blockIdx.x; it < n_items; it += gridDim.x) {
      // the partition of item `it`: one broadcast load from the map written by part_items_kernel
      const int p = (int)a.item_part[it];
      const unsigned long long n_chunks = a.item_off[p + 1] - a.item_off[p], ci = it - a.item_off[p];
      const int64_t P0 = (int64_t)a.part_off[p], P1 = (int64_t)a.part_off[p + 1];
      const int64_t per = (P1 - P0 + (int64_t)n_chunks - 1) / (int64_t)n_chunks;
      const int64_t r0 = P0 + (int64_t)ci * per, r1 = r0 + per < P1 ? r0 + per : P1;
      const bool exclusive = n_chunks == 1;
      // a table no larger than the partition needs: 2 slots per row is always enough
      const uint64_t want = 2ull * (uint64_t)(r1 - r0) + 64;
      const uint32_t Sn = (uint32_t)(want < a.slots ? want : a.slots) & ~7u;   // whole buckets
      F f(a, smem, Sn);
      f.s_spill = &s_spilled;
      __syncthreads();                       // the previous partition's emit is over
      if (tid == 0) { s_count = 0; s_spilled = 0; }
      f.init(tid, T);
      __syncthreads();
      bool missed = false;
      // chunks of UNR * T rows, bounds-checked per row; the next chunk loads while this one is processed
      constexpr int UNR = NV >= 4 ? 1 : 2;
      U u[2][UNR];
      uint64_t raw[2][UNR][NV];
      const int64_t chunk = (int64_t)UNR * T;
      auto load_chunk = [&](int b, int64_t c0) {
#pragma unroll
        for (int s = 0; s < UNR; ++s) {
          const int64_t i = c0 + (int64_t)s * T + tid;
          if (i < r1) {
            u[b][s] = load_u<KK>(a.key, i);
#pragma unroll
            for (int c = 0; c < NV; ++c) raw[b][s][c] = (Sig<SIG>::kStatic || c < n_vals) ? global_val(a.plan, c, sig_vw<SIG>(a.plan, c), i) : 0ull;
          }
        }
      };
      auto process_chunk = [&](int b, int64_t c0) {
        uint32_t miss = 0;
#pragma unroll
        for (int s = 0; s < UNR; s += 2) {
          bool v0 = c0 + (int64_t)s * T + tid < r1, v1 = (s + 1 < UNR) && (c0 + (int64_t)(s + 1) * T + tid < r1);
          if constexpr (sizeof(U) == 8) if (a.skip_empty) {      // padding rows of a spill buffer
            v0 = v0 && u[b][s] != kEmpty64;
            v1 = v1 && u[b][s + 1 < UNR ? s + 1 : s] != kEmpty64;
          }
          miss |= f.pair(v0 ? u[b][s] : (U)0, raw[b][s], v0, v1 ? u[b][s + 1 < UNR ? s + 1 : s] : (U)0, raw[b][s + 1 < UNR ? s + 1 : s], v1, &s_count) << s;
        }
        f.spill(u[b], raw[b], miss, missed);
      };
      int64_t c0 = r0;
      load_chunk(0, c0);
      while (c0 < r1) {
        if (c0 + chunk < r1) load_chunk(1, c0 + chunk);
        process_chunk(0, c0);
        c0 += chunk;
        if (c0 >= r1) break;
        if (c0 + chunk < r1) load_chunk(0, c0 + chunk);
        process_chunk(1, c0);
        c0 += chunk;
      }
      __syncthreads();
      // emit only what this CTA owns exclusively: a whole partition none of whose rows was sent to
      // the global table (otherwise a key could be emitted here AND by the compaction pass)
      if (exclusive && s_spilled == 0u && !a.force_merge) f.flush_emit(tid, T, s_count, &s_base, s_wtot);
      else f.flush_merge(tid, T);
    }
  }
}


template <int KK, int SIG, int BK>
int launch_one(const HashAggLaunch& L, cudaStream_t s) {
  auto kern = L.ring ? hash_agg_kernel<KK, SIG, BK> : hash_agg_ldg_kernel<KK, SIG, BK>;
  HashAggArgs a;
  a.key = L.key; a.plan = L.plan; a.n = L.n; a.part_off = L.part_off; a.item_off = L.item_off; a.item_part = L.item_part; a.n_parts = L.n_parts;
  a.slots = L.slots; a.limit = L.limit; a.spec = L.spec; a.max_probes = L.max_probes > 0 ? L.max_probes : 16;
  a.n_hot = (L.spec || IsPre<KK>::v) ? 0 : std::min(L.n_hot, kMaxHot);
  for (int i = 0; i < kMaxHot; ++i) a.hot[i] = i < a.n_hot ? L.hot[i] : 0ull;
  a.table = L.table; a.cap = L.cap; a.stride = L.stride; a.call = L.call;
  for (int k = 0; k < kMaxKeyCols; ++k) a.out_keys[k] = L.out_keys[k];
  for (int j = 0; j < kMaxAggs; ++j) a.out_aggs[j] = static_cast<uint64_t*>(L.out_aggs[j]);
  a.n_out = L.n_out_aggs; a.out_capacity = L.out_capacity;
  // dynamic shared memory: [ring: stages x stage_bytes][heavy-hitter cells][table]
  HashAggSmem lay = hash_agg_smem_layout(L.key, L.plan, L.key_kind, L.threads, L.hot_reserved && !IsPre<KK>::v, L.stages);
  if (!L.ring) { lay.table_off = 0; lay.hot_off = 0; }     // no ring: the table is all of the dynamic shared memory
  for (int k = 0; k < kMaxKeyCols; ++k) { a.koff[k] = lay.koff[k]; a.kw[k] = lay.kw[k]; }
  for (int c = 0; c < kMaxVals; ++c) { a.voff[c] = lay.voff[c]; a.vw[c] = lay.vw[c]; }
  a.stages = lay.stages; a.stage_bytes = lay.stage_bytes; a.n_src = lay.n_src;
  { const char* e = std::getenv("EIGER_RING_HINT"); a.ring_hint = e ? std::atoi(e) : 1; } a.hot_off = lay.hot_off; a.table_off = lay.table_off;
  a.queue_off = 0;
  a.sp_keys = (L.ring || IsPre<KK>::v) ? nullptr : L.spill_keys; a.sp_cap_chunks = L.spill_cap_chunks; a.sp_lg = L.spill_lg;
  for (int c = 0; c < kMaxVals; ++c) a.sp_vals[c] = L.spill_vals[c];
  a.skip_empty = L.skip_empty; a.force_merge = L.force_merge;
  size_t smem = (size_t)lay.table_off + L.table_smem_bytes;
  if (!L.ring && !IsPre<KK>::v && L.queue_bytes) { a.queue_off = (uint32_t)((smem + 127) & ~(size_t)127); smem = a.queue_off + L.queue_bytes; }
  if (smem > 32 * 1024) EIGER_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<L.blocks, L.threads, smem, s>>>(a);
  count_launch();
  EIGER_CUDA(cudaGetLastError());
  return EIGER_OK;
}

template <int KK, int BK>
int launch_sig_bk(const HashAggLaunch& L, cudaStream_t s) {
  switch (L.sig) {
    case SIG_GENERIC: return launch_one<KK, SIG_GENERIC, BK>(L, s);
    case SIG_SC: return launch_one<KK, SIG_SC, BK>(L, s);
    case SIG_A4I: return launch_one<KK, SIG_A4I, BK>(L, s);
    case SIG_A4F: return launch_one<KK, SIG_A4F, BK>(L, s);
    case SIG_S4C: return launch_one<KK, SIG_S4C, BK>(L, s);
    case SIG_SC32: return launch_one<KK, SIG_SC32, BK>(L, s);
    case SIG_G1: return launch_one<KK, SIG_G1, BK>(L, s);
    default: return EIGER_ERR_ARG;
  }
}
template <int KK>
int launch_sig(const HashAggLaunch& L, cudaStream_t s) {
  using U = typename KeyTraits<KK>::U;
  if constexpr (sizeof(U) == 4) {
    // the narrow-bucket kernels exist for the SUM + COUNT and the generic signature only (compile time)
    if (L.bucket_keys == 2 && L.sig == SIG_SC) return launch_one<KK, SIG_SC, 2>(L, s);
    if (L.bucket_keys == 2 && L.sig == SIG_SC32) return launch_one<KK, SIG_SC32, 2>(L, s);
    if (L.bucket_keys == 2 && L.sig == SIG_GENERIC) return launch_one<KK, SIG_GENERIC, 2>(L, s);
    if (L.bucket_keys == 2 && L.sig == SIG_G1) return launch_one<KK, SIG_G1, 2>(L, s);
  }
  return launch_sig_bk<KK, 16 / (int)sizeof(U)>(L, s);
}

}  // namespace

// one translation unit per group of key kinds
int launch_hash_agg_i32(const HashAggLaunch& L, cudaStream_t s);   // KK_I32
int launch_hash_agg_i64(const HashAggLaunch& L, cudaStream_t s);   // KK_I64, KK_GEN
int launch_hash_agg_pre(const HashAggLaunch& L, cudaStream_t s);   // KK_U32PRE, KK_U64PRE (partition mode)

}  // namespace eiger
