// gq_skeleton.cuh — hand-written sm_100a device code of the fused scan kernel (one translation unit per plan shape).
//
// The plan compiler (gq_codegen.cpp) emits a small prelude of #defines + two row functions (gq_pass / gq_body) and
// splices them at the //@@ROW_FUNCTIONS@@ marker below; everything else — the TMA bulk-copy pipeline, the hash-table
// primitives, the shared-memory low-cardinality aggregation, the reductions — is this file, compiled as-is by NVRTC
// (no headers needed) or by nvcc (build-time check). This is the fused FilterProject -> HashProbe* -> consumer step
// of SURVEY.md §8(a1-a8): predicate and projection are evaluated in registers inside the consuming kernel
// ("fused operations, fewer memory writes"), no selection vector is materialised.
//
// Kernel shape (B200: 148 SMs, 227 KB smem/CTA, TMA):
//   grid  = one persistent CTA per SM; tiles of GQ_TILE rows are dealt round-robin (tile = blockIdx.x + i*gridDim.x)
//   block = GQ_NT consumer threads + 1 producer warp. The producer's lane 0 issues one 1-D bulk copy
//           (cp.async.bulk.shared::cluster.global.mbarrier) per referenced column per tile into a GQ_STAGES-deep ring of
//           shared-memory stages; full/empty mbarriers hand stages to the consumers and back. Consumers read row
//           (tid + j*GQ_NT) of every column from shared memory — consecutive lanes, consecutive elements — so columns
//           of different widths (i8/i32/i64) need no register shuffling and every global access is a full-line burst.
//   tail  = the < GQ_TILE leftover rows are read straight from global memory by one CTA (same row functions).
//
// Prelude macros expected: GQ_NCOL, GQ_NT, GQ_R, GQ_STAGES, GQ_STAGE_BYTES, GQ_COL_OFF(c), GQ_COL_BYTES(c) (bytes per
// element), GQ_CONSUMER, GQ_NAGG, GQ_AGG_OP(a), GQ_LC_CAP, GQ_TARGET_SW, GQ_NDEP, GQ_EVICT_FIRST.

typedef unsigned long long u64;
typedef long long i64;
typedef unsigned int u32;

#define GQ_EMPTY 0x8000000000000000ULL   // empty-slot marker = INT64_MIN; a user key equal to it lives in the side area
#define GQ_TILE (GQ_NT * GQ_R)
#define GQ_NWARP (GQ_NT / 32)
#define GQ_MAXCOL 16
#define GQ_MAXK 48
#define GQ_MAXOUT 12
#define GQ_SIDE_SLOTS 64

#define GQ_C_GLOBAL 0
#define GQ_C_LOWCARD 1
#define GQ_C_HIGHCARD 2
#define GQ_C_BUILD 3
#define GQ_C_MATERIALISE 4

#define GQ_E_CAPACITY 3
#define GQ_E_DUPLICATE 6

#define GQ_OP_SUM 0
#define GQ_OP_MIN 1
#define GQ_OP_MAX 2
#define GQ_OP_COUNT 3

// Device view of a hash table (join table or group-by table). Layout must match gq_internal.h:GqTableDev.
struct GqTableDev {
  u64* slots;        // capacity * slot_words words; word 0 of a slot = key (GQ_EMPTY when free)
  u64 mask;          // capacity - 1 (capacity is a power of two)
  i64* header;       // [0] rows inserted, [1] entries in the side area, [2..] reserved
  u64* side;         // GQ_SIDE_SLOTS slots for rows whose key == GQ_EMPTY (join) / 1 slot (group-by)
  int shift;         // 64 - log2(capacity)
  int slot_words;
  u32 flags;
  u32 pad;
};

// Kernel parameters: one fixed layout for every generated kernel. Must match gq_internal.h:GqParams.
struct GqParams {
  const void* col[GQ_MAXCOL];   // referenced input columns, compacted in plan order
  i64 nrows;
  i64 k[GQ_MAXK];               // predicate bounds and expression literals (kernel is shape-specialised, not value-)
  GqTableDev probe[4];
  GqTableDev target;            // BUILD: table being built; LOWCARD/HIGHCARD: group-by table
  i64* acc;                     // GLOBAL: GQ_NAGG accumulators in device memory (pre-set to identities)
  i64* out[GQ_MAXOUT];          // MATERIALISE: output columns
  i64 out_capacity;
  i64* out_count;
  const i64* hot;               // HIGHCARD: hot list of this batch (hot[0] = count, hot[1..] = keys) or null
  int* err;                     // sticky device error
  int pad;
};

// ---------------------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ u32 gq_smem_addr(const void* p) { return (u32)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void gq_mbar_init(u64* bar, u32 count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(gq_smem_addr(bar)), "r"(count));
}
__device__ __forceinline__ void gq_mbar_expect_tx(u64* bar, u32 bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(gq_smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void gq_mbar_arrive(u64* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(gq_smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void gq_mbar_wait(u64* bar, u32 parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "GQ_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra GQ_DONE_%=;\n"
      "bra GQ_WAIT_%=;\n"
      "GQ_DONE_%=:\n"
      "}\n" ::"r"(gq_smem_addr(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ u64 gq_policy_evict_first() {
  u64 pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
// 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier (TMA engine; SASS: UBLKCP).
__device__ __forceinline__ void gq_bulk_g2s(void* dst, const void* src, u32 bytes, u64* bar, u64 pol) {
#if GQ_EVICT_FIRST
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::
          "r"(gq_smem_addr(dst)), "l"(src), "r"(bytes), "r"(gq_smem_addr(bar)), "l"(pol) : "memory");
#else
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                   "r"(gq_smem_addr(dst)), "l"(src), "r"(bytes), "r"(gq_smem_addr(bar)) : "memory");
#endif
}
__device__ __forceinline__ void gq_consumer_barrier() {   // named barrier 1: the GQ_NT consumer threads only
  asm volatile("bar.sync 1, %0;" ::"n"(GQ_NT) : "memory");
}
__device__ __forceinline__ void gq_ld128(const u64* p, u64& a, u64& b) {   // read-only 128-bit slot load
  asm volatile("ld.global.nc.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p));
}
__device__ __forceinline__ u64 gq_ld_relaxed(const u64* p) {               // sees concurrent CAS results (L2)
  u64 v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}

// ---------------------------------------------------------------------------------------------- wrapping int64
__device__ __forceinline__ i64 gq_add(i64 a, i64 b) { return (i64)((u64)a + (u64)b); }
__device__ __forceinline__ i64 gq_sub(i64 a, i64 b) { return (i64)((u64)a - (u64)b); }
__device__ __forceinline__ i64 gq_mul(i64 a, i64 b) { return (i64)((u64)a * (u64)b); }
__device__ __forceinline__ i64 gq_min(i64 a, i64 b) { return a < b ? a : b; }
__device__ __forceinline__ i64 gq_max(i64 a, i64 b) { return a > b ? a : b; }

__device__ __forceinline__ void gq_set_err(int* err, int code) { atomicCAS(err, 0, code); }

// ---------------------------------------------------------------------------------------------- hash tables
// Open addressing, linear probing, 64-bit CAS on the key word (north_star). Fibonacci hashing of the folded key.
__device__ __forceinline__ u64 gq_hash(i64 key, int shift) {
  u64 x = (u64)key;
  x ^= x >> 32;
  return (x * 0x9E3779B97F4A7C15ULL) >> shift;
}

// HashBuild insert: duplicates are kept as separate slots (multiset, S3) unless `unique` is asserted,
// in which case an equal key sets the sticky GQ_E_DUPLICATE. Payload words are written by the CAS winner; probes only
// run after the building kernel has finished (pipeline boundary), so no reader can see them half-written.
template <int SW, int NPAY>
__device__ __forceinline__ bool gq_ht_insert(const GqTableDev& T, i64 key, const i64* pay, bool unique, int* err) {
  if ((u64)key == GQ_EMPTY) {                     // reserved bit pattern: side area (S14)
    i64 idx = (i64)atomicAdd((u64*)&T.header[1], 1ULL);
    if (unique && idx > 0) { gq_set_err(err, GQ_E_DUPLICATE); return false; }
    if (idx >= GQ_SIDE_SLOTS) { gq_set_err(err, GQ_E_CAPACITY); return false; }
    u64* s = T.side + idx * SW;
    s[0] = (u64)key;
#pragma unroll
    for (int p = 0; p < NPAY; ++p) s[1 + p] = (u64)pay[p];
    return true;
  }
  u64 i = gq_hash(key, T.shift);
  for (u64 n = 0; n <= T.mask; ++n, i = (i + 1) & T.mask) {
    u64* s = T.slots + i * SW;
    u64 prev = atomicCAS(s, GQ_EMPTY, (u64)key);
    if (prev == GQ_EMPTY) {
#pragma unroll
      for (int p = 0; p < NPAY; ++p) s[1 + p] = (u64)pay[p];
      return true;
    }
    if (unique && prev == (u64)key) { gq_set_err(err, GQ_E_DUPLICATE); return false; }
  }
  gq_set_err(err, GQ_E_CAPACITY);
  return false;
}

// HashAggregation insert-or-update: returns the slot of `key`, claiming a free one by CAS if the key is
// new. Aggregate words already hold their identities (table-init kernel), so there is no claimed-but-uninitialised
// window. *won tells the caller it created the group (it then stores the dependent key columns).
template <int SW>
__device__ __forceinline__ u64* gq_ht_upsert(const GqTableDev& T, i64 key, bool* won, int* err) {
  *won = false;
  if ((u64)key == GQ_EMPTY) {
    i64 prev = (i64)atomicExch((u64*)&T.header[1], 1ULL);
    *won = (prev == 0);
    return T.side;
  }
  u64 i = gq_hash(key, T.shift);
  for (u64 n = 0; n <= T.mask; ++n, i = (i + 1) & T.mask) {
    u64* s = T.slots + i * SW;
    u64 k = gq_ld_relaxed(s);
    if (k == (u64)key) return s;
    if (k == GQ_EMPTY) {
      u64 prev = atomicCAS(s, GQ_EMPTY, (u64)key);
      if (prev == GQ_EMPTY) { *won = true; return s; }
      if (prev == (u64)key) return s;
    }
  }
  gq_set_err(err, GQ_E_CAPACITY);
  return nullptr;
}

// Variants that continue from a first slot access already issued by the caller (linear mode: the first CAS / key read
// of all GQ_R rows of a thread are in flight together before any of them is consumed).
template <int SW, int NPAY>
__device__ __forceinline__ bool gq_ht_insert_pre(const GqTableDev& T, i64 key, const i64* pay, bool unique, u64 i,
                                                 u64 prev, int* err) {
  if ((u64)key == GQ_EMPTY) return gq_ht_insert<SW, NPAY>(T, key, pay, unique, err);
  for (u64 n = 0; n <= T.mask; ++n) {
    u64* s = T.slots + i * SW;
    if (prev == GQ_EMPTY) {
#pragma unroll
      for (int p = 0; p < NPAY; ++p) s[1 + p] = (u64)pay[p];
      return true;
    }
    if (unique && prev == (u64)key) { gq_set_err(err, GQ_E_DUPLICATE); return false; }
    i = (i + 1) & T.mask;
    prev = atomicCAS(T.slots + i * SW, GQ_EMPTY, (u64)key);
  }
  gq_set_err(err, GQ_E_CAPACITY);
  return false;
}
template <int SW>
__device__ __forceinline__ u64* gq_ht_upsert_pre(const GqTableDev& T, i64 key, u64 i, u64 k, bool* won, int* err) {
  if ((u64)key == GQ_EMPTY) return gq_ht_upsert<SW>(T, key, won, err);
  *won = false;
  for (u64 n = 0; n <= T.mask; ++n) {
    u64* s = T.slots + i * SW;
    if (k == (u64)key) return s;
    if (k == GQ_EMPTY) {
      u64 prev = atomicCAS(s, GQ_EMPTY, (u64)key);
      if (prev == GQ_EMPTY) { *won = true; return s; }
      if (prev == (u64)key) return s;
    }
    i = (i + 1) & T.mask;
    k = gq_ld_relaxed(T.slots + i * SW);
  }
  gq_set_err(err, GQ_E_CAPACITY);
  return nullptr;
}

// Aggregate update at L2 (RED.ADD / RED.MIN / RED.MAX .64 — results are not read back).
__device__ __forceinline__ void gq_red(const int OP, u64* p, i64 v) {
  if (OP == GQ_OP_SUM || OP == GQ_OP_COUNT) atomicAdd(p, (u64)v);
  else if (OP == GQ_OP_MIN) atomicMin((i64*)p, v);
  else atomicMax((i64*)p, v);
}
__device__ __forceinline__ i64 gq_combine(const int OP, i64 a, i64 b) {
  if (OP == GQ_OP_SUM || OP == GQ_OP_COUNT) return gq_add(a, b);
  if (OP == GQ_OP_MIN) return gq_min(a, b);
  return gq_max(a, b);
}
__device__ __forceinline__ i64 gq_identity(const int OP) {
  if (OP == GQ_OP_MIN) return (i64)0x7FFFFFFFFFFFFFFFLL;
  if (OP == GQ_OP_MAX) return (i64)0x8000000000000000ULL;
  return 0;
}
__device__ __forceinline__ i64 gq_warp_reduce(const int OP, i64 v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = gq_combine(OP, v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// ---------------------------------------------------------------------------------------------- row sources
// A tile staged in shared memory by the producer, or the ragged tail read from global memory.
struct GqSrcSmem {
  const unsigned char* stage;
  int t;   // consumer thread id
  template <class T> __device__ __forceinline__ i64 ld(int /*c*/, int off, int j) const {
    return (i64)((const T*)(stage + off))[t + j * GQ_NT];
  }
};
struct GqSrcGlobal {
  const GqParams* P;
  i64 row0;   // first row of the tail
  int t;
  template <class T> __device__ __forceinline__ i64 ld(int c, int /*off*/, int j) const {
    return (i64)((const T*)P->col[c])[row0 + t + (i64)j * GQ_NT];
  }
};

// ---------------------------------------------------------------------------------------------- consumer state
// Per-thread consumer context. Only the members the selected GQ_CONSUMER uses survive dead-code elimination.
struct GqCtx {
  i64 acc[GQ_NAGG > 0 ? GQ_NAGG : 1];   // GLOBAL: register accumulators
  i64* lc_keys;                         // LOWCARD: shared key table [GQ_LC_CAP + 1]
  i64* lc_acc;                          // LOWCARD: shared accumulators [(GQ_LC_CAP+1) * GQ_NAGG * GQ_NT], lane-private
  int* lc_side_used;
  i64 ninserted;                        // BUILD: rows inserted by this thread
  i64* hot_keys;                        // HIGHCARD + GQ_HOT: shared set of this batch's hot keys [GQ_HOT_POS]
  u64* hot_acc;                         //   CTA-shared accumulators [GQ_HOT_POS][GQ_NAGG]
  int* hot_touched;                     //   entry received at least one row
  int nhot;
  int t;
};

// Low-cardinality group-by: the CTA keeps a tiny open-addressing key table in shared memory (CAS only
// the first time a key is seen); each consumer thread owns a PRIVATE accumulator cell per (group, aggregate), laid
// out [group][agg][thread] so a warp's 32 cells are 32 consecutive 8-byte words: plain conflict-free LDS/add/STS,
// no atomics, no shuffles on the per-row path. Cells are reduced over threads once, at the end, and flushed into the
// global group-by table (the Partial -> Final merge of PAPER.md:154 inside one kernel).
__device__ __forceinline__ int gq_lc_slot(GqCtx& cx, i64 key, int* err) {
  if ((u64)key == GQ_EMPTY) { *cx.lc_side_used = 1; return GQ_LC_CAP; }
  u32 i = (u32)gq_hash(key, 64 - 16) & (GQ_LC_CAP - 1);
  for (int n = 0; n < GQ_LC_CAP; ++n, i = (i + 1) & (GQ_LC_CAP - 1)) {
    i64 k = ((volatile i64*)cx.lc_keys)[i];
    if (k == key) return (int)i;
    if ((u64)k == GQ_EMPTY) {
      u64 prev = atomicCAS((u64*)&cx.lc_keys[i], GQ_EMPTY, (u64)key);
      if (prev == GQ_EMPTY || prev == (u64)key) return (int)i;
    }
  }
  gq_set_err(err, GQ_E_CAPACITY);   // more distinct keys than max_groups
  return -1;
}
__device__ __forceinline__ void gq_lc_update(const int OP, GqCtx& cx, int slot, int a, i64 v) {
  i64* cell = cx.lc_acc + ((slot * GQ_NAGG + a) * GQ_NT + cx.t);
  *cell = gq_combine(OP, *cell, v);
}

// Hot keys of a skewed high-cardinality group-by: rows whose key is in the batch's hot list
// are accumulated in CTA-shared memory and flushed to the global table once per CTA, instead of hammering one L2
// address with hundreds of millions of atomics. 64-bit shared atomics are CAS loops on sm_100 (ATOMS.CAST.SPIN), so
// SUM/COUNT use two native 32-bit ATOMS.ADD with an explicit carry; MIN/MAX compare first and CAS only to improve.
#define GQ_HOT_POS 512
#define GQ_HOT_MAX 256
__device__ __forceinline__ int gq_hot_find(const GqCtx& cx, i64 key) {
  u32 i = (u32)gq_hash(key, 64 - 16) & (GQ_HOT_POS - 1);
  for (int n = 0; n < GQ_HOT_POS; ++n, i = (i + 1) & (GQ_HOT_POS - 1)) {
    const i64 k = cx.hot_keys[i];
    if (k == key) return (int)i;
    if ((u64)k == GQ_EMPTY) return -1;
  }
  return -1;
}
__device__ __forceinline__ void gq_hot_update(const int OP, GqCtx& cx, int pos, int a, i64 v) {
  u64* cell = cx.hot_acc + pos * GQ_NAGG + a;
  if (OP == GQ_OP_SUM || OP == GQ_OP_COUNT) {
    u32* w = (u32*)cell;
    const u32 lo = (u32)(u64)v, hi = (u32)((u64)v >> 32);
    const u32 old = atomicAdd(w, lo);
    const u32 up = hi + ((u32)(old + lo) < old ? 1u : 0u);   // carry out of the low word belongs to THIS addition
    if (up) atomicAdd(w + 1, up);
  } else {
    i64 cur = *(volatile i64*)cell;
    while (OP == GQ_OP_MIN ? v < cur : v > cur) {
      const i64 prev = (i64)atomicCAS(cell, (u64)cur, (u64)v);
      if (prev == cur) break;
      cur = prev;
    }
  }
}

// MATERIALISE: ballot/popc compaction — the lanes that reach this point together reserve a contiguous
// output range with ONE atomic (warp-aggregated), then write their rows side by side.
__device__ __forceinline__ i64 gq_reserve_row(const GqParams& P) {
  u32 m = __activemask();
  int lane = threadIdx.x & 31;
  int leader = __ffs(m) - 1;
  i64 base = 0;
  if (lane == leader) base = (i64)atomicAdd((u64*)P.out_count, (u64)__popc(m));
  base = __shfl_sync(m, base, leader);
  i64 idx = base + __popc(m & ((1u << lane) - 1u));
  if (idx >= P.out_capacity) { gq_set_err(P.err, GQ_E_CAPACITY); return -1; }
  return idx;
}

//@@ROW_FUNCTIONS@@
