// gq_skeleton.cuh — hand-written sm_100a device code of the fused scan kernel (one translation unit per plan shape).
//
// The plan compiler (gq_codegen.cpp) emits a small prelude of #defines + the row code (gq_tile: the GQ_R rows of a
// thread step by step through filter, probes, projection and consumer; or gq_pass / gq_body when a probed table may
// hold duplicate keys) and splices it at the //@@ROW_FUNCTIONS@@ marker below; everything else — the TMA bulk-copy pipeline, the hash-table
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
// element), GQ_CONSUMER, GQ_NAGG, GQ_AGG_OP(a), GQ_LC_G (group cells), GQ_LC_KT (key-table slots), GQ_LC_KEY32,
// GQ_LC_KEY_BITS, GQ_TARGET_SW, GQ_NDEP, GQ_CHECK_DEP, GQ_HOT, GQ_FUSED_FINAL, GQ_DIRECT_AW.

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
#define GQ_GTAB_SLOTS 64

#define GQ_C_GLOBAL 0
#define GQ_C_LOWCARD 1
#define GQ_C_HIGHCARD 2
#define GQ_C_BUILD 3
#define GQ_C_MATERIALISE 4
#define GQ_C_DIRECT 5
#define GQ_C_PARTITION 6
#define GQ_C_SCATTER 7

#define GQ_E_CAPACITY 3
#define GQ_E_DUPLICATE 6
#define GQ_E_DEPENDENT 8
#define GQ_E_KEYRANGE 9

#define GQ_OP_SUM 0
#define GQ_OP_MIN 1
#define GQ_OP_MAX 2
#define GQ_OP_COUNT 3

// Device view of a hash table (join table or group-by table). Layout must match gq_internal.h:GqTableDev.
struct GqTableDev {
  u64* slots;        // capacity * slot_words words; word 0 of a slot = key (GQ_EMPTY when free)
  u64 mask;          // capacity - 1 (capacity: any multiple of 4; a power of two for group-by tables)
  i64* header;       // [0] rows inserted, [1] entries in the side area, [2..] reserved
  u64* side;         // GQ_SIDE_SLOTS slots for rows whose key == GQ_EMPTY (join) / 1 slot (group-by)
  int shift;         // 64 - log2(capacity)
  int slot_words;
  u32 flags;
  u32 bshift;        // log2(slots per 32-byte bucket): probe sequences start on a bucket boundary (join tables)
  i64 base;          // direct-address table (GQ_F_DENSE_KEYS): key_min; then slots = payload rows [range][NPAY],
                     // side = membership entries {bits, rank prefix} per 32 keys, mask = range size - 1
};

// Outputs of the finaliser fused into the scan kernel (gq_pipeline over one batch, LOWCARD / GLOBAL consumers): every
// CTA folds its partial groups into a small context-owned table (LOWCARD: find-or-claim by key, then RED) or writes its
// partial aggregates to `part` (GLOBAL), takes a ticket, and the last CTA emits the dense result (keys, aggregates, AVG,
// group count) and leaves table and ticket zeroed — no separate init / finalise launches. Must match gq_internal.h.
struct GqFinal {
  i64* part;                    // GLOBAL: [grid][NAGG] per-CTA partial aggregates
  u32* ticket;                  // context-owned counter, zero between kernels (reset by the last CTA)
  u64* gtab;                    // LOWCARD: context-owned merge table, all states zero between kernels: word 0 = groups
                                //   claimed, then from word 32 GQ_GTAB_SLOTS slots of 16 words {state, key, aggregates}
  void* out_key[2];
  i64* out_agg[8];
  double* out_avg[8];
  int avg_sum[8], avg_cnt[8];
  int navg, nkeys;
  int key_bits[2], key_dtype[2];
  i64 out_capacity;
  i64* out_n;
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
  const i64* hot;               // HIGHCARD: hot list of this batch (hot[0] = count, hot[32..] = keys) or null
  int* err;                     // sticky device error
  int pad;
  u64* dacc;                    // DIRECT: aggregate words indexed by the slot of the probed unique table
  u64* part;                    // PARTITION: record buffers, [npart][pcap] records of GQ_PART_RW words
  u64* pcur;                    // PARTITION: per-partition append cursors
  i64 pcap;                     // PARTITION: records per partition
  i64 pshift;                   // PARTITION: partition = first slot of the key in the target table >> pshift
  i64 npart;                    // number of partitions
  u32* sc_info;                 // SCATTER: per chunk (partition << 8) | records used
  u32* sc_count;                // SCATTER: chunks per partition (RED)
  u32* sc_ncta;                 // SCATTER: chunks allocated by every CTA
  i64 sc_slab;                  // SCATTER: chunk ids of CTA b are [b * sc_slab, (b + 1) * sc_slab)
  GqFinal fin;                  // GQ_FUSED_FINAL: outputs of the in-kernel finaliser
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
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::
          "r"(gq_smem_addr(dst)), "l"(src), "r"(bytes), "r"(gq_smem_addr(bar)), "l"(pol) : "memory");
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

__device__ __forceinline__ u64 gq_ld_acquire(const u64* p) {
  u64 v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void gq_st_release(u64* p, u64 v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
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
// Join tables are read one 32-byte sector at a time (LDG.256): a "bucket" holds 4 key-only slots, 2 key+payload
// slots or 1 wide slot, and every probe sequence starts on a bucket boundary (T.bshift), so the first fetch examines
// a whole bucket. Slots of a bucket fill in order (an inserter only skips a slot it has seen occupied), hence a
// lookup may stop at the first EMPTY slot.
__device__ __forceinline__ u64 gq_hash(i64 key, int shift) {
  u64 x = (u64)key;
  x ^= x >> 32;
  return (x * 0x9E3779B97F4A7C15ULL) >> shift;
}
// First slot of a key's probe sequence: the top bits of the hash scaled to the capacity (multiply-shift range
// reduction — the capacity need not be a power of two, so a table is sized to its row-count hint, not the next power
// of two above it), aligned down to a bucket boundary.
__device__ __forceinline__ u64 gq_slot0(const GqTableDev& T, i64 key) {
  return (__umul64hi(gq_hash(key, 0), T.mask + 1) >> T.bshift) << T.bshift;
}
__device__ __forceinline__ u64 gq_next(const GqTableDev& T, u64 i, u64 step) {   // capacity is a multiple of step
  i += step;
  return i > T.mask ? 0 : i;
}
__device__ __forceinline__ void gq_ld256(const u64* p, u64 (&w)[4]) {   // one 32-byte sector, read-only path
  asm volatile("ld.global.nc.v4.u64 {%0, %1, %2, %3}, [%4];" : "=l"(w[0]), "=l"(w[1]), "=l"(w[2]), "=l"(w[3]) : "l"(p));
}
__device__ __forceinline__ void gq_ld256_relaxed(const u64* p, u64 (&w)[4]) {   // sees concurrent CAS results (L2)
  asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(w[0]), "=l"(w[1]) : "l"(p) : "memory");
  asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(w[2]), "=l"(w[3]) : "l"(p + 2) : "memory");
}

template <int NW> __device__ __forceinline__ void gq_ld_bucket(const u64* p, u64 (&w)[NW]) {
  gq_ld256(p, *(u64(*)[4])&w[0]);
  if (NW == 8) gq_ld256(p + 4, *(u64(*)[4])&w[NW - 4]);
}
template <int NW> __device__ __forceinline__ void gq_ld_bucket_relaxed(const u64* p, u64 (&w)[NW]) {
  gq_ld256_relaxed(p, *(u64(*)[4])&w[0]);
  if (NW == 8) gq_ld256_relaxed(p + 4, *(u64(*)[4])&w[NW - 4]);
}

// HashBuild insert of one row: duplicates are kept as separate slots (multiset, S3) unless `unique`
// is asserted, in which case an equal key sets the sticky GQ_E_DUPLICATE. Payload words are written by the CAS
// winner; probes only run after the building kernel has finished (pipeline boundary), so no reader can
// see them half-written.
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
  u64 i = gq_slot0(T, key);
  for (u64 n = 0; n <= T.mask; ++n, i = gq_next(T, i, 1)) {
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

// HashAggregation insert-or-update of one row: returns the slot of `key`, claiming a free one by CAS
// if the key is new. Aggregate words already hold their identities (table-init kernel), so there is no
// claimed-but-uninitialised window. *won tells the caller it created the group.
template <int SW>
__device__ __forceinline__ u64* gq_ht_upsert(const GqTableDev& T, i64 key, bool* won, int* err) {
  *won = false;
  if ((u64)key == GQ_EMPTY) {
    i64 prev = (i64)atomicExch((u64*)&T.header[1], 1ULL);
    *won = (prev == 0);
    return T.side;
  }
  u64 i = gq_slot0(T, key);
  for (u64 n = 0; n <= T.mask; ++n, i = gq_next(T, i, 1)) {
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

// ---- GQ_R rows of a thread at once ("linear mode"): the slot accesses of all rows are issued together and resolved
// in rounds, so a thread keeps up to GQ_R random accesses in flight and a round costs ONE memory latency however many
// rows are still unresolved (memory-level parallelism is what bounds the hash phases, not bandwidth).

// HashProbe of a table with unique keys. live[j] is cleared for rows without a match; idx[j] receives
// the matching slot index (capacity = the side entry), pay[j][] its payload words.
template <int SW, int NPAY>
__device__ __forceinline__ void gq_probe_rows(const GqTableDev& T, const i64 (&key)[GQ_R], bool (&live)[GQ_R],
                                              u64 (&idx)[GQ_R], i64 (&pay)[GQ_R][NPAY > 0 ? NPAY : 1]) {
  constexpr int B = SW == 1 ? 4 : SW == 2 ? 4 : 1;   // slots per bucket: 32 bytes, or 64 bytes for key+payload slots
  constexpr int NW = B * SW;                         // words per bucket fetch (4 or 8: one or two LDG.256)
  u64 w[GQ_R][NW];
  u32 pend = 0;
#pragma unroll
  for (int j = 0; j < GQ_R; ++j) {
    idx[j] = 0;
    if (live[j]) {
      if ((u64)key[j] == GQ_EMPTY) {   // reserved key pattern: unique table => at most one side entry (S14)
        if (T.header[1] > 0) {
#pragma unroll
          for (int p = 0; p < NPAY; ++p) pay[j][p] = (i64)T.side[1 + p];
          idx[j] = T.mask + 1;
        } else live[j] = false;
      } else {
        idx[j] = gq_slot0(T, key[j]);
        gq_ld_bucket<NW>(T.slots + idx[j] * SW, w[j]);
        pend |= 1u << j;
      }
    }
  }
  for (u64 round = 0; pend != 0; ++round) {
#pragma unroll
    for (int j = 0; j < GQ_R; ++j) {
      if (pend & (1u << j)) {
        // slots of a bucket fill in order, so a match can never sit behind an EMPTY slot: look for the key in all B
        // slots first, and only without a match ask whether the bucket has a free slot (= the key is absent)
        int hb = -1;
        bool emp = false;
#pragma unroll
        for (int b = 0; b < B; ++b) {
          const u64 kw = w[j][b * SW];
          if (kw == (u64)key[j]) hb = b;
          emp = emp || kw == GQ_EMPTY;
        }
        bool done = true;
        if (hb >= 0) {
          idx[j] += hb;
#pragma unroll
          for (int b = 0; b < B; ++b)
            if (b == hb) {
#pragma unroll
              for (int p = 0; p < NPAY; ++p) pay[j][p] = (i64)w[j][b * SW + 1 + p];
            }
        } else if (emp || round * B > T.mask) live[j] = false;   // free slot seen, or a full table without the key
        else done = false;
        if (done) pend &= ~(1u << j);
        else {
          idx[j] = gq_next(T, idx[j], B);
          gq_ld_bucket<NW>(T.slots + idx[j] * SW, w[j]);
        }
      }
    }
  }
}

// HashBuild insert of GQ_R rows: read the bucket, CAS the first EMPTY slot seen, re-examine on a lost race.
template <int SW, int NPAY>
__device__ __forceinline__ int gq_insert_rows(const GqTableDev& T, const i64 (&key)[GQ_R], const bool (&live)[GQ_R],
                                              const i64 (&pay)[GQ_R][NPAY > 0 ? NPAY : 1], bool unique, int* err) {
  constexpr int B = SW == 1 ? 4 : SW == 2 ? 4 : 1;
  constexpr int NW = B * SW;
  u64 w[GQ_R][NW];
  u64 idx[GQ_R];
  u32 pend = 0;
  int ninserted = 0;
#pragma unroll
  for (int j = 0; j < GQ_R; ++j) {
    idx[j] = 0;
    if (live[j]) {
      if ((u64)key[j] == GQ_EMPTY) { if (gq_ht_insert<SW, NPAY>(T, key[j], pay[j], unique, err)) ++ninserted; }
      else {
        idx[j] = gq_slot0(T, key[j]);
        gq_ld_bucket_relaxed<NW>(T.slots + idx[j] * SW, w[j]);
        pend |= 1u << j;
      }
    }
  }
  for (u64 round = 0; pend != 0; ++round) {
#pragma unroll
    for (int j = 0; j < GQ_R; ++j) {
      if (pend & (1u << j)) {
        int fb = -1;          // first EMPTY slot of the bucket
        bool dup = false;
#pragma unroll
        for (int b = 0; b < B; ++b) {
          const u64 kw = w[j][b * SW];
          if (fb < 0 && kw == GQ_EMPTY) fb = b;
          if (fb < 0 && kw == (u64)key[j]) dup = true;   // an equal key stored before the first free slot
        }
        if (unique && dup) { gq_set_err(err, GQ_E_DUPLICATE); pend &= ~(1u << j); }
        else if (fb >= 0) {
          u64* s = T.slots + (idx[j] + fb) * SW;
          const u64 prev = atomicCAS(s, GQ_EMPTY, (u64)key[j]);
          if (prev == GQ_EMPTY) {
#pragma unroll
            for (int p = 0; p < NPAY; ++p) s[1 + p] = (u64)pay[j][p];
            ++ninserted;
            pend &= ~(1u << j);
          } else {
#pragma unroll
            for (int b = 0; b < B; ++b) if (b == fb) w[j][b * SW] = prev;   // lost the race: look at the bucket again
          }
        } else if (round > 2 * (T.mask + 1)) { gq_set_err(err, GQ_E_CAPACITY); pend &= ~(1u << j); }
        else {
          idx[j] = gq_next(T, idx[j], B);
          gq_ld_bucket_relaxed<NW>(T.slots + idx[j] * SW, w[j]);
        }
      }
    }
  }
  return ninserted;
}

// HashAggregation insert-or-update of GQ_R rows: slot[j] = the group's slot (null on error), won[j] = created it.
template <int SW>
__device__ __forceinline__ void gq_upsert_rows(const GqTableDev& T, const i64 (&key)[GQ_R], const bool (&live)[GQ_R],
                                               u64* (&slot)[GQ_R], bool (&won)[GQ_R], int* err) {
  u64 k[GQ_R], idx[GQ_R];
  u32 pend = 0;
#pragma unroll
  for (int j = 0; j < GQ_R; ++j) {
    slot[j] = nullptr; won[j] = false; idx[j] = 0; k[j] = GQ_EMPTY;
    if (live[j]) {
      if ((u64)key[j] == GQ_EMPTY) slot[j] = gq_ht_upsert<SW>(T, key[j], &won[j], err);
      else {
        idx[j] = gq_slot0(T, key[j]);
        k[j] = gq_ld_relaxed(T.slots + idx[j] * SW);
        pend |= 1u << j;
      }
    }
  }
  for (u64 round = 0; pend != 0; ++round) {
#pragma unroll
    for (int j = 0; j < GQ_R; ++j) {
      if (pend & (1u << j)) {
        u64* s = T.slots + idx[j] * SW;
        if (k[j] == (u64)key[j]) { slot[j] = s; pend &= ~(1u << j); }
        else if (k[j] == GQ_EMPTY) {
          const u64 prev = atomicCAS(s, GQ_EMPTY, (u64)key[j]);
          if (prev == GQ_EMPTY) { won[j] = true; slot[j] = s; pend &= ~(1u << j); }
          else k[j] = prev;                         // somebody else claimed it: same key => next round returns it
        } else if (round > 2 * (T.mask + 1)) { gq_set_err(err, GQ_E_CAPACITY); pend &= ~(1u << j); }
        else {
          idx[j] = gq_next(T, idx[j], 1);
          k[j] = gq_ld_relaxed(T.slots + idx[j] * SW);
        }
      }
    }
  }
}

// ---- direct-address join tables (GQ_F_DENSE_KEYS; SURVEY 8(f) NEXT-3 "dense-key array mode"): the planner
// declared the build keys' range, so slot = key - key_min. The membership bitmap is an array of 64-bit entries, one per
// 32 keys: low word = the 32 membership bits, high word = the number of member keys BEFORE this entry (filled in by
// gq_hash_build_finish). HashBuild sets a bit (RED.OR) and stores the payload row at slot (a duplicate key shows at finish:
// fewer member keys than rows inserted); HashProbe is ONE 8-byte load from an L2-resident array (15 M keys: 3.75 MB) — the probes that miss never reach
// DRAM — plus, on a hit, the payload row. The RANK of the key among the member keys (prefix + popcount) is the slot index
// handed to direct aggregation, so its accumulator array has one slot per build row, not per key of the range.
template <int NPAY>
__device__ __forceinline__ bool gq_dense_insert(const GqTableDev& T, i64 key, const i64* pay, int* err) {
  const u64 idx = (u64)key - (u64)T.base;
  if (idx > T.mask) { gq_set_err(err, GQ_E_KEYRANGE); return false; }
  // Fire-and-forget RED.OR (little-endian: the low word of the entry): no round trip per row. A repeated key sets a bit
  // that is already set, so the member count computed by gq_hash_build_finish falls short of the rows inserted — the
  // duplicate is reported there (GQ_ERR_DUPLICATE_KEY), not here.
  atomicOr((u32*)(T.side + (idx >> 5)), 1u << (u32)(idx & 31));
#pragma unroll
  for (int p = 0; p < NPAY; ++p) T.slots[idx * NPAY + p] = (u64)pay[p];
  return true;
}
template <int NPAY>
__device__ __forceinline__ int gq_dense_insert_rows(const GqTableDev& T, const i64 (&key)[GQ_R], const bool (&live)[GQ_R],
                                                    const i64 (&pay)[GQ_R][NPAY > 0 ? NPAY : 1], int* err) {
  int n = 0;
#pragma unroll
  for (int j = 0; j < GQ_R; ++j)
    if (live[j] && gq_dense_insert<NPAY>(T, key[j], pay[j], err)) ++n;
  return n;
}
// one row: *idx = key - key_min (payload row), *rank = position among the member keys
__device__ __forceinline__ bool gq_dense_find(const GqTableDev& T, i64 key, u64* idx, u64* rank) {
  *idx = (u64)key - (u64)T.base;
  if (*idx > T.mask) return false;
  const u64 e = __ldg(T.side + (*idx >> 5));
  const u32 bits = (u32)e, sh = (u32)(*idx & 31);
  *rank = (e >> 32) + __popc(bits & ((1u << sh) - 1u));
  return (bits >> sh) & 1u;
}
template <int NPAY>
__device__ __forceinline__ void gq_dense_probe_rows(const GqTableDev& T, const i64 (&key)[GQ_R], bool (&live)[GQ_R],
                                                    u64 (&rank)[GQ_R], i64 (&pay)[GQ_R][NPAY > 0 ? NPAY : 1]) {
  u64 e[GQ_R], idx[GQ_R];
#pragma unroll
  for (int j = 0; j < GQ_R; ++j) {                      // the bitmap entries of all rows in flight together
    idx[j] = (u64)key[j] - (u64)T.base;
    live[j] = live[j] && idx[j] <= T.mask;
    e[j] = live[j] ? __ldg(T.side + (idx[j] >> 5)) : 0ULL;
  }
#pragma unroll
  for (int j = 0; j < GQ_R; ++j) {
    const u32 bits = (u32)e[j], sh = (u32)(idx[j] & 31);
    live[j] = live[j] && ((bits >> sh) & 1u);
    rank[j] = (e[j] >> 32) + __popc(bits & ((1u << sh) - 1u));
  }
#pragma unroll
  for (int j = 0; j < GQ_R; ++j) {
    if (live[j]) {
#pragma unroll
      for (int p = 0; p < NPAY; ++p) pay[j][p] = (i64)__ldg(T.slots + idx[j] * NPAY + p);
    }
  }
}

// Dependent key word of a group slot: a trailing key column declared functionally dependent on the
// hashed key is stored, not hashed. Normally the row that created the group stores it. With GQ_F_CHECK_DEPENDENT the
// word starts as GQ_DEP_UNSET and EVERY row CASes its value in: a row that finds a different value stored proves the
// declaration false and sets the sticky GQ_E_DEPENDENT.
#define GQ_DEP_UNSET 0x8000000000000001ULL
__device__ __forceinline__ void gq_dep_store(u64* w, i64 dep, bool won, int* err) {
#if GQ_CHECK_DEP
  const u64 prev = atomicCAS(w, GQ_DEP_UNSET, (u64)dep);
  if (prev != GQ_DEP_UNSET && prev != (u64)dep) gq_set_err(err, GQ_E_DEPENDENT);
#else
  if (won) *w = (u64)dep;
#endif
}

// Aggregate update at L2 (RED.ADD / RED.MIN / RED.MAX .64 — results are not read back).
__device__ __forceinline__ void gq_red(const int OP, u64* p, i64 v) {
  if (OP == GQ_OP_SUM || OP == GQ_OP_COUNT) atomicAdd(p, (u64)v);
  else if (OP == GQ_OP_MIN) atomicMin((i64*)p, v);
  else atomicMax((i64*)p, v);
}
// The same with an L2 cache policy (direct aggregation: the accumulator array should outlive the streamed input in L2).
__device__ __forceinline__ void gq_red_hint(const int OP, u64* p, i64 v, u64 pol) {
  if (OP == GQ_OP_SUM || OP == GQ_OP_COUNT) asm volatile("red.global.add.L2::cache_hint.u64 [%0], %1, %2;" ::"l"(p), "l"(v), "l"(pol) : "memory");
  else if (OP == GQ_OP_MIN) asm volatile("red.global.min.L2::cache_hint.s64 [%0], %1, %2;" ::"l"(p), "l"(v), "l"(pol) : "memory");
  else asm volatile("red.global.max.L2::cache_hint.s64 [%0], %1, %2;" ::"l"(p), "l"(v), "l"(pol) : "memory");
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

// Radix-clustered aggregation, pass A: a surviving row is appended to the record buffer of the
// partition its key's first table slot falls in; pass B (gq_k_part_upsert) then applies the records partition by
// partition, so the slice of the group-by table being updated stays L2-resident. One record = GQ_PART_RW words (key,
// dependent key, aggregate inputs), a multiple of 4 words so that it is written with 32-byte stores.
__device__ __forceinline__ void gq_st256(u64* p, u64 a, u64 b, u64 c, u64 d) {
  asm volatile("st.global.v4.u64 [%0], {%1, %2, %3, %4};" ::"l"(p), "l"(a), "l"(b), "l"(c), "l"(d) : "memory");
}
// The same store with an L2 evict-last policy: a record line (4 records) is completed by four stores that lie far apart
// in time, so it should outlive the streamed input in L2 (C5 pass A 10.1 -> 9.6 ms; the open lines of 148 CTAs x 16384
// partitions still exceed L2, see DESIGN 5.4).
__device__ __forceinline__ u64 gq_policy_evict_last() {
  u64 pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void gq_st256_keep(u64* p, u64 a, u64 b, u64 c, u64 d, u64 pol) {
  asm volatile("st.global.L2::cache_hint.v4.u64 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "l"(a), "l"(b), "l"(c), "l"(d), "l"(pol) : "memory");
}

// Appending is done in CTA-private chunks of GQ_PART_CHUNK records: a shared-memory counter hands out the slots of the
// CTA's open chunk of a partition (ATOMS), and only the thread that finds the chunk exhausted draws the next chunk from
// the partition's global cursor — one global atomic per 32 records instead of one per record (a returned global
// atomic per row caps the scan at ~35 G rows/s). Unused slots of the last chunks are padded with EMPTY-key records at
// the end of the kernel; pass B skips them. Returns the record index inside the partition buffer, or -1 when the
// partition's buffer is full (the caller then processes the row in place).
#define GQ_PART_CHUNK 32u
__device__ __forceinline__ i64 gq_part_reserve(const GqParams& P, u32* st, u64 p) {
  for (;;) {
    const u32 v0 = ((volatile u32*)st)[p];
    if ((v0 & 0xFFFFu) > GQ_PART_CHUNK) {                 // being refilled by another thread, or full
      if ((v0 >> 16) == 0xFFFFu) return -1;
      __nanosleep(64);                                    // the refill is a global atomic away: do not burn issue slots
      continue;
    }
    const u32 v = atomicAdd(&st[p], 1u);
    const u32 used = v & 0xFFFFu;
    if (used < GQ_PART_CHUNK) return (i64)(v >> 16) * GQ_PART_CHUNK + used;
    if (used == GQ_PART_CHUNK) {                          // this thread opens the next chunk and takes its first slot
      const u64 c = atomicAdd(P.pcur + p * 16, 1ULL);
      if (c >= (u64)P.pcap / GQ_PART_CHUNK || c >= 0xFFFFull) {
        ((volatile u32*)st)[p] = 0xFFFF0000u | (GQ_PART_CHUNK + 1u);
        return -1;
      }
      __threadfence_block();
      ((volatile u32*)st)[p] = ((u32)c << 16) | 1u;
      return (i64)c * GQ_PART_CHUNK;
    }
  }
}

// Partitioned shared-memory aggregation, pass A (SCATTER consumer): a surviving row becomes one record
// (key, dependent key, aggregate inputs) appended to a chunk of GQ_PART_CHUNK records that belongs to the partition
// its key hashes to. Chunks are CTA-private and are handed out from a CTA-private range of chunk ids by a
// shared-memory counter, so the per-row path has NO global atomic: one ATOMS on the partition's {chunk : 20, used : 12}
// state word hands out the slots of the open chunk; the thread that finds it exhausted opens the next chunk (one
// ATOMS on the CTA's chunk counter, one fire-and-forget RED on the partition's chunk count, one 4-byte store of the
// chunk's partition). Pass B (gq_psa) finds a partition's chunks through a directory built from those words.
// Returns the record index (chunk id * GQ_PART_CHUNK + slot), or ~0 when the CTA's chunk range is exhausted (cannot
// happen for a range sized rows / GQ_PART_CHUNK + partitions; reported as a capacity error).
#if GQ_SC_CLUSTER > 1
// ---- thread-block clusters (pass A of the partitioned aggregation): the CTAs of a cluster SHARE the open chunk of every
// partition — the state word of partition p lives in the shared memory of CTA (p mod cluster size) and is reached through
// distributed shared memory — so a cluster, not a CTA, owns one open 128-byte record line per partition: 74 clusters x
// 16384 partitions = 155 MB of open lines instead of 310 MB, and more of them are complete when they leave L2.
__device__ __forceinline__ u32 gq_cluster_rank() { u32 r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ u32 gq_cluster_id() { u32 r; asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r)); return r; }
__device__ __forceinline__ u32 gq_mapa(u32 saddr, u32 rank) {
  u32 r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
  return r;
}
__device__ __forceinline__ u32 gq_dsm_ld(u32 a) {
  u32 v;
  asm volatile("ld.volatile.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void gq_dsm_st(u32 a, u32 v) { asm volatile("st.volatile.shared::cluster.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ u32 gq_dsm_add(u32 a, u32 v) {
  u32 o;
  asm volatile("atom.shared::cluster.add.u32 %0, [%1], %2;" : "=r"(o) : "r"(a), "r"(v) : "memory");
  return o;
}
__device__ __forceinline__ void gq_cluster_sync() {   // every thread of every CTA of the cluster, warps converged
  asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// The state words live in the cluster's distributed shared memory: st / next are THIS CTA's arrays; partition p's word is
// word p / GQ_SC_CLUSTER of CTA p mod GQ_SC_CLUSTER, the chunk counter is CTA 0's; chunk ids of cluster c are
// [c * sc_slab, (c + 1) * sc_slab).
__device__ __forceinline__ u32 gq_sc_word(u32* st, u32 p) { return gq_mapa(gq_smem_addr(st + p / GQ_SC_CLUSTER), p % GQ_SC_CLUSTER); }
__device__ __forceinline__ u32 gq_sc_ld(u32 a) { return gq_dsm_ld(a); }
__device__ __forceinline__ u32 gq_sc_add(u32 a) { return gq_dsm_add(a, 1u); }
__device__ __forceinline__ void gq_sc_st(u32 a, u32 v) { gq_dsm_st(a, v); }
__device__ __forceinline__ u32 gq_sc_next(u32* next) { return gq_dsm_add(gq_mapa(gq_smem_addr(next), 0u), 1u); }
__device__ __forceinline__ u64 gq_sc_base(const GqParams& P) { return (u64)gq_cluster_id() * (u64)P.sc_slab; }
#else
__device__ __forceinline__ u32 gq_sc_word(u32* st, u32 p) { return gq_smem_addr(st + p); }
__device__ __forceinline__ u32 gq_sc_ld(u32 a) {
  u32 v;
  asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ u32 gq_sc_add(u32 a) {
  u32 o;
  asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(o) : "r"(a) : "memory");
  return o;
}
__device__ __forceinline__ void gq_sc_st(u32 a, u32 v) { asm volatile("st.volatile.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ u32 gq_sc_next(u32* next) { return atomicAdd(next, 1u); }
__device__ __forceinline__ u64 gq_sc_base(const GqParams& P) { return (u64)blockIdx.x * (u64)P.sc_slab; }
#endif
// A reservation is ONE atomic increment of the partition's word (a "ticket"): used < GQ_PART_CHUNK is a slot of the open
// chunk, used == GQ_PART_CHUNK makes this thread the opener of the next chunk (it takes the first slot and stores the
// new word), used > GQ_PART_CHUNK means the chunk is being opened: poll with loads, then draw again. A thread adds at
// most one stray increment per opening, so the 12-bit field cannot overflow (2 x 1024 threads + 32 < 4096). The three
// phases are separate calls so that a thread's GQ_R tickets are in flight together (half of them are remote shared-memory
// atomics in a cluster) and so that every opener acts before anybody polls (no waiting cycle between rows).
__device__ __forceinline__ u32 gq_scatter_ticket(u32* st, u32 p) { return gq_sc_add(gq_sc_word(st, p)); }
__device__ __forceinline__ u64 gq_scatter_open(const GqParams& P, u32 a, u32* next, u32 p, u32 v) {
  const u32 c = gq_sc_next(next);
  if ((i64)c >= P.sc_slab) { gq_set_err(P.err, GQ_E_CAPACITY); gq_sc_st(a, v & ~0xFFFu); return ~0ULL; }
  const u64 gid = gq_sc_base(P) + c;
  P.sc_info[gid] = (p << 8) | GQ_PART_CHUNK;               // assumed full; part-filled chunks are fixed up at the end
  atomicAdd(P.sc_count + p, 1u);
  gq_sc_st(a, (c << 12) | 1u);
  return gid * GQ_PART_CHUNK;
}
// phase 2 (openers only): returns true when this ticket was the opener's; idx = the record index (or ~0: out of chunks)
__device__ __forceinline__ bool gq_scatter_opener(const GqParams& P, u32* st, u32* next, u32 p, u32 v, u64& idx) {
  if ((v & 0xFFFu) != GQ_PART_CHUNK) return false;
  idx = gq_scatter_open(P, gq_sc_word(st, p), next, p, v);
  return true;
}
// phase 3 (everybody else)
__device__ __forceinline__ u64 gq_scatter_take(const GqParams& P, u32* st, u32* next, u32 p, u32 v) {
  u32 used = v & 0xFFFu;
  if (used < GQ_PART_CHUNK) return (gq_sc_base(P) + (v >> 12)) * GQ_PART_CHUNK + used;
  const u32 a = gq_sc_word(st, p);
  for (;;) {
    while ((gq_sc_ld(a) & 0xFFFu) > GQ_PART_CHUNK) __nanosleep(20);   // the next chunk is being opened
    v = gq_sc_add(a);
    used = v & 0xFFFu;
    if (used < GQ_PART_CHUNK) return (gq_sc_base(P) + (v >> 12)) * GQ_PART_CHUNK + used;
    if (used == GQ_PART_CHUNK) return gq_scatter_open(P, a, next, p, v);
  }
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
  u64* lc_tab;                          // LOWCARD: shared key table [GQ_LC_KT]: {key32, gid} packed, or 64-bit keys
  u32* lc_gid;                          //   group ids of the 64-bit key table [GQ_LC_KT]
  i64* lc_gkey;                         //   key of every group id [GQ_LC_G]
  int* lc_n;                            //   [0] groups so far, [1] insert lock, [2] gid of the reserved-pattern key + 1
  i64* lc_acc;                          //   accumulators [GQ_LC_G][GQ_NAGG][GQ_NT], thread-private cells
  u32* part_st;                         // record append: per-partition {chunk id, used} of this CTA's open chunk
  u32* sc_next;                         // SCATTER: next free chunk of this CTA's chunk range
  int* mat;                             // MATERIALISE: shared [0] rows of the tile so far, [2..3] the tile's output base
  i64 ninserted;                        // BUILD: rows inserted by this thread
  i64* hot_keys;                        // HIGHCARD + GQ_HOT: shared set of this batch's hot keys [GQ_HOT_POS]
  u64* hot_acc;                         //   CTA-shared accumulators [GQ_HOT_POS][GQ_NAGG]
  int* hot_touched;                     //   entry received at least one row
  unsigned char* hot_ovf;               //   bucket was full when a key that hashes to it was inserted [GQ_HOT_POS / 4]
  int nhot;
  int t;
};

// Low-cardinality group-by. The CTA keeps a small key table in shared memory that maps a packed key
// to a dense group id (assigned the first time the key is seen, under a CTA lock — at most GQ_LC_G times per CTA).
// Each consumer thread owns a PRIVATE accumulator cell per (group, aggregate), laid out [group][agg][thread] so a
// warp's 32 cells are 32 consecutive 8-byte words: plain conflict-free LDS / add / STS, no atomics and no shuffles
// on the per-row path. Cells are reduced over threads once, at the end (Partial -> Final of PAPER.md:154 inside one
// kernel). Packed keys narrower than 32 bits use {key32, gid} entries fetched with one LDS.64.
#define GQ_LC_LOG2KT (GQ_LC_KT == 64 ? 6 : GQ_LC_KT == 128 ? 7 : 8)
#define GQ_LC_PENDING 0xFFFFFFFEu   // group id of a key-table position that is claimed but not published yet
// {key32, gid} entries hold the key masked to the packed key width (< 32 bits): a sign-extended single key such as -1
// would otherwise equal the high half of an EMPTY entry (~0). Distinct keys of that width stay distinct when masked.
#define GQ_LC_K32(key) ((u32)(key) & ((1u << GQ_LC_KEY_BITS) - 1u))
__device__ __forceinline__ u32 gq_lc_hash(i64 key) {
#if GQ_LC_KEY32
  return (GQ_LC_K32(key) * 0x9E3779B1u) >> (32 - GQ_LC_LOG2KT);
#else
  return (u32)gq_hash(key, 64 - GQ_LC_LOG2KT);
#endif
}
// Fast path: walk the probe sequence until the key or an empty position (almost always the first position: the table
// has >= 4x more positions than groups). Returns the group id, or -1 if the key is not in the table yet.
__device__ __forceinline__ int gq_lc_find(const GqCtx& cx, i64 key) {
  u32 h = gq_lc_hash(key);
#if GQ_LC_KEY32
  for (int n = 0; n < GQ_LC_KT; ++n, h = (h + 1) & (GQ_LC_KT - 1)) {
    const u64 e = ((volatile u64*)cx.lc_tab)[h];
    if ((u32)(e >> 32) == GQ_LC_K32(key)) return (u32)e == GQ_LC_PENDING ? -1 : (int)(u32)e;
    if (e == ~0ULL) return -1;
  }
#else
  if ((u64)key == GQ_EMPTY) { const int v = ((volatile int*)cx.lc_n)[2]; return v > 0 ? v - 1 : -1; }   // reserved bit pattern: id kept aside
  for (int n = 0; n < GQ_LC_KT; ++n, h = (h + 1) & (GQ_LC_KT - 1)) {
    const u64 k = ((volatile u64*)cx.lc_tab)[h];
    if (k == (u64)key) { const u32 g = ((volatile u32*)cx.lc_gid)[h]; return g == GQ_LC_PENDING ? -1 : (int)g; }
    if (k == GQ_EMPTY) return -1;
  }
#endif
  return -1;
}
// One-probe form for the per-row path: group id if the first position holds the key, else -1 (then gq_lc_slow decides).
__device__ __forceinline__ int gq_lc_find1(const GqCtx& cx, i64 key) {
  const u32 h = gq_lc_hash(key);
#if GQ_LC_KEY32
  const u64 e = ((volatile u64*)cx.lc_tab)[h];
  return ((u32)(e >> 32) == GQ_LC_K32(key) && (u32)e != GQ_LC_PENDING) ? (int)(u32)e : -1;
#else
  const u64 k = ((volatile u64*)cx.lc_tab)[h];
  if (k != (u64)key || k == GQ_EMPTY) return -1;
  const u32 g = ((volatile u32*)cx.lc_gid)[h];
  return g == GQ_LC_PENDING ? -1 : (int)g;
#endif
}
// Slow path (collision, or first sight of a key): the warp handles its needy lanes one key at a time; lane 0 takes
// the CTA lock, walks the probe sequence and inserts the key with the next group id if it is absent. Must be called
// by all 32 lanes of the warp (converged); `need` selects the lanes that want an answer.
// Lock-free insert-or-find of one key by ONE thread: the table position is claimed by CAS with a "pending" group id,
// the winner then draws the next dense id and publishes it; a thread that meets a pending entry of its key waits for
// the id (the winner is always another warp, or this very thread).
__device__ __forceinline__ int gq_lc_new_group(GqCtx& cx, i64 k, int* err) {
  int g = atomicAdd(&cx.lc_n[0], 1);
  if (g >= GQ_LC_G) { gq_set_err(err, GQ_E_CAPACITY); g = 0; }   // more distinct keys than max_groups
  else cx.lc_gkey[g] = k;
  return g;
}
__device__ __forceinline__ int gq_lc_insert_or_find(GqCtx& cx, i64 k, int* err) {
#if !GQ_LC_KEY32
  if ((u64)k == GQ_EMPTY) {                               // reserved bit pattern: its id lives in lc_n[2] (id + 1)
    for (;;) {
      const int v = ((volatile int*)cx.lc_n)[2];
      if (v > 0) return v - 1;
      if (v == 0 && atomicCAS(&cx.lc_n[2], 0, -1) == 0) {
        const int g = gq_lc_new_group(cx, k, err);
        __threadfence_block();
        ((volatile int*)cx.lc_n)[2] = g + 1;
        return g;
      }
    }
  }
#endif
  u32 i = gq_lc_hash(k);
  for (int adv = 0; adv < GQ_LC_KT;) {                     // `continue` re-examines the same position
#if GQ_LC_KEY32
    const u64 e = ((volatile u64*)cx.lc_tab)[i];
    if ((u32)(e >> 32) == GQ_LC_K32(k)) {
      if ((u32)e != GQ_LC_PENDING) return (int)(u32)e;
      continue;                                           // id not published yet: look again
    }
    if (e == ~0ULL) {
      const u64 prev = atomicCAS(&cx.lc_tab[i], ~0ULL, ((u64)GQ_LC_K32(k) << 32) | GQ_LC_PENDING);
      if (prev == ~0ULL) {
        const int g = gq_lc_new_group(cx, k, err);
        __threadfence_block();
        ((volatile u64*)cx.lc_tab)[i] = ((u64)GQ_LC_K32(k) << 32) | (u32)g;
        return g;
      }
      continue;                                           // somebody claimed this position: re-examine it
    }
#else
    const u64 e = ((volatile u64*)cx.lc_tab)[i];
    if (e == (u64)k) {
      const u32 g = ((volatile u32*)cx.lc_gid)[i];
      if (g != GQ_LC_PENDING) return (int)g;
      continue;
    }
    if (e == GQ_EMPTY) {
      const u64 prev = atomicCAS(&cx.lc_tab[i], GQ_EMPTY, (u64)k);   // lc_gid[i] holds GQ_LC_PENDING until published
      if (prev == GQ_EMPTY) {
        const int g = gq_lc_new_group(cx, k, err);
        __threadfence_block();
        ((volatile u32*)cx.lc_gid)[i] = (u32)g;
        return g;
      }
      continue;
    }
#endif
    i = (i + 1) & (GQ_LC_KT - 1);
    ++adv;
  }
  gq_set_err(err, GQ_E_CAPACITY);                         // key table full
  return 0;
}
// One row at a time (row code of plans that probe a table with duplicate keys: rows fan out, so the lanes of a warp
// are not converged here): look the key up, insert it on first sight. gq_lc_insert_or_find is a single-thread,
// lock-free protocol, so it needs no warp cooperation; a lane that meets an entry another lane is still publishing
// re-reads it (independent thread scheduling guarantees the publisher makes progress).
__device__ __forceinline__ int gq_lc_slot(GqCtx& cx, i64 key, int* err) {
  const int g = gq_lc_find(cx, key);
  return g >= 0 ? g : gq_lc_insert_or_find(cx, key, err);
}
// Slow path (collision, or first sight of a key): the needy lanes of the warp are grouped by key (MATCH.ANY); the
// first lane of every group inserts or finds its key — all groups at once, they touch different table positions —
// and hands the id to its group. Must be called by all 32 lanes of the warp (converged).
__device__ __forceinline__ int gq_lc_slow_body(GqCtx& cx, i64 key, bool need, int grp, int* err) {
  const int lane = threadIdx.x & 31;
  const u32 needmask = __ballot_sync(0xffffffffu, need);
  int src = lane, g = 0;
  if (need) {
    const u32 m = __match_any_sync(needmask, key);
    src = __ffs(m) - 1;
    if (src == lane) g = gq_lc_insert_or_find(cx, key, err);
  }
  g = __shfl_sync(0xffffffffu, g, src);
  return need ? g : grp;
}
// Out of line: the per-row code only carries a call, not four inlined copies of the insert protocol.
__device__ __noinline__ int gq_lc_slow_call(u64* tab, u32* gid, i64* gkey, int* n, i64 key, bool need, int grp, int* err) {
  GqCtx c;
  c.lc_tab = tab; c.lc_gid = gid; c.lc_gkey = gkey; c.lc_n = n;
  return gq_lc_slow_body(c, key, need, grp, err);
}
__device__ __forceinline__ int gq_lc_slow(GqCtx& cx, i64 key, bool need, int grp, int* err) {
  return gq_lc_slow_call(cx.lc_tab, cx.lc_gid, cx.lc_gkey, cx.lc_n, key, need, grp, err);
}
__device__ __forceinline__ void gq_lc_update(const int OP, GqCtx& cx, int grp, int a, i64 v) {
  i64* cell = cx.lc_acc + ((grp * GQ_NAGG + a) * GQ_NT + cx.t);
  *cell = gq_combine(OP, *cell, v);
}

// Hot keys of a skewed high-cardinality group-by: rows whose key is in the batch's hot list
// are accumulated in CTA-shared memory and flushed to the global table once per CTA, instead of hammering one L2
// address with hundreds of millions of atomics. 64-bit shared atomics are CAS loops on sm_100 (ATOMS.CAST.SPIN), so
// SUM/COUNT use two native 32-bit ATOMS.ADD with an explicit carry; MIN/MAX compare first and CAS only to improve.
#ifndef GQ_HOT_POS      // (set by the plan compiler: 512 positions for <= 256 keys; pass A of the partitioned aggregation
#define GQ_HOT_POS 512  // takes 2048 positions for <= 1536 keys when they fit beside a 3-stage ring)
#define GQ_HOT_MAX 256
#endif
// The hot set is bucketised: GQ_HOT_POS / 4 buckets of 4 keys (GQ_HOT_POS positions for <= GQ_HOT_MAX keys). A key sits in the bucket
// its hash names unless that bucket was full when it was inserted (then in the next one), so a lookup reads one
// 32-byte bucket (two LDS.128) and almost always stops there: a bucket with a free position was never full. (The
// position-by-position linear probe it replaces was a third of pass A's instructions on C5: every row of a warp walked
// as far as the unluckiest lane.)
__device__ __forceinline__ u32 gq_hot_bucket(i64 key) { return (u32)gq_hash(key, 64 - 16) & (GQ_HOT_POS / 4 - 1); }
__device__ __forceinline__ void gq_hot_insert(GqCtx& cx, i64 key) {   // set-up only; keys are distinct
  u32 b = gq_hot_bucket(key);
  for (int n = 0; n < GQ_HOT_POS / 4; ++n, b = (b + 1) & (GQ_HOT_POS / 4 - 1)) {
    for (int q = 0; q < 4; ++q)
      if (atomicCAS((u64*)&cx.hot_keys[b * 4 + q], GQ_EMPTY, (u64)key) == GQ_EMPTY) return;
    cx.hot_ovf[b] = 1;                                  // the key moves on: lookups that miss here must too
  }
}
// A lookup reads one 32-byte bucket and its overflow flag and stops there unless a key was ever turned away from that
// bucket. (Stopping at the first bucket with an EMPTY position instead cost four more 64-bit compares per row, and at
// 75 % load most rows — the misses — walked on into a second bucket: a quarter of pass A's instructions on C5.)
__device__ __forceinline__ int gq_hot_find(const GqCtx& cx, i64 key) {
  u32 b = gq_hot_bucket(key);
  for (int n = 0; n < GQ_HOT_POS / 4; ++n, b = (b + 1) & (GQ_HOT_POS / 4 - 1)) {
    const longlong2 k01 = *(const longlong2*)&cx.hot_keys[b * 4], k23 = *(const longlong2*)&cx.hot_keys[b * 4 + 2];
    const unsigned char ovf = cx.hot_ovf[b];
    if (k01.x == key) return (int)(b * 4);
    if (k01.y == key) return (int)(b * 4 + 1);
    if (k23.x == key) return (int)(b * 4 + 2);
    if (k23.y == key) return (int)(b * 4 + 3);
    if (!ovf) return -1;
  }
  return -1;
}
// A hot row's update in two phases, so that the shared-memory round trips of its aggregates overlap: gq_hot_issue sends
// the low-word add (SUM / COUNT) or reads the cell (MIN / MAX) and returns what came back; gq_hot_finish propagates the
// carry / runs the compare-and-swap loop.
__device__ __forceinline__ u64 gq_hot_issue(const int OP, GqCtx& cx, int pos, int a, i64 v) {
  u64* cell = cx.hot_acc + pos * GQ_NAGG + a;
  if (OP == GQ_OP_SUM || OP == GQ_OP_COUNT) return (u64)atomicAdd((u32*)cell, (u32)(u64)v);
  return *(volatile u64*)cell;
}
__device__ __forceinline__ void gq_hot_finish(const int OP, GqCtx& cx, int pos, int a, i64 v, u64 got) {
  u64* cell = cx.hot_acc + pos * GQ_NAGG + a;
  if (OP == GQ_OP_SUM || OP == GQ_OP_COUNT) {
    const u32 lo = (u32)(u64)v, hi = (u32)((u64)v >> 32), old = (u32)got;
    const u32 up = hi + ((u32)(old + lo) < old ? 1u : 0u);   // carry out of the low word belongs to THIS addition
    if (up) atomicAdd((u32*)cell + 1, up);
  } else {
    i64 cur = (i64)got;
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

// MATERIALISE, linear mode: one global reservation per CTA and tile. Ballot/popc gives each row its rank inside the
// warp, a shared-memory add gives the warp its offset inside the tile, and thread 0 reserves the tile's output range
// with ONE atomic on the device-side row count (per-warp reservations serialise on that single address: 1.2 ms for
// the 1.09 M output rows of the C2 filter; per-tile ones do not).
__device__ __forceinline__ void gq_materialise_offsets(const GqParams& P, GqCtx& cx, const bool (&live)[GQ_R], i64 (&orow)[GQ_R]) {
  const int lane = threadIdx.x & 31;
  int pre[GQ_R];
  int wtot = 0;
#pragma unroll
  for (int j = 0; j < GQ_R; ++j) {
    const u32 m = __ballot_sync(0xffffffffu, live[j]);
    pre[j] = wtot + __popc(m & ((1u << lane) - 1u));
    wtot += __popc(m);
  }
  int woff = 0;
  if (lane == 0 && wtot) woff = atomicAdd(&cx.mat[0], wtot);
  woff = __shfl_sync(0xffffffffu, woff, 0);
  gq_consumer_barrier();                                  // every warp has added its rows
  if (threadIdx.x == 0) {
    const int tot = ((volatile int*)cx.mat)[0];
    *(volatile i64*)(cx.mat + 2) = tot ? (i64)atomicAdd((u64*)P.out_count, (u64)tot) : 0;
    ((volatile int*)cx.mat)[0] = 0;
  }
  gq_consumer_barrier();                                  // base published, tile counter reset
  const i64 base = *(volatile i64*)(cx.mat + 2);
#pragma unroll
  for (int j = 0; j < GQ_R; ++j) {
    orow[j] = live[j] ? base + woff + pre[j] : -1;
    if (orow[j] >= P.out_capacity) { gq_set_err(P.err, GQ_E_CAPACITY); orow[j] = -1; }
  }
}

//@@ROW_FUNCTIONS@@
