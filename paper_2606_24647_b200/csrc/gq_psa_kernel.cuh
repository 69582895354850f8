// gq_psa_kernel.cuh — pass B of the partitioned shared-memory aggregation (high-cardinality HashAggregation of one
// large batch; PAPER.md:154 group-by, :92 "operator implementation by input size").
// Compiled per plan shape by NVRTC, after the prelude and gq_skeleton.cuh (types, gq_hash, GqFinal).
//
// Pass A (gq_scan, SCATTER consumer) cut the surviving rows into records and appended them to chunks of
// GQ_PART_CHUNK records, each chunk owned by the partition its keys hash to (the top bits of the Fibonacci hash). A
// partition is small enough for ALL its groups to fit a shared-memory hash table, so here:
//   - persistent CTAs draw work items (a partition, or a segment of a heavy partition) from a global queue;
//   - the CTA streams the item's chunks from HBM exactly once (coalesced 32-byte records, GQ_PSA_U chunks in flight
//     per warp) and aggregates them in its shared-memory table: open addressing, linear probing, ATOMS.CAS.64 to
//     claim a key, SUM/COUNT as 32-bit ATOMS.ADD pairs with explicit carry (64-bit shared atomics are CAS loops on
//     sm_100), MIN/MAX as compare-then-CAS — no global atomic and no global table on the per-row path. The 32 records
//     of a chunk go through the table TOGETHER (gq_psa_row: warp-converged probe rounds, straight-line updates): with
//     one data-dependent loop per lane the warp executed every lane's path in turn (12 of 32 lanes active, 490
//     warp instructions per chunk);
//   - then writes its groups straight into the dense output columns (ONE global atomic per item reserves the rows).
// Heavy partitions (hot keys) are cut into segments handled by different CTAs; a segment flushes its partial groups
// into a small global merge table with the ordinary insert-or-update protocol, emitted afterwards by gq_k_finalise.
// Any key distribution stays correct: if a partition holds more distinct keys than the table takes, its key space
// is halved (by a second, bijective hash) and the chunks are streamed again for each half, recursively.
//
// Prelude macros used: GQ_NAGG, GQ_AGG_OP(a), GQ_AGG_SRC(a) (record word of the aggregate's input; unused for COUNT),
// GQ_NDEP, GQ_CHECK_DEP, GQ_TARGET_SW (words per table slot), GQ_PART_RW (words per record), GQ_PSA_LOG2SLOTS,
// GQ_PSA_THREADS, GQ_PSA_U (chunks in flight per warp).

#define GQ_PSA_NW (GQ_PSA_THREADS / 32)            // GQ_PSA_THREADS, GQ_PSA_U (chunks in flight per warp): prelude
#define GQ_PSA_SLOTS (1 << GQ_PSA_LOG2SLOTS)
// Groups a table takes before it gives up (load 0.75). The count is checked once per warp and iteration, so up to
// GQ_PSA_U x GQ_PSA_THREADS further claims may be in flight: a table that fills up completely is caught by the probe
// loop's guard.
#define GQ_PSA_LIMIT (GQ_PSA_SLOTS - GQ_PSA_SLOTS / 4)
#define GQ_PSA_SW GQ_TARGET_SW
#define GQ_PSA_RW GQ_PART_RW
#define GQ_PSA_TABW ((GQ_PSA_SLOTS + 1) * GQ_PSA_SW)  // + the side slot (key == the reserved EMPTY pattern, S14)
#define GQ_PSA_GID_BITS 26                            // directory entry = chunk id | records used << 26

// Must match gq_internal.h:GqPsaParams.
struct GqPsaParams {
  const u64* rec;        // record pool: [chunk][GQ_PART_CHUNK][GQ_PSA_RW]
  const u32* plist;      // directory: chunk entries grouped by partition
  const u32* pstart;     // [partitions + 1] first directory entry of every partition
  const u32* items;      // work items: partition | segment << 16 ... see item_seg
  const u32* item_seg;   // segment index of the item inside its partition (0 for unsplit partitions) | sub-pass << 24
  const u32* nitems;     // device scalar
  u32* work;             // queue cursor (zero before the launch)
  int* err;
  GqTableDev merge;      // global merge table for the segments of split partitions
  u32 seg_chunks;        // chunks per segment (partitions with more chunks are split)
  int hshift;            // partition = hash >> hshift
  int log2sub;           // every partition is aggregated in 2^log2sub sub-passes (work items), one per value of the next hash bits
  int pad;
  GqFinal fin;
};

enum { GQ_PSA_ITEM = 0, GQ_PSA_NG, GQ_PSA_OVF, GQ_PSA_CUR, GQ_PSA_SIDE, GQ_PSA_SP, GQ_PSA_BASE_LO, GQ_PSA_BASE_HI, GQ_PSA_CTLN = 16 };

__device__ __forceinline__ u64 gq_psa_mix(u64 x) {   // bijective finaliser: distinct keys keep distinct values
  x ^= x >> 33; x *= 0xff51afd7ed558ccdULL; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ULL; x ^= x >> 33;
  return x;
}
__device__ __forceinline__ u64 gq_psa_init_word(int q) {    // word q of an empty slot
  if (q == 0) return GQ_EMPTY;
  u64 v = GQ_CHECK_DEP ? GQ_DEP_UNSET : 0ULL;
#pragma unroll
  for (int a = 0; a < GQ_NAGG; ++a) if (q == 1 + GQ_NDEP + a) v = (u64)gq_identity(GQ_AGG_OP(a));
  return v;
}

// One record per lane, all 32 lanes of the warp together (converged): finds or claims the slot of every active
// lane's key and applies the record's aggregate inputs. The probe loop runs until no lane is pending, so the warp
// executes it once per round, not once per lane; new groups are counted with one atomic per warp; the updates are
// straight-line code (SUM/COUNT: a 32-bit ATOMS.ADD and, only when there is a carry or a high word, a second one;
// MIN/MAX: compare first, CAS only to improve).
__device__ __forceinline__ void gq_psa_row(u64* tab, u32* ctl, const u64 (&w)[GQ_PSA_RW], bool act, u64 h, int tshift, int* err, u32* nwon) {
  const u64 key = w[0];
  u64* slot = nullptr;
  bool won = false, side_won = false;
  if (act && key == GQ_EMPTY) {                         // reserved bit pattern (S14): the side slot, counted by GQ_PSA_SIDE
    side_won = atomicExch(&ctl[GQ_PSA_SIDE], 1u) == 0u;
    slot = tab + (size_t)GQ_PSA_SLOTS * GQ_PSA_SW;
  }
  // (the overflow flag is read once per row, not per probed slot: a claim made after the table has given up is harmless,
  // the item is redone anyway)
  bool pend = act && slot == nullptr && !((volatile u32*)ctl)[GQ_PSA_OVF];
  u32 i = (u32)(h >> (tshift - GQ_PSA_LOG2SLOTS)) & (GQ_PSA_SLOTS - 1);
  int n = 0;
  for (; n <= GQ_PSA_SLOTS && __any_sync(0xffffffffu, pend); ++n) {
    if (pend) {
      u64* s = tab + (size_t)i * GQ_PSA_SW;
      const u64 k = *(volatile u64*)s;
      if (k == key) { slot = s; pend = false; }
      else {
        if (k == GQ_EMPTY) {
          const u64 prev = atomicCAS(s, GQ_EMPTY, key);
          if (prev == GQ_EMPTY) { slot = s; won = true; pend = false; }
          else if (prev == key) { slot = s; pend = false; }
        }
        if (pend) i = (i + 1) & (GQ_PSA_SLOTS - 1);
      }
    }
  }
  if (pend) ((volatile u32*)ctl)[GQ_PSA_OVF] = 1u;       // walked the whole table: it is full
  *nwon += won ? 1u : 0u;                               // counted once per warp and iteration by the caller
  if (slot != nullptr) {
#if GQ_NDEP
#if GQ_CHECK_DEP
    { const u64 prev = atomicCAS(slot + 1, GQ_DEP_UNSET, w[1]); if (prev != GQ_DEP_UNSET && prev != w[1]) gq_set_err(err, GQ_E_DEPENDENT); }
#else
    if (won || side_won) *(volatile u64*)(slot + 1) = w[1];
#endif
#endif
    // two phases, so that the shared-memory round trips of the row's aggregates overlap: first every low-word add goes
    // out and every MIN/MAX cell is read, then the carries and the compare-and-swap loops
    u64 got[GQ_NAGG];
#pragma unroll
    for (int a = 0; a < GQ_NAGG; ++a) {
      const int op = GQ_AGG_OP(a);
      u64* cell = slot + 1 + GQ_NDEP + a;
      if (op == GQ_OP_COUNT) got[a] = (u64)atomicAdd((u32*)cell, 1u);
      else if (op == GQ_OP_SUM) got[a] = (u64)atomicAdd((u32*)cell, (u32)w[GQ_AGG_SRC(a)]);
      else got[a] = *(volatile u64*)cell;
    }
#pragma unroll
    for (int a = 0; a < GQ_NAGG; ++a) {
      const int op = GQ_AGG_OP(a);
      u64* cell = slot + 1 + GQ_NDEP + a;
      if (op == GQ_OP_COUNT) {
        if ((u32)got[a] == 0xFFFFFFFFu) atomicAdd((u32*)cell + 1, 1u);
      } else if (op == GQ_OP_SUM) {
        const u64 v = w[GQ_AGG_SRC(a)];
        const u32 lo = (u32)v, hi = (u32)(v >> 32), old = (u32)got[a];
        const u32 up = hi + ((u32)(old + lo) < old ? 1u : 0u);   // the carry out of the low word belongs to THIS addition
        if (up) atomicAdd((u32*)cell + 1, up);
      } else {
        const i64 v = (i64)w[GQ_AGG_SRC(a)];
        i64 cur = (i64)got[a];
        while (op == GQ_OP_MIN ? v < cur : v > cur) {
          const i64 prev = (i64)atomicCAS(cell, (u64)cur, (u64)v);
          if (prev == cur) break;
          cur = prev;
        }
      }
    }
  }
}

__device__ __forceinline__ i64 gq_psa_sext(u64 v, int bits) {
  if (bits >= 64) return (i64)v;
  const u64 m = 1ULL << (bits - 1);
  v &= (1ULL << bits) - 1;
  return (i64)((v ^ m) - m);
}
__device__ __forceinline__ void gq_psa_store_key(void* col, int dtype, i64 idx, i64 v) {
  if (dtype == 1) ((signed char*)col)[idx] = (signed char)v;
  else if (dtype == 2) ((int*)col)[idx] = (int)v;
  else ((i64*)col)[idx] = v;
}
// One dense output row from a table slot: keys unpacked, aggregates, AVG = double(sum)/double(count).
__device__ __forceinline__ void gq_psa_emit(const GqFinal& F, i64 row, u64 key, const u64* slot) {
  const int nhashed = F.nkeys - GQ_NDEP;
  if (nhashed == 1) gq_psa_store_key(F.out_key[0], F.key_dtype[0], row, (i64)key);
  else if (nhashed == 2) {
    gq_psa_store_key(F.out_key[0], F.key_dtype[0], row, gq_psa_sext(key, F.key_bits[0]));
    gq_psa_store_key(F.out_key[1], F.key_dtype[1], row, gq_psa_sext(key >> F.key_bits[0], F.key_bits[1]));
  }
#if GQ_NDEP
  gq_psa_store_key(F.out_key[nhashed], F.key_dtype[nhashed], row, (i64)slot[1]);
#endif
  i64 vals[GQ_NAGG];
#pragma unroll
  for (int a = 0; a < GQ_NAGG; ++a) { vals[a] = (i64)slot[1 + GQ_NDEP + a]; F.out_agg[a][row] = vals[a]; }
  for (int v = 0; v < F.navg; ++v) {
    i64 s = 0, c = 1;
#pragma unroll
    for (int a = 0; a < GQ_NAGG; ++a) { if (a == F.avg_sum[v]) s = vals[a]; if (a == F.avg_cnt[v]) c = vals[a]; }
    F.out_avg[v][row] = (double)s / (double)c;
  }
}

// The records of GQ_PSA_U chunks (directory entries e: chunk id | records used << GQ_PSA_GID_BITS), one record per lane.
__device__ __forceinline__ void gq_psa_load(const GqPsaParams& P, const u32 (&e)[GQ_PSA_U], u64 (&w)[GQ_PSA_U][GQ_PSA_RW], bool (&live)[GQ_PSA_U], int lane) {
#pragma unroll
  for (int u = 0; u < GQ_PSA_U; ++u) {
    live[u] = (u32)lane < (e[u] >> GQ_PSA_GID_BITS);
    const u64* r = P.rec + ((u64)(e[u] & ((1u << GQ_PSA_GID_BITS) - 1u)) * GQ_PART_CHUNK + lane) * GQ_PSA_RW;
#pragma unroll
    for (int q = 0; q < GQ_PSA_RW; q += 4) {
      w[u][q] = w[u][q + 1] = w[u][q + 2] = w[u][q + 3] = 0;
      if (live[u])
        asm volatile("ld.global.nc.L1::no_allocate.v4.u64 {%0, %1, %2, %3}, [%4];"
                     : "=l"(w[u][q]), "=l"(w[u][q + 1]), "=l"(w[u][q + 2]), "=l"(w[u][q + 3]) : "l"(r + q));
    }
  }
}

extern "C" __global__ void __launch_bounds__(GQ_PSA_THREADS, 1) gq_psa(const __grid_constant__ GqPsaParams P) {
  extern __shared__ __align__(128) unsigned char gq_smem[];
  u64* tab = (u64*)gq_smem;
  u64* stack = tab + GQ_PSA_TABW;                     // up to 64 pending key ranges {lo, hi}
  u32* ctl = (u32*)(stack + 2 * 66);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (*(volatile int*)P.err != 0) return;             // sticky error: later kernels are no-ops
  const u32 nitems = *P.nitems;
  for (;;) {
    __syncthreads();
    if (tid == 0) ctl[GQ_PSA_ITEM] = atomicAdd(P.work, 1u);
    __syncthreads();
    const u32 item = ctl[GQ_PSA_ITEM];
    if (item >= nitems) break;
    const u32 part = P.items[item], seg = P.item_seg[item] & 0xFFFFFFu, sub = P.item_seg[item] >> 24;
    const int log2sub = P.log2sub;
    const int tshift = P.hshift - log2sub;              // the table index comes from the hash bits below partition and sub-pass
    const u32 p0 = P.pstart[part], p1 = P.pstart[part + 1];
    const bool split = (p1 - p0) > P.seg_chunks;      // this item is one segment of a heavy partition
    const u32 c0 = split ? p0 + seg * P.seg_chunks : p0;
    const u32 c1 = split ? min(p1, c0 + P.seg_chunks) : p1;
    if (tid == 0) { stack[0] = 0ULL; stack[1] = ~0ULL; ctl[GQ_PSA_SP] = 1; }
    for (int depth_guard = 0;; ++depth_guard) {
      __syncthreads();
      const u32 sp = ctl[GQ_PSA_SP];
      if (sp == 0) break;
      const u64 lo = stack[2 * (sp - 1)], hi = stack[2 * (sp - 1) + 1];
      const bool filt = !(lo == 0ULL && hi == ~0ULL);
      __syncthreads();
      // ---- empty table
      for (int i = tid; i <= GQ_PSA_SLOTS; i += GQ_PSA_THREADS) {
#pragma unroll
        for (int q = 0; q < GQ_PSA_SW; ++q) tab[(size_t)i * GQ_PSA_SW + q] = gq_psa_init_word(q);   // constants after unrolling
      }
      if (tid == 0) { ctl[GQ_PSA_NG] = 0; ctl[GQ_PSA_OVF] = 0; ctl[GQ_PSA_CUR] = 0; ctl[GQ_PSA_SIDE] = 0; ctl[GQ_PSA_SP] = sp - 1; }
      __syncthreads();
      // ---- stream the item's chunks: GQ_PSA_U chunks of 32 records per warp in flight
      // (the directory entries of the NEXT iteration are fetched while this one is processed: the record addresses depend on
      // them, and two dependent global round trips per iteration were 18 % of the kernel's stall samples)
      u32 en[GQ_PSA_U];
      u64 wn[GQ_PSA_U][GQ_PSA_RW];                       // records of the NEXT iteration, loaded while this one is processed
      bool liven[GQ_PSA_U];
      const u32 stride = GQ_PSA_NW * GQ_PSA_U, b0 = c0 + warp * GQ_PSA_U;
#pragma unroll
      for (int u = 0; u < GQ_PSA_U; ++u) { const u32 ci = b0 + u; en[u] = ci < c1 ? __ldg(P.plist + ci) : 0u; }
      gq_psa_load(P, en, wn, liven, lane);
#pragma unroll
      for (int u = 0; u < GQ_PSA_U; ++u) { const u32 ci = b0 + stride + u; en[u] = ci < c1 ? __ldg(P.plist + ci) : 0u; }
      for (u32 b = b0; b < c1; b += stride) {
        if (((volatile u32*)ctl)[GQ_PSA_OVF]) break;
        u64 w[GQ_PSA_U][GQ_PSA_RW];
        bool live[GQ_PSA_U];
#pragma unroll
        for (int u = 0; u < GQ_PSA_U; ++u) {
          live[u] = liven[u];
#pragma unroll
          for (int q = 0; q < GQ_PSA_RW; ++q) w[u][q] = wn[u][q];
        }
        gq_psa_load(P, en, wn, liven, lane);               // iteration b + stride (entries fetched one iteration ago)
#pragma unroll
        for (int u = 0; u < GQ_PSA_U; ++u) { const u32 cn = b + 2 * stride + u; en[u] = cn < c1 ? __ldg(P.plist + cn) : 0u; }
        u32 nwon = 0;
#pragma unroll
        for (int u = 0; u < GQ_PSA_U; ++u) {
          const u64 key = w[u][0];
          const u64 h = gq_hash((i64)key, 0);
          bool act = live[u];
          if (log2sub) act = act && (u32)((h >> tshift) & ((1u << log2sub) - 1u)) == sub;   // another sub-pass owns this key
          if (filt) { const u64 h2 = gq_psa_mix(key); act = act && h2 >= lo && h2 <= hi; }
          gq_psa_row(tab, ctl, w[u], act, h, tshift, P.err, &nwon);
        }
        // new groups of this warp and iteration: one atomic (up to GQ_PSA_U x GQ_PSA_THREADS claims may be uncounted when
        // the bound is checked; a table that fills up meanwhile is caught by the probe loop's guard)
        nwon = __reduce_add_sync(0xffffffffu, nwon);
        if (nwon != 0u && lane == 0 && atomicAdd(&ctl[GQ_PSA_NG], nwon) + nwon > (u32)GQ_PSA_LIMIT) ((volatile u32*)ctl)[GQ_PSA_OVF] = 1u;
      }
      __syncthreads();
      if (ctl[GQ_PSA_OVF]) {
        // more distinct keys than the table takes: halve the key range (second hash) and stream the chunks again
        if (tid == 0) {
          u32 s2 = ctl[GQ_PSA_SP];
          if (lo == hi || s2 + 2 > 64) gq_set_err(P.err, GQ_E_CAPACITY);   // unreachable: one key cannot overflow
          else {
            const u64 mid = lo + (hi - lo) / 2;
            stack[2 * s2] = mid + 1; stack[2 * s2 + 1] = hi; ++s2;
            stack[2 * s2] = lo; stack[2 * s2 + 1] = mid; ++s2;
            ctl[GQ_PSA_SP] = s2;
          }
        }
        continue;
      }
      // ---- the groups of this key range are complete
      const u32 ng = ctl[GQ_PSA_NG] + ctl[GQ_PSA_SIDE];
      if (!split) {
        // dense output rows: one global atomic reserves them
        if (tid == 0) {
          const u64 base = ng ? atomicAdd((u64*)P.fin.out_n, (u64)ng) : 0ULL;
          ctl[GQ_PSA_BASE_LO] = (u32)base; ctl[GQ_PSA_BASE_HI] = (u32)(base >> 32);
          if ((i64)(base + ng) > P.fin.out_capacity) gq_set_err(P.err, GQ_E_CAPACITY);
        }
        __syncthreads();
        const u64 base = (u64)ctl[GQ_PSA_BASE_LO] | ((u64)ctl[GQ_PSA_BASE_HI] << 32);
        for (int i = tid; i <= GQ_PSA_SLOTS; i += GQ_PSA_THREADS) {
          const u64* s = tab + (size_t)i * GQ_PSA_SW;
          const bool have = i < GQ_PSA_SLOTS ? s[0] != GQ_EMPTY : ctl[GQ_PSA_SIDE] != 0;
          if (!have) continue;
          const i64 row = (i64)(base + atomicAdd(&ctl[GQ_PSA_CUR], 1u));
          if (row < P.fin.out_capacity) gq_psa_emit(P.fin, row, i < GQ_PSA_SLOTS ? s[0] : GQ_EMPTY, s);
        }
      } else {
        // one segment of a heavy partition: fold the partial groups into the global merge table
        for (int i = tid; i <= GQ_PSA_SLOTS; i += GQ_PSA_THREADS) {
          const u64* s = tab + (size_t)i * GQ_PSA_SW;
          const bool have = i < GQ_PSA_SLOTS ? s[0] != GQ_EMPTY : ctl[GQ_PSA_SIDE] != 0;
          if (!have) continue;
          bool won;
          u64* g = gq_ht_upsert<GQ_PSA_SW>(P.merge, i < GQ_PSA_SLOTS ? (i64)s[0] : (i64)GQ_EMPTY, &won, P.err);
          if (!g) continue;
#if GQ_NDEP
          gq_dep_store(g + 1, (i64)s[1], won, P.err);
#endif
#pragma unroll
          for (int a = 0; a < GQ_NAGG; ++a) gq_red(GQ_AGG_OP(a), g + 1 + GQ_NDEP + a, (i64)s[1 + GQ_NDEP + a]);
        }
      }
    }
  }
}
