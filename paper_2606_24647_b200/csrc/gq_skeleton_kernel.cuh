// gq_skeleton_kernel.cuh — second half of the fused scan kernel (follows the generated row functions).

// Shared-memory layout (dynamic): [GQ_STAGES stages][full/empty mbarriers][consumer area]
#define GQ_BAR_OFF (GQ_STAGES * GQ_STAGE_BYTES)
#define GQ_CONS_OFF (GQ_BAR_OFF + 2 * GQ_STAGES * 8 + 64)
// LOWCARD consumer area: key table, group ids, group keys, counters, final values, then the private cells
#define GQ_LC_GID_OFF (GQ_LC_KT * 8)
#define GQ_LC_GKEY_OFF (GQ_LC_KT * 12)
#define GQ_LC_N_OFF (GQ_LC_GKEY_OFF + GQ_LC_G * 8)
#define GQ_LC_FIN_OFF (GQ_LC_N_OFF + 16)
#define GQ_LC_HEAD_BYTES ((GQ_LC_FIN_OFF + GQ_LC_G * GQ_NAGG * 8 + 127) / 128 * 128)

template <class Src>
__device__ __forceinline__ void gq_process(const GqParams& P, const Src& src, GqCtx& cx, int nvalid_j, bool full) {
#if GQ_LINEAR
  // generated: the GQ_R rows advance step by step, accesses issued before use
  if (full) gq_tile<Src, true>(P, src, cx, nvalid_j);
  else gq_tile<Src, false>(P, src, cx, nvalid_j);
#else
  // Evaluate the filter for all GQ_R rows first (independent shared-memory loads in flight together), then run the
  // body (probes, projection, consumer) only for passing rows.
  bool pass[GQ_R];
#pragma unroll
  for (int j = 0; j < GQ_R; ++j) pass[j] = (full || j < nvalid_j) ? gq_pass(P, src, j) : false;
#pragma unroll
  for (int j = 0; j < GQ_R; ++j)
    if (pass[j]) gq_body(P, src, j, cx);
#endif
}

__device__ __forceinline__ i64 gq_ldcg(const i64* p) { return __ldcg(p); }

#if GQ_FUSED_FINAL
__device__ __forceinline__ i64 gq_fin_sext(u64 v, int bits) {
  if (bits >= 64) return (i64)v;
  const u64 m = 1ULL << (bits - 1);
  v &= (1ULL << bits) - 1;
  return (i64)((v ^ m) - m);
}
__device__ __forceinline__ void gq_fin_store_key(void* col, int dtype, i64 idx, i64 v) {
  if (dtype == 1) ((signed char*)col)[idx] = (signed char)v;
  else if (dtype == 2) ((int*)col)[idx] = (int)v;
  else ((i64*)col)[idx] = v;
}
// One output row: keys unpacked from the packed key word, aggregates, derived AVG = double(sum) / double(count).
__device__ __forceinline__ void gq_fin_emit(const GqFinal& F, i64 row, i64 key, const i64* vals) {
  if (F.nkeys == 1) gq_fin_store_key(F.out_key[0], F.key_dtype[0], row, key);
  else if (F.nkeys == 2) {
    gq_fin_store_key(F.out_key[0], F.key_dtype[0], row, gq_fin_sext((u64)key, F.key_bits[0]));
    gq_fin_store_key(F.out_key[1], F.key_dtype[1], row, gq_fin_sext((u64)key >> F.key_bits[0], F.key_bits[1]));
  }
#pragma unroll
  for (int a = 0; a < GQ_NAGG; ++a) F.out_agg[a][row] = vals[a];
  for (int v = 0; v < F.navg; ++v) F.out_avg[v][row] = (double)vals[F.avg_sum[v]] / (double)vals[F.avg_cnt[v]];
}
#endif

#if GQ_FUSED_FINAL
// Aggregate words of the context-owned merge table: a representation whose identity is 0 for every operator.
__device__ __forceinline__ u64 gq_gt_enc(const int OP, i64 v) {
  if (OP == GQ_OP_MAX) return (u64)v ^ 0x8000000000000000ULL;          // unsigned order == signed order; INT64_MIN -> 0
  if (OP == GQ_OP_MIN) return ~((u64)v ^ 0x8000000000000000ULL);       // reversed: the maximum of these is the minimum
  return (u64)v;
}
__device__ __forceinline__ i64 gq_gt_dec(const int OP, u64 w) {
  if (OP == GQ_OP_MAX) return (i64)(w ^ 0x8000000000000000ULL);
  if (OP == GQ_OP_MIN) return (i64)(~w ^ 0x8000000000000000ULL);
  return (i64)w;
}
__device__ __forceinline__ u32 gq_atom_add_acq_rel(u32* p, u32 v) {
  u32 old;
  asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], %2;" : "=r"(old) : "l"(p), "r"(v) : "memory");
  return old;
}
#endif

#if GQ_CONSUMER == GQ_C_LOWCARD
// Reduces the GQ_NT private cells of up to four pairs p = group * GQ_NAGG + a (p0, p0 + GQ_NWARP, ...) over the warp's
// lanes, the four chains interleaved (the loads of one pair alone are a dependent LDS/combine chain); every lane gets
// the results.
__device__ __forceinline__ void gq_lc_reduce4(const GqCtx& cx, int p0, int np, int lane, i64 (&v)[4]) {
  int op[4];
  const i64* cells[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const int p = p0 + u * GQ_NWARP;
    const int pc = p < np ? p : p0;
    op[u] = GQ_AGG_OP(pc % GQ_NAGG);
    cells[u] = cx.lc_acc + (size_t)pc * GQ_NT;
    v[u] = gq_identity(op[u]);
  }
#pragma unroll 2
  for (int i = lane; i < GQ_NT; i += 32) {
#pragma unroll
    for (int u = 0; u < 4; ++u) v[u] = gq_combine(op[u], v[u], cells[u][i]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
    for (int u = 0; u < 4; ++u) v[u] = gq_combine(op[u], v[u], __shfl_xor_sync(0xffffffffu, v[u], o));
  }
}
#endif

// One tile into ring stage s: one 1-D TMA bulk copy per referenced column, completion counted on the stage's full barrier.
__device__ __forceinline__ void gq_produce_tile(const GqParams& P, unsigned char* smem, u64* full_bar, int s, i64 tile, u64 pol) {
  gq_mbar_expect_tx(&full_bar[s], (u32)GQ_TX_BYTES);
  unsigned char* st = smem + (size_t)s * GQ_STAGE_BYTES;
#pragma unroll
  for (int c = 0; c < GQ_NCOL; ++c)
    gq_bulk_g2s(st + GQ_COL_OFF(c), (const unsigned char*)P.col[c] + (size_t)tile * GQ_TILE * GQ_COL_BYTES(c),
                (u32)(GQ_TILE * GQ_COL_BYTES(c)), &full_bar[s], pol);
}

extern "C" __global__ void __launch_bounds__(GQ_NT + 32, 1) gq_scan(const __grid_constant__ GqParams P) {
  extern __shared__ __align__(128) unsigned char gq_smem[];
  u64* full_bar = (u64*)(gq_smem + GQ_BAR_OFF);
  u64* empty_bar = full_bar + GQ_STAGES;
  const int tid = threadIdx.x;
  const i64 ntiles = P.nrows / GQ_TILE;                  // full tiles; the remainder is the tail
  // Sticky error: later kernels are no-ops (gq.h "Errors"). Thread 0 reads the flag once, the CTA decides after the
  // set-up barrier below: every thread sees the same value, and the round trip overlaps the shared-memory set-up.
  volatile int* err_seen = (volatile int*)(gq_smem + GQ_BAR_OFF + 2 * GQ_STAGES * 8);
  if (tid == 0) *err_seen = *(volatile int*)P.err;
  // The producer lane initialises the mbarriers and issues the bulk copies of its first GQ_STAGES tiles BEFORE the set-up
  // barrier: the first TMA round trip (~1.8 us cold) overlaps the error-flag load and the shared-memory set-up.
  i64 produced = 0;
  if (tid == GQ_NT) {
    for (int s = 0; s < GQ_STAGES; ++s) { gq_mbar_init(&full_bar[s], 1); gq_mbar_init(&empty_bar[s], GQ_NWARP); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    const u64 pol = gq_policy_evict_first();
    for (i64 tile = blockIdx.x; tile < ntiles && produced < GQ_STAGES; tile += gridDim.x, ++produced)
      gq_produce_tile(P, gq_smem, full_bar, (int)produced, tile, pol);
  }
  GqCtx cx;
  cx.t = tid;
  cx.ninserted = 0;
#if GQ_CONSUMER == GQ_C_LOWCARD
  cx.lc_tab = (u64*)(gq_smem + GQ_CONS_OFF);
  cx.lc_gid = (u32*)(gq_smem + GQ_CONS_OFF + GQ_LC_GID_OFF);
  cx.lc_gkey = (i64*)(gq_smem + GQ_CONS_OFF + GQ_LC_GKEY_OFF);
  cx.lc_n = (int*)(gq_smem + GQ_CONS_OFF + GQ_LC_N_OFF);
  cx.lc_acc = (i64*)(gq_smem + GQ_CONS_OFF + GQ_LC_HEAD_BYTES);
  if (tid < GQ_NT) {
    for (int i = tid; i < GQ_LC_KT; i += GQ_NT) { cx.lc_tab[i] = GQ_LC_KEY32 ? ~0ULL : GQ_EMPTY; cx.lc_gid[i] = 0xFFFFFFFEu; }
    if (tid < 4) cx.lc_n[tid] = 0;
#pragma unroll
    for (int a = 0; a < GQ_NAGG; ++a)
      for (int g = 0; g < GQ_LC_G; ++g) cx.lc_acc[(g * GQ_NAGG + a) * GQ_NT + tid] = gq_identity(GQ_AGG_OP(a));
  }
#endif
#if GQ_CONSUMER == GQ_C_GLOBAL
#pragma unroll
  for (int a = 0; a < GQ_NAGG; ++a) cx.acc[a] = gq_identity(GQ_AGG_OP(a));
#endif
#if GQ_CONSUMER == GQ_C_MATERIALISE
  cx.mat = (int*)(gq_smem + GQ_CONS_OFF);
  if (tid < 4) cx.mat[tid] = 0;
#endif
#if GQ_PART_RW
  cx.part_st = (u32*)(gq_smem + GQ_CONS_OFF + GQ_PART_STATE_OFF);
#if GQ_SC_CLUSTER > 1
  const int nstate = (int)P.npart / GQ_SC_CLUSTER;         // this CTA holds the words of the partitions p with p mod cluster size == its rank
#else
  const int nstate = (int)P.npart;
#endif
  for (int i = tid; i < nstate; i += GQ_NT + 32) cx.part_st[i] = GQ_PART_CHUNK;   // no open chunk yet
#if GQ_CONSUMER == GQ_C_SCATTER
  cx.sc_next = cx.part_st + nstate;
  if (tid == 0) *cx.sc_next = 0;
#endif
#endif
#if GQ_HOT
  cx.hot_keys = (i64*)(gq_smem + GQ_CONS_OFF);
  cx.hot_acc = (u64*)(cx.hot_keys + GQ_HOT_POS);
  cx.hot_touched = (int*)(cx.hot_acc + GQ_HOT_POS * GQ_NAGG);
  cx.hot_ovf = (unsigned char*)(cx.hot_touched + GQ_HOT_POS);
  cx.nhot = 0;
  if (P.hot) { const i64 n = P.hot[0]; cx.nhot = (int)(n < GQ_HOT_MAX ? n : GQ_HOT_MAX); }
  if (cx.nhot > 0) {
    for (int i = tid; i < GQ_HOT_POS; i += GQ_NT + 32) {
      cx.hot_keys[i] = (i64)GQ_EMPTY;
      cx.hot_touched[i] = 0;
      if (i < GQ_HOT_POS / 4) cx.hot_ovf[i] = 0;
#pragma unroll
      for (int a = 0; a < GQ_NAGG; ++a) cx.hot_acc[i * GQ_NAGG + a] = (u64)gq_identity(GQ_AGG_OP(a));
    }
    __syncthreads();
    for (int i = tid; i < cx.nhot; i += GQ_NT + 32) gq_hot_insert(cx, P.hot[32 + i]);   // this batch's hot keys into the shared set (distinct by construction)
  }
#endif
  __syncthreads();
#if GQ_SC_CLUSTER > 1
  gq_cluster_sync();                                     // the peers' state words are initialised before anybody reserves through them
#endif
  if (*err_seen != 0) {
    if (tid == GQ_NT) for (i64 i = 0; i < produced; ++i) gq_mbar_wait(&full_bar[i], 0u);   // copies in flight land before the CTA exits
#if GQ_SC_CLUSTER > 1
    __syncwarp();
    gq_cluster_sync();                                   // a peer that did not see the error may still reserve through this CTA's words
#endif
#if GQ_FUSED_FINAL
    if (tid == 0) {   // keep ticket (and merge table) zeroed for the next kernel
      const u32 t = atomicAdd(P.fin.ticket, 1u);
      if (t == gridDim.x - 1) {
        *P.fin.ticket = 0;
#if GQ_CONSUMER == GQ_C_LOWCARD
        P.fin.gtab[0] = 0;
        for (int i = 0; i < GQ_GTAB_SLOTS * 16; ++i) P.fin.gtab[32 + i] = 0;
#endif
      }
    }
#endif
    return;
  }

  if (tid >= GQ_NT) {
    // ------------------------------------------------------------------ producer warp: TMA bulk copies
    if (tid == GQ_NT) {
      const u64 pol = gq_policy_evict_first();
      i64 it = produced;
      for (i64 tile = blockIdx.x + produced * gridDim.x; tile < ntiles; tile += gridDim.x, ++it) {
        const int s = (int)(it % GQ_STAGES);
        const u32 ph = (u32)((it / GQ_STAGES) & 1);
        gq_mbar_wait(&empty_bar[s], ph ^ 1u);            // the consumers have released the stage
        gq_produce_tile(P, gq_smem, full_bar, s, tile, pol);
      }
    }
#if GQ_SC_CLUSTER > 1
    __syncwarp();
    gq_cluster_sync();                                   // the cluster's final barrier (see the SCATTER epilogue)
#endif
    return;
  }

  // -------------------------------------------------------------------- consumers
  {
    GqSrcSmem src;
    src.t = tid;
    i64 it = 0;
    for (i64 tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
      const int s = (int)(it % GQ_STAGES);
      const u32 ph = (u32)((it / GQ_STAGES) & 1);
      gq_mbar_wait(&full_bar[s], ph);                    // the tile's bytes have landed
      src.stage = gq_smem + (size_t)s * GQ_STAGE_BYTES;
      gq_process(P, src, cx, GQ_R, true);
      __syncwarp();
      if ((tid & 31) == 0) gq_mbar_arrive(&empty_bar[s]);  // this warp is done with the stage
    }
  }
  // ragged tail (< GQ_TILE rows): one CTA reads it straight from global memory
  {
    const i64 row0 = ntiles * GQ_TILE;
    const i64 rem = P.nrows - row0;
    if (rem > 0 && (i64)blockIdx.x == ntiles % gridDim.x) {
      GqSrcGlobal src;
      src.P = &P; src.row0 = row0; src.t = tid;
      // rows tid + j*GQ_NT < rem  <=>  j < ceil((rem - tid) / GQ_NT)
      const int nj = rem > tid ? (int)((rem - tid + GQ_NT - 1) / GQ_NT) : 0;
      gq_process(P, src, cx, nj, false);
    }
  }

  // -------------------------------------------------------------------- consumer epilogues
  const int lane = tid & 31, warp = tid >> 5;
  (void)lane; (void)warp;
#if GQ_CONSUMER == GQ_C_GLOBAL
  {
    // warp shuffle -> shared -> one value per CTA per aggregate
    i64* red = (i64*)(gq_smem + GQ_CONS_OFF);            // [GQ_NAGG][GQ_NWARP], then [4] flags
    int* flag = (int*)(red + GQ_NAGG * GQ_NWARP);
#pragma unroll
    for (int a = 0; a < GQ_NAGG; ++a) {
      i64 v = gq_warp_reduce(GQ_AGG_OP(a), cx.acc[a]);
      if (lane == 0) red[a * GQ_NWARP + warp] = v;
    }
    gq_consumer_barrier();
    if (tid < 32) {
#pragma unroll
      for (int a = 0; a < GQ_NAGG; ++a) {
        i64 v = gq_identity(GQ_AGG_OP(a));
        for (int w = tid; w < GQ_NWARP; w += 32) v = gq_combine(GQ_AGG_OP(a), v, red[a * GQ_NWARP + w]);
        v = gq_warp_reduce(GQ_AGG_OP(a), v);
#if GQ_FUSED_FINAL
        if (tid == 0) P.fin.part[(i64)blockIdx.x * GQ_NAGG + a] = v;
#else
        if (tid == 0) gq_red(GQ_AGG_OP(a), (u64*)&P.acc[a], v);
#endif
      }
    }
#if GQ_FUSED_FINAL
    // last CTA to finish merges the per-CTA partials and writes the single output row
    if (tid == 0) { __threadfence(); flag[0] = (atomicAdd(P.fin.ticket, 1u) == gridDim.x - 1); }
    gq_consumer_barrier();
    if (flag[0]) {
#pragma unroll
      for (int a = 0; a < GQ_NAGG; ++a) {
        i64 v = gq_identity(GQ_AGG_OP(a));
        for (int b = tid; b < (int)gridDim.x; b += GQ_NT) v = gq_combine(GQ_AGG_OP(a), v, gq_ldcg(P.fin.part + (i64)b * GQ_NAGG + a));
        v = gq_warp_reduce(GQ_AGG_OP(a), v);
        if (lane == 0) red[a * GQ_NWARP + warp] = v;
      }
      gq_consumer_barrier();
      if (tid == 0) {
        i64 vals[GQ_NAGG];
#pragma unroll
        for (int a = 0; a < GQ_NAGG; ++a) {
          i64 v = gq_identity(GQ_AGG_OP(a));
          for (int w = 0; w < GQ_NWARP; ++w) v = gq_combine(GQ_AGG_OP(a), v, red[a * GQ_NWARP + w]);
          vals[a] = v;
        }
        if (P.fin.out_capacity >= 1) gq_fin_emit(P.fin, 0, 0, vals);
        else gq_set_err(P.err, GQ_E_CAPACITY);
        *P.fin.out_n = 1;
        *P.fin.ticket = 0;
      }
    }
#endif
  }
#endif
#if GQ_CONSUMER == GQ_C_LOWCARD
  {
    gq_consumer_barrier();
    const int ng = min(((volatile int*)cx.lc_n)[0], GQ_LC_G);   // the counter overshoots when the plan's max_groups is exceeded
#if !GQ_FUSED_FINAL
    // one warp per (group, aggregate): reduce the GQ_NT private cells, merge into the global table
    for (int p0 = warp; p0 < ng * GQ_NAGG; p0 += 4 * GQ_NWARP) {
      i64 v[4];
      gq_lc_reduce4(cx, p0, ng * GQ_NAGG, lane, v);
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int p = p0 + u * GQ_NWARP;
        if (lane == 0 && p < ng * GQ_NAGG) {
          const int g = p / GQ_NAGG, a = p % GQ_NAGG;
          bool won;
          u64* slot = gq_ht_upsert<GQ_TARGET_SW>(P.target, cx.lc_gkey[g], &won, P.err);
          if (slot) gq_red(GQ_AGG_OP(a), slot + 1 + GQ_NDEP + a, v[u]);
        }
      }
    }
#else
    // ---- finaliser fused into the scan: CTA-level reduction -> the CTA's <= GQ_LC_G groups are folded into
    // the context-owned merge table (find-or-claim by key: the claimer stores its values and publishes the slot, later
    // CTAs RED theirs in) -> ticket -> the last CTA only reads the table, emits and zeroes it. Replaces "every CTA
    // writes its partials, the last one folds grid x G of them" (C1: that tail was 6 of 18 us).
    i64* fin = (i64*)(gq_smem + GQ_CONS_OFF + GQ_LC_FIN_OFF);
    u64* gt = P.fin.gtab;
#if GQ_LC_KEY32
    // The first find-or-claim CAS of every group goes out BEFORE the CTA-level reduction and is consumed after it: its
    // round trip to L2 (0.7 us) hides behind the reduction instead of following it.
    u64 st0 = 0;
    if (tid < ng) {
      const i64 key = cx.lc_gkey[tid];
      st0 = atomicCAS(gt + 32 + (u32)gq_hash(key, 64 - 6) * 16, 0ULL, 2ULL | ((u64)GQ_LC_K32(key) << 32));
    }
#endif
    for (int p0 = warp; p0 < ng * GQ_NAGG; p0 += 4 * GQ_NWARP) {
      i64 v[4];
      gq_lc_reduce4(cx, p0, ng * GQ_NAGG, lane, v);
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (lane == 0 && p0 + u * GQ_NWARP < ng * GQ_NAGG) fin[p0 + u * GQ_NWARP] = v[u];
    }
    gq_consumer_barrier();
    if (tid < ng) {
      const i64 key = cx.lc_gkey[tid];
      u32 h = (u32)gq_hash(key, 64 - 6);
      bool done = false;
#if GQ_LC_KEY32
      // Packed keys narrower than 32 bits travel IN the slot's first word (2 | key << 32), and the slot's aggregate words
      // are kept in a form whose identity is ZERO for every operator (gq_gt_enc: MIN/MAX as unsigned maxima of the
      // biased / complemented value), so a zeroed table is a valid empty table for any plan: ONE CAS round trip tells a
      // CTA that the slot is (now) its key's and it can RED straight away — no claim/publish wait.
      const u64 mine = 2ULL | ((u64)GQ_LC_K32(key) << 32);
      for (int n = 0; n < GQ_GTAB_SLOTS && !done; ++n, h = (h + 1) & (GQ_GTAB_SLOTS - 1)) {
        u64* s = gt + 32 + h * 16;
        const u64 st = n == 0 ? st0 : atomicCAS(s, 0ULL, mine);
        if (st != 0 && st != mine) continue;               // another key's slot
        if (st == 0) s[1] = (u64)key;                      // (read by the last CTA only, after every CTA's fence + ticket)
#pragma unroll
        for (int a = 0; a < GQ_NAGG; ++a) {
          const u64 v = gq_gt_enc(GQ_AGG_OP(a), fin[tid * GQ_NAGG + a]);
          if (GQ_AGG_OP(a) == GQ_OP_MIN || GQ_AGG_OP(a) == GQ_OP_MAX) atomicMax(s + 2 + a, v);
          else atomicAdd(s + 2 + a, v);
        }
        done = true;
      }
#else
      for (int n = 0; n < GQ_GTAB_SLOTS && !done; ++n, h = (h + 1) & (GQ_GTAB_SLOTS - 1)) {
        u64* s = gt + 32 + h * 16;
        u64 st = gq_ld_acquire(s);
        if (st == 0) st = atomicCAS(s, 0ULL, 1ULL);
        if (st == 0) {                                     // claimed: store key and values, then publish
          s[1] = (u64)key;
#pragma unroll
          for (int a = 0; a < GQ_NAGG; ++a) s[2 + a] = gq_gt_enc(GQ_AGG_OP(a), fin[tid * GQ_NAGG + a]);
          gq_st_release(s, 2ULL);
          done = true;
          break;
        }
        while (st == 1) st = gq_ld_acquire(s);             // being published by another CTA
        if (s[1] == (u64)key) {
#pragma unroll
          for (int a = 0; a < GQ_NAGG; ++a) {
            const u64 v = gq_gt_enc(GQ_AGG_OP(a), fin[tid * GQ_NAGG + a]);
            if (GQ_AGG_OP(a) == GQ_OP_MIN || GQ_AGG_OP(a) == GQ_OP_MAX) atomicMax(s + 2 + a, v);
            else atomicAdd(s + 2 + a, v);
          }
          done = true;
        }
      }
#endif
      if (!done) gq_set_err(P.err, GQ_E_CAPACITY);
    }
    gq_consumer_barrier();
    // ticket: release (this CTA's table updates, ordered before by the barrier) and acquire (the last CTA reads the table)
    if (tid == 0) cx.lc_n[3] = (gq_atom_add_acq_rel(P.fin.ticket, 1u) == gridDim.x - 1);
    gq_consumer_barrier();
    if (((volatile int*)cx.lc_n)[3]) {
      // (the table is read with ld.cg, after thread 0's acquire and the CTA barrier)
      if (tid < GQ_GTAB_SLOTS) {                            // warps 0 and 1: one slot per lane
        u64* s = gt + 32 + tid * 16;
        i64 wd[2 + GQ_NAGG];                                // state, key and values of the slot: all loads in flight together
#pragma unroll
        for (int i = 0; i < 2 + GQ_NAGG; ++i) wd[i] = __ldcg((const i64*)s + i);
        const bool have = ((u64)wd[0] & 3ULL) == 2ULL;
        const u32 m = __ballot_sync(0xffffffffu, have);
        if (tid == 31) cx.lc_n[2] = __popc(m);            // groups in slots 0..31 (lc_n[2] is free by now)
        asm volatile("bar.sync 2, 64;" ::: "memory");
        const int row = (tid >= 32 ? ((volatile int*)cx.lc_n)[2] : 0) + __popc(m & ((1u << lane) - 1u));
        if (have) {
#pragma unroll
          for (int a = 0; a < GQ_NAGG; ++a) wd[2 + a] = gq_gt_dec(GQ_AGG_OP(a), (u64)wd[2 + a]);
          if (row < P.fin.out_capacity) gq_fin_emit(P.fin, row, wd[1], wd + 2);
          else gq_set_err(P.err, GQ_E_CAPACITY);
#pragma unroll
          for (int i = 0; i < 2 + GQ_NAGG; ++i) s[i] = 0;   // a zeroed slot is an empty slot with identity aggregates
        }
        if (tid == 63) {
          if (row + (have ? 1 : 0) > GQ_LC_G) gq_set_err(P.err, GQ_E_CAPACITY);   // more distinct keys than max_groups
          *P.fin.out_n = row + (have ? 1 : 0); gt[0] = 0; *P.fin.ticket = 0;
        }
      }
    }
#endif
  }
#endif
#if GQ_HOT
  if (cx.nhot > 0) {   // flush the CTA's hot-key partials into the global table (Partial -> Final)
    gq_consumer_barrier();
    for (int pos = tid; pos < GQ_HOT_POS; pos += GQ_NT) {
      if (!cx.hot_touched[pos]) continue;
      bool won;
      u64* slot = gq_ht_upsert<GQ_TARGET_SW>(P.target, cx.hot_keys[pos], &won, P.err);
      if (!slot) continue;
#pragma unroll
      for (int a = 0; a < GQ_NAGG; ++a) gq_red(GQ_AGG_OP(a), slot + 1 + GQ_NDEP + a, (i64)cx.hot_acc[pos * GQ_NAGG + a]);
    }
  }
#endif
#if GQ_CONSUMER == GQ_C_SCATTER
#if GQ_SC_CLUSTER > 1
  {   // every CTA of the cluster has stopped reserving: each records how far the part-filled chunks of ITS partitions got
    __syncwarp();
    gq_cluster_sync();
    const u32 rank = gq_cluster_rank();
    const u64 cbase = (u64)gq_cluster_id() * (u64)P.sc_slab;
    for (int q = tid; q < nstate; q += GQ_NT) {
      const u32 v = cx.part_st[q];
      const u32 used = v & 0xFFFu;
      if (used < GQ_PART_CHUNK) P.sc_info[cbase + (v >> 12)] = (((u32)q * GQ_SC_CLUSTER + rank) << 8) | used;
    }
    if (tid == 0 && rank == 0) { const u32 n = *cx.sc_next; P.sc_ncta[gq_cluster_id()] = n < (u32)P.sc_slab ? n : (u32)P.sc_slab; }
  }
#else
  {   // record how far this CTA's part-filled chunks got, and how many chunks it opened
    gq_consumer_barrier();
    for (int p = tid; p < (int)P.npart; p += GQ_NT) {
      const u32 v = cx.part_st[p];
      const u32 used = v & 0xFFFu;
      if (used < GQ_PART_CHUNK) P.sc_info[(u64)blockIdx.x * (u64)P.sc_slab + (v >> 12)] = ((u32)p << 8) | used;
    }
    if (tid == 0) { const u32 n = *cx.sc_next; P.sc_ncta[blockIdx.x] = n < (u32)P.sc_slab ? n : (u32)P.sc_slab; }
  }
#endif
#elif GQ_PART_RW
  {   // pad the unused slots of this CTA's open chunks with EMPTY-key records (pass B skips them)
    gq_consumer_barrier();
    for (int p = tid; p < (int)P.npart; p += GQ_NT) {
      const u32 v = cx.part_st[p];
      const u32 used = v & 0xFFFFu, chunk = v >> 16;
      if (chunk == 0xFFFFu || used >= GQ_PART_CHUNK || (chunk == 0 && v == GQ_PART_CHUNK)) continue;
      u64* rec = P.part + ((u64)p * (u64)P.pcap + (u64)chunk * GQ_PART_CHUNK) * GQ_PART_RW;
      for (u32 i = used; i < GQ_PART_CHUNK; ++i) rec[(u64)i * GQ_PART_RW] = GQ_EMPTY;
    }
  }
#endif
#if GQ_CONSUMER == GQ_C_BUILD
  {
    i64 v = gq_warp_reduce(GQ_OP_SUM, cx.ninserted);
    if (lane == 0 && v != 0) atomicAdd((u64*)&P.target.header[0], (u64)v);
  }
#endif
}
