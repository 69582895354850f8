// gq_skeleton_kernel.cuh — second half of the fused scan kernel (follows the generated gq_pass / gq_body).

// Shared-memory layout (dynamic): [GQ_STAGES stages][full/empty mbarriers][consumer area]
#define GQ_BAR_OFF (GQ_STAGES * GQ_STAGE_BYTES)
#define GQ_CONS_OFF (GQ_BAR_OFF + 2 * GQ_STAGES * 8 + 64)
#define GQ_LC_KEYS_BYTES (((GQ_LC_CAP + 1) * 8 + 8 + 127) / 128 * 128)

template <class Src>
__device__ __forceinline__ void gq_process(const GqParams& P, const Src& src, GqCtx& cx, int nvalid_j, bool full) {
#if GQ_LINEAR
  gq_tile(P, src, cx, nvalid_j, full);   // generated: the GQ_R rows advance step by step, accesses issued before use
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

extern "C" __global__ void __launch_bounds__(GQ_NT + 32, 1) gq_scan(const __grid_constant__ GqParams P) {
  extern __shared__ __align__(128) unsigned char gq_smem[];
  u64* full_bar = (u64*)(gq_smem + GQ_BAR_OFF);
  u64* empty_bar = full_bar + GQ_STAGES;
  const int tid = threadIdx.x;
  const i64 ntiles = P.nrows / GQ_TILE;                  // full tiles; the remainder is the tail
  if (*(volatile int*)P.err != 0) return;                // sticky error: later kernels are no-ops (gq.h "Errors")

  if (tid == 0) {
    for (int s = 0; s < GQ_STAGES; ++s) { gq_mbar_init(&full_bar[s], 1); gq_mbar_init(&empty_bar[s], GQ_NWARP); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  GqCtx cx;
  cx.t = tid;
  cx.ninserted = 0;
#if GQ_CONSUMER == GQ_C_LOWCARD
  cx.lc_keys = (i64*)(gq_smem + GQ_CONS_OFF);
  cx.lc_side_used = (int*)(cx.lc_keys + GQ_LC_CAP + 1);
  cx.lc_acc = (i64*)(gq_smem + GQ_CONS_OFF + GQ_LC_KEYS_BYTES);
  if (tid < GQ_NT) {
    for (int i = tid; i <= GQ_LC_CAP; i += GQ_NT) cx.lc_keys[i] = (i64)GQ_EMPTY;
    if (tid == 0) *cx.lc_side_used = 0;
#pragma unroll
    for (int a = 0; a < GQ_NAGG; ++a)
      for (int g = 0; g <= GQ_LC_CAP; ++g) cx.lc_acc[(g * GQ_NAGG + a) * GQ_NT + tid] = gq_identity(GQ_AGG_OP(a));
  }
#endif
#if GQ_CONSUMER == GQ_C_GLOBAL
#pragma unroll
  for (int a = 0; a < GQ_NAGG; ++a) cx.acc[a] = gq_identity(GQ_AGG_OP(a));
#endif
#if GQ_HOT
  cx.hot_keys = (i64*)(gq_smem + GQ_CONS_OFF);
  cx.hot_acc = (u64*)(cx.hot_keys + GQ_HOT_POS);
  cx.hot_touched = (int*)(cx.hot_acc + GQ_HOT_POS * GQ_NAGG);
  cx.nhot = 0;
  if (P.hot) { const i64 n = P.hot[0]; cx.nhot = (int)(n < GQ_HOT_MAX ? n : GQ_HOT_MAX); }
  if (cx.nhot > 0) {
    for (int i = tid; i < GQ_HOT_POS; i += GQ_NT + 32) {
      cx.hot_keys[i] = (i64)GQ_EMPTY;
      cx.hot_touched[i] = 0;
#pragma unroll
      for (int a = 0; a < GQ_NAGG; ++a) cx.hot_acc[i * GQ_NAGG + a] = (u64)gq_identity(GQ_AGG_OP(a));
    }
    __syncthreads();
    if (tid < cx.nhot) {   // insert this batch's hot keys into the shared set (distinct by construction)
      const i64 key = P.hot[1 + tid];
      u32 i = (u32)gq_hash(key, 64 - 16) & (GQ_HOT_POS - 1);
      for (int n = 0; n < GQ_HOT_POS; ++n, i = (i + 1) & (GQ_HOT_POS - 1))
        if (atomicCAS((u64*)&cx.hot_keys[i], GQ_EMPTY, (u64)key) == GQ_EMPTY) break;
    }
  }
#endif
  __syncthreads();

  if (tid >= GQ_NT) {
    // ------------------------------------------------------------------ producer warp: TMA bulk copies
    if (tid == GQ_NT) {
      const u64 pol = gq_policy_evict_first();
      i64 it = 0;
      for (i64 tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        const int s = (int)(it % GQ_STAGES);
        const u32 ph = (u32)((it / GQ_STAGES) & 1);
        gq_mbar_wait(&empty_bar[s], ph ^ 1u);            // stage free (first pass through the ring: immediately)
        gq_mbar_expect_tx(&full_bar[s], (u32)GQ_TX_BYTES);
        unsigned char* st = gq_smem + (size_t)s * GQ_STAGE_BYTES;
#pragma unroll
        for (int c = 0; c < GQ_NCOL; ++c)
          gq_bulk_g2s(st + GQ_COL_OFF(c), (const unsigned char*)P.col[c] + (size_t)tile * GQ_TILE * GQ_COL_BYTES(c),
                      (u32)(GQ_TILE * GQ_COL_BYTES(c)), &full_bar[s], pol);
      }
    }
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
#if GQ_CONSUMER == GQ_C_GLOBAL
  {
    // warp shuffle -> shared -> one atomic per CTA per aggregate
    i64* red = (i64*)(gq_smem + GQ_CONS_OFF);            // [GQ_NAGG][GQ_NWARP]
#pragma unroll
    for (int a = 0; a < GQ_NAGG; ++a) {
      i64 v = gq_warp_reduce(GQ_AGG_OP(a), cx.acc[a]);
      if ((tid & 31) == 0) red[a * GQ_NWARP + (tid >> 5)] = v;
    }
    gq_consumer_barrier();
    if (tid < 32) {
#pragma unroll
      for (int a = 0; a < GQ_NAGG; ++a) {
        i64 v = gq_identity(GQ_AGG_OP(a));
        for (int w = tid; w < GQ_NWARP; w += 32) v = gq_combine(GQ_AGG_OP(a), v, red[a * GQ_NWARP + w]);
        v = gq_warp_reduce(GQ_AGG_OP(a), v);
        if (tid == 0) gq_red(GQ_AGG_OP(a), (u64*)&P.acc[a], v);
      }
    }
  }
#endif
#if GQ_CONSUMER == GQ_C_LOWCARD
  {
    gq_consumer_barrier();
    // one thread per (group position, aggregate): reduce the GQ_NT private cells, merge into the global table
    for (int pa = tid; pa < (GQ_LC_CAP + 1) * GQ_NAGG; pa += GQ_NT) {
      const int g = pa / GQ_NAGG, a = pa % GQ_NAGG;
      const bool used = g < GQ_LC_CAP ? ((u64)cx.lc_keys[g] != GQ_EMPTY) : (*cx.lc_side_used != 0);
      if (!used) continue;
      const i64 key = g < GQ_LC_CAP ? cx.lc_keys[g] : (i64)GQ_EMPTY;
      const i64* cells = cx.lc_acc + (size_t)pa * GQ_NT;
      i64 v = 0;
      bool won;
      u64* slot = gq_ht_upsert<GQ_TARGET_SW>(P.target, key, &won, P.err);
      if (!slot) continue;
      // the aggregate's op is only known per `a` at compile time: dispatch over the (few) aggregates
#pragma unroll
      for (int aa = 0; aa < GQ_NAGG; ++aa) {
        if (aa == a) {
          v = gq_identity(GQ_AGG_OP(aa));
          for (int i = 0; i < GQ_NT; ++i) v = gq_combine(GQ_AGG_OP(aa), v, cells[(i + tid) % GQ_NT]);
          gq_red(GQ_AGG_OP(aa), slot + 1 + GQ_NDEP + aa, v);
        }
      }
    }
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
#if GQ_CONSUMER == GQ_C_BUILD
  {
    i64 v = gq_warp_reduce(GQ_OP_SUM, cx.ninserted);
    if ((tid & 31) == 0 && v != 0) atomicAdd((u64*)&P.target.header[0], (u64)v);
  }
#endif
}
