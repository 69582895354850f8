// gq_static.cu — plan-independent sm_100a kernels, compiled by nvcc into libgq.so: hash-table initialisation, the
// HashAggregation finaliser (table -> dense output columns + device-side group count + derived AVG),
// the top-k finaliser (OrderBy/TopN in its smallest form) and the read-roofline probe.
#include <algorithm>

#include "gq_internal.h"

typedef unsigned long long u64;
typedef long long i64;

// ------------------------------------------------------------------------------------------------ table init
// Writes the slot pattern (key = EMPTY, dependent words 0, aggregate identities) with 128-bit stores where the slot
// size allows; zeroes the header (header[1] = header1) and marks side slots empty.
__global__ void gq_k_init_table(u64* slots, i64 nwords, int sw, const __grid_constant__ ulonglong4 pat0,
                                const __grid_constant__ ulonglong4 pat1, const __grid_constant__ ulonglong4 pat2,
                                const __grid_constant__ ulonglong4 pat3, u64* side, i64 nside_words, i64* header, i64 header1) {
  const u64 pat[16] = {pat0.x, pat0.y, pat0.z, pat0.w, pat1.x, pat1.y, pat1.z, pat1.w,
                       pat2.x, pat2.y, pat2.z, pat2.w, pat3.x, pat3.y, pat3.z, pat3.w};
  const i64 stride = (i64)gridDim.x * blockDim.x;
  const i64 t0 = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  // slot sizes are multiples of 2 words (or 1 word: key-only tables) -> pairs of words never straddle the pattern oddly
  if ((sw & 1) == 0) {
    ulonglong2* s2 = (ulonglong2*)slots;
    const i64 npairs = nwords / 2;
    const int pw = sw / 2;
    for (i64 i = t0; i < npairs; i += stride) {
      int k = (int)(i % pw) * 2;
      s2[i] = make_ulonglong2(pat[k], pat[k + 1]);
    }
  } else {
    for (i64 i = t0; i < nwords; i += stride) slots[i] = pat[i % sw];
  }
  for (i64 i = t0; i < nside_words; i += stride) side[i] = pat[i % sw];
  if (t0 < 32) header[t0] = (t0 == 1) ? header1 : 0;
}

cudaError_t gq_launch_init_table(cudaStream_t s, u64* slots, i64 nslots, int sw, const u64* pattern, u64* side,
                                 i64 nside, i64* header, i64 header1, int num_sms) {
  ulonglong4 p[4];
  u64* pp = (u64*)p;
  for (int i = 0; i < 16; ++i) pp[i] = pattern[i % sw];
  i64 nwords = nslots * sw;
  i64 work = (sw & 1) == 0 ? nwords / 2 : nwords;
  int blocks = (int)std::min<i64>((i64)num_sms * 16, std::max<i64>(1, (work + 255) / 256));
  gq_k_init_table<<<blocks, 256, 0, s>>>(slots, nwords, sw, p[0], p[1], p[2], p[3], side, nside * sw, header, header1);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ finalise (dense)
__device__ __forceinline__ i64 gq_sext(u64 v, int bits) {
  if (bits >= 64) return (i64)v;
  u64 m = 1ULL << (bits - 1);
  v &= (1ULL << bits) - 1;
  return (i64)((v ^ m) - m);
}
__device__ __forceinline__ void gq_store_key(void* col, int dtype, i64 idx, i64 v) {
  if (dtype == GQ_I8) ((signed char*)col)[idx] = (signed char)v;
  else if (dtype == GQ_I32) ((int*)col)[idx] = (int)v;
  else ((i64*)col)[idx] = v;
}
// A group as the finalisers see it. Hashed state: slot i of the group-by table (key word, dependent words, aggregate
// words). Direct state: accumulator slot i is a group iff its touch word (a COUNT) is non-zero; key and dependent key
// come from slot i of the join table the scan probed. Index `capacity` (direct) / -2 (hashed) names the side entry.
struct GqGroupRef { u64 key; const u64* dep; const u64* agg; };
__device__ __forceinline__ bool gq_group_at(const GqFinaliseParams& P, i64 i, GqGroupRef* g) {
  if (P.direct) {
    const u64* acc = P.dacc + i * P.daw;
    if (acc[P.dtouch] == 0) return false;
    if (P.jdense) {   // direct-address join table: slot i = rank of the key among the build keys; jside = key of every rank,
      if (i >= P.capacity) return false;   // jslots = payload rows indexed by key - key_min
      g->key = P.jside[i];
      g->dep = P.jslots + (u64)((i64)g->key - P.jbase) * P.jnpay + (P.dep_pay > 0 ? P.dep_pay : 0);
      g->agg = acc;
      return true;
    }
    const u64* js = i < P.capacity ? P.jslots + i * P.jsw : P.jside;
    g->key = i < P.capacity ? js[0] : GQ_EMPTY_KEY;
    g->dep = js + 1 + (P.dep_pay > 0 ? P.dep_pay : 0);
    g->agg = acc;
    return true;
  }
  const u64* s = i == -2 ? P.side : P.slots + i * P.slot_words;
  g->key = i == -2 ? GQ_EMPTY_KEY : s[0];
  g->dep = s + 1;
  g->agg = s + 1 + P.ndep;
  return i == -2 ? P.header[1] != 0 : g->key != GQ_EMPTY_KEY;
}
// Emits one group at output row idx.
__device__ __forceinline__ void gq_emit_group(const GqFinaliseParams& P, const GqGroupRef& g, i64 idx) {
  const int nhashed = P.nkeys - P.ndep;
  if (nhashed == 1) gq_store_key(P.out_key[0], P.key_dtype[0], idx, (i64)g.key);
  else if (nhashed == 2) {
    gq_store_key(P.out_key[0], P.key_dtype[0], idx, gq_sext(g.key, P.key_bits[0]));
    gq_store_key(P.out_key[1], P.key_dtype[1], idx, gq_sext(g.key >> P.key_bits[0], P.key_bits[1]));
  }
  for (int d = 0; d < P.ndep; ++d) gq_store_key(P.out_key[nhashed + d], P.key_dtype[nhashed + d], idx, (i64)g.dep[d]);
  for (int a = 0; a < P.naggs; ++a) P.out_agg[a][idx] = (i64)g.agg[a];
  for (int v = 0; v < P.navg; ++v)
    P.out_avg[v][idx] = (double)(i64)g.agg[P.avg_sum[v]] / (double)(i64)g.agg[P.avg_cnt[v]];
}

// One thread per GQ_FIN_PER slots; block-level compaction: ballot/popc inside warps, shared-memory scan over warps,
// ONE atomicAdd per block on the device-side group count.
#define GQ_FIN_THREADS 256
#define GQ_FIN_PER 4
__global__ void __launch_bounds__(GQ_FIN_THREADS) gq_k_finalise(const __grid_constant__ GqFinaliseParams P) {
  __shared__ int warp_cnt[GQ_FIN_THREADS / 32];
  __shared__ i64 block_base;
  if (*(volatile int*)P.err != 0) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const i64 nblocks_slots = (P.capacity + GQ_FIN_THREADS * GQ_FIN_PER - 1) / (GQ_FIN_THREADS * GQ_FIN_PER);
  for (i64 b = blockIdx.x; b < nblocks_slots; b += gridDim.x) {
    const i64 base = b * (GQ_FIN_THREADS * GQ_FIN_PER);
    GqGroupRef grp[GQ_FIN_PER];
    bool have[GQ_FIN_PER];
    int mine = 0;
#pragma unroll
    for (int j = 0; j < GQ_FIN_PER; ++j) {
      i64 i = base + j * GQ_FIN_THREADS + threadIdx.x;
      have[j] = (i < P.capacity) && gq_group_at(P, i, &grp[j]);
      mine += have[j];
    }
    // exclusive prefix of `mine` inside the block
    int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int n = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += n; }
    if (lane == 31) warp_cnt[warp] = incl;
    __syncthreads();
    if (threadIdx.x == 0) {
      int tot = 0;
      for (int w = 0; w < GQ_FIN_THREADS / 32; ++w) { int c = warp_cnt[w]; warp_cnt[w] = tot; tot += c; }
      block_base = tot ? (i64)atomicAdd((u64*)P.out_n, (u64)tot) : 0;
    }
    __syncthreads();
    i64 idx = block_base + warp_cnt[warp] + (incl - mine);
#pragma unroll
    for (int j = 0; j < GQ_FIN_PER; ++j) {
      if (!have[j]) continue;
      if (idx < P.out_capacity) gq_emit_group(P, grp[j], idx);
      else atomicCAS(P.err, 0, (int)GQ_ERR_CAPACITY);
      ++idx;
    }
    __syncthreads();
  }
  // the side slot: the group whose key equals the reserved EMPTY pattern, or THE group of a key-less aggregation
  GqGroupRef sg;
  if (blockIdx.x == 0 && threadIdx.x == 0 && gq_group_at(P, P.direct ? P.capacity : -2, &sg)) {
    i64 idx = (i64)atomicAdd((u64*)P.out_n, 1ULL);
    if (idx < P.out_capacity) gq_emit_group(P, sg, idx);
    else atomicCAS(P.err, 0, (int)GQ_ERR_CAPACITY);
  }
}

// ------------------------------------------------------------------------------------------------ finalise (top-k)
// Order: aggregate descending, then key tuple ascending — a total order, so the answer is unique.
struct GqCand { i64 val, k0, k1, slot; int valid; };
__device__ __forceinline__ bool gq_better(const GqCand& a, const GqCand& b) {   // a strictly before b
  if (!a.valid) return false;
  if (!b.valid) return true;
  if (a.val != b.val) return a.val > b.val;
  if (a.k0 != b.k0) return a.k0 < b.k0;
  return a.k1 < b.k1;
}
__device__ __forceinline__ GqCand gq_cand_shfl(const GqCand& c, int src) {
  GqCand r;
  r.val = __shfl_sync(0xffffffffu, c.val, src); r.k0 = __shfl_sync(0xffffffffu, c.k0, src);
  r.k1 = __shfl_sync(0xffffffffu, c.k1, src); r.slot = __shfl_sync(0xffffffffu, c.slot, src);
  r.valid = __shfl_sync(0xffffffffu, c.valid, src);
  return r;
}
// Warp-distributed sorted list: lane i holds the i-th best entry. Inserts warp-uniform candidate c.
__device__ __forceinline__ void gq_list_insert(GqCand& mine, const GqCand& c, int lane) {
  unsigned before = __ballot_sync(0xffffffffu, gq_better(mine, c));   // entries that stay ahead of c (a prefix)
  int pos = __popc(before);
  GqCand up;
  up.val = __shfl_up_sync(0xffffffffu, mine.val, 1); up.k0 = __shfl_up_sync(0xffffffffu, mine.k0, 1);
  up.k1 = __shfl_up_sync(0xffffffffu, mine.k1, 1); up.slot = __shfl_up_sync(0xffffffffu, mine.slot, 1);
  up.valid = __shfl_up_sync(0xffffffffu, mine.valid, 1);
  if (lane == pos) mine = c;
  else if (lane > pos) mine = up;
}
__device__ __forceinline__ GqCand gq_make_cand(const GqFinaliseParams& P, const GqGroupRef& g, i64 slot) {
  GqCand c;
  c.valid = 1; c.slot = slot; c.k1 = 0;
  c.val = (i64)g.agg[P.topk_agg];
  const int nhashed = P.nkeys - P.ndep;
  if (nhashed == 2) { c.k0 = gq_sext(g.key, P.key_bits[0]); c.k1 = gq_sext(g.key >> P.key_bits[0], P.key_bits[1]); }
  else { c.k0 = (i64)g.key; if (P.ndep) c.k1 = (i64)g.dep[0]; }
  return c;
}
// Feeds the candidates held by the lanes in `m` (each better than the list's current worst) into the list.
// `kth` = topk - 1: only the first topk entries matter, so admission compares with entry kth (entries behind it are
// pushed-down leftovers that stay sorted and are never read).
__device__ __forceinline__ void gq_list_feed(GqCand& mine, const GqCand& c, bool want, int lane, int kth) {
  unsigned m = __ballot_sync(0xffffffffu, want);
  while (m) {
    int src = __ffs(m) - 1;
    m &= m - 1;
    GqCand b = gq_cand_shfl(c, src);
    GqCand worst = gq_cand_shfl(mine, kth);
    if (gq_better(b, worst)) gq_list_insert(mine, b, lane);
  }
}
#define GQ_TOPK_BLOCKS 592
#define GQ_TOPK_WARPS 8
#define GQ_TOPK_UNROLL 4
// scratch layout: [GQ_TOPK_BLOCKS][32] GqCand lists | [GQ_TOPK_BOUND_BLOCKS] i64 sample maxima | [GQ_TOPK_BLOCKS] int entries per list
#define GQ_TOPK_BOUND_BLOCKS 64
#define GQ_TOPK_BOUND_PER 16
#define GQ_TOPK_NONE ((i64)0x8000000000000000LL)
#define GQ_TOPK_RANK_MAX 1024   // entries the merge ranks by counting (4 x 8 B each in the merge's shared memory)
__device__ __forceinline__ i64* gq_topk_maxima(const GqFinaliseParams& P) { return (i64*)((GqCand*)P.scratch + 32 * GQ_TOPK_BLOCKS); }
__device__ __forceinline__ int* gq_topk_counts(const GqFinaliseParams& P) { return (int*)(gq_topk_maxima(P) + GQ_TOPK_BOUND_BLOCKS); }
// validity and ordering aggregate of slot i (loaded unconditionally: several of these are in flight per thread)
__device__ __forceinline__ void gq_topk_peek(const GqFinaliseParams& P, i64 i, u64& tv, i64& vv) {
  const i64 ii = i < P.capacity ? i : 0;
  if (P.direct) { tv = P.dacc[ii * P.daw + P.dtouch]; vv = (i64)P.dacc[ii * P.daw + P.topk_agg]; }
  else {
    const u64* sl = P.slots + ii * P.slot_words;
    tv = sl[0] != GQ_EMPTY_KEY; vv = (i64)sl[1 + P.ndep + P.topk_agg];
  }
  if (i >= P.capacity) tv = 0;
}
// pass 0: an admission bound for pass 1. Every block takes the maximum of the ordering aggregate over a strided sample of
// the table; the k-th largest of the GQ_TOPK_BOUND_BLOCKS maxima is a value that at least k groups reach, so no group
// below it can be among the first k. (Without it every warp of pass 1 fills and sorts a list of its own first: the scan
// was bound by shuffles, 97 us for 132 MB on C3.)
__global__ void __launch_bounds__(256) gq_k_topk_bound(const __grid_constant__ GqFinaliseParams P) {
  __shared__ i64 wmax[8];
  const i64 nt = (i64)GQ_TOPK_BOUND_BLOCKS * 256;
  const i64 t = (i64)blockIdx.x * 256 + threadIdx.x;
  i64 stride = P.capacity / (nt * GQ_TOPK_BOUND_PER);
  if (stride < 1) stride = 1;
  u64 tv[GQ_TOPK_BOUND_PER];
  i64 vv[GQ_TOPK_BOUND_PER];
#pragma unroll
  for (int u = 0; u < GQ_TOPK_BOUND_PER; ++u) gq_topk_peek(P, ((i64)u * nt + t) * stride, tv[u], vv[u]);
  i64 best = GQ_TOPK_NONE;
#pragma unroll
  for (int u = 0; u < GQ_TOPK_BOUND_PER; ++u) if (tv[u] != 0 && vv[u] > best) best = vv[u];
  for (int o = 16; o > 0; o >>= 1) { const i64 x = __shfl_xor_sync(0xffffffffu, best, o); if (x > best) best = x; }
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) if (wmax[w] > best) best = wmax[w];
    gq_topk_maxima(P)[blockIdx.x] = best;
  }
}
// the k-th largest of the sample maxima (GQ_TOPK_NONE = "no bound" when fewer than k blocks saw a group); warp-uniform
__device__ __forceinline__ i64 gq_topk_bound_value(const GqFinaliseParams& P, int lane) {
  const i64* M = gq_topk_maxima(P);
  const i64 m0 = M[lane], m1 = M[lane + 32];
  int c0 = 0, c1 = 0;
  for (int j = 0; j < 32; ++j) {
    const i64 a = __shfl_sync(0xffffffffu, m0, j), b = __shfl_sync(0xffffffffu, m1, j);
    c0 += (a >= m0) + (b >= m0);
    c1 += (a >= m1) + (b >= m1);
  }
  i64 best = GQ_TOPK_NONE;
  if (c0 >= P.topk && m0 > best) best = m0;
  if (c1 >= P.topk && m1 > best) best = m1;
  for (int o = 16; o > 0; o >>= 1) { const i64 x = __shfl_xor_sync(0xffffffffu, best, o); if (x > best) best = x; }
  return best;
}
// pass 1: every warp scans a strided share of the table (GQ_TOPK_UNROLL chunks of 32 slots in flight) and keeps its
// own best list; lists go to scratch.
__global__ void __launch_bounds__(GQ_TOPK_WARPS * 32, 4) gq_k_topk_scan(const __grid_constant__ GqFinaliseParams P) {
  if (*(volatile int*)P.err != 0) return;
  const int lane = threadIdx.x & 31;
  const int kth = P.topk - 1;
  const i64 gw = (i64)blockIdx.x * GQ_TOPK_WARPS + (threadIdx.x >> 5);
  const i64 nw = (i64)gridDim.x * GQ_TOPK_WARPS;
  GqCand mine; mine.valid = 0; mine.val = 0; mine.k0 = 0; mine.k1 = 0; mine.slot = -1;
  if (gw == 0) {   // the side slot
    GqCand c; c.valid = 0; c.val = 0; c.k0 = 0; c.k1 = 0; c.slot = -1;
    bool want = false;
    GqGroupRef g;
    const i64 si = P.direct ? P.capacity : -2;
    if (lane == 0 && gq_group_at(P, si, &g)) { c = gq_make_cand(P, g, si); want = true; }
    gq_list_feed(mine, c, want, lane, kth);
  }
  // admission bound, warp-uniform: the larger of pass 0's bound and the value of the list's k-th entry; refreshed after
  // every insertion, so the common iteration is two loads, a compare and a vote
  i64 bound = gq_topk_bound_value(P, lane);
  {
    const GqCand w0 = gq_cand_shfl(mine, kth);
    if (w0.valid && w0.val > bound) bound = w0.val;
  }
  for (i64 i0 = gw * 32; i0 < P.capacity; i0 += nw * 32 * GQ_TOPK_UNROLL) {
    // validity word and ordering aggregate of GQ_TOPK_UNROLL slots, loaded unconditionally (all in flight together);
    // the full candidate (keys) is only built for the few slots that can still enter the list
    u64 tv[GQ_TOPK_UNROLL];
    i64 vv[GQ_TOPK_UNROLL];
#pragma unroll
    for (int u = 0; u < GQ_TOPK_UNROLL; ++u) gq_topk_peek(P, i0 + (i64)u * nw * 32 + lane, tv[u], vv[u]);
#pragma unroll
    for (int u = 0; u < GQ_TOPK_UNROLL; ++u) {
      bool want = tv[u] != 0 && vv[u] >= bound;
      if (!__any_sync(0xffffffffu, want)) continue;
      const i64 i = i0 + (i64)u * nw * 32 + lane;
      const GqCand worst = gq_cand_shfl(mine, kth);
      GqCand c; c.valid = 0; c.val = 0; c.k0 = 0; c.k1 = 0; c.slot = -1;
      if (want) {
        GqGroupRef g;
        want = gq_group_at(P, i, &g);
        if (want) { c = gq_make_cand(P, g, i); want = gq_better(c, worst); }
      }
      gq_list_feed(mine, c, want, lane, kth);
      const GqCand w1 = gq_cand_shfl(mine, kth);
      if (w1.valid && w1.val > bound) bound = w1.val;
    }
  }
  // merge the block's GQ_TOPK_WARPS lists into one (warp 0), so pass 2 sees one list per block
  __shared__ GqCand sh[GQ_TOPK_WARPS][32];
  sh[threadIdx.x >> 5][lane] = mine;
  __syncthreads();
  if ((threadIdx.x >> 5) == 0) {
    for (int w = 1; w < GQ_TOPK_WARPS; ++w) {
      GqCand c = sh[w][lane];
      GqCand worst = gq_cand_shfl(mine, kth);
      gq_list_feed(mine, c, c.valid && lane <= kth && gq_better(c, worst), lane, kth);   // entries behind the k-th of a sorted list cannot matter
    }
    ((GqCand*)P.scratch)[(i64)blockIdx.x * 32 + lane] = mine;
    const unsigned have = __ballot_sync(0xffffffffu, mine.valid != 0 && lane <= kth);
    if (lane == 0) gq_topk_counts(P)[blockIdx.x] = __popc(have);
  }
}
// pass 2: one block; every warp merges a strided share of the per-block lists (two lists in flight), warp 0 merges the
// warps' results and writes the first min(k, ngroups) groups in order.
#define GQ_TOPK_MERGE_WARPS 32
__global__ void __launch_bounds__(GQ_TOPK_MERGE_WARPS * 32) gq_k_topk_merge(const __grid_constant__ GqFinaliseParams P, i64 nlists) {
  if (*(volatile int*)P.err != 0) return;
  __shared__ __align__(16) unsigned char shbuf[sizeof(GqCand) * 32 * GQ_TOPK_MERGE_WARPS];
  __shared__ int s_off[GQ_TOPK_BLOCKS + 1], s_wsum[GQ_TOPK_MERGE_WARPS];
  GqCand (*sh)[32] = (GqCand (*)[32])shbuf;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int kth = P.topk - 1;
  const GqCand* in = (const GqCand*)P.scratch;
  // ---- few entries in all lists together (the usual case with pass 0's bound: a few hundred): gather them in shared
  // memory, every thread counts how many entries come before its own, ranks below k are output rows. (Feeding them
  // through sorted warp lists is a chain of ~60 dependent shuffle instructions per entry: 25 us.)
  {
    const int t = threadIdx.x;
    const int c = t < nlists ? gq_topk_counts(P)[t] : 0;   // (nlists = GQ_TOPK_BLOCKS <= blockDim.x)
    int incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int x = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += x; }
    if (lane == 31) s_wsum[warp] = incl;
    __syncthreads();
    int before = 0;
    for (int w = 0; w < warp; ++w) before += s_wsum[w];
    if (t < nlists) s_off[t] = before + incl - c;
    if (t == GQ_TOPK_MERGE_WARPS * 32 - 1) s_off[nlists] = before + incl;
    __syncthreads();
    const int n = s_off[nlists];
    if (n <= GQ_TOPK_RANK_MAX) {
      i64* sv = (i64*)shbuf; i64* sk0 = sv + GQ_TOPK_RANK_MAX; i64* sk1 = sk0 + GQ_TOPK_RANK_MAX; i64* ss = sk1 + GQ_TOPK_RANK_MAX;
      for (int l = warp; l < nlists; l += GQ_TOPK_MERGE_WARPS) {
        const int o = s_off[l];
        if (lane < s_off[l + 1] - o) {
          const GqCand e = in[(i64)l * 32 + lane];
          sv[o + lane] = e.val; sk0[o + lane] = e.k0; sk1[o + lane] = e.k1; ss[o + lane] = e.slot;
        }
      }
      __syncthreads();
      if (t < n) {
        const i64 v = sv[t], k0 = sk0[t], k1 = sk1[t];
        int rank = 0;
        for (int j = 0; j < n; ++j) {
          const i64 a = sv[j], b0 = sk0[j], b1 = sk1[j];
          rank += (a != v) ? (a > v) : (b0 != k0) ? (b0 < k0) : (b1 < k1);
        }
        if (rank < P.topk) {
          GqGroupRef g;
          if (rank < P.out_capacity) { gq_group_at(P, ss[t], &g); gq_emit_group(P, g, rank); }
          else atomicCAS(P.err, 0, (int)GQ_ERR_CAPACITY);
        }
      }
      if (t == 0) *P.out_n = min(n, P.topk);
      return;
    }
    __syncthreads();
  }
  GqCand mine; mine.valid = 0; mine.val = 0; mine.k0 = 0; mine.k1 = 0; mine.slot = -1;
  // lists l = warp, warp + 32, ...: lane j looks at the entry count of the j-th of them, the warp visits the non-empty ones
  // (with pass 0's bound most blocks admit nothing)
  const int* cnt = gq_topk_counts(P);
  for (i64 base = warp; base < nlists; base += 32 * GQ_TOPK_MERGE_WARPS) {
    const i64 lj = base + (i64)lane * GQ_TOPK_MERGE_WARPS;
    unsigned m = __ballot_sync(0xffffffffu, lj < nlists && cnt[lj] > 0);
    while (m) {                                            // four lists in flight: the loads are what this loop waits for
      GqCand c[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        c[u].valid = 0; c[u].val = 0; c[u].k0 = 0; c[u].k1 = 0; c[u].slot = -1;
        if (m) {
          const int j = __ffs(m) - 1;
          m &= m - 1;
          c[u] = in[(base + (i64)j * GQ_TOPK_MERGE_WARPS) * 32 + lane];
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const GqCand worst = gq_cand_shfl(mine, kth);
        gq_list_feed(mine, c[u], c[u].valid && lane <= kth && gq_better(c[u], worst), lane, kth);
      }
    }
  }
  // the warps' lists are merged pairwise (5 rounds of <= k insertions each; one warp taking the 31 others in turn was
  // 310 dependent insertions, most of this kernel's time)
  sh[warp][lane] = mine;
  __syncthreads();
  for (int step = 1; step < GQ_TOPK_MERGE_WARPS; step <<= 1) {
    if ((warp & (2 * step - 1)) == 0) {
      GqCand c = sh[warp + step][lane];
      GqCand worst = gq_cand_shfl(mine, kth);
      gq_list_feed(mine, c, c.valid && lane <= kth && gq_better(c, worst), lane, kth);   // entries behind the k-th of a sorted list cannot matter
      sh[warp][lane] = mine;
    }
    __syncthreads();
  }
  if (warp != 0) return;
  unsigned have = __ballot_sync(0xffffffffu, mine.valid != 0);
  int n = min(__popc(have), P.topk);
  if (lane < n) {
    GqGroupRef g;
    if (lane < P.out_capacity) { gq_group_at(P, mine.slot, &g); gq_emit_group(P, g, lane); }
    else atomicCAS(P.err, 0, (int)GQ_ERR_CAPACITY);
  }
  if (lane == 0) *P.out_n = n;
}

size_t gq_topk_scratch_bytes_impl() { return sizeof(GqCand) * 32 * GQ_TOPK_BLOCKS + 8 * GQ_TOPK_BOUND_BLOCKS + 4 * GQ_TOPK_BLOCKS; }

cudaError_t gq_launch_finalise(cudaStream_t s, const GqFinaliseParams& p, int num_sms, int* nlaunches) {
  if (p.topk > 0) {
    gq_k_topk_bound<<<GQ_TOPK_BOUND_BLOCKS, 256, 0, s>>>(p);
    gq_k_topk_scan<<<GQ_TOPK_BLOCKS, GQ_TOPK_WARPS * 32, 0, s>>>(p);
    gq_k_topk_merge<<<1, GQ_TOPK_MERGE_WARPS * 32, 0, s>>>(p, (i64)GQ_TOPK_BLOCKS);
    *nlaunches = 3;
  } else {
    i64 nb = (p.capacity + GQ_FIN_THREADS * GQ_FIN_PER - 1) / (GQ_FIN_THREADS * GQ_FIN_PER);
    int blocks = (int)std::max<i64>(1, std::min<i64>(nb, (i64)num_sms * 8));
    gq_k_finalise<<<blocks, GQ_FIN_THREADS, 0, s>>>(p);
    *nlaunches = 1;
  }
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ read probe
// Read-only streaming sum: what a pure scan can reach on this box (MEASURED_PEAKS is a copy).
__global__ void __launch_bounds__(512) gq_k_read_probe(const ulonglong2* __restrict__ p, i64 n16, u64* out) {
  u64 acc = 0;
  const i64 stride = (i64)gridDim.x * blockDim.x;
  i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  for (; i + 3 * stride < n16; i += 4 * stride) {
    ulonglong2 a = p[i], b = p[i + stride], c = p[i + 2 * stride], d = p[i + 3 * stride];
    acc += a.x + a.y + b.x + b.y + c.x + c.y + d.x + d.y;
  }
  for (; i < n16; i += stride) { ulonglong2 a = p[i]; acc += a.x + a.y; }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0 && acc) atomicAdd(out, acc);
}
cudaError_t gq_launch_read_probe(cudaStream_t s, const void* data, size_t bytes, u64* out, int num_sms) {
  cudaError_t e = cudaMemsetAsync(out, 0, 8, s);
  if (e != cudaSuccess) return e;
  gq_k_read_probe<<<num_sms * 4, 512, 0, s>>>((const ulonglong2*)data, (i64)(bytes / 16), out);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ partitioned upsert
// Pass B of the radix-clustered aggregation (pass A is the PARTITION consumer of gq_scan): the
// records appended per table partition are applied partition by partition — all CTAs sweep partition p before p + 1 —
// so the slice of the group-by table being updated (capacity / npart slots) stays L2-resident and every insert-or-
// update is an L2 hit instead of a DRAM-random read-modify-write. Same table protocol as the scan kernel: linear
// probing from the multiply-shift slot, 64-bit CAS claims, RED updates on words pre-set to their identities.
#define GQ_PART_THREADS 512
#define GQ_PART_U 4
__device__ __forceinline__ u64 gq_p_ld_relaxed(const u64* p) {
  u64 v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
// All CTAs sweep the partitions in the same order WITHOUT a grid barrier. Measured on C5 (316 M records, 1024
// partitions): free-running 24.7 ms; a grid barrier per partition makes the table traffic compulsory-only (13 GB instead
// of 26 GB of DRAM reads) but takes 173 ms, because a partition's most frequent key then serialises its same-address
// REDs at L2 with nothing else to overlap (barrier every 16 / 64 / 256 partitions: 96 / 71 / 56 ms); combining equal
// keys of a warp in registers before touching the table costs more issue slots than the REDs it saves (78 ms).
__global__ void __launch_bounds__(GQ_PART_THREADS) gq_k_part_upsert(const __grid_constant__ GqPartParams P) {
  if (*(volatile int*)P.err != 0) return;
  const u64 cap = P.mask + 1;
  const int rank = blockIdx.x, nrank = gridDim.x;
  for (int p = 0; p < P.npart; ++p) {
    i64 n = (i64)P.pcur[(i64)p * GQ_PART_CURSOR_STRIDE] * GQ_PART_CHUNK;   // cursors count chunks of GQ_PART_CHUNK records
    if (n > P.pcap) n = P.pcap;
    const u64* base = P.part + (u64)p * (u64)P.pcap * P.rw;
    const i64 step = (i64)nrank * GQ_PART_THREADS * GQ_PART_U;
    // (a C5 partition has chunks for only half of the CTAs; rotating which CTAs take them doubles the active CTAs but
    // lets them spread over more partitions at once: 26.9 ms instead of 21.7 ms — L2 locality matters more here)
    for (i64 r0 = (i64)rank * GQ_PART_THREADS * GQ_PART_U; r0 < n; r0 += step) {
      u64 key[GQ_PART_U], idx[GQ_PART_U], k[GQ_PART_U];
      u64 w[GQ_PART_U][4];                               // first 32 bytes of the record: ONE load (a sector read word by
      bool live[GQ_PART_U];                              // word with a streaming hint is fetched from DRAM once per word)
#pragma unroll
      for (int u = 0; u < GQ_PART_U; ++u) {               // records, then first slot reads: all in flight together
        const i64 r = r0 + (i64)u * GQ_PART_THREADS + threadIdx.x;
        live[u] = r < n;
        const u64* rec = base + (live[u] ? r : 0) * P.rw;
        asm volatile("ld.global.nc.L1::no_allocate.v4.u64 {%0, %1, %2, %3}, [%4];"
                     : "=l"(w[u][0]), "=l"(w[u][1]), "=l"(w[u][2]), "=l"(w[u][3]) : "l"(rec));
        key[u] = w[u][0];
        live[u] = live[u] && key[u] != GQ_EMPTY_KEY;       // padding of a partly used chunk
      }
      if (P.direct) {   // clustered direct aggregation: word 0 of a record IS the accumulator slot
#pragma unroll
        for (int u = 0; u < GQ_PART_U; ++u) {
          if (!live[u]) continue;
          const i64 r = r0 + (i64)u * GQ_PART_THREADS + threadIdx.x;
          const u64* rec = base + r * P.rw;
          u64* slot = P.slots + key[u] * P.sw;
          for (int a = 0; a < P.naggs; ++a) {
            const int sa = P.src[a];
            const i64 v = sa < 0 ? 1 : sa == 1 ? (i64)w[u][1] : sa == 2 ? (i64)w[u][2] : sa == 3 ? (i64)w[u][3] : (i64)__ldg(rec + sa);
            if (P.op[a] == GQ_MIN) atomicMin((i64*)(slot + a), v);
            else if (P.op[a] == GQ_MAX) atomicMax((i64*)(slot + a), v);
            else atomicAdd(slot + a, (u64)v);
          }
          if (P.touch >= 0) atomicAdd(slot + P.touch, 1ULL);
        }
        continue;
      }
#pragma unroll
      for (int u = 0; u < GQ_PART_U; ++u) {
        u64 x = key[u];
        x ^= x >> 32;
        idx[u] = __umul64hi(x * 0x9E3779B97F4A7C15ULL, cap);
        k[u] = live[u] ? gq_p_ld_relaxed(P.slots + idx[u] * P.sw) : 0;
      }
#pragma unroll
      for (int u = 0; u < GQ_PART_U; ++u) {
        if (!live[u]) continue;
        const i64 r = r0 + (i64)u * GQ_PART_THREADS + threadIdx.x;
        u64* slot = nullptr;
        bool won = false;
        for (u64 tries = 0; tries <= 2 * cap; ++tries) {
          u64* s = P.slots + idx[u] * P.sw;
          if (k[u] == key[u]) { slot = s; break; }
          if (k[u] == GQ_EMPTY_KEY) {
            const u64 prev = atomicCAS(s, GQ_EMPTY_KEY, key[u]);
            if (prev == GQ_EMPTY_KEY) { slot = s; won = true; break; }
            k[u] = prev;
            continue;
          }
          idx[u] = idx[u] + 1 > P.mask ? 0 : idx[u] + 1;
          k[u] = gq_p_ld_relaxed(P.slots + idx[u] * P.sw);
        }
        if (!slot) { atomicCAS(P.err, 0, (int)GQ_ERR_CAPACITY); continue; }
        const u64* rec = base + r * P.rw;
        if (P.ndep) {   // dependent key word (see gq_dep_store in the scan skeleton)
          if (P.check_dep) {
            const u64 prev = atomicCAS(slot + 1, GQ_DEP_UNSET, w[u][1]);
            if (prev != GQ_DEP_UNSET && prev != w[u][1]) atomicCAS(P.err, 0, (int)GQ_ERR_DEPENDENT_KEY);
          } else if (won) slot[1] = w[u][1];
        }
        for (int a = 0; a < P.naggs; ++a) {
          const int sa = P.src[a];
          const i64 v = sa < 0 ? 1 : sa == 1 ? (i64)w[u][1] : sa == 2 ? (i64)w[u][2] : sa == 3 ? (i64)w[u][3] : (i64)__ldg(rec + sa);
          u64* w = slot + 1 + P.ndep + a;
          if (P.op[a] == GQ_MIN) atomicMin((i64*)w, v);
          else if (P.op[a] == GQ_MAX) atomicMax((i64*)w, v);
          else atomicAdd(w, (u64)v);
        }
      }
    }
  }
}
cudaError_t gq_launch_part_upsert(cudaStream_t s, const GqPartParams& p, int num_sms) {
  gq_k_part_upsert<<<num_sms * 2, GQ_PART_THREADS, 0, s>>>(p);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ dense-table ranks
// gq_hash_build_finish of a direct-address table: the high word of every bitmap entry := number of member keys before
// it, header[2] := member keys; keyrank[r] := key of rank r (read by the finalisers of direct aggregation). Two
// kernels: per-CTA totals, then every CTA sums the totals before it and scans its own entries.
#define GQ_RANK_THREADS 1024                               // one bitmap entry per thread (gq_internal.h GQ_DENSE_RANK_BLOCK)
__global__ void __launch_bounds__(GQ_RANK_THREADS) gq_k_dense_rank_totals(const u64* entries, i64 nwords, unsigned* totals) {
  __shared__ unsigned warp_sum[GQ_RANK_THREADS / 32];
  const i64 w = (i64)blockIdx.x * GQ_RANK_THREADS + threadIdx.x;
  unsigned c = w < nwords ? __popc((unsigned)entries[w]) : 0u;
  for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
  if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = c;
  __syncthreads();
  if (threadIdx.x == 0) { unsigned t = 0; for (int i = 0; i < GQ_RANK_THREADS / 32; ++i) t += warp_sum[i]; totals[blockIdx.x] = t; }
}
__global__ void __launch_bounds__(GQ_RANK_THREADS) gq_k_dense_rank_apply(u64* entries, i64 nwords, const unsigned* totals, i64 base, u64* keyrank,
                                                                         i64 max_rows, i64* header, int* err) {
  __shared__ unsigned part[GQ_RANK_THREADS];
  __shared__ unsigned block_base;
  const int t = threadIdx.x, lane = t & 31;
  unsigned b = 0;
  for (int i = t; i < (int)blockIdx.x; i += GQ_RANK_THREADS) b += totals[i];
  part[t] = b;
  __syncthreads();
  for (int o = GQ_RANK_THREADS / 2; o > 0; o >>= 1) { if (t < o) part[t] += part[t + o]; __syncthreads(); }
  if (t == 0) block_base = part[0];
  __syncthreads();
  const i64 w = (i64)blockIdx.x * GQ_RANK_THREADS + t;
  const unsigned bits = w < nwords ? (unsigned)entries[w] : 0u;
  const unsigned c = __popc(bits);
  part[t] = c;
  __syncthreads();
  for (int o = 1; o < GQ_RANK_THREADS; o <<= 1) {          // inclusive scan of the per-entry counts
    const unsigned v = t >= o ? part[t - o] : 0;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  const u64 rank0 = (u64)block_base + part[t] - c;         // member keys before this entry
  if (w < nwords) entries[w] = (u64)bits | (rank0 << 32);
  // key of every rank: the warp expands its 32 entries one after the other, lane l taking bit l (coalesced stores)
  for (int k = 0; k < 32; ++k) {
    const unsigned wb = __shfl_sync(0xffffffffu, bits, k);
    const u64 wr = __shfl_sync(0xffffffffu, rank0, k);
    if ((wb >> lane) & 1u) {
      const u64 r = wr + __popc(wb & ((1u << lane) - 1u));
      if ((i64)r < max_rows) keyrank[r] = (u64)(base + (w - lane + k) * 32 + lane);
    }
  }
  if (blockIdx.x == gridDim.x - 1 && t == GQ_RANK_THREADS - 1) {
    const i64 total = (i64)(rank0 + c);
    header[2] = total;
    if (total > max_rows) atomicCAS(err, 0, (int)GQ_ERR_CAPACITY);   // more build rows than max_build_rows promised
    // header[0] = rows the build kernels inserted: more rows than member keys means some key was inserted twice
    if (*(volatile i64*)&header[0] > total) atomicCAS(err, 0, (int)GQ_ERR_DUPLICATE_KEY);
  }
}
cudaError_t gq_launch_dense_rank(cudaStream_t s, unsigned long long* entries, long long nwords, unsigned* totals, long long base,
                                 unsigned long long* keyrank, long long max_rows, long long* header, int* err) {
  const int blocks = (int)((nwords + GQ_RANK_THREADS - 1) / GQ_RANK_THREADS);
  gq_k_dense_rank_totals<<<blocks, GQ_RANK_THREADS, 0, s>>>(entries, nwords, totals);
  gq_k_dense_rank_apply<<<blocks, GQ_RANK_THREADS, 0, s>>>(entries, nwords, totals, base, keyrank, max_rows, header, err);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ state merge
// Partial -> Final between two aggregation states (PAPER.md:154 aggregation modes; Fig. 3: one state per stream; SURVEY
// §8(f) NEXT-2): every group of `src` is inserted into (or found in) `dst` with the ordinary table protocol and its
// aggregate words are combined with RED.ADD / RED.MIN / RED.MAX. The same kernel re-hashes a state into a larger table
// (growth: dst = a freshly initialised table). Direct states (accumulators indexed by the slots of one join table)
// merge word by word.
struct GqMergeParams {
  const u64* sslots; i64 scap; const u64* sside; const i64* sheader;
  u64* dslots; u64 dmask; u64* dside; i64* dheader;
  int sw, ndep, naggs, check_dep, direct, daw;
  int op[GQ_MAX_AGGS + 1];
  int* err;
};
__device__ __forceinline__ void gq_m_red(int op, u64* w, u64 v) {
  if (op == GQ_MIN) atomicMin((i64*)w, (i64)v);
  else if (op == GQ_MAX) atomicMax((i64*)w, (i64)v);
  else atomicAdd(w, v);
}
__global__ void __launch_bounds__(256) gq_k_merge(const __grid_constant__ GqMergeParams P) {
  if (*(volatile int*)P.err != 0) return;
  const i64 stride = (i64)gridDim.x * blockDim.x;
  const i64 t0 = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (P.direct) {   // accumulator arrays over the same join table: slot i of src into slot i of dst (untouched slots hold identities)
    for (i64 i = t0; i <= P.scap; i += stride)
      for (int a = 0; a < P.daw; ++a) {
        const u64 v = P.sslots[i * P.daw + a];
        const int op = a <= P.naggs ? P.op[a] : (int)GQ_SUM;
        if ((op == GQ_MIN && v == 0x7FFFFFFFFFFFFFFFULL) || (op == GQ_MAX && v == 0x8000000000000000ULL) || ((op == GQ_SUM || op == GQ_COUNT_STAR) && v == 0)) continue;
        gq_m_red(op, P.dslots + i * P.daw + a, v);
      }
    return;
  }
  const u64 cap = P.dmask + 1;
  for (i64 i = t0; i < P.scap; i += stride) {
    const u64* s = P.sslots + i * P.sw;
    const u64 key = s[0];
    if (key == GQ_EMPTY_KEY) continue;
    u64 x = key;
    x ^= x >> 32;
    u64 idx = cap > 1 ? __umul64hi(x * 0x9E3779B97F4A7C15ULL, cap) : 0;
    u64* slot = nullptr;
    bool won = false;
    for (u64 tries = 0; tries <= 2 * cap; ++tries) {
      u64* d = P.dslots + idx * P.sw;
      u64 k = gq_p_ld_relaxed(d);
      if (k == GQ_EMPTY_KEY) { const u64 prev = atomicCAS(d, GQ_EMPTY_KEY, key); if (prev == GQ_EMPTY_KEY) { slot = d; won = true; break; } k = prev; }
      if (k == key) { slot = d; break; }
      idx = idx + 1 > P.dmask ? 0 : idx + 1;
    }
    if (!slot) { atomicCAS(P.err, 0, (int)GQ_ERR_CAPACITY); continue; }
    if (P.ndep) {
      if (P.check_dep) {
        const u64 prev = atomicCAS(slot + 1, GQ_DEP_UNSET, s[1]);
        if (prev != GQ_DEP_UNSET && prev != s[1]) atomicCAS(P.err, 0, (int)GQ_ERR_DEPENDENT_KEY);
      } else if (won) slot[1] = s[1];
    }
    for (int a = 0; a < P.naggs; ++a) gq_m_red(P.op[a], slot + 1 + P.ndep + a, s[1 + P.ndep + a]);
  }
  // the side slot: the group whose key is the reserved pattern, or THE group of a key-less aggregation
  if (t0 == 0 && P.sheader[1] != 0) {
    const i64 prev = (i64)atomicExch((u64*)&P.dheader[1], 1ULL);
    if (P.ndep && (prev == 0 || P.check_dep)) P.dside[1] = P.sside[1];
    for (int a = 0; a < P.naggs; ++a) gq_m_red(P.op[a], P.dside + 1 + P.ndep + a, P.sside[1 + P.ndep + a]);
  }
}
__global__ void __launch_bounds__(256) gq_k_count_groups(const u64* slots, i64 cap, int sw, const i64* header, int direct, int daw, int dtouch,
                                                        i64* out) {
  i64 n = 0;
  const i64 stride = (i64)gridDim.x * blockDim.x;
  for (i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x; i < cap + (direct ? 1 : 0); i += stride)
    n += direct ? (slots[i * daw + dtouch] != 0) : (slots[i * sw] != GQ_EMPTY_KEY);
  for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xffffffffu, n, o);
  if ((threadIdx.x & 31) == 0 && n) atomicAdd((u64*)out, (u64)n);
  if (!direct && blockIdx.x == 0 && threadIdx.x == 0 && header[1] != 0) atomicAdd((u64*)out, 1ULL);
}
cudaError_t gq_launch_merge(cudaStream_t s, const unsigned long long* sslots, long long scap, const unsigned long long* sside, const long long* sheader,
                            unsigned long long* dslots, unsigned long long dmask, unsigned long long* dside, long long* dheader, int sw, int ndep,
                            int naggs, const int* op, int check_dep, int direct, int daw, int* err, int num_sms) {
  GqMergeParams p;
  p.sslots = sslots; p.scap = scap; p.sside = sside; p.sheader = sheader; p.dslots = dslots; p.dmask = dmask; p.dside = dside; p.dheader = dheader;
  p.sw = sw; p.ndep = ndep; p.naggs = naggs; p.check_dep = check_dep; p.direct = direct; p.daw = daw; p.err = err;
  for (int a = 0; a <= GQ_MAX_AGGS; ++a) p.op[a] = a < naggs ? op[a] : (int)GQ_SUM;
  const i64 work = std::max<i64>(1, scap);
  const int blocks = (int)std::max<i64>(1, std::min<i64>((work + 255) / 256, (i64)num_sms * 16));
  gq_k_merge<<<blocks, 256, 0, s>>>(p);
  return cudaGetLastError();
}
cudaError_t gq_launch_count_groups(cudaStream_t s, const unsigned long long* slots, long long cap, int sw, const long long* header, int direct, int daw,
                                   int dtouch, long long* out, int num_sms) {
  cudaError_t e = cudaMemsetAsync(out, 0, 8, s);
  if (e != cudaSuccess) return e;
  const int blocks = (int)std::max<i64>(1, std::min<i64>((cap + 255) / 256, (i64)num_sms * 16));
  gq_k_count_groups<<<blocks, 256, 0, s>>>(slots, cap, sw, header, direct, daw, dtouch, out);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ heavy hitters
// Skew handling for high-cardinality group-by: before the fused scan of a large batch, a strided
// sample of the group-key column is counted in a small (key,count) table; keys whose sample count reaches the
// threshold form the batch's hot list. The scan kernel aggregates those keys per CTA in shared memory and flushes
// them once, so the hottest keys no longer serialise hundreds of millions of same-address L2 atomics. The hot list
// only steers WHERE an update is accumulated; results do not depend on it.
__device__ __forceinline__ u64 gq_s_hash(i64 key, int shift) {
  u64 x = (u64)key;
  x ^= x >> 32;
  return (x * 0x9E3779B97F4A7C15ULL) >> shift;
}
// A block first counts its 1024 samples in a shared-memory table and then adds every distinct key ONCE to the global
// sample table: the most frequent key of a Zipf column is 5 % of the samples, and 26 K atomics on one L2 address took
// most of this kernel's 0.1 ms.
#define GQ_HS_THREADS 1024
#define GQ_HS_SLOTS 2048
__global__ void __launch_bounds__(GQ_HS_THREADS) gq_k_hot_sample(const void* keycol, int dtype, i64 nrows, i64 stride, i64 nsample,
                                                                u64* table, u64 mask, int shift) {
  __shared__ u64 skey[GQ_HS_SLOTS];
  __shared__ unsigned scnt[GQ_HS_SLOTS];
  for (int i = threadIdx.x; i < GQ_HS_SLOTS; i += GQ_HS_THREADS) { skey[i] = GQ_EMPTY_KEY; scnt[i] = 0; }
  __syncthreads();
  const i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  const i64 r = t * stride;
  if (t < nsample && r < nrows) {
    const i64 key = dtype == GQ_I8 ? (i64)((const signed char*)keycol)[r] : dtype == GQ_I32 ? (i64)((const int*)keycol)[r]
                                                                                              : ((const i64*)keycol)[r];
    if ((u64)key != GQ_EMPTY_KEY) {
      unsigned i = (unsigned)gq_s_hash(key, 64 - 11);
      for (;; i = (i + 1) & (GQ_HS_SLOTS - 1)) {       // (1024 samples in 2048 slots: a free slot exists)
        u64 k = skey[i];
        if (k == GQ_EMPTY_KEY) k = atomicCAS(&skey[i], GQ_EMPTY_KEY, (u64)key);
        if (k == GQ_EMPTY_KEY || k == (u64)key) { atomicAdd(&scnt[i], 1u); break; }
      }
    }
  }
  __syncthreads();
  for (int q = threadIdx.x; q < GQ_HS_SLOTS; q += GQ_HS_THREADS) {
    const u64 key = skey[q];
    if (key == GQ_EMPTY_KEY) continue;
    u64 i = gq_s_hash((i64)key, shift);
    for (u64 n = 0; n <= mask; ++n, i = (i + 1) & mask) {
      u64* s = table + i * 2;
      u64 k = *(volatile u64*)s;
      if (k != key) {
        if (k != GQ_EMPTY_KEY) continue;
        u64 prev = atomicCAS(s, GQ_EMPTY_KEY, key);
        if (prev != GQ_EMPTY_KEY && prev != key) continue;
      }
      atomicAdd(s + 1, (u64)scnt[q]);
      break;
    }
  }
}
// hot[0] = number of hot keys (<= max_hot), hot[1..31] = histogram of sample counts by floor(log2), hot[32..] = keys.
// The hot list must hold the MOST frequent keys: when more than max_hot keys reach the base threshold, the threshold
// is raised to the smallest power of two that leaves at most max_hot of them.
__global__ void gq_k_hot_hist(const u64* table, i64 nslots, u64 threshold, i64* hot) {
  const i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nslots) return;
  const u64 c = table[i * 2 + 1];
  if (table[i * 2] == GQ_EMPTY_KEY || c < threshold) return;
  int b = 63 - __clzll((long long)c);
  if (b > 31) b = 31;
  if (b < 1) b = 1;
  atomicAdd((u64*)&hot[b], 1ULL);
}
// pass 0 takes every key at or above the raised threshold (at most max_hot of them, by construction); pass 1 fills the
// list up with keys of the bin just below it (sample counts within a factor of two of one another: any subset will do).
__global__ void gq_k_hot_select(const u64* table, i64 nslots, u64 threshold, i64* hot, int max_hot, int pass) {
  const i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nslots) return;
  const u64 k = table[i * 2];
  const u64 c = table[i * 2 + 1];
  if (k == GQ_EMPTY_KEY || c < threshold) return;
  u64 t = threshold, lo = threshold;          // every thread derives the same raised threshold from the histogram
  i64 above = 0;
  for (int b = 31; b >= 1; --b) {
    above += hot[b];
    if (above > max_hot) { const u64 tb = 1ULL << (b + 1); if (tb > t) { t = tb; lo = tb >> 1; if (lo < threshold) lo = threshold; } break; }
  }
  if (pass == 0 ? c < t : (c >= t || c < lo)) return;
  i64 idx = (i64)atomicAdd((u64*)hot, 1ULL);
  if (idx < max_hot) hot[32 + idx] = (i64)k;
}

cudaError_t gq_launch_hot_keys(cudaStream_t s, const void* keycol, int dtype, i64 nrows, u64* table, i64 nslots,
                               i64 nsample, u64 threshold, i64* hot, int max_hot, int num_sms, int* nlaunches) {
  // (key,count) slots: key = EMPTY (0x80..0), count = 0
  u64 pat[16];
  for (int i = 0; i < 16; ++i) pat[i] = (i & 1) ? 0 : GQ_EMPTY_KEY;
  cudaError_t e = gq_launch_init_table(s, table, nslots, 2, pat, table, 0, hot, 0, num_sms);   // header := hot list head (zeroed)
  if (e != cudaSuccess) return e;
  int shift = 64;
  for (i64 c = 1; c < nslots; c <<= 1) --shift;
  const i64 stride = nrows / nsample > 0 ? nrows / nsample : 1;
  gq_k_hot_sample<<<(unsigned)((nsample + GQ_HS_THREADS - 1) / GQ_HS_THREADS), GQ_HS_THREADS, 0, s>>>(keycol, dtype, nrows, stride, nsample, table,
                                                                   (u64)(nslots - 1), shift);
  gq_k_hot_hist<<<(unsigned)((nslots + 255) / 256), 256, 0, s>>>(table, nslots, threshold, hot);
  gq_k_hot_select<<<(unsigned)((nslots + 255) / 256), 256, 0, s>>>(table, nslots, threshold, hot, max_hot, 0);
  gq_k_hot_select<<<(unsigned)((nslots + 255) / 256), 256, 0, s>>>(table, nslots, threshold, hot, max_hot, 1);
  *nlaunches = 5;
  return cudaGetLastError();
}
