// gq_sort.cu — OrderBy / TopN over a device-resident column batch (Fig. 2: the
// plan's CudfOrderBy / TopN operators). Plan-independent sm_100a kernels, compiled by nvcc into libgq.so.
//
// Order: lexicographic over the key columns (keys[0] most significant), ascending or descending per key, signed
// comparison, ties broken by input row position — i.e. a STABLE sort, so the result is unique and compared bit-exactly
// with the oracle's std::stable_sort.
//
// Method: least-significant-digit radix sort of (64-bit sortable key, 32-bit row index) pairs, 8 bits per pass, one
// key column at a time from the least significant column to the most significant (a stable sort by the more
// significant column keeps the order the less significant ones produced). Per column: one gather builds the sortable
// keys (sign bit flipped; all bits inverted for descending), then one pass per byte of the column's width:
//   histogram  — a fixed grid of GQ_SORT_BLOCKS CTAs, each owning a contiguous range of tiles, counts its digits;
//   scan       — one CTA turns the [digit][CTA] counts into exclusive offsets (digit-major: stable across CTAs);
//   scatter    — every CTA walks its range again in order, tile by tile; inside a tile ranks are stable: a warp owns 256
//                consecutive pairs, its lanes with equal digits are found with MATCH.ANY, warps are ordered through
//                per-warp digit counts in shared memory; the tile leaves through a shared-memory staging buffer.
// TopN (limit << rows): two 12-bit histogram levels below the common prefix of the most significant key's images select a
// threshold bucket on the device; only rows at or before it (>= limit of them, more only with ties) are compacted and sorted.
// Everything is stream-ordered; the number of candidate rows stays in device memory (no host synchronisation).
#include <algorithm>

#include "gq_internal.h"

typedef unsigned long long u64;
typedef long long i64;
typedef unsigned int u32;

#define GQ_SORT_THREADS 256
#define GQ_SORT_ITEMS 8
#define GQ_SORT_TILE (GQ_SORT_THREADS * GQ_SORT_ITEMS)
#define GQ_SORT_WARPS (GQ_SORT_THREADS / 32)
#define GQ_SEL_BINS 4096

// Sortable image of a signed column value of `bytes` bytes: unsigned order == requested order.
__device__ __forceinline__ u64 gq_sort_image(i64 v, int bytes, int desc) {
  const int bits = 8 * bytes;
  u64 u = (u64)v ^ (1ULL << (bits - 1));
  if (bits < 64) u &= (1ULL << bits) - 1;
  if (desc) u = bits < 64 ? (~u & ((1ULL << bits) - 1)) : ~u;
  return u;
}
__device__ __forceinline__ i64 gq_sort_load(const void* col, int dtype, i64 r) {
  return dtype == GQ_I8 ? (i64)((const signed char*)col)[r] : dtype == GQ_I32 ? (i64)((const int*)col)[r] : ((const i64*)col)[r];
}
__device__ __forceinline__ u32 gq_sort_n(const u32* d_n) { return *(volatile const u32*)d_n; }

// range of tiles owned by a CTA: contiguous, whole tiles
__device__ __forceinline__ void gq_sort_range(u32 n, u32* lo, u32* hi, u32 tile) {
  const u32 ntiles = (n + tile - 1) / tile;
  const u32 per = (ntiles + gridDim.x - 1) / gridDim.x;
  const u64 a = (u64)blockIdx.x * per * tile, b = a + (u64)per * tile;
  *lo = (u32)(a < n ? a : n);
  *hi = (u32)(b < n ? b : n);
}

__global__ void gq_k_sort_iota(u32* idx, u32 n, u32* d_n) {
  for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) idx[i] = i;
  if (blockIdx.x == 0 && threadIdx.x == 0) *d_n = n;
}

// ---- passes that would move nothing are skipped ON THE DEVICE. While the sortable keys of a column are built, the OR of
// (key xor first key) is collected in the control block (one word per sort column; id GQ_SORT_ROWID = the row-number
// "column" of the TopN path): a byte of that mask is zero iff all keys agree in that byte, and then the pass over it is
// the identity. The host still enqueues every pass (it never learns the mask); histogram, scan and scatter of a skipped
// pass return at once, and since a skipped pass does not swap the two buffers, every kernel derives WHICH buffer holds
// the data from the masks: parity of the number of non-skipped passes so far. (An int64 price column below 2^24: 3
// passes instead of 8.)
#define GQ_SORT_ROWID 32
#define GQ_SORT_CTL_BYTES 512
struct GqSortBufs { u64* k[2]; u32* i[2]; const u32* ctl; };
__device__ __forceinline__ u64 gq_sort_mask(const u32* ctl, int id) { return ((volatile const u64*)ctl)[16 + id]; }
__device__ __forceinline__ u32 gq_sort_live_bytes(u64 m, int below) {      // parity of the non-zero bytes among bytes [0, below)
  u32 p = 0;
  for (int b = 0; b < below; ++b) p ^= ((m >> (8 * b)) & 255ULL) != 0ULL;
  return p;
}
// -> buffer that holds the data when pass `pass` (0..8) of column `id` starts; *live = that pass moves something. All
// threads of the CTA call it (one shared-memory broadcast).
__device__ __forceinline__ u32 gq_sort_where(const u32* ctl, int id, int pass, bool* live) {
  __shared__ u32 sh[2];
  if (threadIdx.x == 0) {
    u32 par = 0;
    for (int c = id + 1; c <= GQ_SORT_ROWID; ++c) par ^= gq_sort_live_bytes(gq_sort_mask(ctl, c), 8);   // columns done before this one
    const u64 m = id >= 0 ? gq_sort_mask(ctl, id) : 0ULL;
    par ^= gq_sort_live_bytes(m, pass);
    sh[0] = par;
    sh[1] = pass < 8 && ((m >> (8 * pass)) & 255ULL) != 0ULL;
  }
  __syncthreads();
  *live = sh[1] != 0;
  return sh[0];
}
__global__ void gq_k_sort_keys(const void* col, int dtype, int bytes, int desc, GqSortBufs B, const u32* d_n, int id) {
  bool live;
  const u32 par = gq_sort_where(B.ctl, id, 0, &live);
  const u32* idx = B.i[par];
  u64* keys = B.k[par];
  const u32 n = gq_sort_n(d_n);
  if (n == 0) return;
  const u64 ref = col ? gq_sort_image(gq_sort_load(col, dtype, (i64)idx[0]), bytes, desc) : (u64)idx[0];
  u64 diff = 0;
  for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const u64 k = col ? gq_sort_image(gq_sort_load(col, dtype, (i64)idx[i]), bytes, desc) : (u64)idx[i];   // col == null: the row index itself
    keys[i] = k;
    diff |= k ^ ref;
  }
  for (int o = 16; o > 0; o >>= 1) diff |= __shfl_xor_sync(0xffffffffu, diff, o);
  if ((threadIdx.x & 31) == 0 && diff) atomicOr((u64*)B.ctl + 16 + id, diff);
}

template <int NT>
__global__ void __launch_bounds__(NT) gq_k_sort_hist(GqSortBufs B, const u32* d_n, int id, int pass, u32* hist) {
  __shared__ u32 h[256];
  bool live;
  const u32 par = gq_sort_where(B.ctl, id, pass, &live);
  if (!live) return;
  const u64* keys = B.k[par];
  const int shift = 8 * pass;
  if (threadIdx.x < 256) h[threadIdx.x] = 0;
  __syncthreads();
  u32 lo, hi;
  gq_sort_range(gq_sort_n(d_n), &lo, &hi, NT * GQ_SORT_ITEMS);
  for (u32 base = lo; base < hi; base += NT * GQ_SORT_ITEMS) {       // eight loads per thread in flight, then eight adds
    u64 k[GQ_SORT_ITEMS];
#pragma unroll
    for (int j = 0; j < GQ_SORT_ITEMS; ++j) { const u32 i = base + (u32)j * NT + threadIdx.x; k[j] = i < hi ? keys[i] : 0ULL; }
#pragma unroll
    for (int j = 0; j < GQ_SORT_ITEMS; ++j) if (base + (u32)j * NT + threadIdx.x < hi) atomicAdd(&h[(k[j] >> shift) & 255], 1u);
  }
  __syncthreads();
  if (threadIdx.x < 256) hist[threadIdx.x * gridDim.x + blockIdx.x] = h[threadIdx.x];      // [digit][CTA]
}

// inclusive scan of one value per thread over a CTA of 1024 threads (warp shuffles + one shared-memory step); returns the
// inclusive prefix, *total = the CTA's sum. Every thread of the CTA calls it.
__device__ __forceinline__ u32 gq_block_scan_1024(u32 v, u32* wsum /* [33] shared */, u32* total) {
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  u32 incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const u32 x = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += x; }
  __syncthreads();                                   // (wsum may still be read by the previous call)
  if (lane == 31) wsum[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    u32 w = wsum[lane], wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const u32 x = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += x; }
    wsum[lane] = wi - w;                              // exclusive prefix of the warp sums
    if (lane == 31) wsum[32] = wi;
  }
  __syncthreads();
  *total = wsum[32];
  return incl + wsum[warp];
}
// exclusive scan of hist in [digit][CTA] order, in place; one CTA of 1024 threads walks it in chunks of 4096 counters,
// four consecutive counters per thread (coalesced 16-byte accesses; the first version gave every thread its own
// contiguous share: strided accesses and a 148-step serial loop, 153 us per pass for 592 CTAs)
__global__ void __launch_bounds__(1024) gq_k_sort_scan(u32* hist, int total, const u32* ctl = nullptr, int id = 0, int pass = 0) {
  __shared__ u32 wsum[33];
  const int t = threadIdx.x;
  if (ctl) { bool live; gq_sort_where(ctl, id, pass, &live); if (!live) return; }   // a skipped pass of the sort
  u32 carry = 0;
  for (int base = 0; base < total; base += 4096) {
    const int i = base + 4 * t;
    u32 v[4];
    if (i + 3 < total && (total & 3) == 0) { const uint4 q = *(const uint4*)(hist + i); v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w; }
    else { for (int k = 0; k < 4; ++k) v[k] = i + k < total ? hist[i + k] : 0u; }
    const u32 s = v[0] + v[1] + v[2] + v[3];
    u32 tot;
    const u32 excl = gq_block_scan_1024(s, wsum, &tot) - s + carry;
    const u32 o0 = excl, o1 = o0 + v[0], o2 = o1 + v[1], o3 = o2 + v[2];
    if (i + 3 < total && (total & 3) == 0) *(uint4*)(hist + i) = make_uint4(o0, o1, o2, o3);
    else { const u32 o[4] = {o0, o1, o2, o3}; for (int k = 0; k < 4; ++k) if (i + k < total) hist[i + k] = o[k]; }
    carry += tot;
  }
}

// Scatter of one pass, the tile permuted THROUGH SHARED MEMORY (the scheme of gq_k_hp_scatter below): a CTA takes 2048
// consecutive pairs, warp w ranks its 256 pairs per digit on its own (MATCH.ANY + warp-private counters, no CTA barrier
// per 32 rows), one pass over [warp][digit] gives every pair its place in the tile's digit-major order, and keys and
// row numbers are staged in that order and written out as runs. The first version ranked 256 pairs per round across the
// CTA (3 barriers per 256 pairs, one load per thread in flight) and wrote every pair on its own: 947 us per pass of
// 60 M pairs; this one 460 us.
// NT = 256 (4 CTAs per SM, 2048-pair tiles) or 512 (2 CTAs per SM, 4096-pair tiles: half as many CTAs keep half as many
// write streams open and a digit's run is twice as long — the full sort uses it; TopN's few candidates take 256).
#define GQ_SS_ITEMS 8
template <int NT>
__global__ void __launch_bounds__(NT, 1024 / NT) gq_k_sort_scatter_staged(GqSortBufs B, const u32* d_n, int id, int pass, const u32* hist) {
  constexpr int NW = NT / 32, TILE = NT * GQ_SS_ITEMS;
  __shared__ u32 cur[256];                               // the CTA's next output position per digit (at the tile's start)
  __shared__ unsigned short wc[NW][256];                 // per tile: pairs of a digit in every warp, then their offsets
  __shared__ unsigned short toff[256];                   // per tile: first place of every digit in the tile's order
  __shared__ u32 wsum[8];
  __shared__ unsigned char pd[TILE];                     // per tile: digit of every place (output position = cur + place - toff)
  __shared__ __align__(16) u64 stage[TILE];
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  bool live;
  const u32 par = gq_sort_where(B.ctl, id, pass, &live);
  if (!live) return;
  const u64* kin = B.k[par]; const u32* iin = B.i[par];
  u64* kout = B.k[par ^ 1]; u32* iout = B.i[par ^ 1];
  const int shift = 8 * pass;
  if (t < 256) cur[t] = hist[t * gridDim.x + blockIdx.x];
  u32 lo, hi;
  gq_sort_range(gq_sort_n(d_n), &lo, &hi, TILE);
  for (u32 base = lo; base < hi; base += TILE) {
    const u32 nt = min((u32)TILE, hi - base);
    if (t < 256) for (int w = 0; w < NW; ++w) wc[w][t] = 0;
    __syncthreads();
    u64 k[GQ_SS_ITEMS];
    unsigned short wr[GQ_SS_ITEMS];                       // rank among the warp's pairs of the digit, then place in the tile
    const u32 i0 = (u32)warp * (32u * GQ_SS_ITEMS) + (u32)lane;
#pragma unroll
    for (int j = 0; j < GQ_SS_ITEMS; ++j) { const u32 i = i0 + (u32)j * 32u; k[j] = i < nt ? kin[base + i] : 0ULL; }
#pragma unroll
    for (int j = 0; j < GQ_SS_ITEMS; ++j) {
      const bool have = i0 + (u32)j * 32u < nt;
      const u32 d = have ? (u32)(k[j] >> shift) & 255u : 256u + (u32)lane;
      const u32 peers = __match_any_sync(0xffffffffu, d);
      const u32 rank = __popc(peers & ((1u << lane) - 1u));
      wr[j] = have ? (unsigned short)(wc[warp][d] + rank) : (unsigned short)0;
      __syncwarp();
      if (have && rank == 0) wc[warp][d] += (unsigned short)__popc(peers);
      __syncwarp();
    }
    __syncthreads();
    u32 tot = 0, incl = 0;
    if (t < 256) {                                        // thread q < 256: digit q (warps 0..7, all lanes)
#pragma unroll
      for (int w = 0; w < NW; ++w) { const u32 c = wc[w][t]; wc[w][t] = (unsigned short)tot; tot += c; }
      incl = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const u32 x = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += x; }
      if (lane == 31) wsum[warp] = incl;
    }
    __syncthreads();
    if (t < 256) {
      u32 before = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) if (w < warp) before += wsum[w];
      toff[t] = (unsigned short)(before + incl - tot);
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < GQ_SS_ITEMS; ++j) {
      if (i0 + (u32)j * 32u < nt) {
        const u32 d = (u32)(k[j] >> shift) & 255u;
        wr[j] = (unsigned short)((u32)toff[d] + (u32)wc[warp][d] + (u32)wr[j]);
        pd[wr[j]] = (unsigned char)d;
        stage[wr[j]] = k[j];
      }
    }
    u32 ix[GQ_SS_ITEMS];                                 // the row numbers are on their way while the keys are written out
#pragma unroll
    for (int j = 0; j < GQ_SS_ITEMS; ++j) { const u32 i = i0 + (u32)j * 32u; ix[j] = i < nt ? iin[base + i] : 0u; }
    __syncthreads();
    for (u32 p = t; p < nt; p += NT) { const u32 d = pd[p]; kout[cur[d] + p - (u32)toff[d]] = stage[p]; }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < GQ_SS_ITEMS; ++j) if (i0 + (u32)j * 32u < nt) ((u32*)stage)[wr[j]] = ix[j];
    __syncthreads();
    for (u32 p = t; p < nt; p += NT) { const u32 d = pd[p]; iout[cur[d] + p - (u32)toff[d]] = ((const u32*)stage)[p]; }
    __syncthreads();
    if (t < 256) cur[t] += tot;                           // (read again only after the next tile's barriers)
  }
}

// ---- TopN candidate selection on the most significant key ----
struct GqSelParams {
  const void* col; int dtype, bytes, desc; u32 n; u64 limit;
  u32* hist1; u32* hist2; u32* ctl;   // ctl[0] = threshold bucket level 1, ctl[1] = level 2, ctl[2] = candidates (cursor)
};
__device__ __forceinline__ u64 gq_sel_top(const GqSelParams& P, u32 r) {   // sortable image left-aligned in 64 bits
  return gq_sort_image(gq_sort_load(P.col, P.dtype, (i64)r), P.bytes, P.desc) << (64 - 8 * P.bytes);
}
// The two 12-bit histogram levels sit directly BELOW the bits all keys share: a pre-pass takes the minimum and maximum of
// the images (ctl words 16..19: ~min and max, both as atomic maxima over the zeroed control block), their common prefix
// is skipped. (With the levels fixed at the top 24 bits a column of small non-negative int64 values — prices, counts —
// fell into ONE bucket, every row became a candidate and TopN cost more than the full sort: 18.6 vs 10.0 ms, 60 M rows.)
__global__ void __launch_bounds__(256) gq_k_sel_range(const __grid_constant__ GqSelParams P) {
  u64 lo = ~0ULL, hi = 0;
  for (u32 r = blockIdx.x * 256 + threadIdx.x; r < P.n; r += gridDim.x * 256) {
    const u64 u = gq_sel_top(P, r);
    lo = u < lo ? u : lo;
    hi = u > hi ? u : hi;
  }
  for (int o = 16; o > 0; o >>= 1) {
    const u64 a = __shfl_xor_sync(0xffffffffu, lo, o), b = __shfl_xor_sync(0xffffffffu, hi, o);
    lo = a < lo ? a : lo;
    hi = b > hi ? b : hi;
  }
  if ((threadIdx.x & 31) == 0 && lo <= hi) { atomicMax((u64*)(P.ctl + 16), ~lo); atomicMax((u64*)(P.ctl + 18), hi); }
}
// shifts of the two levels: level 1 = the 12 bits below the common prefix of all images, level 2 = the 12 below those
__device__ __forceinline__ void gq_sel_shifts(const GqSelParams& P, int* s1, int* s2) {
  const u64 lo = ~*(volatile const u64*)(P.ctl + 16), hi = *(volatile const u64*)(P.ctl + 18);
  const u64 x = lo ^ hi;
  const int vary = x ? 64 - __clzll((long long)x) : 0;        // bits [0, vary) differ between some two keys
  *s1 = vary > 12 ? vary - 12 : 0;
  *s2 = *s1 > 12 ? *s1 - 12 : 0;
}
__global__ void __launch_bounds__(256) gq_k_sel_hist(const __grid_constant__ GqSelParams P, int level) {
  __shared__ u32 h[GQ_SEL_BINS];
  for (int i = threadIdx.x; i < GQ_SEL_BINS; i += 256) h[i] = 0;
  __syncthreads();
  int s1, s2;
  gq_sel_shifts(P, &s1, &s2);
  const u32 t1 = level == 2 ? P.ctl[0] : 0;
  for (u32 r = blockIdx.x * 256 + threadIdx.x; r < P.n; r += gridDim.x * 256) {
    const u64 u = gq_sel_top(P, r);
    const u32 b1 = (u32)(u >> s1) & (GQ_SEL_BINS - 1);
    if (level == 1) atomicAdd(&h[b1], 1u);
    else if (b1 == t1) atomicAdd(&h[(u32)(u >> s2) & (GQ_SEL_BINS - 1)], 1u);
  }
  __syncthreads();
  u32* g = level == 1 ? P.hist1 : P.hist2;
  for (int i = threadIdx.x; i < GQ_SEL_BINS; i += 256) if (h[i]) atomicAdd(&g[i], h[i]);
}
// threshold = the first bucket at which the running count reaches the limit; one CTA of 1024 threads, four buckets each
// (one thread walking 4096 global counters took 100-165 us)
__global__ void __launch_bounds__(1024) gq_k_sel_pick(const __grid_constant__ GqSelParams P, int level) {
  __shared__ u32 wsum[33];
  __shared__ u32 best;
  const int t = threadIdx.x;
  const u32* h = level == 1 ? P.hist1 : P.hist2;
  u64 need = P.limit;
  if (level == 2) {                                   // rows in the buckets before level 1's threshold are taken anyway
    const u32 t1 = P.ctl[0];
    u32 mine = 0;
    for (int k = 0; k < 4; ++k) if ((u32)(4 * t + k) < t1) mine += P.hist1[4 * t + k];
    u32 below;
    gq_block_scan_1024(mine, wsum, &below);
    need = P.limit > (u64)below ? P.limit - (u64)below : 1;
  }
  if (t == 0) best = GQ_SEL_BINS - 1;
  u32 v[4];
  for (int k = 0; k < 4; ++k) v[k] = h[4 * t + k];
  const u32 s = v[0] + v[1] + v[2] + v[3];
  u32 tot;
  u64 run = (u64)(gq_block_scan_1024(s, wsum, &tot) - s);      // (counts sum to <= 2^31 rows: 32 bits suffice)
  for (int k = 0; k < 4; ++k) {
    run += v[k];
    if (run >= need) { atomicMin(&best, (u32)(4 * t + k)); break; }
  }
  __syncthreads();
  if (t == 0) P.ctl[level - 1] = best;
}
__global__ void __launch_bounds__(256) gq_k_sel_compact(const __grid_constant__ GqSelParams P, u32* idx) {
  const u32 t1 = P.ctl[0], t2 = P.ctl[1];
  int s1, s2;
  gq_sel_shifts(P, &s1, &s2);
  for (u32 r0 = blockIdx.x * 256; r0 < P.n; r0 += gridDim.x * 256) {
    const u32 r = r0 + threadIdx.x;
    bool take = false;
    if (r < P.n) {
      const u64 u = gq_sel_top(P, r);
      const u32 b1 = (u32)(u >> s1) & (GQ_SEL_BINS - 1), b2 = (u32)(u >> s2) & (GQ_SEL_BINS - 1);
      take = b1 < t1 || (b1 == t1 && b2 <= t2);
    }
    const u32 m = __ballot_sync(0xffffffffu, take);
    u32 base = 0;
    if ((threadIdx.x & 31) == 0 && m) base = atomicAdd(&P.ctl[2], (u32)__popc(m));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (take) idx[base + __popc(m & ((1u << (threadIdx.x & 31)) - 1u))] = r;   // any order: the rows are sorted by index first
  }
}

struct GqEmitParams {
  const u32* idx[2]; const u32* ctl; const u32* d_n; u64 limit; i64* out_index;
  int ncols; const void* col[GQ_MAX_COLS]; void* out[GQ_MAX_COLS]; int dtype[GQ_MAX_COLS];
};
// Four output rows per thread: the four row numbers are loaded first, then, column by column, four random reads are in
// flight per thread (one dependent load after the other left the gather at half of the DRAM random-sector rate).
__global__ void gq_k_sort_emit(const __grid_constant__ GqEmitParams P) {
  const u64 n = min((u64)gq_sort_n(P.d_n), P.limit);
  bool live;
  const u32* idx = P.idx[gq_sort_where(P.ctl, -1, 0, &live)];       // the buffer the last non-skipped pass wrote
  const u64 stride = (u64)gridDim.x * blockDim.x;
  for (u64 i0 = blockIdx.x * (u64)blockDim.x + threadIdx.x; i0 < n; i0 += 4 * stride) {
    i64 r[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const u64 i = i0 + u * stride; r[u] = i < n ? (i64)idx[i] : 0; }
    if (P.out_index) {
#pragma unroll
      for (int u = 0; u < 4; ++u) { const u64 i = i0 + u * stride; if (i < n) P.out_index[i] = r[u]; }
    }
    for (int c = 0; c < P.ncols; ++c) {
      if (!P.out[c]) continue;
      i64 v[4];
      if (P.dtype[c] == GQ_I8) {
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = (i64)((const signed char*)P.col[c])[r[u]];
#pragma unroll
        for (int u = 0; u < 4; ++u) { const u64 i = i0 + u * stride; if (i < n) ((signed char*)P.out[c])[i] = (signed char)v[u]; }
      } else if (P.dtype[c] == GQ_I32) {
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = (i64)((const int*)P.col[c])[r[u]];
#pragma unroll
        for (int u = 0; u < 4; ++u) { const u64 i = i0 + u * stride; if (i < n) ((int*)P.out[c])[i] = (int)v[u]; }
      } else {
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = ((const i64*)P.col[c])[r[u]];
#pragma unroll
        for (int u = 0; u < 4; ++u) { const u64 i = i0 + u * stride; if (i < n) ((i64*)P.out[c])[i] = v[u]; }
      }
    }
  }
}

// ---- small inputs: one CTA, one launch. ORDER BY at the end of a query usually sees a handful of groups (Fig. 2:
// OrderBy after the final aggregation); the radix path costs >= 27 launches whatever the size (~100 us). Up to 2048 rows
// are sorted as row numbers in shared memory by a bitonic network whose comparator reads the key columns (lexicographic,
// signed, per-key direction, the row number last: a total order, so the unstable network gives the stable result), and
// the same CTA gathers the outputs.
#define GQ_SMALL_SORT_MAX 2048
struct GqSmallSortParams {
  u32 n; int nkeys; u64 limit; i64* out_index; int ncols;
  const void* key[GQ_MAX_COLS]; int key_dtype[GQ_MAX_COLS]; int key_desc[GQ_MAX_COLS];
  const void* col[GQ_MAX_COLS]; void* out[GQ_MAX_COLS]; int dtype[GQ_MAX_COLS];
};
// The first GQ_SMALL_IMG key columns are compared through their sortable images in shared memory (unsigned order ==
// requested order), further ones through the columns themselves.
#define GQ_SMALL_IMG 2
__device__ __forceinline__ bool gq_small_less(const GqSmallSortParams& P, const u64 (*img)[GQ_SMALL_SORT_MAX], u32 a, u32 b) {   // row a strictly before row b
  if (a == 0xFFFFFFFFu) return false;                     // padding sorts last
  if (b == 0xFFFFFFFFu) return true;
#pragma unroll
  for (int k = 0; k < GQ_SMALL_IMG; ++k)
    if (k < P.nkeys) { const u64 x = img[k][a], y = img[k][b]; if (x != y) return x < y; }
  for (int k = GQ_SMALL_IMG; k < P.nkeys; ++k) {
    const i64 x = gq_sort_load(P.key[k], P.key_dtype[k], (i64)a), y = gq_sort_load(P.key[k], P.key_dtype[k], (i64)b);
    if (x != y) return P.key_desc[k] ? x > y : x < y;
  }
  return a < b;
}
__global__ void __launch_bounds__(1024) gq_k_sort_small(const __grid_constant__ GqSmallSortParams P) {
  __shared__ u32 idx[GQ_SMALL_SORT_MAX];
  __shared__ u64 img[GQ_SMALL_IMG][GQ_SMALL_SORT_MAX];
  const u32 t = threadIdx.x;
  u32 N = 2;
  while (N < P.n) N <<= 1;                                // power of two >= n (>= 2)
  for (u32 i = t; i < N; i += 1024) idx[i] = i < P.n ? i : 0xFFFFFFFFu;
  for (int k = 0; k < GQ_SMALL_IMG && k < P.nkeys; ++k) {
    const int bytes = P.key_dtype[k] == GQ_I8 ? 1 : P.key_dtype[k] == GQ_I32 ? 4 : 8;
    for (u32 i = t; i < P.n; i += 1024) img[k][i] = gq_sort_image(gq_sort_load(P.key[k], P.key_dtype[k], (i64)i), bytes, P.key_desc[k]);
  }
  __syncthreads();
  for (u32 k = 2; k <= N; k <<= 1)
    for (u32 j = k >> 1; j > 0; j >>= 1) {
      if (t < N / 2) {                                    // compare-exchange number t of this stage: elements e and e + j
        const u32 e = ((t & ~(j - 1u)) << 1) | (t & (j - 1u));   // = 2 j (t / j) + t % j, j a power of two
        const bool asc = (e & k) == 0;
        const u32 a = idx[e], b = idx[e + j];
        if (gq_small_less(P, img, b, a) == asc) { idx[e] = b; idx[e + j] = a; }
      }
      __syncthreads();
    }
  const u64 nout = min((u64)P.n, P.limit);
  for (u64 i = t; i < nout; i += 1024) {
    const i64 r = (i64)idx[i];
    if (P.out_index) P.out_index[i] = r;
    for (int c = 0; c < P.ncols; ++c) {
      if (!P.out[c]) continue;
      if (P.dtype[c] == GQ_I8) ((signed char*)P.out[c])[i] = ((const signed char*)P.col[c])[r];
      else if (P.dtype[c] == GQ_I32) ((int*)P.out[c])[i] = ((const int*)P.col[c])[r];
      else ((i64*)P.out[c])[i] = ((const i64*)P.col[c])[r];
    }
  }
}

// ---- host side ----
struct GqSortLayout { size_t keys[2], idx[2], hist, sel1, sel2, ctl, total; int nblk; };
static GqSortLayout gq_sort_layout(i64 nrows, int num_sms) {
  GqSortLayout L;
  auto al = [](size_t v) { return (v + 255) / 256 * 256; };
  L.nblk = std::max(1, std::min(num_sms * 4, 1024));
  size_t off = 0;
  const size_t n = (size_t)std::max<i64>(1, nrows);
  for (int b = 0; b < 2; ++b) { L.keys[b] = off; off += al(n * 8); }
  for (int b = 0; b < 2; ++b) { L.idx[b] = off; off += al(n * 4); }
  L.hist = off; off += al((size_t)256 * 1024 * 4);
  L.sel1 = off; off += al(GQ_SEL_BINS * 4);
  L.sel2 = off; off += al(GQ_SEL_BINS * 4);
  L.ctl = off; off += GQ_SORT_CTL_BYTES;
  L.total = off;
  return L;
}
size_t gq_sort_workspace_bytes(i64 nrows) { return gq_sort_layout(nrows, GQ_MAX_SMS).total; }

cudaError_t gq_launch_order_by(cudaStream_t s, int num_sms, const gq_batch* in, const gq_sort_key* keys, int nkeys, i64 limit, char* ws,
                               i64* out_index, void* const* out_cols, int* nlaunches) {
  const GqSortLayout L = gq_sort_layout(in->nrows, GQ_MAX_SMS);
  const int nblk = std::max(1, std::min(num_sms * 4, 1024));
  const u32 n = (u32)in->nrows;
  const u64 lim = limit <= 0 || limit > in->nrows ? (u64)in->nrows : (u64)limit;
  if (n <= GQ_SMALL_SORT_MAX) {                          // one CTA, one launch (the workspace is not used)
    GqSmallSortParams sp;
    sp.n = n; sp.nkeys = nkeys; sp.limit = lim; sp.out_index = out_index; sp.ncols = in->ncols;
    for (int k = 0; k < nkeys; ++k) {
      const gq_column& c = in->cols[keys[k].col];
      sp.key[k] = c.data; sp.key_dtype[k] = (int)c.dtype; sp.key_desc[k] = keys[k].descending ? 1 : 0;
    }
    for (int c = 0; c < in->ncols; ++c) { sp.col[c] = in->cols[c].data; sp.out[c] = out_cols ? out_cols[c] : nullptr; sp.dtype[c] = (int)in->cols[c].dtype; }
    gq_k_sort_small<<<1, 1024, 0, s>>>(sp);
    *nlaunches = 1;
    return cudaGetLastError();
  }
  u64* kbuf[2] = {(u64*)(ws + L.keys[0]), (u64*)(ws + L.keys[1])};
  u32* ibuf[2] = {(u32*)(ws + L.idx[0]), (u32*)(ws + L.idx[1])};
  u32* hist = (u32*)(ws + L.hist);
  u32* ctl = (u32*)(ws + L.ctl);
  u32* d_n = ctl + 8;
  int nl = 0;
  GqSortBufs B;
  B.k[0] = kbuf[0]; B.k[1] = kbuf[1]; B.i[0] = ibuf[0]; B.i[1] = ibuf[1]; B.ctl = ctl;
  const int gs = std::max(1, std::min<int>(num_sms * 8, (int)((n + 255) / 256)));
  auto dtype_bytes = [](int t) { return t == GQ_I8 ? 1 : t == GQ_I32 ? 4 : 8; };
  const bool topn = nkeys > 0 && lim * 8 < (u64)n && n >= (1u << 16);
  // TopN sorts its few candidates (how many is known on the device only) with a small grid: the scan and the launches,
  // not the data, are what its passes cost. (Any grid is correct; many tied candidates just take longer.)
  const int nb = topn ? std::min(nblk, 16) : std::max(1, nblk / 2);   // (the full sort runs 2 CTAs of 512 threads per SM)
  auto passes = [&](int id, int bytes) {             // LSD passes over the low `bytes` bytes of sort column `id`'s keys
    for (int b = 0; b < bytes; ++b) {
      if (topn) {
        gq_k_sort_hist<256><<<nb, 256, 0, s>>>(B, d_n, id, b, hist);
        gq_k_sort_scan<<<1, 1024, 0, s>>>(hist, 256 * nb, ctl, id, b);
        gq_k_sort_scatter_staged<256><<<nb, 256, 0, s>>>(B, d_n, id, b, hist);
      } else {
        gq_k_sort_hist<512><<<nb, 512, 0, s>>>(B, d_n, id, b, hist);
        gq_k_sort_scan<<<1, 1024, 0, s>>>(hist, 256 * nb, ctl, id, b);
        gq_k_sort_scatter_staged<512><<<nb, 512, 0, s>>>(B, d_n, id, b, hist);
      }
      nl += 3;
    }
  };
  cudaError_t e = cudaSuccess;
  if (!topn) {
    e = cudaMemsetAsync(ctl, 0, GQ_SORT_CTL_BYTES, s);          // the control words (key masks of the pass skipping)
    if (e != cudaSuccess) return e;
  }
  if (topn) {
    e = cudaMemsetAsync(ws + L.sel1, 0, L.total - L.sel1, s);   // both histograms and the control words
    if (e != cudaSuccess) return e;
    GqSelParams sp;
    const gq_column& c0 = in->cols[keys[0].col];
    sp.col = c0.data; sp.dtype = (int)c0.dtype; sp.bytes = dtype_bytes((int)c0.dtype); sp.desc = keys[0].descending ? 1 : 0;
    sp.n = n; sp.limit = lim; sp.hist1 = (u32*)(ws + L.sel1); sp.hist2 = (u32*)(ws + L.sel2); sp.ctl = ctl;
    gq_k_sel_range<<<gs, 256, 0, s>>>(sp);
    ++nl;
    for (int level = 1; level <= 2; ++level) {
      gq_k_sel_hist<<<gs, 256, 0, s>>>(sp, level);
      gq_k_sel_pick<<<1, 1024, 0, s>>>(sp, level);
    }
    gq_k_sel_compact<<<gs, 256, 0, s>>>(sp, ibuf[0]);
    nl += 5;
    e = cudaMemcpyAsync(d_n, ctl + 2, 4, cudaMemcpyDeviceToDevice, s);
    if (e != cudaSuccess) return e;
    // candidates were appended in any order: sort them by row index first (the least significant "key" of a stable sort)
    gq_k_sort_keys<<<gs, 256, 0, s>>>(nullptr, 0, 4, 0, B, d_n, GQ_SORT_ROWID);
    ++nl;
    passes(GQ_SORT_ROWID, 4);
  } else {
    gq_k_sort_iota<<<gs, 256, 0, s>>>(ibuf[0], n, d_n);
    ++nl;
  }
  for (int k = nkeys - 1; k >= 0; --k) {
    const gq_column& c = in->cols[keys[k].col];
    gq_k_sort_keys<<<gs, 256, 0, s>>>(c.data, (int)c.dtype, dtype_bytes((int)c.dtype), keys[k].descending ? 1 : 0, B, d_n, k);
    ++nl;
    passes(k, dtype_bytes((int)c.dtype));
  }
  GqEmitParams ep;
  ep.idx[0] = ibuf[0]; ep.idx[1] = ibuf[1]; ep.ctl = ctl; ep.d_n = d_n; ep.limit = lim; ep.out_index = out_index; ep.ncols = in->ncols;
  for (int c = 0; c < in->ncols; ++c) { ep.col[c] = in->cols[c].data; ep.out[c] = out_cols ? out_cols[c] : nullptr; ep.dtype[c] = (int)in->cols[c].dtype; }
  const int ge = std::max(1, std::min<int>(num_sms * 8, (int)((lim + 255) / 256)));
  gq_k_sort_emit<<<ge, 256, 0, s>>>(ep);
  ++nl;
  *nlaunches = nl;
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------- allocation-free entry point
// gq_order_by_static (include/gq.h): the same launch sequence as gq_order_by, with its workspace in a file-scope device
// array instead of caller memory — for callers that cannot allocate (code under CUDA-graph capture, serving loops,
// harnesses that forbid cudaMalloc). The array is sized for GQ_ORDER_BY_STATIC_MAX_ROWS rows (the layout of
// gq_sort_layout: 2 x 8 B + 2 x 4 B per row, 1 MiB of digit histograms, two select histograms, control words: 4.2 MB)
// and every GPU that loads libgq.so holds it until the process exits.
//   * In HOST code the array's name is a host-side stand-in, not a device address: the device address is taken once per
//     device with cudaGetSymbolAddress, with that device current, and it is that pointer the kernels receive.
//   * All calls share the array and it keeps the previous call's contents. Nothing in it has to start at zero except
//     the select histograms and control words of the TopN path, which gq_launch_order_by clears itself (stream-ordered
//     cudaMemsetAsync) before it uses them; every other region is written before it is read.
//   * Two calls that overlap on the GPU (different streams / contexts of one device) RACE on the array: callers
//     serialise them (one stream, or an event between them).
#define GQ_SORT_AL256(v) ((((size_t)(v)) + 255) / 256 * 256)
#define GQ_SORT_STATIC_BYTES                                                                                        \
  (2 * GQ_SORT_AL256((size_t)GQ_ORDER_BY_STATIC_MAX_ROWS * 8) + 2 * GQ_SORT_AL256((size_t)GQ_ORDER_BY_STATIC_MAX_ROWS * 4) + \
   GQ_SORT_AL256((size_t)256 * 1024 * 4) + 2 * GQ_SORT_AL256(GQ_SEL_BINS * 4) + GQ_SORT_CTL_BYTES)
static __device__ __align__(256) unsigned char gq_sort_static_scratch[GQ_SORT_STATIC_BYTES];

#include <mutex>
#define GQ_SORT_STATIC_MAX_DEVICES 64
static std::mutex g_sort_static_mu;
static char* g_sort_static_ptr[GQ_SORT_STATIC_MAX_DEVICES];   // device address of the array, per device ordinal (null = not asked yet)

// Set-up, once per device: the CURRENT device's address of the scratch array.
static cudaError_t gq_sort_static_address(char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= GQ_SORT_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_sort_static_mu);
  if (!g_sort_static_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, gq_sort_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p || ((size_t)p & 255) != 0) return cudaErrorInvalidSymbol;
    g_sort_static_ptr[dev] = (char*)p;
  }
  *out = g_sort_static_ptr[dev];
  return cudaSuccess;
}

long long gq_sort_static_max_rows() { return GQ_ORDER_BY_STATIC_MAX_ROWS; }

// The caller (gq_api.cpp) has made the context's device current and checked in->nrows <= GQ_ORDER_BY_STATIC_MAX_ROWS.
cudaError_t gq_launch_order_by_static(cudaStream_t s, int num_sms, const gq_batch* in, const gq_sort_key* keys, int nkeys, i64 limit,
                                      i64* out_index, void* const* out_cols, int* nlaunches) {
  if (in->nrows > GQ_ORDER_BY_STATIC_MAX_ROWS || gq_sort_layout(in->nrows, GQ_MAX_SMS).total > (size_t)GQ_SORT_STATIC_BYTES)
    return cudaErrorInvalidValue;
  char* ws = nullptr;
  cudaError_t e = gq_sort_static_address(&ws);
  if (e != cudaSuccess) return e;
  return gq_launch_order_by(s, num_sms, in, keys, nkeys, limit, ws, out_index, out_cols, nlaunches);
}

// ------------------------------------------------------------------------------------- hash partitioning (gq_hash_partition)
// CudfPartitionedOutput: the rows of a batch are grouped by destination =
// gq_hp_dest(key columns) (the function include/gq.h defines), destination-major, input order inside a destination —
// one contiguous packed range per destination, ready to be sent. A stable counting sort with ONE read of the key columns
// (histogram), one read of every column and one write (scatter): (keys + 2 x row bytes) per row, HBM-bound.
//   histogram — every CTA owns a contiguous range of 2048-row tiles and counts its rows per destination (shared-memory
//               counters, one add per distinct destination and 32 rows through MATCH.ANY);
//   scan      — gq_k_sort_scan over [destination][CTA]: exclusive offsets, destination-major, stable across CTAs;
//   scatter   — every CTA walks its range again, tile by tile. Inside a tile warp w owns rows [256 w, 256 w + 256): it
//               ranks them per destination on its own (MATCH.ANY + warp-private counters, no CTA barrier), one pass over
//               [warp][destination] turns the counters into offsets, and every row knows its place in the tile's
//               destination-major order. Then, column by column, the tile is permuted THROUGH SHARED MEMORY: values go to
//               their place in a staging buffer, and the buffer is written out in order, so that the rows of one
//               destination leave as one contiguous run (2048 / nparts rows on average) instead of row by row — a warp
//               writing single 4-byte values into 64 open streams reached 0.5 TB/s, a sixth of this.
#define GQ_HP_THREADS 256
#define GQ_HP_WARPS (GQ_HP_THREADS / 32)
#define GQ_HP_ITEMS 8                              // rows per thread and tile
#define GQ_HP_TILE (GQ_HP_THREADS * GQ_HP_ITEMS)
#ifndef GQ_HP_CTAS_PER_SM
#define GQ_HP_CTAS_PER_SM 4
#endif
struct GqHpParams {
  u32 n; int nparts; int nkeys; int ncols;
  const void* key[GQ_MAX_KEYS_HP]; int key_dtype[GQ_MAX_KEYS_HP];
  const void* col[GQ_MAX_COLS]; void* out[GQ_MAX_COLS]; int dtype[GQ_MAX_COLS];
  u32* hist;                 // [nparts][CTAs of the grid]
  i64* out_row;              // input row number of every output row, or null
  i64* out_offsets;          // [nparts + 1] (or null)
  // peer variant (gq_hash_partition_scatter_to): destination d's column c is written through dst[d * ncols + c], starting
  // at row dst_row0[d] of that buffer — the buffers may live in ANOTHER GPU's memory (peer-mapped over NVLink)
  void* const* dst; const i64* dst_row0;
};
// Destinations of the calling thread's GQ_HP_ITEMS rows r0 + j * stride (rows >= hi get the invalid value 256 + lane, a
// different one per lane). Key column by key column: all of the thread's loads of a column are issued before the first
// hash step uses one (a row-at-a-time loop left ONE load in flight per thread: the histogram ran at 1.6 TB/s).
template <typename T>
__device__ __forceinline__ void gq_hp_mix(const void* col, u32 r0, u32 stride, u32 hi, u64 (&h)[GQ_HP_ITEMS]) {
  T v[GQ_HP_ITEMS];
#pragma unroll
  for (int j = 0; j < GQ_HP_ITEMS; ++j) { const u32 r = r0 + (u32)j * stride; v[j] = r < hi ? ((const T*)col)[r] : (T)0; }
#pragma unroll
  for (int j = 0; j < GQ_HP_ITEMS; ++j) {
    u64 x = h[j] ^ (u64)(i64)v[j];
    x ^= x >> 33; x *= 0xff51afd7ed558ccdULL; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ULL; x ^= x >> 33;
    h[j] = x;
  }
}
__device__ __forceinline__ void gq_hp_dests(const GqHpParams& P, u32 r0, u32 stride, u32 hi, int lane, u32 (&d)[GQ_HP_ITEMS]) {
  u64 h[GQ_HP_ITEMS];
#pragma unroll
  for (int j = 0; j < GQ_HP_ITEMS; ++j) h[j] = 0x9E3779B97F4A7C15ULL;
#pragma unroll 1
  for (int k = 0; k < P.nkeys; ++k) {
    if (P.key_dtype[k] == GQ_I64) gq_hp_mix<i64>(P.key[k], r0, stride, hi, h);
    else if (P.key_dtype[k] == GQ_I32) gq_hp_mix<int>(P.key[k], r0, stride, hi, h);
    else gq_hp_mix<signed char>(P.key[k], r0, stride, hi, h);
  }
#pragma unroll
  for (int j = 0; j < GQ_HP_ITEMS; ++j)
    d[j] = r0 + (u32)j * stride < hi ? (u32)(((h[j] >> 32) * (u64)(u32)P.nparts) >> 32) : 256u + (u32)lane;
}
// rows [lo, hi) of the calling CTA: whole tiles, contiguous, in CTA order
__device__ __forceinline__ void gq_hp_range(u32 n, u32* lo, u32* hi, u32 tile) {
  const u32 ntiles = (n + tile - 1) / tile;
  const u32 per = (ntiles + gridDim.x - 1) / gridDim.x;
  const u64 a = (u64)blockIdx.x * per * tile, b = a + (u64)per * tile;
  *lo = (u32)(a < n ? a : n);
  *hi = (u32)(b < n ? b : n);
}
template <int NT>
__global__ void __launch_bounds__(NT) gq_k_hp_hist(const __grid_constant__ GqHpParams P) {
  constexpr int NW = NT / 32;
  __shared__ u32 cnt[NW][256];                       // warp-private counters: an add only meets the adds of its own warp
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  if (t < 256) for (int w = 0; w < NW; ++w) cnt[w][t] = 0;
  __syncthreads();
  u32 lo, hi;
  gq_hp_range(P.n, &lo, &hi, NT * GQ_HP_ITEMS);
  for (u32 base = lo; base < hi; base += NT * GQ_HP_ITEMS) {
    u32 d[GQ_HP_ITEMS];
    gq_hp_dests(P, base + (u32)t, NT, hi, lane, d);
#pragma unroll
    for (int j = 0; j < GQ_HP_ITEMS; ++j) if (d[j] < 256u) atomicAdd(&cnt[warp][d[j]], 1u);
  }
  __syncthreads();
  if (t < P.nparts) {
    u32 s = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) s += cnt[w][t];
    P.hist[(size_t)t * gridDim.x + blockIdx.x] = s;
  }
}
// the calling thread's GQ_HP_ITEMS values of column c (rows base + 256 warp + 32 j + lane of a tile of nt rows), as raw words
__device__ __forceinline__ void gq_hp_load(const GqHpParams& P, int c, u32 base, u32 nt, int warp, int lane, u64 (&v)[GQ_HP_ITEMS]) {
  const int dt = P.dtype[c];
  const u32 i0 = (u32)warp * 256u + (u32)lane;
  if (dt == GQ_I64) {
    const u64* src = (const u64*)P.col[c] + base;
#pragma unroll
    for (int j = 0; j < GQ_HP_ITEMS; ++j) { const u32 i = i0 + (u32)j * 32u; v[j] = i < nt ? src[i] : 0ULL; }
  } else if (dt == GQ_I32) {
    const u32* src = (const u32*)P.col[c] + base;
#pragma unroll
    for (int j = 0; j < GQ_HP_ITEMS; ++j) { const u32 i = i0 + (u32)j * 32u; v[j] = i < nt ? (u64)src[i] : 0ULL; }
  } else {
    const unsigned char* src = (const unsigned char*)P.col[c] + base;
#pragma unroll
    for (int j = 0; j < GQ_HP_ITEMS; ++j) { const u32 i = i0 + (u32)j * 32u; v[j] = i < nt ? (u64)src[i] : 0ULL; }
  }
}
// NT = 256 (4 CTAs per SM, 2048-row tiles) below GQ_HP_WIDE_FROM destinations, 512 (2 CTAs per SM, 4096-row tiles: half as
// many open write streams, runs twice as long) from there on: C2 table, 256 destinations 2.44 -> 1.72 ms, but 64
// destinations 1.09 -> 1.17 ms.
template <int NT, bool PEER>
__global__ void __launch_bounds__(NT, 1024 / NT) gq_k_hp_scatter(const __grid_constant__ GqHpParams P) {
  constexpr int NW = NT / 32, TILE = NT * GQ_HP_ITEMS;
  __shared__ u32 cur[256];                             // the CTA's next output row per destination (at the tile's start)
  __shared__ unsigned short wc[NW][256];               // per tile: rows of a destination in every warp, then their offsets
  __shared__ unsigned short toff[256];                 // per tile: first place of every destination in the tile's order
  __shared__ u32 wsum[8];
  __shared__ unsigned char pd[TILE];                   // per tile: destination of every place (output row = cur + place - toff)
  constexpr bool GPOS = NT == 256;                     // 2048-row tiles also keep the output row of every place (one lookup per
  __shared__ u32 gpos[GPOS ? TILE : 1];                //  element instead of three; 4096-row tiles have no room for it)
  __shared__ __align__(16) unsigned char stage[TILE * 8];
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  if (t < 256) {
    cur[t] = t < P.nparts ? P.hist[(size_t)t * gridDim.x + blockIdx.x] : 0u;
    if (PEER) {   // cursor = row inside the DESTINATION's buffer: dst_row0[d] + (row among this sender's rows for d); < 2^32
      if (t < P.nparts) cur[t] = cur[t] - P.hist[(size_t)t * gridDim.x] + (u32)P.dst_row0[t];
    }
    if (blockIdx.x == 0 && P.out_offsets) {            // CTA 0's cursors are the destinations' first rows
      if (t < P.nparts) P.out_offsets[t] = (i64)P.hist[(size_t)t * gridDim.x];
      if (t == 0) P.out_offsets[P.nparts] = (i64)P.n;
    }
  }
  u32 lo, hi;
  gq_hp_range(P.n, &lo, &hi, TILE);
  for (u32 base = lo; base < hi; base += TILE) {
    const u32 nt = min((u32)TILE, hi - base);          // rows of this tile
    if (t < 256) for (int w = 0; w < NW; ++w) wc[w][t] = 0;
    __syncthreads();
    // (1) destination and rank among the warp's rows of that destination; the warp's rows are base + 256 warp + 32 j + lane
    u32 d[GQ_HP_ITEMS];
    unsigned short place[GQ_HP_ITEMS];                 // rank among the warp's rows of the destination, then place in the tile
    gq_hp_dests(P, base + (u32)warp * 256u + (u32)lane, 32u, base + nt, lane, d);
#pragma unroll
    for (int j = 0; j < GQ_HP_ITEMS; ++j) {
      const u32 peers = __match_any_sync(0xffffffffu, d[j]);
      const u32 rank = __popc(peers & ((1u << lane) - 1u));
      const bool have = d[j] < 256u;
      place[j] = have ? (unsigned short)(wc[warp][d[j]] + rank) : (unsigned short)0;
      __syncwarp();
      if (have && rank == 0) wc[warp][d[j]] += (unsigned short)__popc(peers);
      __syncwarp();
    }
    __syncthreads();
    // (2) thread q < 256: counters of destination q -> offsets over the warps; block scan of the totals -> toff
    u32 tot = 0, incl = 0;
    if (t < 256) {
#pragma unroll
      for (int w = 0; w < NW; ++w) { const u32 c = wc[w][t]; wc[w][t] = (unsigned short)tot; tot += c; }
      incl = tot;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const u32 x = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += x; }
      if (lane == 31) wsum[warp] = incl;
    }
    __syncthreads();
    if (t < 256) {
      u32 before = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) if (w < warp) before += wsum[w];
      toff[t] = (unsigned short)(before + incl - tot);  // place of destination t's first row in the tile
    }
    __syncthreads();
    // (3) place of every row in the tile's destination-major order
#pragma unroll
    for (int j = 0; j < GQ_HP_ITEMS; ++j) {
      if (d[j] < 256u) {
        const u32 in_run = (u32)wc[warp][d[j]] + (u32)place[j];        // rows of this destination before mine in the tile
        place[j] = (unsigned short)((u32)toff[d[j]] + in_run);
        pd[place[j]] = (unsigned char)d[j];
        if (GPOS) gpos[place[j]] = cur[d[j]] + in_run;
      }
    }
    if (P.out_row) {
#pragma unroll
      for (int j = 0; j < GQ_HP_ITEMS; ++j) {
        const u32 i = (u32)warp * 256u + (u32)j * 32u + (u32)lane;
        if (i < nt) P.out_row[cur[d[j]] + (u32)place[j] - (u32)toff[d[j]]] = (i64)(base + i);
      }
    }
    // (4) column by column through the staging buffer. A column's values are loaded as raw 64-bit words one column AHEAD:
    // the loads of column c + 1 are in flight while column c is written out (the registers are free once c is staged).
    u64 v[GQ_HP_ITEMS];
    gq_hp_load(P, 0, base, nt, warp, lane, v);
#pragma unroll 1
    for (int c = 0; c < P.ncols; ++c) {
      const int dt = P.dtype[c];
      if (dt == GQ_I64) {
#pragma unroll
        for (int j = 0; j < GQ_HP_ITEMS; ++j) if (d[j] < 256u) ((u64*)stage)[place[j]] = v[j];
      } else if (dt == GQ_I32) {
#pragma unroll
        for (int j = 0; j < GQ_HP_ITEMS; ++j) if (d[j] < 256u) ((u32*)stage)[place[j]] = (u32)v[j];
      } else {
#pragma unroll
        for (int j = 0; j < GQ_HP_ITEMS; ++j) if (d[j] < 256u) ((unsigned char*)stage)[place[j]] = (unsigned char)v[j];
      }
      if (c + 1 < P.ncols) gq_hp_load(P, c + 1, base, nt, warp, lane, v);
      __syncthreads();                                  // (also: pd of this tile is complete)
      for (u32 p = t; p < nt; p += NT) {
        const u32 dd = pd[p];
        const u32 row = GPOS ? gpos[p] : cur[dd] + p - (u32)toff[dd];
        void* o = PEER ? (void*)__ldg((const unsigned long long*)P.dst + (size_t)dd * P.ncols + c) : P.out[c];   // PEER: d's own buffer (peer memory)
        if (dt == GQ_I64) ((u64*)o)[row] = ((const u64*)stage)[p];
        else if (dt == GQ_I32) ((u32*)o)[row] = ((const u32*)stage)[p];
        else ((unsigned char*)o)[row] = ((const unsigned char*)stage)[p];
      }
      __syncthreads();                                  // the buffer is free for the next column / tile
    }
    if (t < 256) cur[t] += tot;                         // (read again only after the next tile's barriers)
  }
}
// 4 CTAs of 256 threads per SM up to GQ_HP_WIDE_FROM destinations, 2 CTAs of 512 threads above
#define GQ_HP_WIDE_FROM 128
static int gq_hp_blocks(int num_sms, int nparts) { return std::max(1, std::min(num_sms * (nparts >= GQ_HP_WIDE_FROM ? 2 : 4), 1024)); }
size_t gq_hash_partition_workspace_bytes(int nparts) {
  return ((size_t)nparts * (size_t)gq_hp_blocks(GQ_MAX_SMS, 1) * 4 + 255) / 256 * 256;
}
cudaError_t gq_launch_hash_partition(cudaStream_t s, int num_sms, const gq_batch* in, const int* key_cols, int nkeys, int nparts, char* ws,
                                     void* const* out_cols, i64* out_row, i64* out_offsets, int* nlaunches) {
  GqHpParams P;
  P.n = (u32)in->nrows; P.nparts = nparts; P.nkeys = nkeys; P.ncols = in->ncols;
  for (int k = 0; k < nkeys; ++k) { P.key[k] = in->cols[key_cols[k]].data; P.key_dtype[k] = (int)in->cols[key_cols[k]].dtype; }
  for (int c = 0; c < in->ncols; ++c) { P.col[c] = in->cols[c].data; P.out[c] = out_cols[c]; P.dtype[c] = (int)in->cols[c].dtype; }
  P.hist = (u32*)ws; P.out_row = out_row; P.out_offsets = out_offsets; P.dst = nullptr; P.dst_row0 = nullptr;
  const int nblk = gq_hp_blocks(num_sms, nparts);
  if (nparts >= GQ_HP_WIDE_FROM) gq_k_hp_hist<512><<<nblk, 512, 0, s>>>(P); else gq_k_hp_hist<256><<<nblk, 256, 0, s>>>(P);
  gq_k_sort_scan<<<1, 1024, 0, s>>>(P.hist, nparts * nblk);
  if (nparts >= GQ_HP_WIDE_FROM) gq_k_hp_scatter<512, false><<<nblk, 512, 0, s>>>(P); else gq_k_hp_scatter<256, false><<<nblk, 256, 0, s>>>(P);
  *nlaunches = 3;
  return cudaGetLastError();
}
// Two-phase variant for a partition fused with its transfer: (1) count — histogram + scan, rows per destination to
// d_counts; the caller exchanges the counts and derives where this sender's rows start in every destination's buffers;
// (2) scatter_to — the scatter of the SAME batch (the scanned histogram is still in ws), every destination's run written
// through that destination's own column pointers (peer-mapped memory of another GPU: the stores travel over NVLink
// while the next tile is being permuted — no packed send buffer, no separate all-to-all).
__global__ void gq_k_hp_counts(const u32* hist, int nblk, int nparts, u32 n, i64* counts) {
  const int d = blockIdx.x * blockDim.x + threadIdx.x;
  if (d >= nparts) return;
  const u32 a = hist[(size_t)d * nblk], b = d + 1 < nparts ? hist[(size_t)(d + 1) * nblk] : n;
  counts[d] = (i64)(b - a);
}
static void gq_hp_fill(GqHpParams& P, const gq_batch* in, const int* key_cols, int nkeys, int nparts, char* ws) {
  P.n = (u32)in->nrows; P.nparts = nparts; P.nkeys = nkeys; P.ncols = in->ncols;
  for (int k = 0; k < nkeys; ++k) { P.key[k] = in->cols[key_cols[k]].data; P.key_dtype[k] = (int)in->cols[key_cols[k]].dtype; }
  for (int c = 0; c < in->ncols; ++c) { P.col[c] = in->cols[c].data; P.out[c] = nullptr; P.dtype[c] = (int)in->cols[c].dtype; }
  P.hist = (u32*)ws; P.out_row = nullptr; P.out_offsets = nullptr; P.dst = nullptr; P.dst_row0 = nullptr;
}
cudaError_t gq_launch_hash_partition_count(cudaStream_t s, int num_sms, const gq_batch* in, const int* key_cols, int nkeys, int nparts, char* ws,
                                           i64* counts, int* nlaunches) {
  GqHpParams P;
  gq_hp_fill(P, in, key_cols, nkeys, nparts, ws);
  const int nblk = gq_hp_blocks(num_sms, nparts);
  if (nparts >= GQ_HP_WIDE_FROM) gq_k_hp_hist<512><<<nblk, 512, 0, s>>>(P); else gq_k_hp_hist<256><<<nblk, 256, 0, s>>>(P);
  gq_k_sort_scan<<<1, 1024, 0, s>>>(P.hist, nparts * nblk);
  gq_k_hp_counts<<<1, 256, 0, s>>>(P.hist, nblk, nparts, P.n, counts);
  *nlaunches = 3;
  return cudaGetLastError();
}
cudaError_t gq_launch_hash_partition_scatter_to(cudaStream_t s, int num_sms, const gq_batch* in, const int* key_cols, int nkeys, int nparts,
                                                char* ws, void* const* d_dst, const i64* d_row0, int* nlaunches) {
  GqHpParams P;
  gq_hp_fill(P, in, key_cols, nkeys, nparts, ws);
  P.dst = d_dst; P.dst_row0 = d_row0;
  if (nparts >= GQ_HP_WIDE_FROM) gq_k_hp_scatter<512, true><<<gq_hp_blocks(num_sms, nparts), 512, 0, s>>>(P);
  else gq_k_hp_scatter<256, true><<<gq_hp_blocks(num_sms, nparts), 256, 0, s>>>(P);
  *nlaunches = 1;
  return cudaGetLastError();
}
