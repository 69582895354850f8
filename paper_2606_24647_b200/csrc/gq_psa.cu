// gq_psa.cu — directory kernels of the partitioned shared-memory aggregation (between pass A, the SCATTER consumer of
// gq_scan, and pass B, gq_psa): turn the per-partition chunk counts into a directory of chunk ids grouped by
// partition, and into the queue of work items pass B draws from. Plan-independent, compiled by nvcc.
#include <algorithm>

#include "gq_internal.h"

typedef unsigned u32;
typedef unsigned long long u64;

// One CTA. (1) pstart = exclusive prefix sum of pcount; (2) work items, heaviest first, so that the long ones start
// early: the segments of split partitions (more than seg_chunks chunks), then partitions well above the average, then
// the rest; empty partitions produce no item.
#define GQ_DIR_THREADS 1024
__global__ void __launch_bounds__(GQ_DIR_THREADS) gq_k_psa_dir(const __grid_constant__ GqPsaDirParams P) {
  __shared__ u32 part_sum[GQ_DIR_THREADS];
  __shared__ u32 cls_n[3], cls_cur[3];
  const int t = threadIdx.x;
  const int per = (P.npart + GQ_DIR_THREADS - 1) / GQ_DIR_THREADS;
  const int lo = t * per, hi = min(P.npart, lo + per);
  u32 s = 0;
  for (int p = lo; p < hi; ++p) s += P.pcount[p];
  part_sum[t] = s;
  if (t < 3) cls_n[t] = 0;
  __syncthreads();
  for (int o = 1; o < GQ_DIR_THREADS; o <<= 1) {   // inclusive scan of the per-thread sums
    const u32 v = t >= o ? part_sum[t - o] : 0;
    __syncthreads();
    part_sum[t] += v;
    __syncthreads();
  }
  const u32 total = part_sum[GQ_DIR_THREADS - 1];
  u32 run = part_sum[t] - s;
  for (int p = lo; p < hi; ++p) { P.pstart[p] = run; run += P.pcount[p]; }
  if (t == 0) P.pstart[P.npart] = total;
  const u32 big = 4 * (total / (u32)P.npart) + 64;
  auto cls = [&](u32 n) { return n > P.seg_chunks ? 0 : n > big ? 1 : 2; };
  for (int p = lo; p < hi; ++p) {
    const u32 n = P.pcount[p];
    if (n) atomicAdd(&cls_n[cls(n)], (n > P.seg_chunks ? (n + P.seg_chunks - 1) / P.seg_chunks : 1u) * P.nsub);
  }
  __syncthreads();
  if (t == 0) {
    cls_cur[0] = 0; cls_cur[1] = cls_n[0]; cls_cur[2] = cls_n[0] + cls_n[1];
    const u32 n = cls_n[0] + cls_n[1] + cls_n[2];
    if (n > P.max_items) { atomicCAS(P.err, 0, (int)GQ_ERR_CAPACITY); *P.nitems = 0; } else *P.nitems = n;
  }
  __syncthreads();
  if (cls_n[0] + cls_n[1] + cls_n[2] > P.max_items) return;
  for (int p = lo; p < hi; ++p) {
    const u32 n = P.pcount[p];
    if (!n) continue;
    const u32 k = n > P.seg_chunks ? (n + P.seg_chunks - 1) / P.seg_chunks : 1u;
    const u32 at = atomicAdd(&cls_cur[cls(n)], k * P.nsub);   // the sub-passes of a segment are neighbours in the queue: the
    for (u32 i = 0; i < k * P.nsub; ++i) {                     // CTAs that draw them stream the same chunks at the same time (L2)
      P.items[at + i] = (u32)p; P.item_seg[at + i] = (i / P.nsub) | ((i % P.nsub) << 24);
    }
  }
}
cudaError_t gq_launch_psa_dir(cudaStream_t s, const GqPsaDirParams& p) {
  gq_k_psa_dir<<<1, GQ_DIR_THREADS, 0, s>>>(p);
  return cudaGetLastError();
}

// Directory fill: every chunk a pass-A CTA opened (chunk ids [c * slab, c * slab + ncta[c])) is entered under its
// partition as (chunk id | records used << GQ_PSA_GID_BITS); the order inside a partition does not matter.
__global__ void __launch_bounds__(256) gq_k_psa_fill(const u32* info, const u32* ncta, long long slab, const u32* pstart, u32* pfill,
                                                     u32* plist) {
  const u32 c = blockIdx.y;
  const u32 n = ncta[c];
  for (u32 l = blockIdx.x * blockDim.x + threadIdx.x; l < n; l += gridDim.x * blockDim.x) {
    const u64 gid = (u64)c * (u64)slab + l;
    const u32 e = info[gid];
    const u32 p = e >> 8, used = e & 0xFFu;
    const u32 pos = atomicAdd(&pfill[p], 1u);
    plist[pstart[p] + pos] = (u32)gid | (used << GQ_PSA_GID_BITS);
  }
}
cudaError_t gq_launch_psa_fill(cudaStream_t s, const u32* info, const u32* ncta, int nctas, long long slab, const u32* pstart,
                               u32* pfill, u32* plist) {
  const unsigned bx = (unsigned)std::min<long long>(64, std::max<long long>(1, (slab + 255) / 256));
  gq_k_psa_fill<<<dim3(bx, (unsigned)nctas), 256, 0, s>>>(info, ncta, slab, pstart, pfill, plist);
  return cudaGetLastError();
}
