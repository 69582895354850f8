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
  // (npart <= 16384: a thread's <= 16 counts are read once, all loads in flight together, and kept in registers)
  u32 cnt[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) cnt[i] = (i < per && lo + i < hi) ? P.pcount[lo + i] : 0u;
  u32 s = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += cnt[i];
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
#pragma unroll
  for (int i = 0; i < 16; ++i) if (i < per && lo + i < hi) { P.pstart[lo + i] = run; run += cnt[i]; }
  if (t == 0) P.pstart[P.npart] = total;
  const u32 big = 4 * (total / (u32)P.npart) + 64;
  auto cls = [&](u32 n) { return n > P.seg_chunks ? 0 : n > big ? 1 : 2; };
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const u32 n = cnt[i];
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
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const u32 n = cnt[i];
    const int p = lo + i;
    if (!n) continue;
    const u32 k = n > P.seg_chunks ? (n + P.seg_chunks - 1) / P.seg_chunks : 1u;
    const u32 at = atomicAdd(&cls_cur[cls(n)], k * P.nsub);   // the sub-passes of a segment are neighbours in the queue: the
    for (u32 i = 0; i < k * P.nsub; ++i) {                     // CTAs that draw them stream the same chunks at the same time (L2)
      P.items[at + i] = (u32)p; P.item_seg[at + i] = (i / P.nsub) | ((i % P.nsub) << 24);
    }
  }
}
cudaError_t gq_launch_psa_dir(cudaStream_t s, const GqPsaDirParams& p) {
  if (p.npart > 16 * GQ_DIR_THREADS) return cudaErrorInvalidValue;   // a thread keeps its <= 16 counts in registers
  gq_k_psa_dir<<<1, GQ_DIR_THREADS, 0, s>>>(p);
  return cudaGetLastError();
}

// Directory fill: every chunk a pass-A CTA opened (chunk ids [c * slab, c * slab + ncta[c])) is entered under its
// partition as (chunk id | records used << GQ_PSA_GID_BITS); the order inside a partition does not matter.
__global__ void __launch_bounds__(256) gq_k_psa_fill(const u32* info, const u32* ncta, long long slab, const u32* pstart, u32* pfill,
                                                     u32* plist) {
  const u32 c = blockIdx.y;
  const u32 n = ncta[c];
  // four chunks per thread and iteration: the kernel is a chain of dependent L2 round trips (word -> counter -> start ->
  // store), so it is the number of chains in flight that sets its speed
  for (u32 l0 = (blockIdx.x * blockDim.x + threadIdx.x) * 4u; l0 < n; l0 += gridDim.x * blockDim.x * 4u) {
    const u64 gid0 = (u64)c * (u64)slab + l0;
    u32 e[4], pos[4], st[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) e[u] = l0 + u < n ? info[gid0 + u] : 0u;
#pragma unroll
    for (int u = 0; u < 4; ++u) if (l0 + u < n) { pos[u] = atomicAdd(&pfill[(e[u] >> 8) * GQ_PSA_FILL_STRIDE], 1u); st[u] = pstart[e[u] >> 8]; }
#pragma unroll
    for (int u = 0; u < 4; ++u) if (l0 + u < n) plist[st[u] + pos[u]] = (u32)(gid0 + u) | ((e[u] & 0xFFu) << GQ_PSA_GID_BITS);
  }
}
cudaError_t gq_launch_psa_fill(cudaStream_t s, const u32* info, const u32* ncta, int nctas, long long slab, const u32* pstart,
                               u32* pfill, u32* plist) {
  const unsigned bx = (unsigned)std::min<long long>(64, std::max<long long>(1, (slab + 1023) / 1024));
  gq_k_psa_fill<<<dim3(bx, (unsigned)nctas), 256, 0, s>>>(info, ncta, slab, pstart, pfill, plist);
  return cudaGetLastError();
}
