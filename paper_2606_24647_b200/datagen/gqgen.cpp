// gqgen — seeded, integer-only, counter-based generator of synthetic analytical columns.
//
// Serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench) with identical bytes. It holds NONE of the
// method's arithmetic (no filter, join, hash or aggregate lives here) — SURVEY.md §8(d) "Generator (subsystem 1)".
// The tables it produces stand in for the dbgen-generated TPC-H-like tables the paper measures on
// (PAPER.md:45, :59); only their shapes (row counts, key fan-out 1..7, day ranges, cents-scaled prices) are taken
// from BASELINE.json. Every value is a pure function of (seed, stream, index), so the bytes do not depend on the
// thread count used to fill a column.
//
// Build: g++ -O2 -shared -fPIC -pthread gqgen.cpp -o libgqgen.so   (no CUDA, no oracle, no library headers)
#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <thread>
#include <vector>

namespace {

typedef unsigned __int128 u128;

// SplitMix64 output function (public domain, Steele/Lea/Flood) on a counter. stream separates columns.
inline uint64_t mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}
inline uint64_t rnd(uint64_t seed, uint64_t stream, uint64_t i) {
  uint64_t s = mix64(seed + 0x632BE59BD9B4E019ULL * (stream + 1));
  return mix64(s + (i + 1) * 0x9E3779B97F4A7C15ULL);
}
// uniform integer in [0, span) by multiply-high (span >= 1)
inline uint64_t below(uint64_t r, uint64_t span) { return (uint64_t)(((u128)r * (u128)span) >> 64); }

template <class F>
void parallel_for(int64_t n, int nthreads, F f) {
  if (nthreads <= 1 || n < (1 << 16)) { f(0, n); return; }
  std::vector<std::thread> th;
  int64_t chunk = (n + nthreads - 1) / nthreads;
  for (int t = 0; t < nthreads; ++t) {
    int64_t a = t * chunk, b = std::min<int64_t>(n, a + chunk);
    if (a >= b) break;
    th.emplace_back([=] { f(a, b); });
  }
  for (auto& x : th) x.join();
}

template <class T>
void fill_uniform(uint64_t seed, uint64_t stream, int64_t lo, int64_t hi, int64_t n, T* out, int nthreads) {
  const uint64_t span = (uint64_t)(hi - lo) + 1;
  parallel_for(n, nthreads, [=](int64_t a, int64_t b) {
    for (int64_t i = a; i < b; ++i) out[i] = (T)(lo + (int64_t)below(rnd(seed, stream, (uint64_t)i), span));
  });
}

}  // namespace

extern "C" {

int gqgen_hw_threads() { unsigned n = std::thread::hardware_concurrency(); return n ? (int)n : 1; }

// i.i.d. uniform integers in the closed range [lo, hi]; value i depends only on (seed, stream, i).
void gqgen_uniform_i64(uint64_t seed, uint64_t stream, int64_t lo, int64_t hi, int64_t n, int64_t* out, int nthreads) {
  fill_uniform<int64_t>(seed, stream, lo, hi, n, out, nthreads);
}
void gqgen_uniform_i32(uint64_t seed, uint64_t stream, int64_t lo, int64_t hi, int64_t n, int32_t* out, int nthreads) {
  fill_uniform<int32_t>(seed, stream, lo, hi, n, out, nthreads);
}
void gqgen_uniform_i8(uint64_t seed, uint64_t stream, int64_t lo, int64_t hi, int64_t n, int8_t* out, int nthreads) {
  fill_uniform<int8_t>(seed, stream, lo, hi, n, out, nthreads);
}

// Fisher–Yates shuffle of an int64 array in place with the stream's RNG (sequential by definition).
void gqgen_shuffle_i64(uint64_t seed, uint64_t stream, int64_t n, int64_t* a) {
  for (int64_t i = n - 1; i >= 1; --i) {
    int64_t j = (int64_t)below(rnd(seed, stream, (uint64_t)i), (uint64_t)i + 1);
    int64_t t = a[i]; a[i] = a[j]; a[j] = t;
  }
}

// out = Fisher–Yates permutation of 1..n (unique keys of dim / cust / orders tables).
void gqgen_permutation_i64(uint64_t seed, uint64_t stream, int64_t n, int64_t* out) {
  for (int64_t i = 0; i < n; ++i) out[i] = i + 1;
  gqgen_shuffle_i64(seed, stream, n, out);
}

// out[i] = domain[uniform index]  (e.g. orders.custkey uniform over cust keys, i.i.d.)
void gqgen_pick_i64(uint64_t seed, uint64_t stream, const int64_t* domain, int64_t ndomain, int64_t n, int64_t* out,
                    int nthreads) {
  parallel_for(n, nthreads, [=](int64_t a, int64_t b) {
    for (int64_t i = a; i < b; ++i) out[i] = domain[below(rnd(seed, stream, (uint64_t)i), (uint64_t)ndomain)];
  });
}

// Foreign-key column with bounded fan-out: dim position k gets c_k in {1..7} fact rows, counts
// adjusted cyclically so that sum c_k == nfact exactly; emitted in dim order, then (unless clustered) Fisher–Yates
// shuffled. Requires ndim <= nfact <= 7*ndim. Returns 0 on success, -1 if that does not hold.
int gqgen_fanout_fk(uint64_t seed, uint64_t stream_counts, uint64_t stream_shuffle, const int64_t* dimkeys,
                    int64_t ndim, int64_t nfact, int clustered, int64_t* out) {
  if (ndim <= 0 || nfact < ndim || nfact > 7 * ndim) return -1;
  std::vector<uint8_t> c((size_t)ndim);
  int64_t total = 0;
  for (int64_t k = 0; k < ndim; ++k) {
    c[(size_t)k] = (uint8_t)(1 + below(rnd(seed, stream_counts, (uint64_t)k), 7));
    total += c[(size_t)k];
  }
  int64_t d = nfact - total;
  for (int64_t k = 0; d != 0; k = (k + 1 == ndim ? 0 : k + 1)) {
    if (d > 0 && c[(size_t)k] < 7) { ++c[(size_t)k]; --d; }
    else if (d < 0 && c[(size_t)k] > 1) { --c[(size_t)k]; ++d; }
  }
  int64_t w = 0;
  for (int64_t k = 0; k < ndim; ++k)
    for (int r = 0; r < c[(size_t)k]; ++r) out[w++] = dimkeys[k];
  if (!clustered) gqgen_shuffle_i64(seed, stream_shuffle, nfact, out);
  return 0;
}

// Zipf(s = 1) keys over N distinct values: P(rank r) = (1/r)/H_N; rank by inverse CDF on
// u = (rnd >> 11) * 2^-53 with a binary64 CDF accumulated sequentially r = 1..N (cdf[N] forced to 1.0);
// key = 1 + ((rank-1) * 2654435761 mod N). A guide table only narrows the search range; it returns the same rank
// as a plain binary search.
void gqgen_zipf_keys(uint64_t seed, uint64_t stream, int64_t N, int64_t n, int64_t* out, int nthreads) {
  std::vector<double> cdf((size_t)N + 1);
  double h = 0.0;
  for (int64_t r = 1; r <= N; ++r) h += 1.0 / (double)r;
  double acc = 0.0;
  cdf[0] = 0.0;
  for (int64_t r = 1; r <= N; ++r) { acc += 1.0 / (double)r; cdf[(size_t)r] = acc / h; }
  cdf[(size_t)N] = 1.0;
  // guide[g] = smallest r with cdf[r] > g / G  (search for u in [g/G, (g+1)/G) starts there)
  const int64_t G = 1 << 20;
  std::vector<int64_t> guide((size_t)G + 1);
  {
    int64_t r = 1;
    for (int64_t g = 0; g <= G; ++g) {
      double edge = (double)g / (double)G;
      while (r < N && !(cdf[(size_t)r] > edge)) ++r;
      guide[(size_t)g] = r;
    }
  }
  const double* cd = cdf.data();
  const int64_t* gd = guide.data();
  parallel_for(n, nthreads, [=](int64_t a, int64_t b) {
    for (int64_t i = a; i < b; ++i) {
      double u = (double)(rnd(seed, stream, (uint64_t)i) >> 11) * (1.0 / 9007199254740992.0);
      int64_t g = (int64_t)(u * (double)G);
      int64_t lo = gd[g], hi = gd[g + 1];  // answer in [lo, hi]
      while (lo < hi) {
        int64_t mid = lo + (hi - lo) / 2;
        if (cd[mid] > u) hi = mid; else lo = mid + 1;
      }
      out[i] = 1 + (int64_t)((((uint64_t)(lo - 1)) * 2654435761ULL) % (uint64_t)N);
    }
  });
}

// Column checksum used to freeze the generator (tests/golden): wrapping u64 sum, xor, min, max of the values
// sign-extended to int64. elem_bytes in {1,4,8}.
void gqgen_checksum(const void* data, int elem_bytes, int64_t n, uint64_t* out4) {
  uint64_t s = 0, x = 0; int64_t mn = INT64_MAX, mx = INT64_MIN;
  for (int64_t i = 0; i < n; ++i) {
    int64_t v = elem_bytes == 1 ? (int64_t)((const int8_t*)data)[i]
              : elem_bytes == 4 ? (int64_t)((const int32_t*)data)[i] : ((const int64_t*)data)[i];
    s += (uint64_t)v; x ^= (uint64_t)v; mn = std::min(mn, v); mx = std::max(mx, v);
  }
  out4[0] = s; out4[1] = x; out4[2] = (uint64_t)mn; out4[3] = (uint64_t)mx;
}

}  // extern "C"
