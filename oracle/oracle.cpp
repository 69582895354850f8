// oracle.cpp — plain, slow, single-threaded CPU oracle.  TEST INFRASTRUCTURE ONLY (see oracle.h).
//
// Every function is the textbook definition of the operator the paper names, written out row by row
// (SURVEY.md §8(c) definitions 1-8; PAPER.md:112-116 operators, :92 inner join, :59 no nulls, :154 aggregation):
//   1 Filter    pass(r) = AND_i pred_i(r), values sign-extended to int64 (S21)
//   2 Project   postfix program in uint64 wrapping arithmetic (S6), shadowed in __int128 to flag overflow
//   3 Join      multiset { (p,b) : pass(p) and pass(b) and p.fk == b.key } (S2-S4); brute-force double loop beside it
//   4 Chain     definition 3 applied step by step; each match appends the build side's payload columns
//   5 Group by  map from key tuple to SUM (wrapping) / COUNT / MIN / MAX in int64 (S19); output sorted by key tuple
//   6 Global    zero key columns => exactly one group, present even with zero surviving rows: (SUM 0, COUNT 0) (S9)
//   8 Top-k     order (aggregate descending, key tuple ascending) (S11), first min(k, ngroups)
// Build: g++ -O2 -std=c++17 -shared -fPIC oracle.cpp -o liboracle.so   (no CUDA, no product headers)
// Pins (tests/test_oracle_*.py): hand-computed worked examples T1-T5 (tests/golden/), brute-force nested-loop join,
// invariants I1-I7, closed-form pass fractions, pandas/numpy group-by and merge as an independent third opinion.
#include "oracle.h"

#include <algorithm>
#include <array>
#include <cstdint>
#include <map>
#include <unordered_map>
#include <vector>

typedef __int128 i128;

struct ocl_result {
  std::vector<std::vector<int64_t>> cols;
  int64_t nrows = 0;
  int64_t input_rows = 0;
  int32_t overflow = 0;
};

namespace {

int64_t cell(const ocl_column& c, int64_t r) {
  switch (c.dtype) {
    case OCL_I8: return (int64_t)((const int8_t*)c.data)[r];
    case OCL_I32: return (int64_t)((const int32_t*)c.data)[r];
    default: return ((const int64_t*)c.data)[r];
  }
}

bool pred_ok(const ocl_pred& p, int64_t x) {
  switch (p.op) {
    case OCL_LT: return x < p.lo;
    case OCL_LE: return x <= p.lo;
    case OCL_GT: return x > p.lo;
    case OCL_GE: return x >= p.lo;
    case OCL_EQ: return x == p.lo;
    case OCL_NE: return x != p.lo;
    case OCL_RANGE_CO: return p.lo <= x && x < p.hi;
    case OCL_RANGE_CC: return p.lo <= x && x <= p.hi;
  }
  return false;
}

bool in_i64(i128 v) { return v >= (i128)INT64_MIN && v <= (i128)INT64_MAX; }

// A "row" is the vector of its column values: the table's own columns followed by appended payload columns.
typedef std::vector<int64_t> Row;

Row base_row(const ocl_table& t, int64_t r) {
  Row v((size_t)t.ncols);
  for (int c = 0; c < t.ncols; ++c) v[(size_t)c] = cell(t.cols[c], r);
  return v;
}

bool row_passes(const Row& row, const ocl_pred* preds, int npred) {
  for (int i = 0; i < npred; ++i)
    if (!pred_ok(preds[i], row[(size_t)preds[i].col])) return false;
  return true;
}

// Postfix evaluation: wrapping uint64 value + exact shadow (shadow saturates the flag, not the value).
int64_t eval_expr(const ocl_expr& e, const Row& row, int32_t* overflow, bool* ok) {
  std::vector<uint64_t> st;
  std::vector<i128> sh;
  for (int i = 0; i < e.ntoks; ++i) {
    const ocl_tok& t = e.toks[i];
    if (t.op == OCL_X_COL) {
      if (t.arg < 0 || (size_t)t.arg >= row.size()) { *ok = false; return 0; }
      st.push_back((uint64_t)row[(size_t)t.arg]); sh.push_back((i128)row[(size_t)t.arg]);
    } else if (t.op == OCL_X_CONST) {
      st.push_back((uint64_t)t.arg); sh.push_back((i128)t.arg);
    } else {
      if (st.size() < 2) { *ok = false; return 0; }
      uint64_t b = st.back(); st.pop_back(); uint64_t a = st.back(); st.pop_back();
      i128 sb = sh.back(); sh.pop_back(); i128 sa = sh.back(); sh.pop_back();
      uint64_t r; i128 s;
      if (t.op == OCL_X_ADD) { r = a + b; s = sa + sb; }
      else if (t.op == OCL_X_SUB) { r = a - b; s = sa - sb; }
      else if (t.op == OCL_X_MUL) { r = a * b; s = sa * sb; }
      else { *ok = false; return 0; }
      if (!in_i64(s)) { *overflow = 1; s = (i128)(int64_t)r; }  // keep shadow bounded; flag is sticky
      st.push_back(r); sh.push_back(s);
    }
  }
  if (st.size() != 1) { *ok = false; return 0; }
  return (int64_t)st[0];
}

// A built relation: key -> payload tuples of every surviving build row (multimap: duplicates kept, S3).
struct Relation {
  std::unordered_multimap<int64_t, std::vector<int64_t>> map;
  int npayload = 0;
};

// Inner-join expansion (definitions 3 and 4): all rows obtained from `row` by matching probe steps s..n-1 in order.
void expand(const Row& row, const ocl_probe* probes, int nprobes, int s, const std::vector<Relation>& rels,
            std::vector<Row>* out) {
  if (s == nprobes) { out->push_back(row); return; }
  const Relation& rel = rels[(size_t)probes[s].build];
  auto range = rel.map.equal_range(row[(size_t)probes[s].key_col]);
  for (auto it = range.first; it != range.second; ++it) {
    Row ext = row;
    ext.insert(ext.end(), it->second.begin(), it->second.end());
    expand(ext, probes, nprobes, s + 1, rels, out);
  }
}

bool probes_valid(const ocl_probe* probes, int nprobes, int ncols, int nearlier, const std::vector<Relation>& rels) {
  int width = ncols;
  for (int s = 0; s < nprobes; ++s) {
    if (probes[s].build < 0 || probes[s].build >= nearlier) return false;
    if (probes[s].key_col < 0 || probes[s].key_col >= width) return false;
    width += rels[(size_t)probes[s].build].npayload;
  }
  return true;
}

struct Acc { int64_t v[8]; i128 exact[8]; };  // exact[] = running SUM without wrap (overflow flag only)

}  // namespace

extern "C" {

ocl_result* ocl_run_query(const ocl_query* q) {
  if (!q || q->nkeys < 0 || q->nkeys > 2 || q->naggs < 0 || q->naggs > 8) return nullptr;
  ocl_result* res = new ocl_result();
  std::vector<Relation> rels;
  // ---- build relations in order (HashBuild consumes its whole input before any probe) ----
  for (int b = 0; b < q->nbuilds; ++b) {
    const ocl_build& bd = q->builds[b];
    if (!probes_valid(bd.probes, bd.nprobes, bd.in.ncols, b, rels)) { delete res; return nullptr; }
    Relation rel; rel.npayload = bd.npayload;
    for (int64_t r = 0; r < bd.in.nrows; ++r) {
      Row row = base_row(bd.in, r);
      for (int i = 0; i < bd.npred; ++i)
        if (bd.preds[i].col < 0 || bd.preds[i].col >= bd.in.ncols) { delete res; return nullptr; }
      if (!row_passes(row, bd.preds, bd.npred)) continue;
      std::vector<Row> joined;
      expand(row, bd.probes, bd.nprobes, 0, rels, &joined);
      for (const Row& j : joined) {
        if (bd.key_col < 0 || (size_t)bd.key_col >= j.size()) { delete res; return nullptr; }
        std::vector<int64_t> pay;
        for (int p = 0; p < bd.npayload; ++p) {
          if (bd.payload_cols[p] < 0 || (size_t)bd.payload_cols[p] >= j.size()) { delete res; return nullptr; }
          pay.push_back(j[(size_t)bd.payload_cols[p]]);
        }
        rel.map.emplace(j[(size_t)bd.key_col], pay);
      }
    }
    rels.push_back(std::move(rel));
  }
  // ---- scan the fact side: filter -> probes -> project -> group ----
  if (!probes_valid(q->probes, q->nprobes, q->in.ncols, q->nbuilds, rels)) { delete res; return nullptr; }
  typedef std::array<int64_t, 2> Key;
  std::map<Key, Acc> groups;
  auto fresh = [&]() {
    Acc a;
    for (int i = 0; i < 8; ++i) { a.v[i] = 0; a.exact[i] = 0; }
    for (int i = 0; i < q->naggs; ++i)
      a.v[i] = q->aggs[i].op == OCL_MIN ? INT64_MAX : q->aggs[i].op == OCL_MAX ? INT64_MIN : 0;
    return a;
  };
  if (q->nkeys == 0) groups[Key{0, 0}] = fresh();  // definition 6
  for (int i = 0; i < q->npred; ++i)
    if (q->preds[i].col < 0 || q->preds[i].col >= q->in.ncols) { delete res; return nullptr; }
  for (int64_t r = 0; r < q->in.nrows; ++r) {
    Row row = base_row(q->in, r);
    if (!row_passes(row, q->preds, q->npred)) continue;
    std::vector<Row> joined;
    expand(row, q->probes, q->nprobes, 0, rels, &joined);
    for (const Row& j : joined) {
      ++res->input_rows;
      std::vector<int64_t> ev((size_t)q->nexpr);
      bool ok = true;
      for (int e = 0; e < q->nexpr; ++e) ev[(size_t)e] = eval_expr(q->exprs[e], j, &res->overflow, &ok);
      if (!ok) { delete res; return nullptr; }
      Key k{0, 0};
      for (int c = 0; c < q->nkeys; ++c) {
        if (q->key_cols[c] < 0 || (size_t)q->key_cols[c] >= j.size()) { delete res; return nullptr; }
        k[(size_t)c] = j[(size_t)q->key_cols[c]];
      }
      auto it = groups.find(k);
      if (it == groups.end()) it = groups.emplace(k, fresh()).first;
      Acc& a = it->second;
      for (int i = 0; i < q->naggs; ++i) {
        const ocl_agg& g = q->aggs[i];
        if (g.op == OCL_COUNT_STAR) { a.v[i] += 1; continue; }
        if (g.expr < 0 || g.expr >= q->nexpr) { delete res; return nullptr; }
        int64_t x = ev[(size_t)g.expr];
        if (g.op == OCL_SUM) {
          a.v[i] = (int64_t)((uint64_t)a.v[i] + (uint64_t)x);
          a.exact[i] += (i128)x;
          if (!in_i64(a.exact[i])) { res->overflow = 1; a.exact[i] = (i128)a.v[i]; }
        } else if (g.op == OCL_MIN) a.v[i] = std::min(a.v[i], x);
        else if (g.op == OCL_MAX) a.v[i] = std::max(a.v[i], x);
        else { delete res; return nullptr; }
      }
    }
  }
  // ---- emit: key tuple ascending (std::map order), or top-k by (aggregate desc, key asc) ----
  std::vector<std::pair<Key, Acc>> rows(groups.begin(), groups.end());
  if (q->topk > 0) {
    if (q->topk_agg < 0 || q->topk_agg >= q->naggs) { delete res; return nullptr; }
    const int ta = q->topk_agg;
    std::stable_sort(rows.begin(), rows.end(), [ta](const std::pair<Key, Acc>& x, const std::pair<Key, Acc>& y) {
      if (x.second.v[ta] != y.second.v[ta]) return x.second.v[ta] > y.second.v[ta];
      return x.first < y.first;
    });
    if ((int64_t)rows.size() > q->topk) rows.resize((size_t)q->topk);
  }
  res->nrows = (int64_t)rows.size();
  res->cols.assign((size_t)(q->nkeys + q->naggs), std::vector<int64_t>((size_t)res->nrows));
  for (int64_t g = 0; g < res->nrows; ++g) {
    for (int c = 0; c < q->nkeys; ++c) res->cols[(size_t)c][(size_t)g] = rows[(size_t)g].first[(size_t)c];
    for (int i = 0; i < q->naggs; ++i) res->cols[(size_t)(q->nkeys + i)][(size_t)g] = rows[(size_t)g].second.v[i];
  }
  return res;
}

ocl_result* ocl_filter_project(const ocl_table* in, const ocl_pred* preds, int32_t npred, const ocl_expr* exprs,
                               int32_t nexpr) {
  ocl_result* res = new ocl_result();
  res->cols.assign((size_t)nexpr, std::vector<int64_t>());
  for (int i = 0; i < npred; ++i)
    if (preds[i].col < 0 || preds[i].col >= in->ncols) { delete res; return nullptr; }
  for (int64_t r = 0; r < in->nrows; ++r) {
    Row row = base_row(*in, r);
    if (!row_passes(row, preds, npred)) continue;
    bool ok = true;
    for (int e = 0; e < nexpr; ++e) res->cols[(size_t)e].push_back(eval_expr(exprs[e], row, &res->overflow, &ok));
    if (!ok) { delete res; return nullptr; }
    ++res->nrows;
  }
  res->input_rows = res->nrows;
  return res;
}

static ocl_result* pairs_result(std::vector<std::pair<int64_t, int64_t>>& pairs) {
  std::sort(pairs.begin(), pairs.end());
  ocl_result* res = new ocl_result();
  res->nrows = res->input_rows = (int64_t)pairs.size();
  res->cols.assign(2, std::vector<int64_t>(pairs.size()));
  for (size_t i = 0; i < pairs.size(); ++i) { res->cols[0][i] = pairs[i].first; res->cols[1][i] = pairs[i].second; }
  return res;
}

ocl_result* ocl_join_pairs(const ocl_table* build, const ocl_pred* bpreds, int32_t nbpred, int32_t bkey,
                           const ocl_table* probe, const ocl_pred* ppreds, int32_t nppred, int32_t pkey) {
  std::unordered_multimap<int64_t, int64_t> m;
  for (int64_t b = 0; b < build->nrows; ++b) {
    Row row = base_row(*build, b);
    if (row_passes(row, bpreds, nbpred)) m.emplace(row[(size_t)bkey], b);
  }
  std::vector<std::pair<int64_t, int64_t>> pairs;
  for (int64_t p = 0; p < probe->nrows; ++p) {
    Row row = base_row(*probe, p);
    if (!row_passes(row, ppreds, nppred)) continue;
    auto range = m.equal_range(row[(size_t)pkey]);
    for (auto it = range.first; it != range.second; ++it) pairs.emplace_back(p, it->second);
  }
  return pairs_result(pairs);
}

ocl_result* ocl_join_pairs_bruteforce(const ocl_table* build, const ocl_pred* bpreds, int32_t nbpred, int32_t bkey,
                                      const ocl_table* probe, const ocl_pred* ppreds, int32_t nppred, int32_t pkey) {
  std::vector<std::pair<int64_t, int64_t>> pairs;
  for (int64_t p = 0; p < probe->nrows; ++p) {
    Row pr = base_row(*probe, p);
    if (!row_passes(pr, ppreds, nppred)) continue;
    for (int64_t b = 0; b < build->nrows; ++b) {
      Row br = base_row(*build, b);
      if (!row_passes(br, bpreds, nbpred)) continue;
      if (pr[(size_t)pkey] == br[(size_t)bkey]) pairs.emplace_back(p, b);
    }
  }
  return pairs_result(pairs);
}

ocl_result* ocl_order_by(const ocl_table* in, const ocl_sort_key* keys, int32_t nkeys, int64_t limit) {
  if (!in || nkeys < 0 || (nkeys > 0 && !keys)) return nullptr;
  for (int32_t k = 0; k < nkeys; ++k) if (keys[k].col < 0 || keys[k].col >= in->ncols) return nullptr;
  std::vector<int64_t> order((size_t)in->nrows);
  for (int64_t r = 0; r < in->nrows; ++r) order[(size_t)r] = r;
  std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) {
    for (int32_t k = 0; k < nkeys; ++k) {
      const int64_t x = cell(in->cols[keys[k].col], a), y = cell(in->cols[keys[k].col], b);
      if (x != y) return keys[k].descending ? x > y : x < y;
    }
    return false;                                          // equal key tuples: stable_sort keeps input order
  });
  const int64_t n = (limit <= 0 || limit > in->nrows) ? in->nrows : limit;
  ocl_result* res = new ocl_result();
  res->nrows = n;
  res->input_rows = in->nrows;
  res->cols.assign((size_t)in->ncols + 1, std::vector<int64_t>((size_t)n));
  for (int64_t i = 0; i < n; ++i) {
    res->cols[0][(size_t)i] = order[(size_t)i];
    for (int32_t c = 0; c < in->ncols; ++c) res->cols[(size_t)c + 1][(size_t)i] = cell(in->cols[c], order[(size_t)i]);
  }
  return res;
}

// Hash partitioning (PAPER.md:160, :174 CudfPartitionedOutput; DESIGN reading R-HP): the definition
// written out. destination(row) follows include/gq.h: h := 0x9E3779B97F4A7C15; for every key column, in order,
// h := fmix64(h XOR value) with the 64-bit finaliser of MurmurHash3 (x ^= x >> 33; x *= 0xff51afd7ed558ccd; x ^= x >> 33;
// x *= 0xc4ceb9fe1a85ec53; x ^= x >> 33); destination = floor((h div 2^32) * nparts / 2^32). Rows are emitted destination
// by destination, input order inside one destination.
ocl_result* ocl_hash_partition(const ocl_table* in, const int32_t* key_cols, int32_t nkeys, int32_t nparts) {
  if (!in || nkeys < 1 || !key_cols || nparts < 1) return nullptr;
  for (int32_t k = 0; k < nkeys; ++k) if (key_cols[k] < 0 || key_cols[k] >= in->ncols) return nullptr;
  std::vector<int64_t> dest((size_t)in->nrows);
  for (int64_t r = 0; r < in->nrows; ++r) {
    uint64_t h = 0x9E3779B97F4A7C15ULL;
    for (int32_t k = 0; k < nkeys; ++k) {
      uint64_t x = h ^ (uint64_t)cell(in->cols[key_cols[k]], r);
      x ^= x >> 33;
      x *= 0xff51afd7ed558ccdULL;
      x ^= x >> 33;
      x *= 0xc4ceb9fe1a85ec53ULL;
      x ^= x >> 33;
      h = x;
    }
    dest[(size_t)r] = (int64_t)(((h >> 32) * (uint64_t)nparts) >> 32);
  }
  ocl_result* res = new ocl_result();
  res->nrows = in->nrows;
  res->input_rows = in->nrows;
  res->cols.assign((size_t)in->ncols + 2, std::vector<int64_t>());
  for (int64_t d = 0; d < nparts; ++d)
    for (int64_t r = 0; r < in->nrows; ++r)
      if (dest[(size_t)r] == d) {
        res->cols[0].push_back(d);
        res->cols[1].push_back(r);
        for (int32_t c = 0; c < in->ncols; ++c) res->cols[(size_t)c + 2].push_back(cell(in->cols[c], r));
      }
  return res;
}

int64_t ocl_result_nrows(const ocl_result* r) { return r->nrows; }
int32_t ocl_result_ncols(const ocl_result* r) { return (int32_t)r->cols.size(); }
const int64_t* ocl_result_col(const ocl_result* r, int32_t c) { return r->cols[(size_t)c].data(); }
int64_t ocl_result_input_rows(const ocl_result* r) { return r->input_rows; }
int32_t ocl_result_overflow(const ocl_result* r) { return r->overflow; }
double ocl_avg(int64_t sum, int64_t count) { return (double)sum / (double)count; }
void ocl_result_free(ocl_result* r) { delete r; }

}  // extern "C"
