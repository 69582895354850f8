// gq_codegen.cpp — plan-time translation of one scan shape into a fused CUDA kernel source.
//
// This is the "expression compilation at plan creation time" of PAPER.md:124/:152 (TypedExpr -> fused AST), done
// B200-first: the whole FilterProject -> HashProbe* -> consumer chain of a plan becomes ONE kernel. The generator
// emits a prelude of #defines plus two straight-line row functions (gq_pass, gq_body) and splices them between the
// two halves of the hand-written skeleton (gq_skeleton.cuh / gq_skeleton_kernel.cuh). Predicate bounds and literals
// stay runtime parameters (GqParams::k), so a kernel is specialised by plan SHAPE, not by constants.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <map>
#include <sstream>

#include "gq_internal.h"

extern const char gq_skeleton_a[];
extern const char gq_skeleton_b[];
extern const char gq_skeleton_psa[];

int gq_dtype_bytes(gq_dtype t) { return t == GQ_I8 ? 1 : t == GQ_I32 ? 4 : t == GQ_I64 ? 8 : 0; }
static const char* ctype(gq_dtype t) { return t == GQ_I8 ? "signed char" : t == GQ_I32 ? "int" : "long long"; }

static uint64_t fnv1a(const std::string& s) {
  uint64_t h = 1469598103934665603ULL;
  for (unsigned char c : s) { h ^= c; h *= 1099511628211ULL; }
  return h;
}

namespace {
struct Gen {
  const GqScanSpec& sp;
  std::string* msg;
  int ncols_in;
  std::vector<int> compact;           // input column -> kernel column (or -1)
  std::vector<int> cols;              // kernel column -> input column
  std::vector<long long> consts;
  std::vector<int> vcol_probe, vcol_pay;  // virtual column -> (probe step, payload index)
  std::string sfx;                        // "" (one row at a time) or "[j]" (linear mode: GQ_R rows in register arrays)
  bool linear = false;

  Gen(const GqScanSpec& s, std::string* m) : sp(s), msg(m), ncols_in((int)s.in_dtype.size()) {
    compact.assign((size_t)ncols_in, -1);
    for (size_t s2 = 0; s2 < sp.probes.size(); ++s2)
      for (int p = 0; p < sp.probes[s2].npayload; ++p) { vcol_probe.push_back((int)s2); vcol_pay.push_back(p); }
  }
  bool fail(const std::string& m) { if (msg) *msg = m; return false; }
  int row_width() const { return ncols_in + (int)vcol_probe.size(); }
  // number of row columns visible BEFORE probe step s
  int width_before_probe(int s) const {
    int w = ncols_in;
    for (int i = 0; i < s; ++i) w += sp.probes[(size_t)i].npayload;
    return w;
  }
  bool use_col(int c) {                                   // register an input column as referenced
    if (c < 0 || c >= row_width()) return fail("column index out of range");
    if (c >= ncols_in) return true;
    if (compact[(size_t)c] < 0) {
      if ((int)cols.size() >= GQ_MAXCOL) return fail("too many referenced input columns");
      compact[(size_t)c] = (int)cols.size();
      cols.push_back(c);
    }
    return true;
  }
  std::string val(int c) const {                          // name of the row value of column c
    char b[32];
    if (c < ncols_in) snprintf(b, sizeof b, "v%d", c);
    else if (linear) {   // payload word of probe step s: py<s>[j][p]
      snprintf(b, sizeof b, "py%d[j][%d]", vcol_probe[(size_t)(c - ncols_in)], vcol_pay[(size_t)(c - ncols_in)]);
      return b;
    } else snprintf(b, sizeof b, "y%d_%d", vcol_probe[(size_t)(c - ncols_in)], vcol_pay[(size_t)(c - ncols_in)]);
    return std::string(b) + sfx;
  }
  std::string konst(long long v) {   // equal literals share one parameter slot, so common subexpressions stay common
    size_t i = 0;
    while (i < consts.size() && consts[i] != v) ++i;
    if (i == consts.size()) {
      if ((int)consts.size() >= GQ_MAXK) { fail("too many constants"); return "0"; }
      consts.push_back(v);
    }
    return "P.k[" + std::to_string(i) + "]";
  }
  std::string load(int c) const {                         // typed load of input column c for row slot j
    int kc = compact[(size_t)c];
    std::ostringstream o;
    o << (sfx.empty() ? "const i64 v" : "v") << c << sfx << " = src.template ld<" << ctype(sp.in_dtype[(size_t)c]) << ">(" << kc
      << ", GQ_COL_OFF(" << kc << "), j);";
    return o.str();
  }
  bool expr(const std::vector<gq_xtok>& toks, std::string* out) {
    std::vector<std::string> st;
    if (toks.empty() || (int)toks.size() > GQ_MAX_TOKS) return fail("expression length out of range");
    for (const gq_xtok& t : toks) {
      if (t.op == GQ_X_COL) {
        if (t.arg < 0 || t.arg >= row_width()) return fail("expression column out of range");
        st.push_back(val((int)t.arg));
      } else if (t.op == GQ_X_CONST) st.push_back(konst(t.arg));
      else if (t.op == GQ_X_ADD || t.op == GQ_X_SUB || t.op == GQ_X_MUL) {
        if (st.size() < 2) return fail("malformed postfix expression");
        std::string b = st.back(); st.pop_back();
        std::string a = st.back(); st.pop_back();
        const char* f = t.op == GQ_X_ADD ? "gq_add" : t.op == GQ_X_SUB ? "gq_sub" : "gq_mul";
        st.push_back(std::string(f) + "(" + a + ", " + b + ")");
      } else return fail("unknown expression token");
    }
    if (st.size() != 1) return fail("malformed postfix expression");
    *out = st[0];
    return true;
  }
};
}  // namespace


// ---- filter condition of one predicate, shared by both modes ----
static bool pred_cond(Gen& g, const gq_pred& p, std::string* c) {
  const std::string v = g.val(p.col);
  const std::string klo = g.konst(p.lo);   // sequenced: lo before hi (operands of + are unsequenced)
  const std::string khi = (p.op == GQ_RANGE_CO || p.op == GQ_RANGE_CC) ? g.konst(p.hi) : std::string();
  switch (p.op) {
    case GQ_LT: *c = v + " < " + klo; break;
    case GQ_LE: *c = v + " <= " + klo; break;
    case GQ_GT: *c = v + " > " + klo; break;
    case GQ_GE: *c = v + " >= " + klo; break;
    case GQ_EQ: *c = v + " == " + klo; break;
    case GQ_NE: *c = v + " != " + klo; break;
    case GQ_RANGE_CO: *c = v + " >= " + klo + " && " + v + " < " + khi; break;
    case GQ_RANGE_CC: *c = v + " >= " + klo + " && " + v + " <= " + khi; break;
    default: return g.fail("unknown comparison");
  }
  return true;
}

// ---- key expression shared by both modes: one hashed 64-bit word (+ optional dependent column) ----
static gq_status key_exprs(Gen& g, const GqScanSpec& sp, std::string* keyx, std::string* depx, std::string* msg) {
  const int nk = (int)sp.key_cols.size();
  if (nk < 1 || nk > GQ_MAX_KEYS || sp.ndep < 0 || sp.ndep >= nk) { if (msg) *msg = "bad key columns"; return GQ_ERR_INVALID_ARG; }
  if (nk - sp.ndep == 1) *keyx = g.val(sp.key_cols[0]);
  else {  // two hashed keys packed into one 64-bit word: key0 in the low bits
    auto dt = [&](int c) { return c < g.ncols_in ? sp.in_dtype[(size_t)c]
                                                  : sp.probes[(size_t)g.vcol_probe[(size_t)(c - g.ncols_in)]].pay_dtype[g.vcol_pay[(size_t)(c - g.ncols_in)]]; };
    int b0 = 8 * gq_dtype_bytes(dt(sp.key_cols[0])), b1 = 8 * gq_dtype_bytes(dt(sp.key_cols[1]));
    if (b0 + b1 > 64) { if (msg) *msg = "packed key wider than 64 bits: declare a dependent key (ndependent)"; return GQ_ERR_UNSUPPORTED; }
    char buf[256];
    snprintf(buf, sizeof buf, "(i64)((((u64)%s) & 0x%llxULL) | ((((u64)%s) & 0x%llxULL) << %d))", g.val(sp.key_cols[0]).c_str(),
             (unsigned long long)((b0 == 64) ? ~0ULL : ((1ULL << b0) - 1)), g.val(sp.key_cols[1]).c_str(),
             (unsigned long long)((1ULL << b1) - 1), b0);
    *keyx = buf;
  }
  if (sp.ndep == 1) *depx = g.val(sp.key_cols[(size_t)nk - 1]);
  return GQ_OK;
}

// ---- linear mode: gq_tile processes the GQ_R rows of a thread step by step. Every hash-table step hands all GQ_R
// rows to one skeleton helper (gq_probe_rows / gq_upsert_rows / gq_insert_rows) that keeps their slot accesses in
// flight together and resolves them in rounds.
static gq_status emit_linear(Gen& g, const GqScanSpec& sp, std::ostringstream& o, std::string* msg) {
  g.sfx = "[j]";
  g.linear = true;
  const int nprobe = (int)sp.probes.size();
  const int nagg = (int)sp.aggs.size();
  const char* LOOP = "#pragma unroll\n  for (int j = 0; j < GQ_R; ++j) ";
  // Dense form (low-cardinality consumer): in a full tile every load, expression and cell update is unconditional and
  // a filtered-out row contributes the aggregate's identity to group 0 — straight-line code, so the compiler can
  // interleave the GQ_R rows of a thread. The other consumers skip the work of filtered-out rows.
  const bool dense = sp.consumer == GQ_C_LOWCARD;
  const char* GUARD = dense ? "if (FULL || live[j]) " : "if (live[j]) ";
  o << "template <class Src, bool FULL> __device__ __forceinline__ void gq_tile(const GqParams& P, const Src& src, GqCtx& cx, int nvalid) {\n";
  o << "  bool live[GQ_R];\n";
  for (int c : g.cols) o << "  i64 v" << c << "[GQ_R]" << (dense ? " = {}" : "") << ";\n";
  // ---- filter: all rows first, so the shared-memory loads of the GQ_R rows overlap ----
  o << "  " << LOOP << "{\n    live[j] = FULL || j < nvalid;\n";
  std::vector<bool> loaded(g.compact.size(), false);
  for (const gq_pred& p : sp.preds) {
    if (dense) {
      if (!loaded[(size_t)p.col]) { o << "    " << GUARD << "{ " << g.load(p.col) << " }\n"; loaded[(size_t)p.col] = true; }
      o << "    { ";
    } else {
      o << "    if (live[j]) { ";
      if (!loaded[(size_t)p.col]) { o << g.load(p.col) << " "; loaded[(size_t)p.col] = true; }
    }
    std::string c;
    if (!pred_cond(g, p, &c)) return GQ_ERR_INVALID_ARG;
    o << "live[j] = " << (dense ? "live[j] && " : "") << "(" << c << "); }\n";
  }
  o << "  }\n";
  // ---- remaining input columns of surviving rows ----
  {
    bool any = false;
    for (int c : g.cols) any = any || !loaded[(size_t)c];
    if (any) {
      o << "  " << LOOP << GUARD << "{\n";
      for (int c : g.cols) if (!loaded[(size_t)c]) o << "    " << g.load(c) << "\n";
      o << "  }\n";
    }
  }
  // a row column as a whole GQ_R array (input columns are arrays already; payloads are copied out)
  int ntmp = 0;
  auto as_array = [&](int c) -> std::string {
    if (c < g.ncols_in) return "v" + std::to_string(c);
    const std::string nm = "ka" + std::to_string(ntmp++);
    o << "  i64 " << nm << "[GQ_R];\n  " << LOOP << nm << "[j] = " << g.val(c) << ";\n";
    return nm;
  };
  // ---- projection, emitted after the probe steps ----
  bool projected = false;
  auto emit_projection = [&]() -> bool {
    projected = true;
    if (sp.exprs.empty()) return true;
    for (size_t e = 0; e < sp.exprs.size(); ++e) o << "  i64 e" << e << "[GQ_R];\n";
    o << "  " << LOOP << (dense ? "" : "if (live[j]) ") << "{\n";
    for (size_t e = 0; e < sp.exprs.size(); ++e) {
      std::string x;
      if (!g.expr(sp.exprs[e], &x)) return false;
      o << "    e" << e << "[j] = " << x << ";\n";
    }
    o << "  }\n";
    return true;
  };
  // ---- probe steps ----
  for (int s = 0; s < nprobe; ++s) {
    const GqProbeSpec& ps = sp.probes[(size_t)s];
    const std::string S = std::to_string(s);
    const std::string karr = as_array(ps.key_col);
    o << "  u64 pi" << S << "[GQ_R]; i64 py" << S << "[GQ_R][" << (ps.npayload > 0 ? ps.npayload : 1) << "];\n";
    if (ps.dense) o << "  gq_dense_probe_rows<" << ps.npayload << ">(P.probe[" << S << "], " << karr << ", live, pi" << S << ", py" << S << ");\n";
    else o << "  gq_probe_rows<" << ps.slot_words << ", " << ps.npayload << ">(P.probe[" << S << "], " << karr << ", live, pi" << S
      << ", py" << S << ");\n";
    o << "  (void)pi" << S << "; (void)py" << S << ";\n";
  }
  if (!projected && !emit_projection()) return GQ_ERR_INVALID_ARG;
  std::string keyx, depx;
  if (sp.consumer == GQ_C_LOWCARD || sp.consumer == GQ_C_HIGHCARD || sp.consumer == GQ_C_PARTITION || sp.consumer == GQ_C_SCATTER) {
    gq_status st = key_exprs(g, sp, &keyx, &depx, msg);
    if (st != GQ_OK) return st;
  }
  auto aggval = [&](const gq_agg& a) { return a.op == GQ_COUNT_STAR ? std::string("1") : "e" + std::to_string(a.expr) + "[j]"; };
  // hot keys of a skewed batch (DESIGN 5.4): rows whose key is in the batch's hot list are aggregated in CTA-shared
  // memory and leave the row set; the CTA flushes its partial groups once, at the end of the kernel
  auto emit_hot = [&]() {
    o << "#if GQ_HOT\n  if (cx.nhot > 0) {\n  int hpos[GQ_R];\n  " << LOOP << "hpos[j] = live[j] ? gq_hot_find(cx, tkey[j]) : -1;\n"
      << "  " << LOOP << "{\n      const int hp = hpos[j];\n      if (hp >= 0) {\n";
    for (int a = 0; a < nagg; ++a)
      o << "        const u64 hg" << a << " = gq_hot_issue(" << (int)sp.aggs[(size_t)a].op << ", cx, hp, " << a << ", " << aggval(sp.aggs[(size_t)a]) << ");\n";
    for (int a = 0; a < nagg; ++a)
      o << "        gq_hot_finish(" << (int)sp.aggs[(size_t)a].op << ", cx, hp, " << a << ", " << aggval(sp.aggs[(size_t)a]) << ", hg" << a << ");\n";
    o << "        cx.hot_touched[hp] = 1;\n        live[j] = false;\n      }\n    }\n  }\n#endif\n";
  };
  switch (sp.consumer) {
    case GQ_C_GLOBAL:
      o << "  " << LOOP << "if (live[j]) {\n";
      for (int a = 0; a < nagg; ++a)
        o << "    cx.acc[" << a << "] = gq_combine(" << (int)sp.aggs[(size_t)a].op << ", cx.acc[" << a << "], " << aggval(sp.aggs[(size_t)a]) << ");\n";
      o << "  }\n";
      break;
    case GQ_C_LOWCARD:
      // group id: one LDS on the fast path; first sights and collisions take the (rare, warp-converged) slow path
      o << "  int grp[GQ_R]; i64 lk[GQ_R]; bool need[GQ_R]; bool anyneed = false;\n";
      o << "  " << LOOP << "{\n    lk[j] = " << keyx << ";\n    const int g1 = gq_lc_find1(cx, lk[j]);\n"
        << "    grp[j] = live[j] ? g1 : 0;\n    need[j] = live[j] && g1 < 0;\n    anyneed = anyneed || need[j];\n  }\n";
      // (keys inserted while serving an earlier row are picked up by a second one-probe look before asking again)
      o << "  if (__any_sync(0xffffffffu, anyneed)) {\n  " << LOOP << "{\n"
        << "      if (need[j]) { const int g2 = gq_lc_find1(cx, lk[j]); if (g2 >= 0) { grp[j] = g2; need[j] = false; } }\n"
        << "      if (__any_sync(0xffffffffu, need[j])) grp[j] = gq_lc_slow(cx, lk[j], need[j], grp[j], P.err);\n    }\n  }\n";
      o << "  " << LOOP << "{\n";
      for (int a = 0; a < nagg; ++a) {
        const int op = (int)sp.aggs[(size_t)a].op;
        o << "    gq_lc_update(" << op << ", cx, grp[j], " << a << ", live[j] ? " << aggval(sp.aggs[(size_t)a]) << " : gq_identity(" << op << "));\n";
      }
      o << "  }\n";
      break;
    case GQ_C_PARTITION:
    case GQ_C_HIGHCARD: {
      o << "  i64 tkey[GQ_R];\n  " << LOOP << "tkey[j] = " << keyx << ";\n";
      emit_hot();
      if (sp.consumer == GQ_C_PARTITION) {
        // pass A of the radix-clustered aggregation: append (key, dependent key, aggregate inputs) to the record
        // buffer of the key's table partition; rows that do not fit (or carry the reserved key pattern) fall through
        // to the ordinary insert-or-update below, so any skew stays correct
        const int rw = sp.part_rw;
        o << "  u64 pidx[GQ_R], ppart[GQ_R];\n";
        o << "  " << LOOP << "{\n    pidx[j] = ~0ULL; ppart[j] = 0;\n    if (live[j] && (u64)tkey[j] != GQ_EMPTY) {\n"
          << "      ppart[j] = gq_slot0(P.target, tkey[j]) >> P.pshift;\n      pidx[j] = (u64)gq_part_reserve(P, cx.part_st, ppart[j]);\n    }\n  }\n";
        o << "  " << LOOP << "if (live[j] && pidx[j] != ~0ULL) {\n    u64* rec = P.part + (ppart[j] * (u64)P.pcap + pidx[j]) * " << rw << ";\n";
        std::vector<std::string> words;
        words.push_back("(u64)tkey[j]");
        if (sp.ndep == 1) words.push_back("(u64)" + depx);
        for (int e : sp.part_exprs) words.push_back("(u64)e" + std::to_string(e) + "[j]");
        while ((int)words.size() < rw) words.push_back("0ULL");
        for (int w = 0; w < rw; w += 4)
          o << "    gq_st256(rec + " << w << ", " << words[(size_t)w] << ", " << words[(size_t)w + 1] << ", " << words[(size_t)w + 2] << ", " << words[(size_t)w + 3] << ");\n";
        o << "    live[j] = false;\n  }\n";
      }
      o << "  u64* slot[GQ_R]; bool won[GQ_R];\n";
      o << "  gq_upsert_rows<" << sp.target_sw << ">(P.target, tkey, live, slot, won, P.err);\n";
      o << "  " << LOOP << "if (live[j] && slot[j]) {\n";
      if (sp.ndep == 1) o << "    gq_dep_store(slot[j] + 1, " << depx << ", won[j], P.err);\n";
      for (int a = 0; a < nagg; ++a)
        o << "    gq_red(" << (int)sp.aggs[(size_t)a].op << ", slot[j] + " << (1 + sp.ndep + a) << ", " << aggval(sp.aggs[(size_t)a]) << ");\n";
      o << "  }\n";
      break;
    }
    case GQ_C_SCATTER: {
      // pass A of the partitioned shared-memory aggregation: one record per surviving row, appended to a CTA-private
      // chunk of the partition the key hashes to (P.pshift = 64 - log2(partitions)); no table is touched here
      const int rw = sp.part_rw;
      o << "  i64 tkey[GQ_R];\n  " << LOOP << "tkey[j] = " << keyx << ";\n";
      emit_hot();
      o << "  u64 ridx[GQ_R]; u32 rpart[GQ_R], rtick[GQ_R]; bool ropen[GQ_R];\n";
      o << "  " << LOOP << "{\n    ridx[j] = ~0ULL; ropen[j] = false; rpart[j] = (u32)(gq_hash(tkey[j], 0) >> P.pshift);\n"
        << "    rtick[j] = live[j] ? gq_scatter_ticket(cx.part_st, rpart[j]) : 0u;\n  }\n";
      o << "  " << LOOP << "if (live[j]) ropen[j] = gq_scatter_opener(P, cx.part_st, cx.sc_next, rpart[j], rtick[j], ridx[j]);\n";
      o << "  " << LOOP << "if (live[j] && !ropen[j]) ridx[j] = gq_scatter_take(P, cx.part_st, cx.sc_next, rpart[j], rtick[j]);\n";
      o << "  const u64 keep = gq_policy_evict_last();\n";
      o << "  " << LOOP << "if (ridx[j] != ~0ULL) {\n    u64* rec = P.part + ridx[j] * " << rw << ";\n";
      std::vector<std::string> words;
      words.push_back("(u64)tkey[j]");
      if (sp.ndep == 1) words.push_back("(u64)" + depx);
      for (int e : sp.part_exprs) words.push_back("(u64)e" + std::to_string(e) + "[j]");
      while ((int)words.size() < rw) words.push_back("0ULL");
      for (int w = 0; w < rw; w += 4)
        o << "    gq_st256_keep(rec + " << w << ", " << words[(size_t)w] << ", " << words[(size_t)w + 1] << ", " << words[(size_t)w + 2] << ", " << words[(size_t)w + 3] << ", keep);\n";
      o << "  }\n";
      break;
    }
    case GQ_C_DIRECT: {
      // group == matched slot of probe step direct_step (SURVEY §8(d) note on C3): no key compare, no CAS
      if (sp.direct_step < 0 || sp.direct_step >= nprobe || sp.direct_aw < nagg) { if (msg) *msg = "bad direct aggregation spec"; return GQ_ERR_INVALID_ARG; }
      if (sp.part_rw > 0) {
        // clustered: append (accumulator slot, aggregate inputs) to the record buffer of the slot's slice of the array
        // (P.pshift = log2 slots per slice); pass B applies the records slice by slice. Rows that do not fit their
        // buffer fall through to the in-place REDs below.
        const int rw = sp.part_rw;
        o << "  u64 pidx[GQ_R], ppart[GQ_R];\n";
        o << "  " << LOOP << "{\n    pidx[j] = ~0ULL; ppart[j] = 0;\n    if (live[j]) {\n"
          << "      ppart[j] = pi" << sp.direct_step << "[j] >> P.pshift;\n      pidx[j] = (u64)gq_part_reserve(P, cx.part_st, ppart[j]);\n    }\n  }\n";
        o << "  " << LOOP << "if (live[j] && pidx[j] != ~0ULL) {\n    u64* rec = P.part + (ppart[j] * (u64)P.pcap + pidx[j]) * " << rw << ";\n";
        std::vector<std::string> words;
        words.push_back("pi" + std::to_string(sp.direct_step) + "[j]");
        for (int e : sp.part_exprs) words.push_back("(u64)e" + std::to_string(e) + "[j]");
        while ((int)words.size() < rw) words.push_back("0ULL");
        for (int w = 0; w < rw; w += 4)
          o << "    gq_st256(rec + " << w << ", " << words[(size_t)w] << ", " << words[(size_t)w + 1] << ", " << words[(size_t)w + 2] << ", " << words[(size_t)w + 3] << ");\n";
        o << "    live[j] = false;\n  }\n";
      }
      o << "  const u64 keep = gq_policy_evict_last();\n";
      o << "  " << LOOP << "if (live[j]) {\n    u64* acc = P.dacc + pi" << sp.direct_step << "[j] * " << sp.direct_aw << ";\n";
      for (int a = 0; a < nagg; ++a)
        o << "    gq_red_hint(" << (int)sp.aggs[(size_t)a].op << ", acc + " << a << ", " << aggval(sp.aggs[(size_t)a]) << ", keep);\n";
      if (sp.direct_touch) o << "    gq_red_hint(3, acc + " << nagg << ", 1, keep);\n";
      o << "  }\n";
      break;
    }
    case GQ_C_BUILD: {
      const int np = (int)sp.payload_cols.size();
      const std::string karr = as_array(sp.build_key_col);
      o << "  i64 bpay[GQ_R][" << (np > 0 ? np : 1) << "];\n";
      if (np > 0) {
        o << "  " << LOOP << "if (live[j]) {\n";
        for (int p = 0; p < np; ++p) o << "    bpay[j][" << p << "] = " << g.val(sp.payload_cols[(size_t)p]) << ";\n";
        o << "  }\n";
      }
      if (sp.dense_target) o << "  cx.ninserted += gq_dense_insert_rows<" << np << ">(P.target, " << karr << ", live, bpay, P.err);\n";
      else o << "  cx.ninserted += gq_insert_rows<" << sp.target_sw << ", " << np << ">(P.target, " << karr << ", live, bpay, "
        << (sp.unique ? "true" : "false") << ", P.err);\n";
      break;
    }
    case GQ_C_MATERIALISE:
      if (sp.exprs.size() > GQ_MAXOUT) { if (msg) *msg = "too many output columns"; return GQ_ERR_UNSUPPORTED; }
      o << "  i64 orow[GQ_R];\n  gq_materialise_offsets(P, cx, live, orow);\n";
      o << "  " << LOOP << "if (orow[j] >= 0) {\n";
      for (size_t e = 0; e < sp.exprs.size(); ++e) o << "    P.out[" << e << "][orow[j]] = e" << e << "[j];\n";
      o << "  }\n";
      break;
    default: if (msg) *msg = "unknown consumer"; return GQ_ERR_INVALID_ARG;
  }
  o << "}\n\n";
  g.sfx.clear();
  g.linear = false;
  return GQ_OK;
}

gq_status gq_codegen(const GqScanSpec& sp, GqKernelInfo* out, std::string* msg) {
  Gen g(sp, msg);
  const int nprobe = (int)sp.probes.size();
  const int nagg = (int)sp.aggs.size();
  if ((int)sp.preds.size() > GQ_MAX_PREDS || nprobe > GQ_MAX_PROBES || (int)sp.exprs.size() > GQ_MAX_EXPRS ||
      nagg > GQ_MAX_AGGS) { if (msg) *msg = "plan exceeds GQ_MAX_* limits"; return GQ_ERR_UNSUPPORTED; }

  // ---- 1. referenced columns: predicate columns first (they are read for every row) ----
  for (const gq_pred& p : sp.preds) {
    if (p.col < 0 || p.col >= g.ncols_in) { if (msg) *msg = "predicate column must be an input column"; return GQ_ERR_INVALID_ARG; }
    if (!g.use_col(p.col)) return GQ_ERR_INVALID_ARG;
  }
  for (int s = 0; s < nprobe; ++s) {
    if (sp.probes[(size_t)s].key_col < 0 || sp.probes[(size_t)s].key_col >= g.width_before_probe(s)) {
      if (msg) *msg = "probe key column out of range"; return GQ_ERR_INVALID_ARG; }
    if (!g.use_col(sp.probes[(size_t)s].key_col)) return GQ_ERR_INVALID_ARG;
  }
  for (const auto& e : sp.exprs)
    for (const gq_xtok& t : e)
      if (t.op == GQ_X_COL && !g.use_col((int)t.arg)) return GQ_ERR_INVALID_ARG;
  for (int c : sp.key_cols) if (!g.use_col(c)) return GQ_ERR_INVALID_ARG;
  if (sp.consumer == GQ_C_BUILD) {
    if (!g.use_col(sp.build_key_col)) return GQ_ERR_INVALID_ARG;
    for (int c : sp.payload_cols) if (!g.use_col(c)) return GQ_ERR_INVALID_ARG;
  }
  for (const gq_agg& a : sp.aggs)
    if (a.op != GQ_COUNT_STAR && (a.expr < 0 || a.expr >= (int)sp.exprs.size())) {
      if (msg) *msg = "aggregate names a missing expression"; return GQ_ERR_INVALID_ARG; }
  if (g.cols.empty()) {  // a kernel needs at least one column to define rows; count(*)-only plans read column 0
    if (g.ncols_in == 0) { if (msg) *msg = "batch has no columns"; return GQ_ERR_INVALID_ARG; }
    g.use_col(0);
  }

  // ---- 2. tiling: consumer threads, rows per thread, stages under the 227 KB shared-memory budget ----
  const int ncol = (int)g.cols.size();
  int row_bytes = 0;
  for (int c : g.cols) row_bytes += gq_dtype_bytes(sp.in_dtype[(size_t)c]);
  // Hash phases are bound by memory latency, not bandwidth (profiles/r1_hash_phases.md): 24 consumer warps x 2 rows
  // hide more of it than 16 x 4 (C4 1.56 -> 1.13 ms). Pure scans: 20 warps x 2 rows (C2 0.242 -> 0.238 ms).
  const bool hashing = nprobe > 0 || sp.consumer == GQ_C_BUILD || sp.consumer == GQ_C_HIGHCARD || sp.consumer == GQ_C_DIRECT ||
                       sp.consumer == GQ_C_PARTITION || sp.consumer == GQ_C_SCATTER;
  int nt = hashing ? 768 : 640;
  const bool tablebound = sp.consumer == GQ_C_HIGHCARD && nprobe == 0;   // DRAM-random bound (C5): 16 warps x 4 rows measured best
  if (tablebound) nt = 512;
  // Pass A of the partitioned aggregation waits on shared-memory (in a cluster: remote) atomics and on its hot-key probe,
  // not on DRAM: every extra warp hides more of it (C5 pass A, consumer threads 640 / 768 / 896 / 992: 10.2 / 9.4 / 8.8 / 8.3 ms).
  if (sp.consumer == GQ_C_SCATTER) nt = 992;
  long long cons_bytes = 256;
  int lc_kt = 64, lc_key32 = 0;
  if (sp.consumer == GQ_C_GLOBAL) cons_bytes = 8LL * nagg * (nt / 32) + 256;
  if (sp.consumer == GQ_C_LOWCARD) {
    if (sp.lc_cap < 1 || sp.lc_cap > 64) { if (msg) *msg = "low-cardinality path needs 1..64 groups"; return GQ_ERR_INVALID_ARG; }
    lc_kt = sp.lc_cap <= 16 ? 64 : sp.lc_cap <= 32 ? 128 : 256;
    lc_key32 = sp.lc_key_bits > 0 && sp.lc_key_bits < 32;
    const long long head = (lc_kt * 12LL + sp.lc_cap * 8LL + 16 + 8LL * sp.lc_cap * nagg + 127) / 128 * 128;
    // thread-private cells: as many consumer threads as leave room for a 3-stage ring of one-row-per-thread tiles
    for (nt = 256; nt > 128; nt /= 2)   // 8 warps x GQ_R independent rows per thread; cells cost 8 B x groups x aggregates per thread
      if (head + 8LL * sp.lc_cap * nagg * nt + 3LL * ((row_bytes * nt + 127) / 128 * 128 + 128 * ncol) + 1024 <= GQ_SMEM_LIMIT) break;
    cons_bytes = head + 8LL * sp.lc_cap * nagg * nt;
  }
  bool all_unique = true;
  for (const GqProbeSpec& ps : sp.probes) all_unique = all_unique && ps.unique;
  const bool use_hot = sp.hot && (sp.consumer == GQ_C_HIGHCARD || sp.consumer == GQ_C_PARTITION || sp.consumer == GQ_C_SCATTER) && all_unique;   // linear mode only
  // hot set: 512 positions (<= 256 keys); pass A takes 2048 (<= 1536 keys: on a Zipf(1) key column every doubling of the
  // hot set keeps another 4 % of the rows out of the record stream) when a 3-stage ring of one-row-per-thread tiles
  // still fits beside it and the partition state words
  int hot_pos = 512;
  if (use_hot && sp.consumer == GQ_C_SCATTER) {
    long long st1 = 0;
    for (int c : g.cols) st1 += ((long long)nt * gq_dtype_bytes(sp.in_dtype[(size_t)c]) + 127) / 128 * 128;
    const long long hb = 2048LL * (8 + 8 * nagg + 4) + 2048 / 4 + 256 + 128 + (sp.part_states / std::max(1, sp.cluster)) * 4LL + 64;
    if (GQ_SMEM_LIMIT - hb - 2 * 4 * 8 - 64 - 128 >= 3 * st1) hot_pos = 2048;
  }
  if (use_hot) cons_bytes = hot_pos * 8LL + (long long)hot_pos * nagg * 8 + hot_pos * 4LL + hot_pos / 4 + 256;   // keys, accumulators, touched, bucket overflow flags
  long long part_state_off = 0;
  if (sp.part_rw > 0) {   // partition state words (+ the CTA's chunk counter)
    if (sp.part_states < 1 || sp.part_states > 16384) { if (msg) *msg = "bad partition count"; return GQ_ERR_INVALID_ARG; }
    part_state_off = (cons_bytes + 127) / 128 * 128;
    cons_bytes = part_state_off + (sp.part_states / std::max(1, sp.cluster)) * 4LL + 64;   // a cluster's CTAs split the state words
  }
  int r = tablebound ? 4 : 2, stages = 0;
  // small inputs: smaller tiles so that every SM still gets several tiles
  if (sp.nrows_hint > 0 && sp.nrows_hint < (long long)sp.num_sms * 8 * nt * 2) r = 1;
  if (sp.consumer == GQ_C_LOWCARD) r = (sp.nrows_hint > 0 && sp.nrows_hint < (long long)sp.num_sms * nt * 4) ? 1 : 4;   // straight-line rows: ILP
  if (sp.consumer == GQ_C_MATERIALISE && !hashing && !(sp.nrows_hint > 0 && sp.nrows_hint < (long long)sp.num_sms * 8 * nt * 2)) r = 4;   // two CTA barriers per tile: bigger tiles
  long long stage_bytes = 0;
  for (;; r /= 2) {
    stage_bytes = 0;
    for (int c : g.cols) stage_bytes += ((long long)nt * r * gq_dtype_bytes(sp.in_dtype[(size_t)c]) + 127) / 128 * 128;
    long long avail = GQ_SMEM_LIMIT - cons_bytes - 2 * 4 * 8 - 64 - 128;
    stages = (int)std::min<long long>(4, avail / stage_bytes);
    if (stages >= 3 || r == 1) break;
  }
  if (stages < 1) { if (msg) *msg = "plan does not fit shared memory"; return GQ_ERR_UNSUPPORTED; }

  // ---- 3. prelude ----
  std::ostringstream o;
  o << "// generated by gq_codegen — plan-shape specialised prelude\n";
  // (part of the source, hence of the kernel's identity: two plans that differ only in their shared-memory carve-up,
  // e.g. in the number of partition state words, must not share a cached kernel and its launch configuration)
  if (use_hot) o << "#define GQ_HOT_POS " << hot_pos << "\n#define GQ_HOT_MAX " << (hot_pos == 2048 ? 1536 : 256) << "\n";
  o << "#define GQ_SC_CLUSTER " << (sp.consumer == GQ_C_SCATTER ? std::max(1, sp.cluster) : 1) << "\n";
  o << "#define GQ_SMEM_BYTES " << (stages * stage_bytes + 2 * stages * 8 + 64 + cons_bytes + 128) << "\n";
  o << "#define GQ_NCOL " << ncol << "\n#define GQ_NT " << nt << "\n#define GQ_R " << r << "\n#define GQ_STAGES "
    << stages << "\n#define GQ_STAGE_BYTES " << stage_bytes << "\n#define GQ_CONSUMER " << sp.consumer << "\n";
  o << "#define GQ_NAGG " << nagg << "\n#define GQ_LC_G " << (sp.lc_cap > 0 ? sp.lc_cap : 1) << "\n#define GQ_LC_KT " << lc_kt
    << "\n#define GQ_LC_KEY32 " << lc_key32 << "\n#define GQ_TARGET_SW "
    << (sp.target_sw > 0 ? sp.target_sw : 1) << "\n#define GQ_NDEP " << sp.ndep << "\n#define GQ_CHECK_DEP " << (sp.check_dep ? 1 : 0) << "\n#define GQ_LC_KEY_BITS " << (lc_key32 ? sp.lc_key_bits : 1) << "\n#define GQ_HOT " << (use_hot ? 1 : 0)
    << "\n#define GQ_PART_RW " << sp.part_rw << "\n#define GQ_PART_STATE_OFF " << part_state_off << "\n#define GQ_FUSED_FINAL " << (sp.fused_final ? 1 : 0) << "\n#define GQ_DIRECT_AW " << (sp.direct_aw > 0 ? sp.direct_aw : 1) << "\n";
  {
    long long off = 0, tx = 0;
    std::ostringstream offs, bytes;
    offs << "#define GQ_COL_OFF(c) (";
    bytes << "#define GQ_COL_BYTES(c) (";
    for (int i = 0; i < ncol; ++i) {
      int b = gq_dtype_bytes(sp.in_dtype[(size_t)g.cols[(size_t)i]]);
      offs << "(c) == " << i << " ? " << off << " : ";
      bytes << "(c) == " << i << " ? " << b << " : ";
      off += ((long long)nt * r * b + 127) / 128 * 128;
      tx += (long long)nt * r * b;
    }
    offs << "0)\n";
    bytes << "0)\n";
    o << offs.str() << bytes.str() << "#define GQ_TX_BYTES " << tx << "\n";
    o << "#define GQ_AGG_OP(a) (";
    for (int a = 0; a < nagg; ++a) o << "(a) == " << a << " ? " << (int)sp.aggs[(size_t)a].op << " : ";
    o << "0)\n";
  }
  o << gq_skeleton_a << "\n";

  // Linear mode: every probed table has unique keys, so a row yields at most one output row and the GQ_R rows of a
  // thread can advance through the steps together, with the first (usually only) slot access of every row issued
  // before any is consumed (memory-level parallelism for the random accesses). Non-unique probes fan rows out and
  // use the nested one-row-at-a-time form.
  bool linear = true;
  for (const GqProbeSpec& ps : sp.probes) linear = linear && ps.unique;
  o << "#define GQ_LINEAR " << (linear ? 1 : 0) << "\n";
  if (linear) {
    gq_status lst = emit_linear(g, sp, o, msg);
    if (lst != GQ_OK) return lst;
  } else {
    // ---- 4. gq_pass: the filter ----
    o << "template <class Src> __device__ __forceinline__ bool gq_pass(const GqParams& P, const Src& src, int j) {\n";
    {
      std::vector<bool> loaded(g.compact.size(), false);
      for (const gq_pred& p : sp.preds) {
        if (!loaded[(size_t)p.col]) { o << "  " << g.load(p.col) << "\n"; loaded[(size_t)p.col] = true; }
        std::string c;
        if (!pred_cond(g, p, &c)) return GQ_ERR_INVALID_ARG;
        o << "  if (!(" << c << ")) return false;\n";
      }
    }
    o << "  return true;\n}\n\n";

    // ---- 5. gq_body: probes, projection, consumer ----
    o << "template <class Src> __device__ __forceinline__ void gq_body(const GqParams& P, const Src& src, int j, GqCtx& cx) {\n";
    {
      // every input column referenced beyond the filter
      std::vector<bool> need(g.compact.size(), false);
      auto mark = [&](int c) { if (c < g.ncols_in) need[(size_t)c] = true; };
      for (const auto& p : sp.probes) mark(p.key_col);
      for (const auto& e : sp.exprs) for (const gq_xtok& t : e) if (t.op == GQ_X_COL) mark((int)t.arg);
      for (int c : sp.key_cols) mark(c);
      if (sp.consumer == GQ_C_BUILD) { mark(sp.build_key_col); for (int c : sp.payload_cols) mark(c); }
      for (size_t c = 0; c < need.size(); ++c) if (need[c]) o << "  " << g.load((int)c) << "\n";
    }
    std::string ind = "  ";
    for (int s = 0; s < nprobe; ++s) {   // one open-addressing lookup loop per probe step, nested
      const GqProbeSpec& ps = sp.probes[(size_t)s];
      const int sw = ps.slot_words;
      o << ind << "{ // probe step " << s << "\n";
      ind += "  ";
      o << ind << "const GqTableDev& T" << s << " = P.probe[" << s << "];\n";
      o << ind << "const i64 pk" << s << " = " << g.val(ps.key_col) << ";\n";
      if (ps.dense) {   // direct-address table: at most one match, found with one bit test
        o << ind << "for (int n" << s << " = 0; n" << s << " < 1; ++n" << s << ") {\n";
        ind += "  ";
        o << ind << "u64 i" << s << ", rk" << s << ";\n" << ind << "if (!gq_dense_find(T" << s << ", pk" << s << ", &i" << s << ", &rk" << s << ")) break;\n"
          << ind << "(void)rk" << s << ";\n";
        for (int p = 0; p < ps.npayload; ++p)
          o << ind << "const i64 y" << s << "_" << p << " = (i64)__ldg(T" << s << ".slots + i" << s << " * " << ps.npayload << " + " << p << ");\n";
        continue;
      }
      o << ind << "const bool sd" << s << " = ((u64)pk" << s << " == GQ_EMPTY);\n";
      o << ind << "i64 ns" << s << " = 0; if (sd" << s << ") ns" << s << " = gq_min(T" << s << ".header[1], GQ_SIDE_SLOTS);\n";
      o << ind << "u64 i" << s << " = gq_slot0(T" << s << ", pk" << s << ");\n";
      o << ind << "for (u64 n" << s << " = 0; n" << s << " <= T" << s << ".mask; ++n" << s << ") {\n";
      ind += "  ";
      o << ind << "const u64* s" << s << "; u64 w" << s << " = 0;\n";
      o << ind << "if (sd" << s << ") { if ((i64)n" << s << " >= ns" << s << ") break; s" << s << " = T" << s
        << ".side + n" << s << " * " << sw << ";" << (sw == 2 ? " w" + std::to_string(s) + " = s" + std::to_string(s) + "[1];" : "")
        << " }\n";
      o << ind << "else {\n";
      o << ind << "  s" << s << " = T" << s << ".slots + i" << s << " * " << sw << "; i" << s << " = gq_next(T" << s << ", i" << s << ", 1);\n";
      if (sw == 2) o << ind << "  u64 kw; gq_ld128(s" << s << ", kw, w" << s << ");\n";
      else o << ind << "  const u64 kw = __ldg(s" << s << ");\n";
      o << ind << "  if (kw == GQ_EMPTY) break;\n";
      o << ind << "  if (kw != (u64)pk" << s << ") continue;\n";
      o << ind << "}\n";
      for (int p = 0; p < ps.npayload; ++p) {
        if (sw == 2) o << ind << "const i64 y" << s << "_" << p << " = (i64)w" << s << ";\n";
        else o << ind << "const i64 y" << s << "_" << p << " = (i64)__ldg(s" << s << " + " << (1 + p) << ");\n";
      }
      if (ps.npayload == 0) o << ind << "(void)w" << s << ";\n";
    }
    // projection
    for (size_t e = 0; e < sp.exprs.size(); ++e) {
      std::string x;
      if (!g.expr(sp.exprs[e], &x)) return GQ_ERR_INVALID_ARG;
      o << ind << "const i64 e" << e << " = " << x << ";\n";
    }
    // group key
    std::string keyx, depx;
    if (sp.consumer == GQ_C_LOWCARD || sp.consumer == GQ_C_HIGHCARD) {
      gq_status kst = key_exprs(g, sp, &keyx, &depx, msg);
      if (kst != GQ_OK) return kst;
    }
    auto aggval = [&](const gq_agg& a) { return a.op == GQ_COUNT_STAR ? std::string("1") : "e" + std::to_string(a.expr); };
    switch (sp.consumer) {
      case GQ_C_GLOBAL:
        for (int a = 0; a < nagg; ++a)
          o << ind << "cx.acc[" << a << "] = gq_combine(" << (int)sp.aggs[(size_t)a].op << ", cx.acc[" << a << "], "
            << aggval(sp.aggs[(size_t)a]) << ");\n";
        break;
      case GQ_C_LOWCARD:
        o << ind << "const int grp = gq_lc_slot(cx, " << keyx << ", P.err);\n" << ind << "if (grp >= 0) {\n";
        for (int a = 0; a < nagg; ++a)
          o << ind << "  gq_lc_update(" << (int)sp.aggs[(size_t)a].op << ", cx, grp, " << a << ", " << aggval(sp.aggs[(size_t)a]) << ");\n";
        o << ind << "}\n";
        break;
      case GQ_C_HIGHCARD:
        o << ind << "bool won; u64* slot = gq_ht_upsert<" << sp.target_sw << ">(P.target, " << keyx << ", &won, P.err);\n";
        o << ind << "if (slot) {\n";
        if (sp.ndep == 1) o << ind << "  gq_dep_store(slot + 1, " << depx << ", won, P.err);\n";
        for (int a = 0; a < nagg; ++a)
          o << ind << "  gq_red(" << (int)sp.aggs[(size_t)a].op << ", slot + " << (1 + sp.ndep + a) << ", " << aggval(sp.aggs[(size_t)a]) << ");\n";
        o << ind << "}\n";
        break;
      case GQ_C_BUILD: {
        const int np = (int)sp.payload_cols.size();
        o << ind << "const i64 pay[" << (np > 0 ? np : 1) << "] = {";
        for (int p = 0; p < np; ++p) o << (p ? ", " : "") << g.val(sp.payload_cols[(size_t)p]);
        if (np == 0) o << "0";
        o << "};\n";
        if (sp.dense_target) o << ind << "if (gq_dense_insert<" << np << ">(P.target, " << g.val(sp.build_key_col) << ", pay, P.err)) ++cx.ninserted;\n";
        else o << ind << "if (gq_ht_insert<" << sp.target_sw << ", " << np << ">(P.target, " << g.val(sp.build_key_col) << ", pay, "
          << (sp.unique ? "true" : "false") << ", P.err)) ++cx.ninserted;\n";
        break;
      }
      case GQ_C_MATERIALISE:
        if (sp.exprs.size() > GQ_MAXOUT) { if (msg) *msg = "too many output columns"; return GQ_ERR_UNSUPPORTED; }
        o << ind << "const i64 orow = gq_reserve_row(P);\n" << ind << "if (orow >= 0) {\n";
        for (size_t e = 0; e < sp.exprs.size(); ++e) o << ind << "  P.out[" << e << "][orow] = e" << e << ";\n";
        o << ind << "}\n";
        break;
      default: if (msg) *msg = "consumer not available for plans that probe a table with duplicate keys"; return GQ_ERR_UNSUPPORTED;
    }
    for (int s = nprobe - 1; s >= 0; --s) {
      if (sp.probes[(size_t)s].unique) o << ind << "break;  // unique build keys: first match is the only match\n";
      ind.resize(ind.size() - 2);
      o << ind << "}\n";
      ind.resize(ind.size() - 2);
      o << ind << "}\n";
    }
    o << "}\n\n";

  }
  o << gq_skeleton_b << "\n";

  out->source = o.str();
  char hb[32];
  snprintf(hb, sizeof hb, "%016llx", (unsigned long long)fnv1a(out->source));
  out->hash = hb;
  out->threads = nt + 32;
  out->tile_rows = nt * r;
  out->cluster = sp.consumer == GQ_C_SCATTER ? std::max(1, sp.cluster) : 1;
  out->smem_bytes = (int)(stages * stage_bytes + 2 * stages * 8 + 64 + cons_bytes + 128);
  out->cols = g.cols;
  out->consts = g.consts;
  if ((int)g.consts.size() > GQ_MAXK) { if (msg) *msg = "too many constants"; return GQ_ERR_UNSUPPORTED; }
  return GQ_OK;
}

// Pass B of the partitioned shared-memory aggregation (gq_psa_kernel.cuh), specialised by the plan's aggregate list,
// record layout and table slot layout. `src[a]` = record word holding the input of aggregate a (unused for COUNT).
gq_status gq_codegen_psa(const GqScanSpec& sp, int log2slots, const int* src, int threads, GqKernelInfo* out, std::string* msg) {
  const int nagg = (int)sp.aggs.size();
  if (nagg < 1 || nagg > GQ_MAX_AGGS || sp.part_rw < 4 || sp.part_rw % 4 || sp.target_sw < 2 || log2slots < 6 || log2slots > 16 ||
      (threads != 512 && threads != 1024)) {
    if (msg) *msg = "bad partitioned-aggregation spec"; return GQ_ERR_INVALID_ARG; }
  std::ostringstream o;
  o << "// generated by gq_codegen_psa — plan-shape specialised prelude\n";
  // the scan skeleton's macros: only its types and hash-table primitives are used here
  o << "#define GQ_NCOL 1\n#define GQ_NT 512\n#define GQ_R 1\n#define GQ_STAGES 1\n#define GQ_STAGE_BYTES 128\n#define GQ_CONSUMER 2\n"
    << "#define GQ_LC_G 1\n#define GQ_LC_KT 64\n#define GQ_LC_KEY32 0\n#define GQ_LC_KEY_BITS 1\n#define GQ_HOT 0\n#define GQ_PART_STATE_OFF 0\n"
    << "#define GQ_FUSED_FINAL 0\n#define GQ_DIRECT_AW 1\n#define GQ_COL_OFF(c) 0\n#define GQ_COL_BYTES(c) 8\n#define GQ_TX_BYTES 0\n";
  o << "#define GQ_NAGG " << nagg << "\n#define GQ_TARGET_SW " << sp.target_sw << "\n#define GQ_NDEP " << sp.ndep << "\n#define GQ_CHECK_DEP "
    << (sp.check_dep ? 1 : 0) << "\n#define GQ_PART_RW " << sp.part_rw << "\n#define GQ_PSA_LOG2SLOTS " << log2slots << "\n#define GQ_PSA_THREADS " << threads
    << "\n#define GQ_PSA_U " << (threads == 1024 ? 2 : 4) << "\n";
  o << "#define GQ_AGG_OP(a) (";
  for (int a = 0; a < nagg; ++a) o << "(a) == " << a << " ? " << (int)sp.aggs[(size_t)a].op << " : ";
  o << "0)\n#define GQ_AGG_SRC(a) (";
  for (int a = 0; a < nagg; ++a) o << "(a) == " << a << " ? " << (src[a] < 0 ? 0 : src[a]) << " : ";
  o << "0)\n";
  o << gq_skeleton_a << "\n" << gq_skeleton_psa << "\n";
  out->source = o.str();
  char hb[32];
  snprintf(hb, sizeof hb, "%016llx", (unsigned long long)fnv1a(out->source));
  out->hash = hb;
  out->entry = "gq_psa";
  out->threads = threads;
  out->tile_rows = 0;
  out->smem_bytes = (int)((((1LL << log2slots) + 1) * sp.target_sw + 2 * 66) * 8 + 64);   // table, range stack, control words
  if (out->smem_bytes > GQ_SMEM_LIMIT) { if (msg) *msg = "partitioned-aggregation table does not fit shared memory"; return GQ_ERR_UNSUPPORTED; }
  return GQ_OK;
}
