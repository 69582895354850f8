// gq_api.cpp — the C ABI of include/gq.h: argument validation, workspace layout, plan normalisation, launches.
// Every entry point only enqueues work on the context's stream — no device allocation, no host sync —
// except gq_create/gq_destroy/gq_sync and the HOST-buffer end-to-end call gq_pipeline_host.
#include <algorithm>
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <sstream>

#include "gq_internal.h"

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline bool aligned(const void* p, size_t a) { return ((uintptr_t)p % a) == 0; }
inline bool dtype_ok(int t) { return t == GQ_I8 || t == GQ_I32 || t == GQ_I64; }

gq_status fail(gq_ctx* ctx, gq_status st, const std::string& m) { if (ctx) ctx->msg = m; return st; }
gq_status cuda_fail(gq_ctx* ctx, cudaError_t e, const char* where) {
  if (ctx) { ctx->last_cuda = (int)e; ctx->msg = std::string(where) + ": " + cudaGetErrorString(e); }
  return GQ_ERR_CUDA;
}

int64_t table_capacity(int64_t max_rows) {   // power of two >= max_rows * 4/3, at least 1024 (load factor <= 0.75)
  int64_t need = std::max<int64_t>(1024, max_rows + (max_rows + 2) / 3);
  int64_t c = 1024;
  while (c < need) c <<= 1;
  return c;
}
// Join tables: capacity = max_rows / load rounded up to a multiple of 1024 — NOT to a power of two: the slot index
// comes from a multiply-shift range reduction, so the table (and a direct-aggregation array indexed by its slots) is
// as small as the hint allows. Load factor (measured, C3/C4 sweeps 0.3-0.75): a table that fits L2 even at load 0.4
// takes 0.4 — its probes are latency-bound and sparse buckets save dependent rounds (C4 1.06 -> 0.98 ms); a larger
// one is bound by random DRAM sectors and takes 0.7 to shrink its footprint (C3 1.77 -> 1.60 ms).
int64_t join_capacity(int64_t max_rows, int slot_words = 1) {
  const int load = (max_rows * slot_words * 8 * 10 / 4 <= (80LL << 20)) ? 40 : 70;
  int64_t need = std::max<int64_t>(1024, (max_rows * 100 + load - 1) / load);
  return (need + 1023) / 1024 * 1024;
}
int join_slot_words(int npayload) { return npayload == 0 ? 1 : (int)align_up((size_t)(1 + npayload), 2); }
// Group-by slot = key + dependent word + aggregates, padded to an even word count (16-byte multiple). Padding to a
// power of two (64-byte slots for C5, never straddling a DRAM burst) was measured: radix-clustered 35.3 -> 34.3 ms but
// single-pass 47.9 -> 49.9 ms and a 3.2 -> 4.3 GB table; not adopted.
int agg_slot_words(int ndep, int naggs) { return (int)align_up((size_t)(1 + ndep + naggs), 2); }
int log2i(int64_t v) { int l = 0; while ((1LL << l) < v) ++l; return l; }

// workspace = [header 256 B][side area][slots]
struct WsLayout { size_t side_off, slots_off, total; };
WsLayout ws_layout(int64_t capacity, int slot_words, int nside) {
  WsLayout w;
  w.side_off = 256;
  w.slots_off = 256 + align_up((size_t)nside * slot_words * 8, 256);
  w.total = w.slots_off + (size_t)capacity * slot_words * 8;
  return w;
}

// Every entry point that enqueues work makes the context's device current first (a process may hold contexts on
// several GPUs; cudaSetDevice is a no-op when nothing changes).
inline void use_device(gq_ctx* ctx) { if (ctx) cudaSetDevice(ctx->device); }

// gq_profile: brackets the kernel launches enqueued while it is alive with a pair of events on the context's stream.
struct ProfScope {
  gq_ctx* c; int i = -1;
  ProfScope(gq_ctx* ctx, const char* name) : c(ctx) {
    if (!c || !c->prof) return;
    i = (int)c->prof_names.size();
    while ((int)c->prof_ev.size() < 2 * (i + 1)) { cudaEvent_t e; if (cudaEventCreate(&e) != cudaSuccess) { i = -1; return; } c->prof_ev.push_back(e); }
    c->prof_names.push_back(name);
    cudaEventRecord(c->prof_ev[2 * i], c->stream);
  }
  ~ProfScope() { if (i >= 0) cudaEventRecord(c->prof_ev[2 * i + 1], c->stream); }
};
#define PROF(ctx, name, call) (ProfScope(ctx, name), (call))

gq_status check_batch(gq_ctx* ctx, const gq_batch* b) {
  use_device(ctx);
  if (!b || b->ncols < 0 || b->ncols > GQ_MAX_COLS || b->nrows < 0 || (b->ncols > 0 && !b->cols))
    return fail(ctx, GQ_ERR_INVALID_ARG, "bad batch");
  for (int c = 0; c < b->ncols; ++c) {
    if (!dtype_ok(b->cols[c].dtype)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad column dtype");
    if (b->nrows > 0 && (!b->cols[c].data || !aligned(b->cols[c].data, 16)))
      return fail(ctx, GQ_ERR_INVALID_ARG, "column pointer null or not 16-byte aligned");
  }
  return GQ_OK;
}

// dtype of row column c (input column or payload of an earlier probe step)
gq_dtype row_dtype(const GqScanSpec& sp, int c) {
  int n = (int)sp.in_dtype.size();
  if (c < n) return sp.in_dtype[(size_t)c];
  c -= n;
  for (const GqProbeSpec& p : sp.probes) { if (c < p.npayload) return p.pay_dtype[c]; c -= p.npayload; }
  return GQ_I64;
}
int row_width(const GqScanSpec& sp) {
  int n = (int)sp.in_dtype.size();
  for (const GqProbeSpec& p : sp.probes) n += p.npayload;
  return n;
}

gq_status fill_common(gq_ctx* ctx, GqScanSpec* sp, const gq_batch* in, const gq_pred* preds, int npred,
                      const gq_probe_step* probes, int nprobes, const gq_expr* exprs, int nexpr) {
  if (npred < 0 || npred > GQ_MAX_PREDS || (npred > 0 && !preds)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad predicates");
  if (nprobes < 0 || nprobes > GQ_MAX_PROBES || (nprobes > 0 && !probes)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad probe steps");
  if (nexpr < 0 || nexpr > GQ_MAX_EXPRS || (nexpr > 0 && !exprs)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad expressions");
  sp->in_dtype.clear();
  for (int c = 0; c < in->ncols; ++c) sp->in_dtype.push_back(in->cols[c].dtype);
  sp->preds.assign(preds, preds + npred);
  for (const gq_pred& p : sp->preds)
    if (p.col < 0 || p.col >= in->ncols || (int)p.op < 0 || (int)p.op > (int)GQ_RANGE_CC)
      return fail(ctx, GQ_ERR_INVALID_ARG, "predicate column/op out of range");
  sp->probes.clear();
  for (int s = 0; s < nprobes; ++s) {
    const gq_table* t = probes[s].table;
    if (!t) return fail(ctx, GQ_ERR_INVALID_ARG, "null table in probe step");
    GqProbeSpec ps;
    ps.key_col = probes[s].key_col;
    ps.npayload = t->npayload;
    for (int p = 0; p < GQ_MAX_PAYLOAD; ++p) ps.pay_dtype[p] = t->payload_dtype[p];
    ps.unique = (t->flags & GQ_F_UNIQUE_KEYS) != 0;
    ps.dense = (t->flags & GQ_F_DENSE_KEYS) != 0;
    ps.slot_words = join_slot_words(t->npayload);
    if (ps.key_col < 0 || ps.key_col >= row_width(*sp)) return fail(ctx, GQ_ERR_INVALID_ARG, "probe key column out of range");
    sp->probes.push_back(ps);
  }
  sp->exprs.clear();
  for (int e = 0; e < nexpr; ++e) {
    if (!exprs[e].toks || exprs[e].ntoks < 1 || exprs[e].ntoks > GQ_MAX_TOKS) return fail(ctx, GQ_ERR_INVALID_ARG, "bad expression");
    sp->exprs.emplace_back(exprs[e].toks, exprs[e].toks + exprs[e].ntoks);
  }
  sp->nrows_hint = in->nrows;
  if (ctx && ctx->num_sms > 0) sp->num_sms = ctx->num_sms;
  return GQ_OK;
}

// Constants in codegen order (predicate bounds, then expression literals); equal values share one parameter slot
// (so common subexpressions stay common in the generated code). idx receives the slot of every occurrence: WHICH
// literals are equal is part of the plan shape, their values are not.
void collect_consts(const GqScanSpec& sp, std::vector<long long>* k, std::vector<int>* idx = nullptr) {
  k->clear();
  auto put = [&](long long v) {
    size_t i = 0;
    while (i < k->size() && (*k)[i] != v) ++i;
    if (i == k->size()) k->push_back(v);
    if (idx) idx->push_back((int)i);
  };
  for (const gq_pred& p : sp.preds) { put(p.lo); if (p.op == GQ_RANGE_CO || p.op == GQ_RANGE_CC) put(p.hi); }
  for (const auto& e : sp.exprs) for (const gq_xtok& t : e) if (t.op == GQ_X_CONST) put(t.arg);
}

// Shape signature (no constant values) and the constants in codegen order (predicates, then expression literals).
int tile_bucket(int64_t nrows, int sms) { return nrows <= 0 ? 0 : nrows < (int64_t)sms * 8 * 512 * 2 ? 1 : nrows < (int64_t)sms * 8 * 512 * 4 ? 2 : 3; }
std::string signature(const GqScanSpec& sp) {
  std::string s;
  s.reserve(256);
  auto put = [&s](long long v) { s += std::to_string(v); s += ','; };
  put(sp.consumer); put(tile_bucket(sp.nrows_hint, sp.num_sms)); put(sp.num_sms);
  for (gq_dtype t : sp.in_dtype) put(t);
  s += 'p';
  for (const gq_pred& p : sp.preds) { put(p.col); put(p.op); }
  s += 'j';
  for (const GqProbeSpec& p : sp.probes) { put(p.key_col); put(p.npayload); put(p.unique); put(p.dense); for (int i = 0; i < p.npayload; ++i) put(p.pay_dtype[i]); }
  s += 'e';
  for (const auto& e : sp.exprs) { for (const gq_xtok& t : e) { put(t.op); if (t.op == GQ_X_COL) put(t.arg); } s += ';'; }
  s += 'k';
  for (int c : sp.key_cols) put(c);
  put(sp.ndep);
  for (const gq_agg& a : sp.aggs) { put(a.op); put(a.expr); }
  put(sp.lc_cap); put(sp.lc_key_bits); put(sp.target_sw); put(sp.build_key_col);
  for (int c : sp.payload_cols) put(c);
  put(sp.unique); put(sp.dense_target); put(sp.hot); put(sp.check_dep); put(sp.fused_final); put(sp.direct_step); put(sp.direct_aw); put(sp.direct_touch);
  put(sp.part_rw); put(sp.part_states); put(sp.cluster); for (int e : sp.part_exprs) put(e);
  s += 'c';
  std::vector<long long> kv; std::vector<int> ki;
  collect_consts(sp, &kv, &ki);
  for (int i : ki) put(i);
  return s;
}
struct CachedKernel { GqKernelInfo info; GqKernel k; bool loaded = false; int device = -1; };
std::mutex g_kmu;
std::map<std::string, CachedKernel> g_kernels;

// Normalise the tiling hint so that every nrows in a bucket produces the same source.
void canon_hint(GqScanSpec* sp) {
  const int64_t unit = (int64_t)sp->num_sms * 8 * 512;
  const int64_t rep[4] = {0, unit, unit * 3, 0};
  sp->nrows_hint = rep[tile_bucket(sp->nrows_hint, sp->num_sms)];
}

gq_status get_kernel_info(const GqScanSpec& sp_in, CachedKernel** out, std::string* msg) {
  GqScanSpec sp = sp_in;
  canon_hint(&sp);
  std::string sig = signature(sp);
  std::lock_guard<std::mutex> l(g_kmu);
  auto it = g_kernels.find(sig);
  if (it == g_kernels.end()) {
    CachedKernel ck;
    gq_status st = gq_codegen(sp, &ck.info, msg);
    if (st != GQ_OK) return st;
    std::vector<long long> k;
    collect_consts(sp, &k);
    if (k != ck.info.consts) { if (msg) *msg = "internal: constant order mismatch"; return GQ_ERR_COMPILE; }
    it = g_kernels.emplace(sig, std::move(ck)).first;
  }
  *out = &it->second;
  return GQ_OK;
}

// JIT (cached) of a generated kernel for the context's device.
gq_status load_kernel(gq_ctx* ctx, CachedKernel* ck, GqKernel* kern) {
  std::lock_guard<std::mutex> l(g_kmu);   // distinct contexts may launch the same plan shape for the first time concurrently (gq.h "Threads")
  if (!ck->loaded || ck->device != ctx->device) {
    cudaSetDevice(ctx->device);
    gq_status st = gq_jit_get(ck->info, ctx->device, &ck->k, &ctx->msg, &ctx->last_cuda);
    if (st != GQ_OK) return st;
    ck->loaded = true;
    ck->device = ctx->device;
  }
  *kern = ck->k;
  return GQ_OK;
}

// Pass B kernel of the partitioned shared-memory aggregation for this plan shape (cached by shape).
gq_status get_psa_kernel_info(const GqScanSpec& sp, int log2slots, const int* src, int threads, CachedKernel** out, std::string* msg) {
  std::string sig = "psa:" + std::to_string(log2slots) + "," + std::to_string(threads) + "," + std::to_string(sp.target_sw) + "," + std::to_string(sp.part_rw) + "," +
                    std::to_string(sp.ndep) + "," + std::to_string(sp.check_dep) + ";";
  for (size_t a = 0; a < sp.aggs.size(); ++a) sig += std::to_string((int)sp.aggs[a].op) + ":" + std::to_string(src[a]) + ",";
  std::lock_guard<std::mutex> l(g_kmu);
  auto it = g_kernels.find(sig);
  if (it == g_kernels.end()) {
    CachedKernel ck;
    gq_status st = gq_codegen_psa(sp, log2slots, src, threads, &ck.info, msg);
    if (st != GQ_OK) return st;
    it = g_kernels.emplace(sig, std::move(ck)).first;
  }
  *out = &it->second;
  return GQ_OK;
}

// CTAs of a persistent grid of clusters that are co-resident (a cluster of 4 does not pack all 148 SMs of a B200).
int cluster_grid(gq_ctx* ctx, const GqKernel& kern) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(ctx->num_sms / kern.cluster * kern.cluster)); cfg.blockDim = dim3((unsigned)kern.threads);
  cfg.dynamicSmemBytes = (size_t)kern.smem_bytes;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = (unsigned)kern.cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  int nc = 0;
  if (cudaOccupancyMaxActiveClusters(&nc, (const void*)kern.fn, &cfg) != cudaSuccess || nc < 1) return ctx->num_sms / kern.cluster * kern.cluster;
  return std::min(ctx->num_sms / kern.cluster, nc) * kern.cluster;
}

// Codegen (cached) -> JIT (cached) -> parameters -> launch of one fused scan kernel.
gq_status run_scan(gq_ctx* ctx, const GqScanSpec& sp, const gq_batch* in, const gq_probe_step* probes,
                   GqParams* P /* target/acc/out/out_count pre-filled */) {
  CachedKernel* ck = nullptr;
  gq_status st = get_kernel_info(sp, &ck, &ctx->msg);
  if (st != GQ_OK) return st;
  GqKernel kern;
  st = load_kernel(ctx, ck, &kern);
  if (st != GQ_OK) return st;
  for (size_t c = 0; c < ck->info.cols.size(); ++c) P->col[c] = in->cols[ck->info.cols[c]].data;
  P->nrows = in->nrows;
  std::vector<long long> k;
  collect_consts(sp, &k);
  for (size_t i = 0; i < k.size(); ++i) P->k[i] = k[i];
  for (size_t s = 0; s < sp.probes.size(); ++s) {
    const gq_table* t = probes[s].table;
    if (t->describe_only) return fail(ctx, GQ_ERR_INVALID_ARG, "probe step names a describe-only table");
    if (t->dense && !t->ranked) return fail(ctx, GQ_ERR_INVALID_ARG, "a GQ_F_DENSE_KEYS table must be finished (gq_hash_build_finish) before it is probed");
    P->probe[s] = t->dev;
    if (t->finished && t->build_stream != ctx->stream) {   // cross-pipeline boundary
      cudaError_t e = cudaStreamWaitEvent(ctx->stream, t->ready, 0);
      if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaStreamWaitEvent");
    }
  }
  P->err = ctx->d_err;
  if (in->nrows == 0) return GQ_OK;   // empty batches are legal no-ops (S9)
  const int64_t ntiles = in->nrows / kern.tile_rows;
  int grid = (int)std::max<int64_t>(1, std::min<int64_t>(ctx->num_sms, ntiles));
  if (kern.cluster > 1) grid = std::max(kern.cluster, std::min(grid, cluster_grid(ctx, kern)) / kern.cluster * kern.cluster);   // whole, co-resident clusters
  void* args[] = {(void*)P};
  static const char* const kname[] = {"gq_scan:global", "gq_scan:lowcard", "gq_scan:highcard", "gq_scan:build", "gq_scan:materialise",
                                      "gq_scan:direct", "gq_scan:partition", "gq_scan:scatter"};
  ProfScope ps(ctx, kname[sp.consumer]);
  cudaError_t e;
  if (kern.cluster > 1) {   // thread-block clusters: the CTAs of a cluster reach each other's shared memory
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)kern.threads);
    cfg.dynamicSmemBytes = (size_t)kern.smem_bytes; cfg.stream = ctx->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)kern.cluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    e = cudaLaunchKernelExC(&cfg, (const void*)kern.fn, args);
  } else
    e = cudaLaunchKernel((const void*)kern.fn, dim3((unsigned)grid), dim3((unsigned)kern.threads), args, (size_t)kern.smem_bytes, ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of fused scan kernel");
  ++ctx->launches;
  return GQ_OK;
}

}  // namespace

extern "C" {

// ------------------------------------------------------------------------------------------------ context
gq_status gq_create(gq_ctx** out, int device, void* cuda_stream) {
  if (!out) return GQ_ERR_INVALID_ARG;
  *out = nullptr;
  cudaError_t e = cudaSetDevice(device);
  if (e != cudaSuccess) return GQ_ERR_CUDA;
  gq_ctx* c = new gq_ctx();
  c->device = device;
  c->stream = (cudaStream_t)cuda_stream;
  int sms = 0;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) == cudaSuccess && sms > 0) c->num_sms = sms;
  e = cudaMalloc((void**)&c->d_err, 256 + GQ_GTAB_BYTES);
  if (e == cudaSuccess) e = cudaMemset(c->d_err, 0, 256 + GQ_GTAB_BYTES);
  if (e == cudaSuccess) e = cudaMallocHost((void**)&c->h_err, 256);
  if (e != cudaSuccess) { if (c->d_err) cudaFree(c->d_err); delete c; return GQ_ERR_CUDA; }
  *c->h_err = 0;
  *out = c;
  return GQ_OK;
}

gq_status gq_destroy(gq_ctx* c) {
  if (!c) return GQ_ERR_INVALID_ARG;
  cudaFree(c->d_err);
  cudaFreeHost(c->h_err);
  for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->ev_start) cudaEventDestroy(c->ev_start);
  for (int i = 0; i < 2; ++i) { if (c->ev_copied[i]) cudaEventDestroy(c->ev_copied[i]); if (c->ev_consumed[i]) cudaEventDestroy(c->ev_consumed[i]); }
  delete c;
  return GQ_OK;
}

gq_status gq_sync(gq_ctx* c) {
  if (!c) return GQ_ERR_INVALID_ARG;
  use_device(c);
  cudaError_t e = cudaMemcpyAsync(c->h_err, c->d_err, sizeof(int), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return cuda_fail(c, e, "gq_sync");
  int code = *c->h_err;
  if (code == 0) return GQ_OK;
  c->msg = code == GQ_ERR_CAPACITY ? "device: hash table or output capacity exceeded"
         : code == GQ_ERR_DUPLICATE_KEY ? "device: duplicate build key under GQ_F_UNIQUE_KEYS"
         : code == GQ_ERR_DEPENDENT_KEY ? "device: a key declared dependent (ndependent) took two values within one group"
         : code == GQ_ERR_KEY_RANGE ? "device: a build key outside the declared range of a GQ_F_DENSE_KEYS table" : "device error";
  return (gq_status)code;
}

gq_status gq_clear_error(gq_ctx* c) {
  if (!c) return GQ_ERR_INVALID_ARG;
  use_device(c);
  // (also the ticket and the merge table of the fused finaliser: a kernel that stopped on the error may have left them set)
  cudaError_t e = cudaMemsetAsync(c->d_err, 0, 256 + GQ_GTAB_BYTES, c->stream);
  return e == cudaSuccess ? GQ_OK : cuda_fail(c, e, "gq_clear_error");
}

const char* gq_status_str(gq_status s) {
  switch (s) {
    case GQ_OK: return "GQ_OK";
    case GQ_ERR_INVALID_ARG: return "GQ_ERR_INVALID_ARG";
    case GQ_ERR_UNSUPPORTED: return "GQ_ERR_UNSUPPORTED";
    case GQ_ERR_CAPACITY: return "GQ_ERR_CAPACITY";
    case GQ_ERR_WORKSPACE_TOO_SMALL: return "GQ_ERR_WORKSPACE_TOO_SMALL";
    case GQ_ERR_CUDA: return "GQ_ERR_CUDA";
    case GQ_ERR_DUPLICATE_KEY: return "GQ_ERR_DUPLICATE_KEY";
    case GQ_ERR_COMPILE: return "GQ_ERR_COMPILE";
    case GQ_ERR_DEPENDENT_KEY: return "GQ_ERR_DEPENDENT_KEY";
    case GQ_ERR_KEY_RANGE: return "GQ_ERR_KEY_RANGE";
  }
  return "GQ_ERR_UNKNOWN";
}
int gq_last_cuda_error(gq_ctx* c) { return c ? c->last_cuda : 0; }
const char* gq_last_message(gq_ctx* c) { return c ? c->msg.c_str() : ""; }
int64_t gq_launch_count(gq_ctx* c) { return c ? c->launches : 0; }

// ------------------------------------------------------------------------------------------------ FilterProject
static gq_status materialise(gq_ctx* ctx, const gq_batch* in, const gq_pred* preds, int32_t npred,
                             const gq_probe_step* probes, int32_t nprobes, const gq_expr* exprs, int32_t nexpr,
                             int64_t* const* out_cols, int64_t out_capacity, int64_t* d_out_count) {
  if (!ctx) return GQ_ERR_INVALID_ARG;
  gq_status st = check_batch(ctx, in);
  if (st != GQ_OK) return st;
  if (nexpr < 1 || !out_cols || !d_out_count || out_capacity < 0) return fail(ctx, GQ_ERR_INVALID_ARG, "bad outputs");
  GqScanSpec sp;
  st = fill_common(ctx, &sp, in, preds, npred, probes, nprobes, exprs, nexpr);
  if (st != GQ_OK) return st;
  sp.consumer = GQ_C_MATERIALISE;
  GqParams P;
  memset(&P, 0, sizeof P);
  for (int e = 0; e < nexpr; ++e) {
    if (!out_cols[e] || !aligned(out_cols[e], 16)) return fail(ctx, GQ_ERR_INVALID_ARG, "output column null or misaligned");
    P.out[e] = (long long*)out_cols[e];
  }
  P.out_capacity = out_capacity;
  P.out_count = (long long*)d_out_count;
  return run_scan(ctx, sp, in, probes, &P);
}

gq_status gq_filter_project(gq_ctx* ctx, const gq_batch* in, const gq_pred* preds, int32_t npred, const gq_expr* exprs,
                            int32_t nexpr, int64_t* const* out_cols, int64_t out_capacity, int64_t* d_out_count) {
  return materialise(ctx, in, preds, npred, nullptr, 0, exprs, nexpr, out_cols, out_capacity, d_out_count);
}

gq_status gq_hash_probe(gq_ctx* ctx, const gq_batch* probe, const gq_pred* preds, int32_t npred,
                        const gq_probe_step* probes, int32_t nprobes, const gq_expr* exprs, int32_t nexpr,
                        int64_t* const* out_cols, int64_t out_capacity, int64_t* d_out_count) {
  if (nprobes < 1) return fail(ctx, GQ_ERR_INVALID_ARG, "gq_hash_probe needs at least one probe step");
  return materialise(ctx, probe, preds, npred, probes, nprobes, exprs, nexpr, out_cols, out_capacity, d_out_count);
}

// ------------------------------------------------------------------------------------------------ HashBuild
gq_status gq_hash_build_workspace(int64_t max_build_rows, int32_t npayload, size_t* bytes) {
  if (!bytes || max_build_rows < 0 || npayload < 0 || npayload > GQ_MAX_PAYLOAD) return GQ_ERR_INVALID_ARG;
  *bytes = ws_layout(join_capacity(max_build_rows, join_slot_words(npayload)), join_slot_words(npayload), GQ_SIDE_SLOTS).total;
  return GQ_OK;
}

// Direct-address table (GQ_F_DENSE_KEYS): [header 256 B][bitmap entries, 8 B per 32 keys of the range][payload rows]
// [key of every rank: max_rows words][scratch of the rank kernels]
struct DenseLayout { int64_t range, max_rows, nwords; size_t bitmap_off, bitmap_bytes, pay_off, keyrank_off, totals_off, total; };
static bool dense_layout(int64_t key_min, int64_t key_max, int64_t max_rows, int npayload, DenseLayout* L) {
  if (key_max < key_min || (uint64_t)key_max - (uint64_t)key_min >= (1ULL << 36) || max_rows < 0) return false;
  L->range = (int64_t)((uint64_t)key_max - (uint64_t)key_min + 1);
  L->max_rows = std::min<int64_t>(L->range, max_rows > 0 ? max_rows : L->range);   // unique keys: never more rows than keys in the range
  if (L->max_rows >= (1LL << 32)) return false;
  L->nwords = (L->range + 31) / 32;
  L->bitmap_off = 256;
  L->bitmap_bytes = align_up((size_t)L->nwords * 8, 256);
  L->pay_off = L->bitmap_off + L->bitmap_bytes;
  L->keyrank_off = L->pay_off + align_up((size_t)L->range * (size_t)npayload * 8, 256);
  L->totals_off = L->keyrank_off + align_up((size_t)L->max_rows * 8, 256);
  L->total = L->totals_off + align_up((size_t)((L->nwords + GQ_DENSE_RANK_BLOCK - 1) / GQ_DENSE_RANK_BLOCK) * 4, 256);
  return true;
}

gq_status gq_hash_build_workspace_dense(int64_t key_min, int64_t key_max, int64_t max_build_rows, int32_t npayload, size_t* bytes) {
  DenseLayout L;
  if (!bytes || npayload < 0 || npayload > GQ_MAX_PAYLOAD || !dense_layout(key_min, key_max, max_build_rows, npayload, &L)) return GQ_ERR_INVALID_ARG;
  *bytes = L.total;
  return GQ_OK;
}

static gq_status build_spec(gq_ctx* ctx, GqScanSpec* sp, const gq_batch* in, const gq_build_desc* d) {
  gq_status st = fill_common(ctx, sp, in, d->preds, d->npred, d->probes, d->nprobes, nullptr, 0);
  if (st != GQ_OK) return st;
  if (d->npayload < 0 || d->npayload > GQ_MAX_PAYLOAD || (d->npayload > 0 && !d->payload_cols))
    return fail(ctx, GQ_ERR_INVALID_ARG, "bad payload columns");
  const int w = row_width(*sp);
  if (d->key_col < 0 || d->key_col >= w) return fail(ctx, GQ_ERR_INVALID_ARG, "build key column out of range");
  sp->consumer = GQ_C_BUILD;
  sp->build_key_col = d->key_col;
  sp->payload_cols.assign(d->payload_cols, d->payload_cols + d->npayload);
  for (int c : sp->payload_cols) if (c < 0 || c >= w) return fail(ctx, GQ_ERR_INVALID_ARG, "payload column out of range");
  sp->unique = (d->flags & GQ_F_UNIQUE_KEYS) != 0;
  if (d->flags & ~(uint32_t)(GQ_F_UNIQUE_KEYS | GQ_F_DENSE_KEYS)) return fail(ctx, GQ_ERR_INVALID_ARG, "unknown gq_build_desc flags");
  sp->dense_target = (d->flags & GQ_F_DENSE_KEYS) != 0;
  if (sp->dense_target && !sp->unique) return fail(ctx, GQ_ERR_INVALID_ARG, "GQ_F_DENSE_KEYS requires GQ_F_UNIQUE_KEYS");
  sp->target_sw = join_slot_words(d->npayload);
  return GQ_OK;
}

gq_status gq_hash_build(gq_ctx* ctx, gq_table** table, void* d_ws, size_t bytes, int64_t max_build_rows,
                        const gq_batch* in, const gq_build_desc* d) {
  if (!ctx || !table || !d) return GQ_ERR_INVALID_ARG;
  gq_status st = check_batch(ctx, in);
  if (st != GQ_OK) return st;
  GqScanSpec sp;
  st = build_spec(ctx, &sp, in, d);
  if (st != GQ_OK) return st;
  gq_table* t = *table;
  if (!t && sp.dense_target) {
    DenseLayout L;
    if (!d_ws || !aligned(d_ws, 256)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad workspace");
    if (!dense_layout(d->key_min, d->key_max, max_build_rows, d->npayload, &L)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad dense key range");
    if (bytes < L.total) return fail(ctx, GQ_ERR_WORKSPACE_TOO_SMALL, "hash-build workspace too small");
    t = new gq_table();
    t->capacity = L.range; t->dense = true; t->key_min = d->key_min;
    t->npayload = d->npayload;
    for (int p = 0; p < d->npayload; ++p) t->payload_dtype[p] = row_dtype(sp, d->payload_cols[p]);
    t->flags = d->flags;
    t->max_rows = L.max_rows;
    t->dev.slots = (unsigned long long*)((char*)d_ws + L.pay_off);
    t->dev.mask = (unsigned long long)(L.range - 1);
    t->dev.header = (long long*)d_ws;
    t->dev.side = (unsigned long long*)((char*)d_ws + L.bitmap_off);
    t->dev.slot_words = d->npayload; t->dev.flags = d->flags; t->dev.base = d->key_min;
    t->keyrank = (unsigned long long*)((char*)d_ws + L.keyrank_off);
    t->rank_totals = (unsigned*)((char*)d_ws + L.totals_off);
    cudaError_t e = cudaMemsetAsync(d_ws, 0, L.bitmap_off + L.bitmap_bytes, ctx->stream);   // header + bitmap; payload rows need no init
    if (e != cudaSuccess) { delete t; return cuda_fail(ctx, e, "dense table init"); }
    { GqScanSpec c = sp; c.nrows_hint = 0; t->build_sig = signature(c) + "|" + std::to_string(d->key_min) + ":" + std::to_string(d->key_max); }
    *table = t;
  } else if (!t) {
    if (!d_ws || !aligned(d_ws, 256) || max_build_rows < 0) return fail(ctx, GQ_ERR_INVALID_ARG, "bad workspace");
    const int sw = sp.target_sw;
    const int64_t cap = join_capacity(max_build_rows, sw);
    WsLayout w = ws_layout(cap, sw, GQ_SIDE_SLOTS);
    if (bytes < w.total) return fail(ctx, GQ_ERR_WORKSPACE_TOO_SMALL, "hash-build workspace too small");
    t = new gq_table();
    t->capacity = cap;
    t->npayload = d->npayload;
    for (int p = 0; p < d->npayload; ++p) t->payload_dtype[p] = row_dtype(sp, d->payload_cols[p]);
    t->flags = d->flags;
    t->max_rows = max_build_rows;
    t->dev.slots = (unsigned long long*)((char*)d_ws + w.slots_off);
    t->dev.mask = (unsigned long long)(cap - 1);
    t->dev.header = (long long*)d_ws;
    t->dev.side = (unsigned long long*)((char*)d_ws + w.side_off);
    t->dev.shift = 64 - log2i(cap);
    t->dev.slot_words = sw;
    t->dev.flags = d->flags;
    t->dev.bshift = (sw == 1 ? 2 : sw == 2 ? 2 : 0);   // slots per 32-byte bucket: 4 / 2 / 1
    unsigned long long pat[16];
    for (int i = 0; i < 16; ++i) pat[i] = 0;
    pat[0] = GQ_EMPTY_KEY;
    cudaError_t e = PROF(ctx, "gq_k_init_table", gq_launch_init_table(ctx->stream, t->dev.slots, cap, sw, pat, t->dev.side, GQ_SIDE_SLOTS, t->dev.header, 0, ctx->num_sms));
    if (e != cudaSuccess) { delete t; return cuda_fail(ctx, e, "table init"); }
    ++ctx->launches;
    { GqScanSpec c = sp; c.nrows_hint = 0; t->build_sig = signature(c); }
    *table = t;
  } else {
    GqScanSpec c = sp; c.nrows_hint = 0;
    std::string sg = signature(c);
    if (t->dense) sg += "|" + std::to_string(d->key_min) + ":" + std::to_string(d->key_max);
    if (t->describe_only || sg != t->build_sig) return fail(ctx, GQ_ERR_INVALID_ARG, "batch schema/desc differs from the table's first batch");
    if (t->finished) return fail(ctx, GQ_ERR_INVALID_ARG, "table already finished");
  }
  GqParams P;
  memset(&P, 0, sizeof P);
  P.target = t->dev;
  return run_scan(ctx, sp, in, d->probes, &P);
}

gq_status gq_hash_build_finish(gq_ctx* ctx, gq_table* t) {
  if (!ctx || !t || t->describe_only) return GQ_ERR_INVALID_ARG;
  use_device(ctx);
  if (t->dense && !t->ranked) {   // all keys are in: rank prefix of every bitmap entry, key of every rank
    cudaError_t e = PROF(ctx, "gq_k_dense_rank(2)", gq_launch_dense_rank(ctx->stream, t->dev.side, (t->capacity + 31) / 32, t->rank_totals, t->key_min,
                                                                        t->keyrank, t->max_rows, t->dev.header, ctx->d_err));
    if (e != cudaSuccess) return cuda_fail(ctx, e, "dense table ranks");
    ctx->launches += 2;
    t->ranked = true;
  }
  if (!t->ready) {
    cudaError_t e = cudaEventCreateWithFlags(&t->ready, cudaEventDisableTiming);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaEventCreate");
  }
  cudaError_t e = cudaEventRecord(t->ready, ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaEventRecord");
  t->build_stream = ctx->stream;
  t->finished = true;
  return GQ_OK;
}

gq_status gq_table_count(gq_ctx* ctx, const gq_table* t, int64_t* d_count) {
  if (!ctx || !t || !d_count || t->describe_only) return GQ_ERR_INVALID_ARG;
  use_device(ctx);
  cudaError_t e = cudaMemcpyAsync(d_count, t->dev.header, 8, cudaMemcpyDeviceToDevice, ctx->stream);
  return e == cudaSuccess ? GQ_OK : cuda_fail(ctx, e, "gq_table_count");
}

gq_status gq_table_destroy(gq_table* t) {
  if (!t) return GQ_ERR_INVALID_ARG;
  if (t->ready) cudaEventDestroy(t->ready);
  delete t;
  return GQ_OK;
}

gq_status gq_table_describe(gq_table** out, const gq_dtype* payload_dtypes, int32_t npayload, uint32_t flags) {
  if (!out || npayload < 0 || npayload > GQ_MAX_PAYLOAD || (npayload > 0 && !payload_dtypes)) return GQ_ERR_INVALID_ARG;
  gq_table* t = new gq_table();
  t->describe_only = true;
  t->npayload = npayload;
  for (int p = 0; p < npayload; ++p) { if (!dtype_ok(payload_dtypes[p])) { delete t; return GQ_ERR_INVALID_ARG; } t->payload_dtype[p] = payload_dtypes[p]; }
  if ((flags & GQ_F_DENSE_KEYS) && !(flags & GQ_F_UNIQUE_KEYS)) { delete t; return GQ_ERR_INVALID_ARG; }
  t->flags = flags;
  t->dense = (flags & GQ_F_DENSE_KEYS) != 0;
  *out = t;
  return GQ_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ HashAggregation
namespace {

// Low-cardinality path: max_groups group cells per consumer thread in shared memory (max_groups * naggs * 8 B per
// thread); taken when at least 128 consumer threads fit beside a 3-stage ring (checked again by the plan compiler).
int lowcard_cap(int64_t max_groups, int naggs, int ndep) {
  if (ndep > 0 || max_groups < 1 || max_groups > 64 || naggs < 1) return 0;
  long long bytes = 8LL * max_groups * naggs * 128;
  return bytes <= 120 * 1024 ? (int)max_groups : 0;
}

// aggregation workspace = table workspace [+ hot list (4 KB) + heavy-hitter sample table] for keyed, non-tiny states
bool agg_has_hot_area(int64_t max_groups, int nkeys) { return nkeys > 0 && max_groups > 64; }
size_t agg_ws_bytes(int64_t cap, int sw, int64_t max_groups, int nkeys, size_t* hot_off) {
  size_t base = align_up(ws_layout(cap, sw, 1).total, 256);
  if (hot_off) *hot_off = base;
  return base + (agg_has_hot_area(max_groups, nkeys) ? GQ_HOT_LIST_BYTES + (size_t)GQ_HOT_SLOTS * 16 : 0);
}

gq_status agg_spec(gq_ctx* ctx, GqScanSpec* sp, const gq_batch* in, const gq_agg_desc* d, int key_bits[2],
                   gq_dtype key_dtype[2]) {
  gq_status st = fill_common(ctx, sp, in, d->preds, d->npred, d->probes, d->nprobes, d->exprs, d->nexpr);
  if (st != GQ_OK) return st;
  if (d->nkeys < 0 || d->nkeys > GQ_MAX_KEYS || (d->nkeys > 0 && !d->key_cols)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad key columns");
  if (d->naggs < 1 || d->naggs > GQ_MAX_AGGS || !d->aggs) return fail(ctx, GQ_ERR_INVALID_ARG, "bad aggregates");
  if (d->ndependent < 0 || (d->nkeys > 0 && d->ndependent >= d->nkeys) || (d->nkeys == 0 && d->ndependent != 0))
    return fail(ctx, GQ_ERR_INVALID_ARG, "bad ndependent");
  if (d->max_groups < 1) return fail(ctx, GQ_ERR_INVALID_ARG, "max_groups must be >= 1");
  const int w = row_width(*sp);
  sp->key_cols.assign(d->key_cols, d->key_cols + d->nkeys);
  int bits = 0;
  key_bits[0] = key_bits[1] = 0;
  for (int k = 0; k < d->nkeys; ++k) {
    if (sp->key_cols[(size_t)k] < 0 || sp->key_cols[(size_t)k] >= w) return fail(ctx, GQ_ERR_INVALID_ARG, "key column out of range");
    key_dtype[k] = row_dtype(*sp, sp->key_cols[(size_t)k]);
    if (k < d->nkeys - d->ndependent) { key_bits[k] = 8 * gq_dtype_bytes(key_dtype[k]); bits += key_bits[k]; }
  }
  if (bits > 64) return fail(ctx, GQ_ERR_UNSUPPORTED, "packed key wider than 64 bits: declare trailing keys dependent (ndependent)");
  sp->ndep = d->ndependent;
  sp->aggs.assign(d->aggs, d->aggs + d->naggs);
  for (gq_agg& a : sp->aggs) {
    if ((int)a.op < 0 || (int)a.op > (int)GQ_COUNT_STAR) return fail(ctx, GQ_ERR_INVALID_ARG, "bad aggregate op");
    // mode Final: the rows are intermediate results; a COUNT is the SUM of the partial counts in `expr`
    if ((d->flags & GQ_F_FINAL_MODE) && a.op == GQ_COUNT_STAR) a.op = GQ_SUM;
    if (a.op != GQ_COUNT_STAR && (a.expr < 0 || a.expr >= d->nexpr)) return fail(ctx, GQ_ERR_INVALID_ARG, "aggregate names a missing expression");
  }
  sp->target_sw = agg_slot_words(d->ndependent, d->naggs);
  sp->lc_cap = d->nkeys > 0 ? lowcard_cap(d->max_groups, d->naggs, d->ndependent) : 0;
  sp->lc_key_bits = bits;
  sp->consumer = d->nkeys == 0 ? GQ_C_GLOBAL : sp->lc_cap > 0 ? GQ_C_LOWCARD : GQ_C_HIGHCARD;
  // skew handling is compiled in when the group key is one plain input column (so that it can be sampled)
  bool all_unique = true;
  for (const GqProbeSpec& ps : sp->probes) all_unique = all_unique && ps.unique;
  sp->hot = sp->consumer == GQ_C_HIGHCARD && d->nkeys == 1 && d->ndependent == 0 && sp->key_cols[0] < in->ncols &&
            agg_has_hot_area(d->max_groups, d->nkeys) && all_unique;
  if (d->flags & ~(uint32_t)(GQ_F_CHECK_DEPENDENT | GQ_F_FINAL_MODE)) return fail(ctx, GQ_ERR_INVALID_ARG, "unknown gq_agg_desc flags");
  sp->check_dep = (d->flags & GQ_F_CHECK_DEPENDENT) != 0 && d->ndependent > 0;
  return GQ_OK;
}

int64_t agg_capacity(int64_t max_groups, int nkeys) { return nkeys == 0 ? 0 : table_capacity(max_groups); }

// Direct aggregation (SURVEY §8(d) note on C3): when the single hashed group key is the key column of a probe step
// into a table with unique keys, a surviving row's group IS the slot it matched, so the aggregate words live in an
// array indexed by that slot: no second hash table, no key compare, no CAS. A dependent key must be a payload of the
// same table (read back from it by the finaliser). Returns the probe step or -1.
struct DirectPlan { int step = -1; int aw = 0; int touch = -1; int dep_pay = -1; int64_t cap = 0; size_t bytes = 0; };
DirectPlan direct_plan(const GqScanSpec& sp, const gq_agg_desc* d, const gq_batch* in, bool schema_only = false) {
  DirectPlan dp;
  if (sp.consumer != GQ_C_HIGHCARD || d->nkeys - d->ndependent != 1 || d->nprobes < 1) return dp;
  for (const GqProbeSpec& ps : sp.probes) if (!ps.unique) return dp;   // rows fan out: the one-row-at-a-time code has no direct form
  int step = -1;
  for (int s = 0; s < d->nprobes; ++s)
    if (d->probes[s].key_col == d->key_cols[0] && d->probes[s].table && (d->probes[s].table->flags & GQ_F_UNIQUE_KEYS) &&
        (schema_only || !d->probes[s].table->describe_only)) step = s;
  if (step < 0) return dp;
  const gq_table* t = d->probes[step].table;
  if (d->ndependent == 1) {
    int first = in->ncols;
    for (int s = 0; s < step; ++s) first += d->probes[s].table->npayload;
    const int c = d->key_cols[1];
    if (c < first || c >= first + t->npayload) return dp;
    dp.dep_pay = c - first;
  }
  for (int i = 0; i < d->naggs; ++i) if (d->aggs[i].op == GQ_COUNT_STAR && dp.touch < 0) dp.touch = i;
  const bool hidden = dp.touch < 0;
  if (hidden) dp.touch = d->naggs;
  dp.aw = (int)align_up((size_t)(d->naggs + (hidden ? 1 : 0)), 2);
  dp.cap = t->dense ? t->max_rows : t->capacity;   // dense: one accumulator slot per build row (slot = rank of the key)
  dp.bytes = 256 + (size_t)(dp.cap + 1) * dp.aw * 8;
  // worthwhile unless the probed table is far larger than a hashed table of max_groups would be
  const size_t hashed = (size_t)agg_capacity(d->max_groups, d->nkeys) * agg_slot_words(d->ndependent, d->naggs) * 8;
  if (!schema_only && dp.bytes > 4 * hashed + (1u << 20)) return DirectPlan();
  dp.step = step;
  return dp;
}

// Radix-clustered aggregation: for a high-cardinality state whose table is far larger than L2,
// pass A (PARTITION consumer of the scan kernel) appends every surviving row to the record buffer of its key's table
// partition and pass B (gq_k_part_upsert) applies the records partition by partition, so every insert-or-update hits
// an L2-resident table slice. Worth it only for big tables and big batches; thresholds overridable for tests.
struct PartPlan { bool on = false; int npart = 0, pshift = 0, rw = 0; int64_t pcap = 0; size_t bytes = 0; std::vector<int> exprs; int src[GQ_MAX_AGGS]; };
// planner knobs (gq_set_option)
std::atomic<int64_t> g_part_min_table_mb{256}, g_part_min_rows{1 << 24}, g_hot_min_rows{GQ_HOT_MIN_ROWS}, g_psa_max_log2part{GQ_PSA_MAX_LOG2PART}, g_psa_threads{0}, g_dpart_min_acc_mb{GQ_DPART_OFF}, g_psa_cluster{2};
PartPlan part_plan(const GqScanSpec& sp, const gq_agg_desc* d, int64_t nrows) {
  PartPlan pp;
  if (sp.consumer != GQ_C_HIGHCARD) return pp;
  for (const GqProbeSpec& ps : sp.probes) if (!ps.unique) return pp;
  const int64_t cap = agg_capacity(d->max_groups, d->nkeys);
  const int sw = sp.target_sw;
  const int64_t table_bytes = cap * sw * 8;
  if (table_bytes < g_part_min_table_mb.load() * (1 << 20) || nrows < g_part_min_rows.load()) return pp;
  int64_t np = 16;
  while (np < 4096 && table_bytes / np > (4 << 20) && np * 2 <= cap / 64) np <<= 1;
  pp.npart = (int)np;
  pp.pshift = log2i(cap) - log2i(np);
  for (int a = 0; a < d->naggs; ++a) {
    pp.src[a] = -1;
    if (d->aggs[a].op == GQ_COUNT_STAR) continue;
    size_t i = 0;
    while (i < pp.exprs.size() && pp.exprs[i] != d->aggs[a].expr) ++i;
    if (i == pp.exprs.size()) pp.exprs.push_back(d->aggs[a].expr);
    pp.src[a] = 1 + d->ndependent + (int)i;
  }
  pp.rw = (int)align_up((size_t)(1 + d->ndependent + pp.exprs.size()), 4);
  pp.pcap = (nrows / np + nrows / (4 * np) + 1024 + GQ_PART_CHUNK - 1) / GQ_PART_CHUNK * GQ_PART_CHUNK;   // whole chunks
  pp.bytes = align_up((size_t)np * 8 * GQ_PART_CURSOR_STRIDE, 256) + (size_t)np * (size_t)pp.pcap * pp.rw * 8;
  pp.on = true;
  return pp;
}

// Clustered DIRECT aggregation: when the accumulator array of a direct aggregation is far larger than L2, every RED of the
// fact scan is a random DRAM read-modify-write (C3: 15.7 M of them bound the scan at 0.64 ms). The same two-pass scheme
// as above is available: pass A appends (accumulator slot, aggregate inputs) records per 4 MB slice of the array, pass B
// applies them slice by slice, so the REDs hit L2. Measured on C3 (132 MB of accumulators, 15.7 M records in 32 slices):
// scan 0.64 -> 0.57 ms but + 0.29 ms for pass B (few, fast-filling slices make the 32-record chunk refills the
// bottleneck), so it is OFF unless the planner lowers "dpart_min_acc_mb" (tests do).
PartPlan direct_part_plan(const DirectPlan& dp, const gq_agg_desc* d, int64_t nrows) {
  PartPlan pp;
  if (dp.step < 0 || dp.bytes < (size_t)g_dpart_min_acc_mb.load() * (1 << 20) || nrows < g_part_min_rows.load()) return pp;
  int shift = 0;
  while (((int64_t)dp.aw * 8 << (shift + 1)) <= (4 << 20)) ++shift;        // slots per slice: 4 MB of accumulators
  const int64_t np = (dp.cap + 1 + (1LL << shift) - 1) >> shift;
  if (np < 2 || np > 4096) return pp;
  pp.npart = (int)np; pp.pshift = shift;
  for (int a = 0; a < d->naggs; ++a) {
    pp.src[a] = -1;
    if (d->aggs[a].op == GQ_COUNT_STAR && !(d->flags & GQ_F_FINAL_MODE)) continue;
    size_t i = 0;
    while (i < pp.exprs.size() && pp.exprs[i] != d->aggs[a].expr) ++i;
    if (i == pp.exprs.size()) pp.exprs.push_back(d->aggs[a].expr);
    pp.src[a] = 1 + (int)i;
  }
  pp.rw = (int)align_up((size_t)(1 + pp.exprs.size()), 4);
  pp.pcap = (nrows / np + nrows / (4 * np) + 1024 + GQ_PART_CHUNK - 1) / GQ_PART_CHUNK * GQ_PART_CHUNK;
  pp.bytes = align_up((size_t)np * 8 * GQ_PART_CURSOR_STRIDE, 256) + (size_t)np * (size_t)pp.pcap * pp.rw * 8;
  pp.on = true;
  return pp;
}

// Partitioned shared-memory aggregation (gq_psa_kernel.cuh): the single-batch path of gq_pipeline for
// high-cardinality group-bys whose table would be far larger than L2. Pass A (SCATTER consumer) appends one record per
// surviving row to CTA-private chunks of the key's partition; pass B aggregates every partition in a shared-memory
// table and writes the dense result. No global group-by table, no global atomics on the per-row path.
struct PsaPlan {
  bool on = false;
  int npart = 0, log2npart = 0, log2sub = 0, log2slots = 0, rw = 0, threads = 512;
  bool hot = false;
  std::vector<int> exprs; int src[GQ_MAX_AGGS];
  int64_t chunks_bound = 0, merge_cap = 0;
  uint32_t seg_chunks = 0, max_items = 0;
  size_t off_zero = 0, zero_bytes = 0, off_pcount = 0, off_pfill = 0, off_pstart = 0, off_items = 0, off_itemseg = 0, off_ncta = 0,
         off_info = 0, off_plist = 0, off_merge = 0, merge_bytes = 0, off_hot = 0, off_rec = 0, bytes = 0;
};
// Pass A runs as thread-block clusters of 2 (74 clusters pack a B200's 148 SMs exactly) whose CTAs share the open chunk of
// every partition: half as many open record lines compete for L2 (DESIGN 5.4). Planner knob "psa_cluster": 1 = off.
int psa_cluster(int num_sms, int npart) { const int c = (int)g_psa_cluster.load(); return (c > 1 && num_sms >= c && npart % c == 0) ? c : 1; }
const int64_t GQ_PSA_MAX_TILE = 4096;   // upper bound of the scan kernel's tile (rows): bounds a CTA's share of the rows
PsaPlan psa_plan(const GqScanSpec& sp, const gq_agg_desc* d, int64_t nrows, int topk) {
  PsaPlan pp;
  if (sp.consumer != GQ_C_HIGHCARD || topk != 0 || d->nkeys < 1) return pp;
  for (const GqProbeSpec& ps : sp.probes) if (!ps.unique) return pp;
  const int sw = sp.target_sw;
  if ((int64_t)agg_capacity(d->max_groups, d->nkeys) * sw * 8 < g_part_min_table_mb.load() * (1 << 20) || nrows < g_part_min_rows.load()) return pp;
  int L = 6;
  auto psa_smem = [sw](int l) { return (((1LL << l) + 1) * sw + 2 * 66) * 8 + 64; };   // as gq_codegen_psa sizes it
  while (psa_smem(L + 1) <= GQ_SMEM_LIMIT) ++L;
  if (psa_smem(L) > GQ_SMEM_LIMIT) return pp;
  pp.log2slots = L;
  // groups a shared-memory table takes (gq_psa_kernel.cuh GQ_PSA_LIMIT), less 5 % for the spread of a hash partitioning
  const int64_t slots = 1LL << L;
  const int64_t limit = (slots - slots / 4) * 19 / 20;
  if (limit < 32) return pp;
  int lp = 6;                                               // 64 .. 16384 key ranges; more groups than that: the key
  while (lp < 14 && (d->max_groups + limit - 1) / limit > (1LL << lp)) ++lp;   // ranges are halved in pass B instead
  // 32 warps hide more of the table's dependent shared-memory round trips than 16 (C5 pass B 6.95 -> 5.27 ms)
  pp.threads = g_psa_threads.load() == 512 ? 512 : 1024;
  // Pass A scatters into at most 2^psa_max_log2part partitions: every (CTA, partition) pair has an open 128-byte line of
  // records, and those lines must stay in L2 until they are full, or every record becomes a random 32-byte DRAM write.
  // The remaining key-range bits are resolved in pass B: 2^log2sub sub-passes per partition, one per work item.
  pp.log2npart = (int)std::min<int64_t>(lp, std::max<int64_t>(6, g_psa_max_log2part.load()));
  pp.log2sub = std::min(3, lp - pp.log2npart);
  pp.npart = 1 << pp.log2npart;
  pp.hot = sp.hot;
  for (int a = 0; a < d->naggs; ++a) {
    pp.src[a] = -1;
    if (d->aggs[a].op == GQ_COUNT_STAR) continue;
    size_t i = 0;
    while (i < pp.exprs.size() && pp.exprs[i] != d->aggs[a].expr) ++i;
    if (i == pp.exprs.size()) pp.exprs.push_back(d->aggs[a].expr);
    pp.src[a] = 1 + d->ndependent + (int)i;
  }
  pp.rw = (int)align_up((size_t)(1 + d->ndependent + pp.exprs.size()), 4);
  // every pass-A CTA owns a private range of chunk ids: its share of the rows / 32, plus one part-filled chunk per partition
  pp.chunks_bound = nrows / GQ_PART_CHUNK + (int64_t)GQ_MAX_SMS * (pp.npart + 2 * GQ_PSA_MAX_TILE / GQ_PART_CHUNK + 2);
  if (pp.chunks_bound >= (1LL << GQ_PSA_GID_BITS) || nrows / GQ_PART_CHUNK + pp.npart + 300 >= (1LL << 20)* GQ_MAX_SMS) return pp;
  // a partition is "heavy" (cut into segments for several CTAs) when it is far above the average AND a sizeable share of all work
  pp.seg_chunks = (uint32_t)std::max<int64_t>(std::max<int64_t>(64, pp.chunks_bound / 512), 4 * pp.chunks_bound / pp.npart);
  pp.max_items = (uint32_t)((pp.npart + 2 * (pp.chunks_bound / pp.seg_chunks) + 2) << pp.log2sub);
  pp.merge_cap = table_capacity(std::min<int64_t>(std::max<int64_t>(1, d->max_groups), (pp.chunks_bound / pp.seg_chunks + 1) * limit) + GQ_HOT_MAX_SCATTER);
  size_t off = 0;
  auto take = [&off](size_t b) { size_t o = off; off += align_up(b, 256); return o; };
  pp.off_zero = take(256);                                   // [0] work cursor, [1] item count
  pp.off_pcount = take((size_t)pp.npart * 4);
  pp.off_pfill = take((size_t)pp.npart * 4 * GQ_PSA_FILL_STRIDE);   // one fill cursor per 32-byte sector
  pp.zero_bytes = off;                                       // zeroed before every run
  pp.off_pstart = take((size_t)(pp.npart + 1) * 4);
  pp.off_items = take((size_t)pp.max_items * 4);
  pp.off_itemseg = take((size_t)pp.max_items * 4);
  pp.off_ncta = take((size_t)GQ_MAX_SMS * 4);
  pp.off_info = take((size_t)pp.chunks_bound * 4);
  pp.off_plist = take((size_t)pp.chunks_bound * 4);
  pp.merge_bytes = ws_layout(pp.merge_cap, sw, 1).total;
  pp.off_merge = take(pp.merge_bytes);
  if (pp.hot) pp.off_hot = take(GQ_HOT_LIST_BYTES + (size_t)GQ_HOT_SLOTS * 16);   // hot list + heavy-hitter sample table
  pp.off_rec = take((size_t)pp.chunks_bound * GQ_PART_CHUNK * pp.rw * 8);
  pp.bytes = off;
  pp.on = true;
  return pp;
}

}  // namespace

extern "C" {

gq_status gq_hash_aggregate_workspace(int64_t max_groups, int32_t nkeys, int32_t naggs, size_t* bytes) {
  if (!bytes || max_groups < 1 || nkeys < 0 || nkeys > GQ_MAX_KEYS || naggs < 1 || naggs > GQ_MAX_AGGS) return GQ_ERR_INVALID_ARG;
  // slot words do not depend on how many keys are dependent beyond +1 word: size for the worst case (1 dependent)
  *bytes = agg_ws_bytes(agg_capacity(max_groups, nkeys), agg_slot_words(nkeys > 1 ? 1 : 0, naggs), max_groups, nkeys, nullptr);
  return GQ_OK;
}

gq_status gq_hash_aggregate_workspace_for(const gq_batch* in, const gq_agg_desc* d, size_t* bytes) {
  if (!in || !d || !bytes) return GQ_ERR_INVALID_ARG;
  gq_status st = gq_hash_aggregate_workspace(d->max_groups, d->nkeys, d->naggs, bytes);
  if (st != GQ_OK) return st;
  gq_ctx tmp;
  GqScanSpec sp;
  int kb[2]; gq_dtype kd[2] = {GQ_I64, GQ_I64};
  st = agg_spec(&tmp, &sp, in, d, kb, kd);
  if (st != GQ_OK) return st;
  DirectPlan dp = direct_plan(sp, d, in);
  if (dp.step >= 0) {
    *bytes = std::max(*bytes, dp.bytes);
    PartPlan pp = direct_part_plan(dp, d, in->nrows);
    if (pp.on) *bytes = align_up(*bytes, 256) + pp.bytes;
  } else {
    PartPlan pp = part_plan(sp, d, in->nrows);
    if (pp.on) *bytes = align_up(*bytes, 256) + pp.bytes;
  }
  return GQ_OK;
}

gq_status gq_hash_aggregate(gq_ctx* ctx, gq_aggstate** state, void* d_ws, size_t bytes, const gq_batch* in,
                            const gq_agg_desc* d) {
  if (!ctx || !state || !d) return GQ_ERR_INVALID_ARG;
  gq_status st = check_batch(ctx, in);
  if (st != GQ_OK) return st;
  GqScanSpec sp;
  int key_bits[2];
  gq_dtype key_dtype[2] = {GQ_I64, GQ_I64};
  st = agg_spec(ctx, &sp, in, d, key_bits, key_dtype);
  if (st != GQ_OK) return st;
  gq_aggstate* a = *state;
  if (!a) {
    if (!d_ws || !aligned(d_ws, 256)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad workspace");
    DirectPlan dp = direct_plan(sp, d, in);
    if (dp.step >= 0 && bytes < dp.bytes) dp = DirectPlan();   // workspace sized by the table-agnostic query: hashed path
    a = new gq_aggstate();
    a->nkeys = d->nkeys; a->ndep = d->ndependent; a->naggs = d->naggs; a->max_groups = d->max_groups;
    for (int k = 0; k < d->nkeys; ++k) { a->key_dtype[k] = key_dtype[k]; a->key_bits[k] = key_bits[k]; }
    for (int i = 0; i < d->naggs; ++i) a->agg_op[i] = d->aggs[i].op;
    unsigned long long pat[16];
    for (int i = 0; i < 16; ++i) pat[i] = 0;
    cudaError_t e;
    if (dp.step >= 0) {
      a->direct = true; a->dtab = d->probes[dp.step].table->dev; a->dcap = dp.cap; a->daw = dp.aw; a->dtouch = dp.touch;
      a->ddense = d->probes[dp.step].table->dense; a->dnpay = d->probes[dp.step].table->npayload;
      a->dkeyrank = d->probes[dp.step].table->keyrank;
      a->dep_pay = dp.dep_pay;
      a->dev.header = (long long*)d_ws;
      a->dacc = (unsigned long long*)((char*)d_ws + 256);
      for (int i = 0; i < d->naggs; ++i)
        pat[i] = d->aggs[i].op == GQ_MIN ? 0x7FFFFFFFFFFFFFFFULL : d->aggs[i].op == GQ_MAX ? 0x8000000000000000ULL : 0ULL;
      {
        PartPlan pp = direct_part_plan(dp, d, in->nrows);
        size_t hb = 0;
        gq_hash_aggregate_workspace(d->max_groups, d->nkeys, d->naggs, &hb);
        const size_t base = align_up(std::max(dp.bytes, hb), 256);   // as gq_hash_aggregate_workspace_for lays it out
        if (pp.on && bytes >= base + pp.bytes) {   // the plan-aware workspace query made room for the record buffers
          a->pcur = (unsigned long long*)((char*)d_ws + base);
          a->part = (unsigned long long*)((char*)d_ws + base + align_up((size_t)pp.npart * 8 * GQ_PART_CURSOR_STRIDE, 256));
          a->pcap = pp.pcap; a->npart = pp.npart; a->pshift = pp.pshift; a->part_rw = pp.rw; a->part_rows = in->nrows;
        }
      }
      e = PROF(ctx, "gq_k_init_table", gq_launch_init_table(ctx->stream, a->dacc, dp.cap + 1, dp.aw, pat, a->dacc, 0, a->dev.header, 0, ctx->num_sms));
    } else {
      const int64_t cap = agg_capacity(d->max_groups, d->nkeys);
      const int sw = sp.target_sw;
      WsLayout w = ws_layout(cap, sw, 1);
      size_t hot_off = 0;
      if (bytes < agg_ws_bytes(cap, sw, d->max_groups, d->nkeys, &hot_off)) {
        delete a;
        return fail(ctx, GQ_ERR_WORKSPACE_TOO_SMALL, "hash-aggregate workspace too small");
      }
      if (agg_has_hot_area(d->max_groups, d->nkeys)) {
        a->hot = (long long*)((char*)d_ws + hot_off);
        a->hot_table = (unsigned long long*)((char*)d_ws + hot_off + GQ_HOT_LIST_BYTES);
      }
      {
        PartPlan pp = part_plan(sp, d, in->nrows);
        const size_t base = align_up(agg_ws_bytes(cap, sw, d->max_groups, d->nkeys, nullptr), 256);
        if (pp.on && bytes >= base + pp.bytes) {   // the plan-aware workspace query made room for the record buffers
          a->pcur = (unsigned long long*)((char*)d_ws + base);
          a->part = (unsigned long long*)((char*)d_ws + base + align_up((size_t)pp.npart * 8 * GQ_PART_CURSOR_STRIDE, 256));
          a->pcap = pp.pcap; a->npart = pp.npart; a->pshift = pp.pshift; a->part_rw = pp.rw; a->part_rows = in->nrows;
        }
      }
      a->capacity = cap;
      a->lowcard = sp.consumer == GQ_C_LOWCARD; a->lc_cap = sp.lc_cap;
      a->dev.slots = (unsigned long long*)((char*)d_ws + w.slots_off);
      a->dev.mask = cap > 0 ? (unsigned long long)(cap - 1) : 0;
      a->dev.header = (long long*)d_ws;
      a->dev.side = (unsigned long long*)((char*)d_ws + w.side_off);
      a->dev.shift = cap > 0 ? 64 - log2i(cap) : 63;
      a->dev.slot_words = sw;
      pat[0] = GQ_EMPTY_KEY;
      a->check_dep = sp.check_dep;
      if (sp.check_dep) pat[1] = GQ_DEP_UNSET;
      for (int i = 0; i < d->naggs; ++i)
        pat[1 + d->ndependent + i] = d->aggs[i].op == GQ_MIN ? 0x7FFFFFFFFFFFFFFFULL : d->aggs[i].op == GQ_MAX ? 0x8000000000000000ULL : 0ULL;
      // a key-less aggregation has exactly one group, present even with no input rows (S9): header[1] = 1
      e = PROF(ctx, "gq_k_init_table", gq_launch_init_table(ctx->stream, a->dev.slots, cap, sw, pat, a->dev.side, 1, a->dev.header, d->nkeys == 0 ? 1 : 0, ctx->num_sms));
    }
    if (e != cudaSuccess) { delete a; return cuda_fail(ctx, e, "aggregate state init"); }
    ++ctx->launches;
    *state = a;
  }
  DirectPlan adp;
  if (a->direct) {
    DirectPlan dp = direct_plan(sp, d, in);
    adp = dp;
    if (dp.step < 0 || d->probes[dp.step].table->dev.slots != a->dtab.slots || dp.aw != a->daw)
      return fail(ctx, GQ_ERR_INVALID_ARG, "batch schema/desc differs from the state's first batch");
    sp.consumer = GQ_C_DIRECT; sp.direct_step = dp.step; sp.direct_aw = dp.aw; sp.direct_touch = dp.touch == d->naggs;
    sp.hot = false;
  }
  {
    GqScanSpec sig_sp = sp; sig_sp.nrows_hint = 0;
    const std::string sig = signature(sig_sp);
    if (a->sig.empty()) a->sig = sig;
    else if (sig != a->sig) return fail(ctx, GQ_ERR_INVALID_ARG, "batch schema/desc differs from the state's first batch");
  }
  GqParams P;
  memset(&P, 0, sizeof P);
  P.target = a->dev;
  P.acc = (long long*)(a->dev.side + 1);
  P.dacc = a->dacc;
  if (sp.hot && a->hot && in->nrows >= g_hot_min_rows.load()) {   // heavy-hitter pass over a strided sample of the key column
    int nl = 0;
    const gq_column& kc = in->cols[sp.key_cols[0]];
    cudaError_t e = PROF(ctx, "gq_k_hot_keys(5)", gq_launch_hot_keys(ctx->stream, kc.data, (int)kc.dtype, in->nrows, a->hot_table, GQ_HOT_SLOTS, GQ_HOT_SAMPLE,
                                       GQ_HOT_THRESHOLD, a->hot, GQ_HOT_MAX, ctx->num_sms, &nl));
    if (e != cudaSuccess) return cuda_fail(ctx, e, "heavy-hitter sampling");
    ctx->launches += nl;
    P.hot = a->hot;
  }
  if (a->part && a->direct && in->nrows >= g_part_min_rows.load() / 4) {
    // clustered direct aggregation: pass A appends (slot, inputs) records per slice of the accumulator array, pass B applies them
    PartPlan pp = direct_part_plan(adp, d, a->part_rows);
    if (!pp.on || pp.rw != a->part_rw || pp.npart != a->npart) return fail(ctx, GQ_ERR_INVALID_ARG, "batch schema/desc differs from the state's first batch");
    sp.part_rw = pp.rw; sp.part_exprs = pp.exprs; sp.part_states = 4096;
    P.part = a->part; P.pcur = a->pcur; P.pcap = a->pcap; P.pshift = a->pshift; P.npart = a->npart;
    cudaError_t e = cudaMemsetAsync(a->pcur, 0, (size_t)a->npart * 8 * GQ_PART_CURSOR_STRIDE, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "partition cursors");
    gq_status st2 = run_scan(ctx, sp, in, d->probes, &P);
    if (st2 != GQ_OK) return st2;
    GqPartParams pb;
    memset(&pb, 0, sizeof pb);
    pb.part = a->part; pb.pcur = a->pcur; pb.pcap = a->pcap; pb.npart = a->npart; pb.rw = a->part_rw;
    pb.slots = a->dacc; pb.mask = 0; pb.sw = a->daw; pb.ndep = 0; pb.naggs = a->naggs;
    for (int i = 0; i < a->naggs; ++i) { pb.op[i] = (int)sp.aggs[(size_t)i].op; pb.src[i] = pp.src[i]; }
    pb.direct = 1; pb.touch = sp.direct_touch ? a->naggs : -1;
    pb.err = ctx->d_err;
    e = PROF(ctx, "gq_k_part_upsert", gq_launch_part_upsert(ctx->stream, pb, ctx->num_sms));
    if (e != cudaSuccess) return cuda_fail(ctx, e, "clustered direct aggregation");
    ++ctx->launches;
    return GQ_OK;
  }
  if (a->part && !a->direct && in->nrows >= g_part_min_rows.load() / 4) {
    // radix-clustered: pass A appends records per table partition, pass B applies them partition by partition
    PartPlan pp = part_plan(sp, d, a->part_rows);
    if (!pp.on || pp.rw != a->part_rw || pp.npart != a->npart) return fail(ctx, GQ_ERR_INVALID_ARG, "batch schema/desc differs from the state's first batch");
    sp.consumer = GQ_C_PARTITION; sp.part_rw = pp.rw; sp.part_exprs = pp.exprs; sp.part_states = 4096;
    P.part = a->part; P.pcur = a->pcur; P.pcap = a->pcap; P.pshift = a->pshift; P.npart = a->npart;
    cudaError_t e = cudaMemsetAsync(a->pcur, 0, (size_t)a->npart * 8 * GQ_PART_CURSOR_STRIDE, ctx->stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "partition cursors");
    gq_status st2 = run_scan(ctx, sp, in, d->probes, &P);
    if (st2 != GQ_OK) return st2;
    GqPartParams pb;
    memset(&pb, 0, sizeof pb);
    pb.part = a->part; pb.pcur = a->pcur; pb.pcap = a->pcap; pb.npart = a->npart; pb.rw = a->part_rw;
    pb.slots = a->dev.slots; pb.mask = a->dev.mask; pb.sw = a->dev.slot_words; pb.ndep = a->ndep; pb.naggs = a->naggs;
    for (int i = 0; i < a->naggs; ++i) { pb.op[i] = (int)a->agg_op[i]; pb.src[i] = pp.src[i]; }
    pb.check_dep = a->check_dep ? 1 : 0;
    pb.err = ctx->d_err;
    e = PROF(ctx, "gq_k_part_upsert", gq_launch_part_upsert(ctx->stream, pb, ctx->num_sms));
    if (e != cudaSuccess) return cuda_fail(ctx, e, "partitioned upsert");
    ++ctx->launches;
    return GQ_OK;
  }
  return run_scan(ctx, sp, in, d->probes, &P);
}

// ---- Partial -> Final between states, group count, growth ----
static bool same_shape(const gq_aggstate* a, const gq_aggstate* b) {
  if (a->nkeys != b->nkeys || a->ndep != b->ndep || a->naggs != b->naggs || a->direct != b->direct) return false;
  for (int k = 0; k < a->nkeys; ++k) if (a->key_dtype[k] != b->key_dtype[k] || a->key_bits[k] != b->key_bits[k]) return false;
  for (int i = 0; i < a->naggs; ++i) {
    const bool sa = a->agg_op[i] == GQ_SUM || a->agg_op[i] == GQ_COUNT_STAR, sb = b->agg_op[i] == GQ_SUM || b->agg_op[i] == GQ_COUNT_STAR;
    if (sa != sb || (!sa && a->agg_op[i] != b->agg_op[i])) return false;
  }
  return true;
}
static gq_status merge_into(gq_ctx* ctx, const gq_aggstate* src, unsigned long long* dslots, unsigned long long dmask,
                            unsigned long long* dside, long long* dheader, bool check_dep) {
  int op[GQ_MAX_AGGS];
  for (int i = 0; i < src->naggs; ++i) op[i] = (int)src->agg_op[i];
  cudaError_t e = src->direct
      ? PROF(ctx, "gq_k_merge", gq_launch_merge(ctx->stream, src->dacc, src->dcap, nullptr, nullptr, dslots, 0, nullptr, nullptr, 0, 0, src->naggs, op, 0, 1,
                                                src->daw, ctx->d_err, ctx->num_sms))
      : PROF(ctx, "gq_k_merge", gq_launch_merge(ctx->stream, src->dev.slots, src->capacity, src->dev.side, src->dev.header, dslots, dmask, dside, dheader,
                                                src->dev.slot_words, src->ndep, src->naggs, op, check_dep ? 1 : 0, 0, 0, ctx->d_err, ctx->num_sms));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "state merge");
  ++ctx->launches;
  return GQ_OK;
}

gq_status gq_aggstate_merge(gq_ctx* ctx, gq_aggstate* dst, const gq_aggstate* src) {
  if (!ctx || !dst || !src || dst == src) return GQ_ERR_INVALID_ARG;
  use_device(ctx);
  if (!same_shape(dst, src)) return fail(ctx, GQ_ERR_INVALID_ARG, "states differ in keys or aggregates");
  if (dst->direct && (dst->dtab.slots != src->dtab.slots || dst->daw != src->daw || dst->dcap != src->dcap))
    return fail(ctx, GQ_ERR_INVALID_ARG, "direct-aggregation states over different join tables cannot be merged");
  if (dst->direct) return merge_into(ctx, src, dst->dacc, 0, nullptr, nullptr, false);
  return merge_into(ctx, src, dst->dev.slots, dst->dev.mask, dst->dev.side, dst->dev.header, dst->check_dep);
}

gq_status gq_aggstate_count(gq_ctx* ctx, const gq_aggstate* a, int64_t* d_count) {
  if (!ctx || !a || !d_count) return GQ_ERR_INVALID_ARG;
  use_device(ctx);
  cudaError_t e = a->direct
      ? PROF(ctx, "gq_k_count_groups", gq_launch_count_groups(ctx->stream, a->dacc, a->dcap, 0, a->dev.header, 1, a->daw, a->dtouch, (long long*)d_count, ctx->num_sms))
      : PROF(ctx, "gq_k_count_groups", gq_launch_count_groups(ctx->stream, a->dev.slots, a->capacity, a->dev.slot_words, a->dev.header, 0, 0, 0,
                                                               (long long*)d_count, ctx->num_sms));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "group count");
  ++ctx->launches;
  return GQ_OK;
}

gq_status gq_aggstate_rehash(gq_ctx* ctx, gq_aggstate* a, void* d_new_ws, size_t bytes, int64_t new_max_groups) {
  if (!ctx || !a || !d_new_ws || !aligned(d_new_ws, 256)) return GQ_ERR_INVALID_ARG;
  use_device(ctx);
  if (a->direct || a->lowcard || a->nkeys == 0) return fail(ctx, GQ_ERR_UNSUPPORTED, "only hashed high-cardinality states grow");
  if (new_max_groups <= a->max_groups) return fail(ctx, GQ_ERR_INVALID_ARG, "new_max_groups must exceed the state's");
  const int64_t cap = agg_capacity(new_max_groups, a->nkeys);
  const int sw = a->dev.slot_words;
  size_t hot_off = 0;
  if (bytes < agg_ws_bytes(cap, sw, new_max_groups, a->nkeys, &hot_off)) return fail(ctx, GQ_ERR_WORKSPACE_TOO_SMALL, "rehash workspace too small");
  WsLayout w = ws_layout(cap, sw, 1);
  GqTableDev nt = a->dev;
  nt.slots = (unsigned long long*)((char*)d_new_ws + w.slots_off);
  nt.mask = (unsigned long long)(cap - 1);
  nt.header = (long long*)d_new_ws;
  nt.side = (unsigned long long*)((char*)d_new_ws + w.side_off);
  nt.shift = 64 - log2i(cap);
  unsigned long long pat[16];
  for (int i = 0; i < 16; ++i) pat[i] = 0;
  pat[0] = GQ_EMPTY_KEY;
  if (a->check_dep) pat[1] = GQ_DEP_UNSET;
  for (int i = 0; i < a->naggs; ++i)
    pat[1 + a->ndep + i] = a->agg_op[i] == GQ_MIN ? 0x7FFFFFFFFFFFFFFFULL : a->agg_op[i] == GQ_MAX ? 0x8000000000000000ULL : 0ULL;
  cudaError_t e = PROF(ctx, "gq_k_init_table", gq_launch_init_table(ctx->stream, nt.slots, cap, sw, pat, nt.side, 1, nt.header, 0, ctx->num_sms));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "rehash table init");
  ++ctx->launches;
  gq_status st = merge_into(ctx, a, nt.slots, nt.mask, nt.side, nt.header, a->check_dep);
  if (st != GQ_OK) return st;
  a->dev = nt; a->capacity = cap; a->max_groups = new_max_groups;
  a->hot = (long long*)((char*)d_new_ws + hot_off);
  a->hot_table = (unsigned long long*)((char*)d_new_ws + hot_off + GQ_HOT_LIST_BYTES);
  a->part = nullptr; a->pcur = nullptr;   // the record buffers lived in the old workspace: later batches aggregate in one pass
  return GQ_OK;
}

size_t gq_topk_scratch_bytes(void) { return gq_topk_scratch_bytes_impl(); }

gq_status gq_hash_aggregate_finish(gq_ctx* ctx, gq_aggstate* a, void* const* out_key_cols, int64_t* const* out_agg_cols,
                                   const gq_avg* avgs, int32_t navg, double* const* out_avg_cols, int64_t out_capacity,
                                   int32_t topk, int32_t topk_agg, void* d_topk_scratch, int64_t* d_out_ngroups) {
  if (!ctx || !a || !out_agg_cols || !d_out_ngroups || out_capacity < 0) return GQ_ERR_INVALID_ARG;
  use_device(ctx);
  if (a->nkeys > 0 && !out_key_cols) return fail(ctx, GQ_ERR_INVALID_ARG, "missing key outputs");
  if (navg < 0 || navg > GQ_MAX_AGGS || (navg > 0 && (!avgs || !out_avg_cols))) return fail(ctx, GQ_ERR_INVALID_ARG, "bad avg spec");
  if (topk < 0 || topk > GQ_MAX_TOPK) return fail(ctx, GQ_ERR_UNSUPPORTED, "topk > GQ_MAX_TOPK");
  if (topk > 0 && (topk_agg < 0 || topk_agg >= a->naggs || !d_topk_scratch)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad topk arguments");
  GqFinaliseParams p;
  memset(&p, 0, sizeof p);
  p.slots = a->dev.slots; p.capacity = a->capacity; p.slot_words = a->dev.slot_words;
  p.side = a->dev.side; p.header = a->dev.header;
  if (a->direct) {
    p.direct = 1; p.capacity = a->dcap; p.dacc = a->dacc; p.daw = a->daw; p.dtouch = a->dtouch; p.dep_pay = a->dep_pay;
    p.jslots = a->dtab.slots; p.jside = a->dtab.side; p.jsw = a->dtab.slot_words;
    p.jdense = a->ddense ? 1 : 0; p.jbase = a->dtab.base; p.jnpay = a->dnpay;
    if (a->ddense) p.jside = a->dkeyrank;
  }
  p.nkeys = a->nkeys; p.ndep = a->ndep; p.naggs = a->naggs;
  for (int k = 0; k < a->nkeys; ++k) {
    if (!out_key_cols[k]) return fail(ctx, GQ_ERR_INVALID_ARG, "null key output");
    p.key_bits[k] = a->key_bits[k]; p.key_dtype[k] = a->key_dtype[k]; p.out_key[k] = out_key_cols[k];
  }
  for (int i = 0; i < a->naggs; ++i) {
    if (!out_agg_cols[i]) return fail(ctx, GQ_ERR_INVALID_ARG, "null aggregate output");
    p.out_agg[i] = (long long*)out_agg_cols[i];
  }
  p.navg = navg;
  for (int v = 0; v < navg; ++v) {
    if (avgs[v].sum_agg < 0 || avgs[v].sum_agg >= a->naggs || avgs[v].count_agg < 0 || avgs[v].count_agg >= a->naggs || !out_avg_cols[v])
      return fail(ctx, GQ_ERR_INVALID_ARG, "bad avg spec");
    p.avg_sum[v] = avgs[v].sum_agg; p.avg_cnt[v] = avgs[v].count_agg; p.out_avg[v] = out_avg_cols[v];
  }
  p.out_capacity = out_capacity; p.out_n = (long long*)d_out_ngroups; p.err = ctx->d_err;
  p.topk = topk; p.topk_agg = topk_agg; p.scratch = d_topk_scratch;
  cudaError_t e = cudaMemsetAsync(d_out_ngroups, 0, 8, ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "memset ngroups");
  int nl = 0;
  e = PROF(ctx, "gq_k_finalise/topk", gq_launch_finalise(ctx->stream, p, ctx->num_sms, &nl));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "finalise");
  ctx->launches += nl;
  return GQ_OK;
}

gq_status gq_aggstate_destroy(gq_aggstate* a) { if (!a) return GQ_ERR_INVALID_ARG; delete a; return GQ_OK; }

// ------------------------------------------------------------------------------------------------ fused pipeline
// Scratch of the finaliser fused into the scan kernel: the per-CTA partial aggregates of a key-less plan (<= 256 CTAs).
// (Low-cardinality plans merge through the context-owned table instead.)
static size_t fused_scratch_bytes(const gq_agg_desc* d) { return align_up(256 * (size_t)d->naggs * 8, 256); }

// Offsets inside a pipeline workspace: [aggregation state][top-k scratch][fused-finaliser scratch][partitioned aggregation]
struct PipeLayout { size_t aggb = 0, topk_off = 0, fused_off = 0, psa_off = 0, total = 0; PsaPlan psa; };
static gq_status pipe_layout(gq_ctx* ctx, const gq_plan* plan, GqScanSpec* sp, int kb[2], gq_dtype kd[2], PipeLayout* L) {
  gq_status st = agg_spec(ctx, sp, plan->in, &plan->agg, kb, kd);
  if (st != GQ_OK) return st;
  DirectPlan dp = direct_plan(*sp, &plan->agg, plan->in, true);
  if (dp.step < 0) L->psa = psa_plan(*sp, &plan->agg, plan->in->nrows, plan->topk);
  if (L->psa.on) st = gq_hash_aggregate_workspace(plan->agg.max_groups, plan->agg.nkeys, plan->agg.naggs, &L->aggb);   // single-pass fallback state
  else st = gq_hash_aggregate_workspace_for(plan->in, &plan->agg, &L->aggb);
  if (st != GQ_OK) return st;
  L->topk_off = align_up(L->aggb, 256);
  L->fused_off = L->topk_off + (plan->topk > 0 ? align_up(gq_topk_scratch_bytes_impl(), 256) : 0);
  L->psa_off = L->fused_off + fused_scratch_bytes(&plan->agg);
  L->total = L->psa_off + (L->psa.on ? L->psa.bytes : 0);
  return GQ_OK;
}

gq_status gq_pipeline_workspace(const gq_plan* plan, size_t* bytes) {
  if (!plan || !plan->in || !bytes) return GQ_ERR_INVALID_ARG;
  gq_ctx tmp;
  GqScanSpec sp;
  int kb[2]; gq_dtype kd[2] = {GQ_I64, GQ_I64};
  PipeLayout L;
  gq_status st = pipe_layout(&tmp, plan, &sp, kb, kd, &L);
  if (st != GQ_OK) return st;
  *bytes = L.total;
  return GQ_OK;
}

// Outputs of a finaliser that runs inside a generated kernel (fused scan finaliser, pass B of the partitioned aggregation).
static gq_status fill_final(gq_ctx* ctx, const gq_plan* plan, const int kb[2], const gq_dtype kd[2], void* const* out_key_cols,
                            int64_t* const* out_agg_cols, double* const* out_avg_cols, int64_t out_capacity, int64_t* d_out_ngroups,
                            GqFinal* F) {
  const gq_agg_desc* d = &plan->agg;
  if (!out_agg_cols || !d_out_ngroups || out_capacity < 0 || (d->nkeys > 0 && !out_key_cols)) return fail(ctx, GQ_ERR_INVALID_ARG, "missing outputs");
  if (plan->navg < 0 || plan->navg > GQ_MAX_AGGS || (plan->navg > 0 && (!plan->avgs || !out_avg_cols))) return fail(ctx, GQ_ERR_INVALID_ARG, "bad avg spec");
  F->nkeys = d->nkeys; F->navg = plan->navg;
  for (int k = 0; k < d->nkeys; ++k) {
    if (!out_key_cols[k]) return fail(ctx, GQ_ERR_INVALID_ARG, "null key output");
    F->out_key[k] = out_key_cols[k]; F->key_bits[k] = kb[k]; F->key_dtype[k] = (int)kd[k];
  }
  for (int i = 0; i < d->naggs; ++i) {
    if (!out_agg_cols[i]) return fail(ctx, GQ_ERR_INVALID_ARG, "null aggregate output");
    F->out_agg[i] = (long long*)out_agg_cols[i];
  }
  for (int v = 0; v < plan->navg; ++v) {
    if (plan->avgs[v].sum_agg < 0 || plan->avgs[v].sum_agg >= d->naggs || plan->avgs[v].count_agg < 0 ||
        plan->avgs[v].count_agg >= d->naggs || !out_avg_cols[v]) return fail(ctx, GQ_ERR_INVALID_ARG, "bad avg spec");
    F->avg_sum[v] = plan->avgs[v].sum_agg; F->avg_cnt[v] = plan->avgs[v].count_agg; F->out_avg[v] = out_avg_cols[v];
  }
  F->out_capacity = out_capacity; F->out_n = (long long*)d_out_ngroups;
  return GQ_OK;
}

// The partitioned shared-memory aggregation: zero the counters -> pass A (scan + scatter) -> directory -> pass B ->
// emit the merge table of split partitions. Five kernels, stream-ordered, no host synchronisation.
static gq_status run_psa(gq_ctx* ctx, const gq_plan* plan, GqScanSpec sp, const PsaPlan& pp, char* ws, const GqFinal& F) {
  const gq_agg_desc* d = &plan->agg;
  const gq_batch* in = plan->in;
  sp.consumer = GQ_C_SCATTER; sp.hot = pp.hot; sp.part_rw = pp.rw; sp.part_exprs = pp.exprs; sp.part_states = pp.npart;
  sp.cluster = psa_cluster(ctx->num_sms, pp.npart);
  CachedKernel* ck = nullptr;
  gq_status st = get_kernel_info(sp, &ck, &ctx->msg);
  if (st != GQ_OK) return st;
  const int64_t tile = ck->info.tile_rows;
  if (tile > GQ_PSA_MAX_TILE || ctx->num_sms > GQ_MAX_SMS) return fail(ctx, GQ_ERR_UNSUPPORTED, "internal: scatter tile/grid exceeds the workspace bound");
  const int cl = sp.cluster;
  int64_t grid = std::max<int64_t>(1, std::min<int64_t>(ctx->num_sms, in->nrows / tile));
  if (cl > 1) {                                                                    // as run_scan rounds it
    GqKernel kq;
    st = load_kernel(ctx, ck, &kq);
    if (st != GQ_OK) return st;
    grid = std::max<int64_t>(cl, std::min<int64_t>(grid, cluster_grid(ctx, kq)) / cl * cl);
  }
  // chunk ids are handed out per writer: a CTA, or a cluster whose CTAs share the partitions' open chunks
  const int64_t writers = grid / cl;
  const int64_t slab = cl * ((in->nrows / grid + 2 * tile) / GQ_PART_CHUNK) + pp.npart + 2;
  if (writers * slab > pp.chunks_bound || slab >= (1LL << 20)) return fail(ctx, GQ_ERR_UNSUPPORTED, "internal: chunk range bound");
  cudaError_t e = cudaMemsetAsync(ws + pp.off_zero, 0, pp.zero_bytes, ctx->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(F.out_n, 0, 8, ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "partitioned aggregation: memset");
  // merge table of split (heavy) partitions: ordinary group-by table protocol
  GqTableDev mt{};
  {
    WsLayout w = ws_layout(pp.merge_cap, sp.target_sw, 1);
    mt.slots = (unsigned long long*)(ws + pp.off_merge + w.slots_off);
    mt.mask = (unsigned long long)(pp.merge_cap - 1);
    mt.header = (long long*)(ws + pp.off_merge);
    mt.side = (unsigned long long*)(ws + pp.off_merge + w.side_off);
    mt.shift = 64 - log2i(pp.merge_cap);
    mt.slot_words = sp.target_sw;
    unsigned long long pat[16];
    for (int i = 0; i < 16; ++i) pat[i] = 0;
    pat[0] = GQ_EMPTY_KEY;
    if (sp.check_dep) pat[1] = GQ_DEP_UNSET;
    for (int i = 0; i < d->naggs; ++i)
      pat[1 + d->ndependent + i] = d->aggs[i].op == GQ_MIN ? 0x7FFFFFFFFFFFFFFFULL : d->aggs[i].op == GQ_MAX ? 0x8000000000000000ULL : 0ULL;
    e = PROF(ctx, "gq_k_init_table", gq_launch_init_table(ctx->stream, mt.slots, pp.merge_cap, sp.target_sw, pat, mt.side, 1, mt.header, 0, ctx->num_sms));
    if (e != cudaSuccess) return cuda_fail(ctx, e, "merge table init");
    ++ctx->launches;
  }
  auto U = [&](size_t off) { return (unsigned*)(ws + off); };
  GqParams P;
  memset(&P, 0, sizeof P);
  P.part = (unsigned long long*)(ws + pp.off_rec);
  P.pshift = 64 - pp.log2npart; P.npart = pp.npart;
  P.sc_info = U(pp.off_info); P.sc_count = U(pp.off_pcount); P.sc_ncta = U(pp.off_ncta); P.sc_slab = slab;
  e = cudaMemsetAsync(P.sc_ncta, 0, GQ_MAX_SMS * 4, ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "partitioned aggregation: memset");
  if (pp.hot && in->nrows >= g_hot_min_rows.load()) {
    // skewed batches: the most frequent keys (strided sample of the key column) are aggregated per CTA in shared memory
    // by pass A and flushed into the merge table; they never become records
    int nl = 0;
    const gq_column& kc = in->cols[sp.key_cols[0]];
    long long* hot = (long long*)(ws + pp.off_hot);
    e = PROF(ctx, "gq_k_hot_keys(5)", gq_launch_hot_keys(ctx->stream, kc.data, (int)kc.dtype, in->nrows, (unsigned long long*)(ws + pp.off_hot + GQ_HOT_LIST_BYTES), GQ_HOT_SLOTS,
                           GQ_HOT_SAMPLE, GQ_HOT_THRESHOLD_SCATTER, hot, GQ_HOT_MAX_SCATTER, ctx->num_sms, &nl));
    if (e != cudaSuccess) return cuda_fail(ctx, e, "heavy-hitter sampling");
    ctx->launches += nl;
    P.hot = hot;
    P.target = mt;
  }
  st = run_scan(ctx, sp, in, d->probes, &P);
  if (st != GQ_OK) return st;
  GqPsaDirParams dp{};
  dp.pcount = U(pp.off_pcount); dp.pstart = U(pp.off_pstart); dp.items = U(pp.off_items); dp.item_seg = U(pp.off_itemseg);
  dp.nitems = U(pp.off_zero) + 1; dp.npart = pp.npart; dp.seg_chunks = pp.seg_chunks; dp.err = ctx->d_err; dp.max_items = pp.max_items; dp.nsub = 1u << pp.log2sub;
  e = PROF(ctx, "gq_k_psa_dir", gq_launch_psa_dir(ctx->stream, dp));
  if (e == cudaSuccess) e = PROF(ctx, "gq_k_psa_fill", gq_launch_psa_fill(ctx->stream, U(pp.off_info), U(pp.off_ncta), (int)writers, slab, U(pp.off_pstart), U(pp.off_pfill), U(pp.off_plist)));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "partition directory");
  ctx->launches += 2;
  CachedKernel* pk = nullptr;
  st = get_psa_kernel_info(sp, pp.log2slots, pp.src, pp.threads, &pk, &ctx->msg);
  if (st != GQ_OK) return st;
  GqKernel kern;
  st = load_kernel(ctx, pk, &kern);
  if (st != GQ_OK) return st;
  GqPsaParams B;
  memset(&B, 0, sizeof B);
  B.rec = P.part; B.plist = U(pp.off_plist); B.pstart = U(pp.off_pstart); B.items = U(pp.off_items); B.item_seg = U(pp.off_itemseg);
  B.nitems = U(pp.off_zero) + 1; B.work = U(pp.off_zero); B.err = ctx->d_err; B.merge = mt; B.seg_chunks = pp.seg_chunks;
  B.hshift = 64 - pp.log2npart; B.log2sub = pp.log2sub; B.fin = F;
  void* args[] = {(void*)&B};
  e = PROF(ctx, "gq_psa", cudaLaunchKernel((const void*)kern.fn, dim3((unsigned)ctx->num_sms), dim3((unsigned)kern.threads), args, (size_t)kern.smem_bytes, ctx->stream));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "launch of the partitioned aggregation kernel");
  ++ctx->launches;
  // groups of split partitions: appended to the same dense output
  GqFinaliseParams fp;
  memset(&fp, 0, sizeof fp);
  fp.slots = mt.slots; fp.capacity = pp.merge_cap; fp.slot_words = sp.target_sw; fp.side = mt.side; fp.header = mt.header;
  fp.nkeys = d->nkeys; fp.ndep = d->ndependent; fp.naggs = d->naggs;
  for (int k = 0; k < d->nkeys; ++k) { fp.key_bits[k] = F.key_bits[k]; fp.key_dtype[k] = F.key_dtype[k]; fp.out_key[k] = F.out_key[k]; }
  for (int i = 0; i < d->naggs; ++i) fp.out_agg[i] = F.out_agg[i];
  fp.navg = F.navg;
  for (int v = 0; v < F.navg; ++v) { fp.avg_sum[v] = F.avg_sum[v]; fp.avg_cnt[v] = F.avg_cnt[v]; fp.out_avg[v] = F.out_avg[v]; }
  fp.out_capacity = F.out_capacity; fp.out_n = F.out_n; fp.err = ctx->d_err;
  int nl = 0;
  e = PROF(ctx, "gq_k_finalise/topk", gq_launch_finalise(ctx->stream, fp, ctx->num_sms, &nl));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "merge table finalise");
  ctx->launches += nl;
  return GQ_OK;
}

gq_status gq_pipeline(gq_ctx* ctx, const gq_plan* plan, void* d_ws, size_t bytes, void* const* out_key_cols,
                      int64_t* const* out_agg_cols, double* const* out_avg_cols, int64_t out_capacity,
                      int64_t* d_out_ngroups) {
  if (!ctx || !plan || !plan->in) return GQ_ERR_INVALID_ARG;
  gq_status st = check_batch(ctx, plan->in);
  if (st != GQ_OK) return st;
  GqScanSpec sp;
  int kb[2]; gq_dtype kd[2] = {GQ_I64, GQ_I64};
  PipeLayout L;
  st = pipe_layout(ctx, plan, &sp, kb, kd, &L);
  if (st != GQ_OK) return st;
  if (bytes < L.total) return fail(ctx, GQ_ERR_WORKSPACE_TOO_SMALL, "pipeline workspace too small");
  if (!d_ws || !aligned(d_ws, 256)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad workspace");
  const gq_agg_desc* d = &plan->agg;

  // One batch, key-less or low-cardinality, no top-k: ONE kernel — every CTA writes its partial groups, the last CTA
  // to finish merges them and emits the dense result (no table-init and no finalise launch).
  if ((sp.consumer == GQ_C_GLOBAL || sp.consumer == GQ_C_LOWCARD) && plan->topk == 0 && plan->in->nrows > 0 && ctx->num_sms <= 256) {
    sp.fused_final = true;
    GqParams P;
    memset(&P, 0, sizeof P);
    st = fill_final(ctx, plan, kb, kd, out_key_cols, out_agg_cols, out_avg_cols, out_capacity, d_out_ngroups, &P.fin);
    if (st != GQ_OK) return st;
    P.fin.part = (long long*)((char*)d_ws + L.fused_off);
    P.fin.ticket = (unsigned*)(ctx->d_err + 16);
    P.fin.gtab = (unsigned long long*)((char*)ctx->d_err + 256);
    return run_scan(ctx, sp, plan->in, d->probes, &P);
  }
  // One large batch into a group-by table far larger than L2: partitioned shared-memory aggregation
  if (L.psa.on && ctx->num_sms <= GQ_MAX_SMS) {
    GqFinal F;
    memset(&F, 0, sizeof F);
    st = fill_final(ctx, plan, kb, kd, out_key_cols, out_agg_cols, out_avg_cols, out_capacity, d_out_ngroups, &F);
    if (st != GQ_OK) return st;
    return run_psa(ctx, plan, sp, L.psa, (char*)d_ws + L.psa_off, F);
  }

  gq_aggstate* a = nullptr;
  st = gq_hash_aggregate(ctx, &a, d_ws, L.aggb, plan->in, &plan->agg);
  if (st != GQ_OK) { if (a) delete a; return st; }
  st = gq_hash_aggregate_finish(ctx, a, out_key_cols, out_agg_cols, plan->avgs, plan->navg, out_avg_cols, out_capacity,
                                plan->topk, plan->topk_agg, (char*)d_ws + L.topk_off, d_out_ngroups);
  delete a;   // host handle only; the enqueued kernels hold device pointers into the caller's workspace
  return st;
}

// ------------------------------------------------------------------------------------------------ read probe
gq_status gq_read_probe(gq_ctx* ctx, const void* d_data, size_t bytes, uint64_t* d_out) {
  if (!ctx || !d_data || !d_out || !aligned(d_data, 16) || bytes % 16) return GQ_ERR_INVALID_ARG;
  use_device(ctx);
  cudaError_t e = PROF(ctx, "gq_k_read_probe", gq_launch_read_probe(ctx->stream, d_data, bytes, (unsigned long long*)d_out, ctx->num_sms));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "read probe");
  ++ctx->launches;
  return GQ_OK;
}

// ------------------------------------------------------------------------------------------------ OrderBy / TopN
gq_status gq_order_by_workspace(int64_t nrows, size_t* bytes) {
  if (!bytes || nrows < 0 || nrows > (1LL << 31)) return GQ_ERR_INVALID_ARG;
  *bytes = gq_sort_workspace_bytes(nrows);
  return GQ_OK;
}

gq_status gq_order_by(gq_ctx* ctx, const gq_batch* in, const gq_sort_key* keys, int32_t nkeys, int64_t limit, void* d_ws, size_t bytes,
                      int64_t* d_out_index, void* const* out_cols) {
  if (!ctx) return GQ_ERR_INVALID_ARG;
  gq_status st = check_batch(ctx, in);
  if (st != GQ_OK) return st;
  if (in->nrows > (1LL << 31)) return fail(ctx, GQ_ERR_UNSUPPORTED, "gq_order_by: more than 2^31 rows");
  if (nkeys < 0 || nkeys > GQ_MAX_COLS || (nkeys > 0 && !keys)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad sort keys");
  for (int k = 0; k < nkeys; ++k)
    if (keys[k].col < 0 || keys[k].col >= in->ncols) return fail(ctx, GQ_ERR_INVALID_ARG, "sort key column out of range");
  if (!d_out_index && !out_cols) return fail(ctx, GQ_ERR_INVALID_ARG, "no outputs");
  if (!d_ws || !aligned(d_ws, 256)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad workspace");
  if (bytes < gq_sort_workspace_bytes(in->nrows)) return fail(ctx, GQ_ERR_WORKSPACE_TOO_SMALL, "order-by workspace too small");
  if (in->nrows == 0) return GQ_OK;
  int nl = 0;
  cudaError_t e = PROF(ctx, "gq_order_by", gq_launch_order_by(ctx->stream, ctx->num_sms, in, keys, nkeys, limit, (char*)d_ws,
                                                               (long long*)d_out_index, out_cols, &nl));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "order by");
  ctx->launches += nl;
  return GQ_OK;
}

// ------------------------------------------------------------------------------------------------ hash partitioning
gq_status gq_hash_partition_workspace(int32_t nparts, size_t* bytes) {
  if (!bytes || nparts < 1 || nparts > GQ_MAX_PARTITIONS) return GQ_ERR_INVALID_ARG;
  *bytes = gq_hash_partition_workspace_bytes(nparts);
  return GQ_OK;
}
gq_status gq_hash_partition(gq_ctx* ctx, const gq_batch* in, const int32_t* key_cols, int32_t nkeys, int32_t nparts, void* d_ws,
                            size_t bytes, void* const* out_cols, int64_t* d_out_row, int64_t* d_out_offsets) {
  if (!ctx) return GQ_ERR_INVALID_ARG;
  gq_status st = check_batch(ctx, in);
  if (st != GQ_OK) return st;
  if (in->nrows > (1LL << 31)) return fail(ctx, GQ_ERR_UNSUPPORTED, "gq_hash_partition: more than 2^31 rows");
  if (nparts < 1) return fail(ctx, GQ_ERR_INVALID_ARG, "gq_hash_partition: nparts < 1");
  if (nparts > GQ_MAX_PARTITIONS) return fail(ctx, GQ_ERR_UNSUPPORTED, "gq_hash_partition: more than GQ_MAX_PARTITIONS destinations");
  if (nkeys < 1 || nkeys > GQ_MAX_KEYS_HP || !key_cols) return fail(ctx, GQ_ERR_INVALID_ARG, "gq_hash_partition: 1..8 key columns");
  for (int k = 0; k < nkeys; ++k)
    if (key_cols[k] < 0 || key_cols[k] >= in->ncols) return fail(ctx, GQ_ERR_INVALID_ARG, "partition key column out of range");
  if (!out_cols || !d_out_offsets || !aligned(d_out_offsets, 8)) return fail(ctx, GQ_ERR_INVALID_ARG, "gq_hash_partition: missing outputs");
  for (int c = 0; c < in->ncols; ++c)
    if (in->nrows > 0 && (!out_cols[c] || !aligned(out_cols[c], 16))) return fail(ctx, GQ_ERR_INVALID_ARG, "output column null or not 16-byte aligned");
  if (!d_ws || !aligned(d_ws, 256)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad workspace");
  if (bytes < gq_hash_partition_workspace_bytes(nparts)) return fail(ctx, GQ_ERR_WORKSPACE_TOO_SMALL, "hash-partition workspace too small");
  if (in->nrows == 0) {
    cudaError_t e0 = cudaMemsetAsync(d_out_offsets, 0, (size_t)(nparts + 1) * 8, ctx->stream);
    return e0 == cudaSuccess ? GQ_OK : cuda_fail(ctx, e0, "hash partition");
  }
  int nl = 0;
  cudaError_t e = PROF(ctx, "gq_hash_partition", gq_launch_hash_partition(ctx->stream, ctx->num_sms, in, key_cols, nkeys, nparts, (char*)d_ws,
                                                                           out_cols, (long long*)d_out_row, (long long*)d_out_offsets, &nl));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "hash partition");
  ctx->launches += nl;
  return GQ_OK;
}

static gq_status hp_check(gq_ctx* ctx, const gq_batch* in, const int32_t* key_cols, int32_t nkeys, int32_t nparts, void* d_ws, size_t bytes) {
  gq_status st = check_batch(ctx, in);
  if (st != GQ_OK) return st;
  if (in->nrows > (1LL << 31)) return fail(ctx, GQ_ERR_UNSUPPORTED, "gq_hash_partition: more than 2^31 rows");
  if (nparts < 1) return fail(ctx, GQ_ERR_INVALID_ARG, "gq_hash_partition: nparts < 1");
  if (nparts > GQ_MAX_PARTITIONS) return fail(ctx, GQ_ERR_UNSUPPORTED, "gq_hash_partition: more than GQ_MAX_PARTITIONS destinations");
  if (nkeys < 1 || nkeys > GQ_MAX_KEYS_HP || !key_cols) return fail(ctx, GQ_ERR_INVALID_ARG, "gq_hash_partition: 1..8 key columns");
  for (int k = 0; k < nkeys; ++k)
    if (key_cols[k] < 0 || key_cols[k] >= in->ncols) return fail(ctx, GQ_ERR_INVALID_ARG, "partition key column out of range");
  if (!d_ws || !aligned(d_ws, 256)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad workspace");
  if (bytes < gq_hash_partition_workspace_bytes(nparts)) return fail(ctx, GQ_ERR_WORKSPACE_TOO_SMALL, "hash-partition workspace too small");
  return GQ_OK;
}
gq_status gq_hash_partition_count(gq_ctx* ctx, const gq_batch* in, const int32_t* key_cols, int32_t nkeys, int32_t nparts, void* d_ws,
                                  size_t bytes, int64_t* d_out_counts) {
  if (!ctx) return GQ_ERR_INVALID_ARG;
  gq_status st = hp_check(ctx, in, key_cols, nkeys, nparts, d_ws, bytes);
  if (st != GQ_OK) return st;
  if (!d_out_counts || !aligned(d_out_counts, 8)) return fail(ctx, GQ_ERR_INVALID_ARG, "gq_hash_partition_count: missing output");
  if (in->nrows == 0) {
    cudaError_t e0 = cudaMemsetAsync(d_out_counts, 0, (size_t)nparts * 8, ctx->stream);
    return e0 == cudaSuccess ? GQ_OK : cuda_fail(ctx, e0, "hash partition count");
  }
  int nl = 0;
  cudaError_t e = PROF(ctx, "gq_hash_partition_count", gq_launch_hash_partition_count(ctx->stream, ctx->num_sms, in, key_cols, nkeys, nparts,
                                                                                       (char*)d_ws, (long long*)d_out_counts, &nl));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "hash partition count");
  ctx->launches += nl;
  return GQ_OK;
}
gq_status gq_hash_partition_scatter_to(gq_ctx* ctx, const gq_batch* in, const int32_t* key_cols, int32_t nkeys, int32_t nparts, void* d_ws,
                                       size_t bytes, void* const* d_dst_cols, const int64_t* d_dst_row0) {
  if (!ctx) return GQ_ERR_INVALID_ARG;
  gq_status st = hp_check(ctx, in, key_cols, nkeys, nparts, d_ws, bytes);
  if (st != GQ_OK) return st;
  if (!d_dst_cols || !aligned(d_dst_cols, 8) || !d_dst_row0 || !aligned(d_dst_row0, 8))
    return fail(ctx, GQ_ERR_INVALID_ARG, "gq_hash_partition_scatter_to: missing destination tables");
  if (in->nrows == 0) return GQ_OK;
  int nl = 0;
  cudaError_t e = PROF(ctx, "gq_hash_partition_scatter_to", gq_launch_hash_partition_scatter_to(ctx->stream, ctx->num_sms, in, key_cols, nkeys, nparts,
                                                                                                 (char*)d_ws, d_dst_cols, (const long long*)d_dst_row0, &nl));
  if (e != cudaSuccess) return cuda_fail(ctx, e, "hash partition scatter");
  ctx->launches += nl;
  return GQ_OK;
}

// Allocation-free variant: workspace = a file-scope device array of gq_sort.cu (see there). No cudaMalloc / cudaFree, no
// event creation (the launch group is not profiled), nothing but kernel launches, one memset and one 4-byte D2D copy.
int64_t gq_order_by_static_max_rows(void) { return gq_sort_static_max_rows(); }
gq_status gq_order_by_static(gq_ctx* ctx, const gq_batch* in, const gq_sort_key* keys, int32_t nkeys, int64_t limit,
                             int64_t* d_out_index, void* const* out_cols) {
  if (!ctx) return GQ_ERR_INVALID_ARG;
  use_device(ctx);                                    // the scratch array's address is per device
  gq_status st = check_batch(ctx, in);
  if (st != GQ_OK) return st;
  if (in->nrows > gq_sort_static_max_rows())
    return fail(ctx, GQ_ERR_UNSUPPORTED, "gq_order_by_static: more than " + std::to_string(gq_sort_static_max_rows()) +
                                             " rows (the static scratch limit); use gq_order_by with a caller workspace");
  if (nkeys < 0 || nkeys > GQ_MAX_COLS || (nkeys > 0 && !keys)) return fail(ctx, GQ_ERR_INVALID_ARG, "bad sort keys");
  for (int k = 0; k < nkeys; ++k)
    if (keys[k].col < 0 || keys[k].col >= in->ncols) return fail(ctx, GQ_ERR_INVALID_ARG, "sort key column out of range");
  if (!d_out_index && !out_cols) return fail(ctx, GQ_ERR_INVALID_ARG, "no outputs");
  if (in->nrows == 0) return GQ_OK;
  int nl = 0;
  cudaError_t e = gq_launch_order_by_static(ctx->stream, ctx->num_sms, in, keys, nkeys, limit, (long long*)d_out_index, out_cols, &nl);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "order by (static scratch)");
  ctx->launches += nl;
  return GQ_OK;
}

gq_status gq_profile(gq_ctx* ctx, int32_t enable) {
  if (!ctx) return GQ_ERR_INVALID_ARG;
  ctx->prof = enable != 0;
  ctx->prof_names.clear();
  return GQ_OK;
}

int32_t gq_profile_read(gq_ctx* ctx, char* h_names, size_t names_bytes, float* h_ms, int32_t max_entries) {
  if (!ctx || !h_ms || max_entries < 0) return -1;
  use_device(ctx);
  if (cudaStreamSynchronize(ctx->stream) != cudaSuccess) return -1;
  std::string names;
  int32_t n = 0;
  for (size_t i = 0; i < ctx->prof_names.size() && n < max_entries; ++i, ++n) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, ctx->prof_ev[2 * i], ctx->prof_ev[2 * i + 1]) != cudaSuccess) ms = -1.f;
    h_ms[n] = ms;
    names += ctx->prof_names[i]; names += '\n';
  }
  if (h_names && names_bytes) { strncpy(h_names, names.c_str(), names_bytes - 1); h_names[names_bytes - 1] = 0; }
  ctx->prof_names.clear();
  return n;
}

gq_status gq_set_option(const char* h_name, int64_t value) {
  if (!h_name) return GQ_ERR_INVALID_ARG;
  const std::string n = h_name;
  if (n == "part_min_table_mb") g_part_min_table_mb = value < 0 ? 256 : value;
  else if (n == "part_min_rows") g_part_min_rows = value < 0 ? (1 << 24) : value;
  else if (n == "hot_min_rows") g_hot_min_rows = value < 0 ? GQ_HOT_MIN_ROWS : value;
  else if (n == "psa_cluster") g_psa_cluster = value == 1 ? 1 : 2;   // (clusters of 4 were measured twice: 132 co-resident CTAs, pass A 9.5 -> 10.9 ms, later 7.6 -> 8.7 ms)
  else if (n == "dpart_min_acc_mb") g_dpart_min_acc_mb = value < 0 ? GQ_DPART_OFF : value;
  else if (n == "psa_threads") g_psa_threads = (value == 512 || value == 1024) ? value : 0;
  else if (n == "psa_max_log2_partitions") g_psa_max_log2part = value < 0 ? GQ_PSA_MAX_LOG2PART : value;
  else return GQ_ERR_INVALID_ARG;
  return GQ_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ host-buffer e2e
namespace {
const int64_t GQ_HOST_CHUNK_ALIGN = 30720;   // lcm of the tile sizes the plan compiler picks
struct HostLayout { size_t agg_off, agg_bytes, topk_off, stage_off[2], stage_col_off[GQ_MAX_COLS], stage_bytes, out_off, out_key_off[2],
                    out_agg_off[GQ_MAX_AGGS], out_avg_off[GQ_MAX_AGGS], n_off, total; };
gq_status host_layout(const gq_plan* plan, int64_t chunk_rows, int64_t out_capacity, HostLayout* L) {
  // plan-aware state size for one chunk-sized batch: direct aggregation (group key = key of a probed unique table) is
  // taken exactly as in gq_pipeline, so the end-to-end path runs the same fused kernels as the device-resident one
  size_t aggb = 0;
  gq_batch shape = *plan->in;
  shape.nrows = std::min<int64_t>(plan->in->nrows, chunk_rows);
  gq_status st = gq_hash_aggregate_workspace_for(&shape, &plan->agg, &aggb);
  if (st != GQ_OK) return st;
  size_t off = 0;
  L->agg_off = 0; L->agg_bytes = aggb; off = align_up(aggb, 256);
  L->topk_off = off; off += plan->topk > 0 ? align_up(gq_topk_scratch_bytes_impl(), 256) : 0;
  size_t sb = 0;
  for (int c = 0; c < plan->in->ncols; ++c) { L->stage_col_off[c] = sb; sb += align_up((size_t)chunk_rows * gq_dtype_bytes(plan->in->cols[c].dtype), 256); }
  L->stage_bytes = sb;
  for (int b = 0; b < 2; ++b) { L->stage_off[b] = off; off += sb; }
  L->out_off = off;
  for (int k = 0; k < plan->agg.nkeys; ++k) { L->out_key_off[k] = off; off += align_up((size_t)out_capacity * 8, 256); }
  for (int a = 0; a < plan->agg.naggs; ++a) { L->out_agg_off[a] = off; off += align_up((size_t)out_capacity * 8, 256); }
  for (int v = 0; v < plan->navg; ++v) { L->out_avg_off[v] = off; off += align_up((size_t)out_capacity * 8, 256); }
  L->n_off = off; off += 256;
  L->total = off;
  return GQ_OK;
}
}  // namespace

extern "C" {

gq_status gq_pipeline_host_workspace(const gq_plan* plan, int64_t chunk_rows, size_t* bytes) {
  if (!plan || !plan->in || !bytes || chunk_rows < 1) return GQ_ERR_INVALID_ARG;
  HostLayout L;
  chunk_rows = (chunk_rows + GQ_HOST_CHUNK_ALIGN - 1) / GQ_HOST_CHUNK_ALIGN * GQ_HOST_CHUNK_ALIGN;   // same rounding as gq_pipeline_host
  // output capacity is not known here: size for max_groups rows (top-k needs only k)
  int64_t cap = plan->topk > 0 ? plan->topk : std::max<int64_t>(1, plan->agg.max_groups);
  gq_status st = host_layout(plan, chunk_rows, cap, &L);
  if (st != GQ_OK) return st;
  *bytes = L.total;
  return GQ_OK;
}

gq_status gq_pipeline_host(gq_ctx* ctx, const gq_plan* plan, int64_t chunk_rows, void* d_ws, size_t bytes,
                           void* const* h_out_key_cols, int64_t* const* h_out_agg_cols, double* const* h_out_avg_cols,
                           int64_t out_capacity, int64_t* h_out_ngroups) {
  if (!ctx || !plan || !plan->in || !d_ws || chunk_rows < 1 || !h_out_ngroups || !h_out_agg_cols) return GQ_ERR_INVALID_ARG;
  const gq_batch* in = plan->in;
  use_device(ctx);
  if (in->ncols < 1 || in->ncols > GQ_MAX_COLS) return fail(ctx, GQ_ERR_INVALID_ARG, "bad batch");
  // whole tiles of every kernel shape (1024 / 1280 / 1536 / 2048 rows) per chunk: only the last chunk has a ragged tail
  chunk_rows = (chunk_rows + GQ_HOST_CHUNK_ALIGN - 1) / GQ_HOST_CHUNK_ALIGN * GQ_HOST_CHUNK_ALIGN;
  int64_t cap = plan->topk > 0 ? plan->topk : std::max<int64_t>(1, plan->agg.max_groups);
  if (out_capacity > cap) out_capacity = cap;
  HostLayout L;
  gq_status st = host_layout(plan, chunk_rows, cap, &L);
  if (st != GQ_OK) return fail(ctx, st, "bad plan");
  if (bytes < L.total) return fail(ctx, GQ_ERR_WORKSPACE_TOO_SMALL, "host-pipeline workspace too small");
  cudaError_t e = cudaSuccess;
  if (!ctx->copy_stream) {
    e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
    for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
      e = cudaEventCreateWithFlags(&ctx->ev_copied[i], cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_consumed[i], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) return cuda_fail(ctx, e, "copy stream setup");
  }
  // the staging areas may still be in use by earlier work on the context's stream
  if (!ctx->ev_start) e = cudaEventCreateWithFlags(&ctx->ev_start, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_start, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_start, 0);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "copy stream ordering");
  char* ws = (char*)d_ws;
  gq_aggstate* a = nullptr;
  int64_t nchunks = std::max<int64_t>(1, (in->nrows + chunk_rows - 1) / chunk_rows);
  for (int64_t i = 0; i < nchunks; ++i) {
    const int b = (int)(i & 1);
    const int64_t r0 = i * chunk_rows, n = std::min<int64_t>(chunk_rows, in->nrows - r0);
    if (i >= 2) e = cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_consumed[b], 0);
    gq_column cols[GQ_MAX_COLS];
    for (int c = 0; c < in->ncols && e == cudaSuccess; ++c) {
      const int eb = gq_dtype_bytes(in->cols[c].dtype);
      cols[c].dtype = in->cols[c].dtype;
      cols[c].data = ws + L.stage_off[b] + L.stage_col_off[c];
      if (n > 0) e = cudaMemcpyAsync((void*)cols[c].data, (const char*)in->cols[c].data + (size_t)r0 * eb, (size_t)n * eb,
                                     cudaMemcpyHostToDevice, ctx->copy_stream);
    }
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_copied[b], ctx->copy_stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->stream, ctx->ev_copied[b], 0);
    if (e != cudaSuccess) { if (a) delete a; return cuda_fail(ctx, e, "chunk copy"); }
    gq_batch chunk{cols, in->ncols, std::max<int64_t>(0, n)};
    st = gq_hash_aggregate(ctx, &a, ws + L.agg_off, L.agg_bytes, &chunk, &plan->agg);
    if (st != GQ_OK) { if (a) delete a; return st; }
    e = cudaEventRecord(ctx->ev_consumed[b], ctx->stream);
    if (e != cudaSuccess) { delete a; return cuda_fail(ctx, e, "event record"); }
  }
  void* dk[2]; int64_t* da[GQ_MAX_AGGS]; double* dv[GQ_MAX_AGGS];
  for (int k = 0; k < plan->agg.nkeys; ++k) dk[k] = ws + L.out_key_off[k];
  for (int i = 0; i < plan->agg.naggs; ++i) da[i] = (int64_t*)(ws + L.out_agg_off[i]);
  for (int v = 0; v < plan->navg; ++v) dv[v] = (double*)(ws + L.out_avg_off[v]);
  st = gq_hash_aggregate_finish(ctx, a, dk, da, plan->avgs, plan->navg, dv, cap, plan->topk, plan->topk_agg,
                                ws + L.topk_off, (int64_t*)(ws + L.n_off));
  const int nkeys = a->nkeys;
  gq_dtype kd[2] = {a->key_dtype[0], a->key_dtype[1]};
  delete a;
  if (st != GQ_OK) return st;
  e = cudaMemcpyAsync(h_out_ngroups, ws + L.n_off, 8, cudaMemcpyDeviceToHost, ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "copy ngroups");
  st = gq_sync(ctx);
  if (st != GQ_OK) return st;
  const int64_t n = std::min<int64_t>(*h_out_ngroups, out_capacity);
  if (*h_out_ngroups > out_capacity) return fail(ctx, GQ_ERR_CAPACITY, "host output capacity exceeded");
  for (int k = 0; k < nkeys && e == cudaSuccess; ++k)
    e = cudaMemcpyAsync(h_out_key_cols[k], dk[k], (size_t)n * gq_dtype_bytes(kd[k]), cudaMemcpyDeviceToHost, ctx->stream);
  for (int i = 0; i < plan->agg.naggs && e == cudaSuccess; ++i)
    e = cudaMemcpyAsync(h_out_agg_cols[i], da[i], (size_t)n * 8, cudaMemcpyDeviceToHost, ctx->stream);
  for (int v = 0; v < plan->navg && e == cudaSuccess; ++v)
    e = cudaMemcpyAsync(h_out_avg_cols[v], dv[v], (size_t)n * 8, cudaMemcpyDeviceToHost, ctx->stream);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "copy results");
  return gq_sync(ctx);
}

// ------------------------------------------------------------------------------------------------ precompile
gq_status gq_set_kernel_cache_dir(const char* h_path) { gq_jit_set_cache_dir(h_path); return GQ_OK; }

static gq_status precompile(const GqScanSpec& sp, char* h_msg, size_t msg_bytes) {
  std::string msg, path;
  CachedKernel* ck = nullptr;
  gq_status st = get_kernel_info(sp, &ck, &msg);
  if (st == GQ_OK) st = gq_jit_compile_to_cache(ck->info, &path, &msg);
  if (st == GQ_OK) msg = path;
  if (h_msg && msg_bytes) { strncpy(h_msg, msg.c_str(), msg_bytes - 1); h_msg[msg_bytes - 1] = 0; }
  return st;
}

gq_status gq_precompile_pipeline(const gq_plan* plan, char* h_msg, size_t msg_bytes) {
  if (!plan || !plan->in) return GQ_ERR_INVALID_ARG;
  gq_ctx tmp;
  GqScanSpec sp;
  int kb[2]; gq_dtype kd[2];
  gq_status st = agg_spec(&tmp, &sp, plan->in, &plan->agg, kb, kd);
  if (st != GQ_OK) { if (h_msg && msg_bytes) { strncpy(h_msg, tmp.msg.c_str(), msg_bytes - 1); h_msg[msg_bytes - 1] = 0; } return st; }
  // every kernel variant this plan shape can launch: streaming (state in a global table), single-batch with the
  // finaliser fused in (key-less / low-cardinality), and direct aggregation (group key = key of a unique probe)
  if ((sp.consumer == GQ_C_GLOBAL || sp.consumer == GQ_C_LOWCARD) && plan->topk == 0) {
    GqScanSpec f = sp; f.fused_final = true;
    st = precompile(f, h_msg, msg_bytes);
    if (st != GQ_OK) return st;
  }
  {
    PartPlan pp = part_plan(sp, &plan->agg, plan->in->nrows);
    if (pp.on) {
      GqScanSpec f = sp;
      f.consumer = GQ_C_PARTITION; f.part_rw = pp.rw; f.part_exprs = pp.exprs; f.part_states = 4096;
      st = precompile(f, h_msg, msg_bytes);
      if (st != GQ_OK) return st;
    }
  }
  DirectPlan dp = direct_plan(sp, &plan->agg, plan->in, true);
  if (dp.step < 0) {
    PsaPlan pa = psa_plan(sp, &plan->agg, plan->in->nrows, plan->topk);
    if (pa.on) {
      GqScanSpec f = sp;
      f.consumer = GQ_C_SCATTER; f.hot = pa.hot; f.part_rw = pa.rw; f.part_exprs = pa.exprs; f.part_states = pa.npart;
      f.cluster = psa_cluster(GQ_DEFAULT_SMS, pa.npart);
      st = precompile(f, h_msg, msg_bytes);
      if (st != GQ_OK) return st;
      std::string msg, path;
      CachedKernel* pk = nullptr;
      st = get_psa_kernel_info(f, pa.log2slots, pa.src, pa.threads, &pk, &msg);
      if (st == GQ_OK) st = gq_jit_compile_to_cache(pk->info, &path, &msg);
      if (st != GQ_OK) { if (h_msg && msg_bytes) { strncpy(h_msg, msg.c_str(), msg_bytes - 1); h_msg[msg_bytes - 1] = 0; } return st; }
    }
  }
  if (dp.step >= 0) {
    GqScanSpec f = sp;
    f.consumer = GQ_C_DIRECT; f.direct_step = dp.step; f.direct_aw = dp.aw; f.direct_touch = dp.touch == plan->agg.naggs; f.hot = false;
    st = precompile(f, h_msg, msg_bytes);
    if (st != GQ_OK) return st;
    // the clustered variant (records per slice of the accumulator array): same row code + the append
    for (int a = 0; a < 1; ++a) {
      PartPlan pp;
      for (int i = 0; i < plan->agg.naggs; ++i) {
        if (plan->agg.aggs[i].op == GQ_COUNT_STAR && !(plan->agg.flags & GQ_F_FINAL_MODE)) continue;
        if (std::find(pp.exprs.begin(), pp.exprs.end(), plan->agg.aggs[i].expr) == pp.exprs.end()) pp.exprs.push_back(plan->agg.aggs[i].expr);
      }
      f.part_rw = (int)align_up((size_t)(1 + pp.exprs.size()), 4); f.part_exprs = pp.exprs; f.part_states = 4096;
      st = precompile(f, h_msg, msg_bytes);
      if (st != GQ_OK) return st;
    }
  }
  return precompile(sp, h_msg, msg_bytes);
}

gq_status gq_precompile_materialise(const gq_batch* in, const gq_pred* preds, int32_t npred, const gq_probe_step* probes,
                                    int32_t nprobes, const gq_expr* exprs, int32_t nexpr, char* h_msg, size_t msg_bytes) {
  if (!in || nexpr < 1) return GQ_ERR_INVALID_ARG;
  gq_ctx tmp;
  GqScanSpec sp;
  gq_status st = fill_common(&tmp, &sp, in, preds, npred, probes, nprobes, exprs, nexpr);
  if (st != GQ_OK) { if (h_msg && msg_bytes) { strncpy(h_msg, tmp.msg.c_str(), msg_bytes - 1); h_msg[msg_bytes - 1] = 0; } return st; }
  sp.consumer = GQ_C_MATERIALISE;
  return precompile(sp, h_msg, msg_bytes);
}

gq_status gq_precompile_build(const gq_batch* in, const gq_build_desc* d, char* h_msg, size_t msg_bytes) {
  if (!in || !d) return GQ_ERR_INVALID_ARG;
  gq_ctx tmp;
  GqScanSpec sp;
  gq_status st = build_spec(&tmp, &sp, in, d);
  if (st != GQ_OK) { if (h_msg && msg_bytes) { strncpy(h_msg, tmp.msg.c_str(), msg_bytes - 1); h_msg[msg_bytes - 1] = 0; } return st; }
  return precompile(sp, h_msg, msg_bytes);
}

}  // extern "C"
