// gq_internal.h — host-side internals of libgq.so (not part of the ABI).
#ifndef GQ_INTERNAL_H
#define GQ_INTERNAL_H
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "../../include/gq.h"

#define GQ_EMPTY_KEY 0x8000000000000000ULL
#define GQ_MAXCOL 16
#define GQ_MAXK 48
#define GQ_MAXOUT 12
#define GQ_SMEM_LIMIT 232448   // 227 KB opt-in dynamic shared memory per CTA on sm_100
#define GQ_DEFAULT_SMS 148     // B200; used only when a plan is compiled ahead of time without a device attached
#define GQ_GTAB_SLOTS 64        // merge table of the fused low-cardinality finaliser: 64 slots of 16 words {state, key, aggregates}
#define GQ_GTAB_BYTES (256 + GQ_GTAB_SLOTS * 128)
#define GQ_DEP_UNSET 0x8000000000000001ULL   // dependent-key word of a slot nobody has stored yet (GQ_F_CHECK_DEPENDENT)

enum { GQ_C_GLOBAL = 0, GQ_C_LOWCARD = 1, GQ_C_HIGHCARD = 2, GQ_C_BUILD = 3, GQ_C_MATERIALISE = 4, GQ_C_DIRECT = 5, GQ_C_PARTITION = 6, GQ_C_SCATTER = 7 };

// ---- device-visible structs: layouts must match gq_skeleton.cuh ----
struct GqTableDev {
  unsigned long long* slots;
  unsigned long long mask;
  long long* header;
  unsigned long long* side;
  int shift;
  int slot_words;
  unsigned flags;
  unsigned bshift;             // log2(slots per 32-byte bucket) for join tables, 0 for aggregation tables
  long long base;              // direct-address (GQ_F_DENSE_KEYS) tables: key_min; slots = payload rows, side = bitmap,
                               // mask = range size - 1
};
struct GqFinal {
  long long* part;
  unsigned* ticket;
  unsigned long long* gtab;
  void* out_key[2];
  long long* out_agg[8];
  double* out_avg[8];
  int avg_sum[8], avg_cnt[8];
  int navg, nkeys;
  int key_bits[2], key_dtype[2];
  long long out_capacity;
  long long* out_n;
};
struct GqParams {
  const void* col[GQ_MAXCOL];
  long long nrows;
  long long k[GQ_MAXK];
  GqTableDev probe[4];
  GqTableDev target;
  long long* acc;
  long long* out[GQ_MAXOUT];
  long long out_capacity;
  long long* out_count;
  const long long* hot;        // HIGHCARD: hot list of this batch (hot[0] = count, hot[32..] = keys) or null
  int* err;
  int pad;
  unsigned long long* dacc;    // DIRECT: aggregate words indexed by slot of the probed unique table
  unsigned long long* part;    // PARTITION: record buffers
  unsigned long long* pcur;    // PARTITION: append cursors
  long long pcap;
  long long pshift;
  long long npart;
  unsigned* sc_info;           // SCATTER (pass A of the partitioned shared-memory aggregation): see gq_skeleton.cuh
  unsigned* sc_count;
  unsigned* sc_ncta;
  long long sc_slab;
  GqFinal fin;
};

// ---- handles ----
struct gq_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  int* d_err = nullptr;        // sticky device error; d_err + 16 = ticket counter of the fused finaliser;
                               // (char*)d_err + 256 = merge table of the fused low-cardinality finaliser (GQ_GTAB_BYTES)
  int* h_err = nullptr;        // pinned mirror
  int num_sms = GQ_DEFAULT_SMS;
  int last_cuda = 0;
  int64_t launches = 0;
  std::string msg;
  bool prof = false;           // gq_profile: every kernel launch group is bracketed by a pair of events
  std::vector<cudaEvent_t> prof_ev;      //   2 events per recorded group (reused across reads)
  std::vector<std::string> prof_names;   //   names of the groups recorded since the last gq_profile_read
  cudaStream_t copy_stream = nullptr;   // gq_pipeline_host: H2D copies overlap the scan of the previous chunk
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_consumed[2] = {nullptr, nullptr}, ev_start = nullptr;
};

struct gq_table {
  bool describe_only = false;
  GqTableDev dev{};
  int64_t capacity = 0;
  int npayload = 0;
  gq_dtype payload_dtype[GQ_MAX_PAYLOAD] = {GQ_I64, GQ_I64, GQ_I64};
  uint32_t flags = 0;
  int64_t max_rows = 0;
  bool dense = false;          // GQ_F_DENSE_KEYS: direct-address table over [key_min, key_min + capacity)
  int64_t key_min = 0;
  unsigned long long* keyrank = nullptr;   //   key of every rank (max_rows entries), filled by gq_hash_build_finish
  unsigned* rank_totals = nullptr;         //   scratch of the rank kernels
  bool ranked = false;
  std::string build_sig;       // shape signature of the first batch (later batches must match)
  cudaEvent_t ready = nullptr; // recorded by gq_hash_build_finish
  cudaStream_t build_stream = nullptr;
  bool finished = false;
};

struct gq_aggstate {
  GqTableDev dev{};
  int64_t capacity = 0;        // 0 when nkeys == 0
  int nkeys = 0, ndep = 0, naggs = 0;
  gq_dtype key_dtype[GQ_MAX_KEYS] = {GQ_I64, GQ_I64};
  int key_bits[GQ_MAX_KEYS] = {64, 0};  // packed widths (0 for a dependent key)
  gq_aggop agg_op[GQ_MAX_AGGS] = {};
  int64_t max_groups = 0;
  bool lowcard = false;
  int lc_cap = 0;
  bool check_dep = false;      // GQ_F_CHECK_DEPENDENT
  bool direct = false;         // aggregate words indexed by the slot of a probed unique table (no keys stored)
  GqTableDev dtab{};           //   that table
  bool ddense = false; int dnpay = 0;   //   ... is a direct-address table with dnpay payload words per row
  const unsigned long long* dkeyrank = nullptr;   //   ... its key-of-rank array (accumulator slot = rank of the key)
  int64_t dcap = 0;            //   its capacity (the accumulator array has dcap + 1 slots: the last is the side entry)
  int daw = 0, dtouch = -1, dep_pay = -1;   // words per accumulator slot, word that marks a touched slot, payload = dep key
  unsigned long long* dacc = nullptr;
  unsigned long long* part = nullptr;  // radix-clustered mode: record buffers and cursors (in the workspace)
  unsigned long long* pcur = nullptr;
  int64_t pcap = 0; int npart = 0, pshift = 0, part_rw = 0;
  int64_t part_rows = 0;               //   rows the buffers were sized for
  long long* hot = nullptr;            // hot list (in the workspace)
  unsigned long long* hot_table = nullptr;
  std::string sig;
};

// ---- normalised plan of one fused scan kernel ----
struct GqProbeSpec {
  int key_col;                 // index into the row (input columns, then payloads of earlier probes)
  int npayload;
  gq_dtype pay_dtype[GQ_MAX_PAYLOAD];
  bool unique;
  bool dense;                  // direct-address table (GQ_F_DENSE_KEYS)
  int slot_words;
};
struct GqScanSpec {
  std::vector<gq_dtype> in_dtype;                 // batch schema
  std::vector<gq_pred> preds;
  std::vector<GqProbeSpec> probes;
  std::vector<std::vector<gq_xtok>> exprs;
  int consumer = GQ_C_GLOBAL;
  std::vector<int> key_cols;                      // LOWCARD / HIGHCARD
  int ndep = 0;
  std::vector<gq_agg> aggs;
  int lc_cap = 0;                                 // LOWCARD: number of group cells (= max_groups)
  int lc_key_bits = 0;                            // LOWCARD: packed key width
  bool fused_final = false;                       // LOWCARD / GLOBAL: finaliser fused into the scan kernel
  int direct_step = -1;                           // DIRECT: probe step whose matched slot is the group
  int direct_aw = 0;                              // DIRECT: words per accumulator slot
  bool direct_touch = false;                      // DIRECT: hidden COUNT word marks touched slots
  int part_states = 0;                            // PARTITION / SCATTER: partition state words in shared memory
  int part_rw = 0;                                // PARTITION / SCATTER: words per record (multiple of 4)
  std::vector<int> part_exprs;                    // PARTITION: expressions stored in a record, in word order
  int target_sw = 0;                              // slot words of the target table
  int build_key_col = 0;                          // BUILD
  std::vector<int> payload_cols;
  bool unique = false;
  bool dense_target = false;                      // BUILD into a direct-address table
  bool hot = false;                               // HIGHCARD: per-CTA shared-memory aggregation of hot keys
  bool check_dep = false;                         // GQ_F_CHECK_DEPENDENT: every row verifies the dependent key
  int cluster = 1;                                // SCATTER: CTAs per thread-block cluster sharing the partitions' open chunks
  int num_sms = GQ_DEFAULT_SMS;                   // tiling heuristics: SM count of the context's device
  int64_t nrows_hint = 0;                         // tiling heuristic only
};

struct GqKernelInfo {
  std::string entry = "gq_scan";   // kernel name
  std::string source;          // full translation unit
  std::string hash;            // 16 hex digits of the source hash
  int threads = 0;             // GQ_NT + 32
  int smem_bytes = 0;
  int tile_rows = 0;
  int cluster = 1;             // thread-block cluster size the kernel must be launched with
  std::vector<int> cols;       // compacted column list: original input column index per kernel column
  std::vector<long long> consts;  // values for GqParams::k
};

// gq_codegen.cpp
gq_status gq_codegen(const GqScanSpec& spec, GqKernelInfo* out, std::string* msg);
gq_status gq_codegen_psa(const GqScanSpec& spec, int log2slots, const int* src, int threads, GqKernelInfo* out, std::string* msg);
int gq_dtype_bytes(gq_dtype t);
// gq_jit.cpp
struct GqKernel { cudaKernel_t fn = nullptr; int threads = 0; int smem_bytes = 0; int tile_rows = 0; int cluster = 1; };
gq_status gq_jit_compile_to_cache(const GqKernelInfo& info, std::string* cubin_path, std::string* msg);
gq_status gq_jit_get(const GqKernelInfo& info, int device, GqKernel* out, std::string* msg, int* cuda_err);
void gq_jit_set_cache_dir(const char* path);
// gq_static.cu
struct GqFinaliseParams {
  const unsigned long long* slots; long long capacity; int slot_words;
  const unsigned long long* side; const long long* header;
  // direct mode: groups = touched accumulator slots; keys / dependent key come from the join table
  int direct; const unsigned long long* dacc; int daw, dtouch, dep_pay;
  const unsigned long long* jslots; const unsigned long long* jside; int jsw;
  int jdense; long long jbase; int jnpay;        // direct-address join table: key = jbase + i, payload row i of jnpay words
  int nkeys, ndep, naggs;
  int key_bits[2]; int key_dtype[2];
  void* out_key[2]; long long* out_agg[GQ_MAX_AGGS];
  int navg; int avg_sum[GQ_MAX_AGGS]; int avg_cnt[GQ_MAX_AGGS]; double* out_avg[GQ_MAX_AGGS];
  long long out_capacity; long long* out_n; int* err;
  int topk, topk_agg; void* scratch;
};
cudaError_t gq_launch_init_table(cudaStream_t s, unsigned long long* slots, long long nslots, int slot_words,
                                 const unsigned long long* pattern, unsigned long long* side, long long nside,
                                 long long* header, long long header1, int num_sms);
cudaError_t gq_launch_finalise(cudaStream_t s, const GqFinaliseParams& p, int num_sms, int* nlaunches);
cudaError_t gq_launch_read_probe(cudaStream_t s, const void* data, size_t bytes, unsigned long long* out, int num_sms);
#define GQ_PART_CHUNK 32            // records per CTA-private append chunk (cursors count chunks)
#define GQ_PART_CURSOR_STRIDE 16   // one append cursor per 128-byte line: atomics to one line serialise at L2
struct GqPartParams {
  const unsigned long long* part; const unsigned long long* pcur; long long pcap; int npart; int rw;
  unsigned long long* slots; unsigned long long mask; int sw; int ndep; int naggs;
  int op[GQ_MAX_AGGS]; int src[GQ_MAX_AGGS];   // src = record word of the aggregate's input, -1 = COUNT(*)
  int check_dep;
  int direct, touch;   // direct: record word 0 = accumulator slot of `slots` (sw words per slot, aggregate a at word a); touch = hidden COUNT word or -1
  int* err;
};
cudaError_t gq_launch_part_upsert(cudaStream_t s, const GqPartParams& p, int num_sms);
cudaError_t gq_launch_merge(cudaStream_t s, const unsigned long long* sslots, long long scap, const unsigned long long* sside, const long long* sheader,
                            unsigned long long* dslots, unsigned long long dmask, unsigned long long* dside, long long* dheader, int sw, int ndep,
                            int naggs, const int* op, int check_dep, int direct, int daw, int* err, int num_sms);
cudaError_t gq_launch_count_groups(cudaStream_t s, const unsigned long long* slots, long long cap, int sw, const long long* header, int direct, int daw,
                                   int dtouch, long long* out, int num_sms);
cudaError_t gq_launch_dense_rank(cudaStream_t s, unsigned long long* entries, long long nwords, unsigned* totals, long long base,
                                 unsigned long long* keyrank, long long max_rows, long long* header, int* err);
#define GQ_DENSE_RANK_BLOCK 1024         // bitmap entries per CTA of the rank kernels
size_t gq_topk_scratch_bytes_impl();
// gq_sort.cu
size_t gq_sort_workspace_bytes(long long nrows);
cudaError_t gq_launch_order_by(cudaStream_t s, int num_sms, const gq_batch* in, const gq_sort_key* keys, int nkeys, long long limit,
                               char* ws, long long* out_index, void* const* out_cols, int* nlaunches);
#define GQ_MAX_KEYS_HP 8                        // key columns of gq_hash_partition
size_t gq_hash_partition_workspace_bytes(int nparts);
cudaError_t gq_launch_hash_partition(cudaStream_t s, int num_sms, const gq_batch* in, const int* key_cols, int nkeys, int nparts, char* ws,
                                     void* const* out_cols, long long* out_row, long long* out_offsets, int* nlaunches);
cudaError_t gq_launch_hash_partition_count(cudaStream_t s, int num_sms, const gq_batch* in, const int* key_cols, int nkeys, int nparts, char* ws,
                                           long long* counts, int* nlaunches);
cudaError_t gq_launch_hash_partition_scatter_to(cudaStream_t s, int num_sms, const gq_batch* in, const int* key_cols, int nkeys, int nparts,
                                                char* ws, void* const* d_dst, const long long* d_row0, int* nlaunches);
#define GQ_ORDER_BY_STATIC_MAX_ROWS (1 << 17)   // rows gq_order_by_static takes (its scratch is a 4.2 MB file-scope device array)
long long gq_sort_static_max_rows();
cudaError_t gq_launch_order_by_static(cudaStream_t s, int num_sms, const gq_batch* in, const gq_sort_key* keys, int nkeys, long long limit,
                                      long long* out_index, void* const* out_cols, int* nlaunches);
cudaError_t gq_launch_hot_keys(cudaStream_t s, const void* keycol, int dtype, long long nrows, unsigned long long* table,
                               long long nslots, long long nsample, unsigned long long threshold, long long* hot,
                               int max_hot, int num_sms, int* nlaunches);
// ---- partitioned shared-memory aggregation (gq_psa_kernel.cuh, gq_psa.cu) ----
#define GQ_MAX_SMS 160               // workspace sizing bound for the per-CTA chunk ranges of pass A
#define GQ_DPART_OFF (1LL << 40)      // accumulator arrays smaller than this many MB are never clustered: off by default
#define GQ_PSA_MAX_LOG2PART 14        // default cap on pass-A partitions (planner knob "psa_max_log2_partitions")
#define GQ_PSA_GID_BITS 26           // directory entry = chunk id | records used << 26
struct GqPsaParams {                 // must match gq_psa_kernel.cuh
  const unsigned long long* rec; const unsigned* plist; const unsigned* pstart; const unsigned* items; const unsigned* item_seg;
  const unsigned* nitems; unsigned* work; int* err; GqTableDev merge; unsigned seg_chunks; int hshift; int log2sub; int pad; GqFinal fin;
};
struct GqPsaDirParams {
  const unsigned* pcount; unsigned* pstart; unsigned* items; unsigned* item_seg; unsigned* nitems; int npart; unsigned seg_chunks;
  int* err; unsigned max_items; unsigned nsub;
};
cudaError_t gq_launch_psa_dir(cudaStream_t s, const GqPsaDirParams& p);
#define GQ_PSA_FILL_STRIDE 8   // words between the fill cursors of two partitions (atomics on one L2 sector serialise)
cudaError_t gq_launch_psa_fill(cudaStream_t s, const unsigned* info, const unsigned* ncta, int nctas, long long slab,
                               const unsigned* pstart, unsigned* pfill, unsigned* plist);
#define GQ_HOT_MAX 256               // hot keys per batch of the global-table paths (shared set of 512 positions per CTA)
#define GQ_HOT_MAX_SCATTER 1536      // ... of pass A of the partitioned aggregation (2048 positions, when they fit shared memory)
#define GQ_HOT_LIST_BYTES 16384      // hot list: 32 header words + keys
#define GQ_HOT_SAMPLE (1LL << 19)    // sampled rows
#define GQ_HOT_SLOTS (1LL << 20)     // (key,count) sample table slots (16 B each)
#define GQ_HOT_THRESHOLD 128         // sample count that makes a key hot (share >= 2^-12): global-table paths
#define GQ_HOT_THRESHOLD_SCATTER 16  // ... pass A: every row kept out of the record stream pays (share >= 2^-15)
#define GQ_HOT_MIN_ROWS (1LL << 22)  // batches smaller than this skip the heavy-hitter pass
#endif
