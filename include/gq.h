/* gq.h — C ABI of the B200-native columnar query hot path (libgq.so).
 *
 * Scope (BASELINE.json north_star): the work the paper's cuDF operators do once data is in GPU
 * memory — FilterProject -> HashBuild/HashProbe (inner equi-join) -> HashAggregation over device-resident column
 * batches ("Accelerating Presto with GPUs", §3.2; operator model lines 112-116, 122-127).
 *
 * Model, as the paper states it:
 *   - operators consume BATCHES of rows held as columns in device memory, together with the CUDA stream that orders
 *     work on them (CudfVector = table + stream); a call only ENQUEUES work on the context's stream and
 *     returns — "GPU operators return immediately ... without blocking";
 *   - HashBuild consumes its whole input before HashProbe starts; streams are synchronised only at such pipeline
 *     boundaries;
 *   - HashAggregation accumulates over many input batches, then emits; here the state is a true
 *     streaming hash table (no concatenate-and-reaggregate work-around);
 *   - expressions are compiled at plan-creation time into fused code: every distinct plan shape
 *     is translated once into one fused sm_100a kernel (filter + probes + projection + consumer), cached by shape;
 *   - running out of (table) memory is an error, never a spill or a silent partial result.
 *
 * Conventions
 *   Pointers   : every `data`, output column, workspace and count pointer is a DEVICE pointer unless its name starts
 *                with `h_` or the doc says HOST. Descriptor structs and the arrays they point to are HOST memory and
 *                are read during the call only.
 *   Ownership  : the caller owns all columns, outputs and workspaces and must keep them alive until the enqueued work
 *                has completed on the context's stream. The library owns only small host handles and the context's
 *                few KB of device scratch (sticky error, ticket and merge table of the fused finalisers). No call
 *                allocates or frees device memory after gq_create.
 *   Alignment  : column and output pointers 16-byte aligned; workspaces 256-byte aligned.
 *   Types      : signed int8 / int32 / int64 columns, no NULLs, no strings, no floating point input.
 *                All arithmetic is wrapping two's-complement int64; aggregates and COUNT are int64.
 *   Order      : row order of multi-row outputs and group order are unspecified (SQL gives none); top-k output is
 *                ordered (aggregate descending, key ascending).
 *   Errors     : host-detectable problems return at once with nothing enqueued. Device-detected problems (table or
 *                output capacity exceeded, duplicate key under GQ_F_UNIQUE_KEYS) set a sticky flag in device memory;
 *                later kernels of that context become no-ops; gq_sync() returns the code.
 *   Threads    : one context = one stream; distinct contexts may be used concurrently (Fig. 3).
 */
#ifndef GQ_H
#define GQ_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  GQ_OK = 0,
  GQ_ERR_INVALID_ARG = 1,          /* null pointer, bad dtype/index, misaligned pointer, malformed expression */
  GQ_ERR_UNSUPPORTED = 2,          /* valid request outside the implemented envelope (limits below) */
  GQ_ERR_CAPACITY = 3,             /* hash table / output buffer full (device-detected, sticky) */
  GQ_ERR_WORKSPACE_TOO_SMALL = 4,
  GQ_ERR_CUDA = 5,                 /* CUDA runtime error: see gq_last_cuda_error */
  GQ_ERR_DUPLICATE_KEY = 6,        /* GQ_F_UNIQUE_KEYS asserted but a duplicate build key was seen (sticky) */
  GQ_ERR_COMPILE = 7,              /* plan-time kernel compilation failed: see gq_last_message */
  GQ_ERR_DEPENDENT_KEY = 8,        /* GQ_F_CHECK_DEPENDENT: a key declared dependent took two values in one group (sticky) */
  GQ_ERR_KEY_RANGE = 9             /* GQ_F_DENSE_KEYS: a build key outside [key_min, key_max] was seen (sticky) */
} gq_status;

typedef enum { GQ_I8 = 1, GQ_I32 = 2, GQ_I64 = 3 } gq_dtype;
typedef struct { const void* data; gq_dtype dtype; } gq_column;                 /* DEVICE pointer, borrowed */
typedef struct { const gq_column* cols; int32_t ncols; int64_t nrows; } gq_batch; /* one batch of rows (SoA) */

/* Filter = AND of predicates `col <op> const` on INPUT columns; npred == 0 => every row passes. One-sided
 * operators compare with `lo`. */
typedef enum { GQ_LT = 0, GQ_LE, GQ_GT, GQ_GE, GQ_EQ, GQ_NE, GQ_RANGE_CO /* lo<=x<hi */, GQ_RANGE_CC /* lo<=x<=hi */ } gq_cmp;
typedef struct { int32_t col; gq_cmp op; int64_t lo, hi; } gq_pred;

/* Projection = postfix program over the row's columns; int64 wrapping + - *. `arg` = column index for GQ_X_COL,
 * literal for GQ_X_CONST. Column indices >= batch.ncols name payload columns appended by probe steps, in order. */
typedef enum { GQ_X_COL = 0, GQ_X_CONST, GQ_X_ADD, GQ_X_SUB, GQ_X_MUL } gq_xop;
typedef struct { gq_xop op; int64_t arg; } gq_xtok;
typedef struct { const gq_xtok* toks; int32_t ntoks; } gq_expr;

typedef enum { GQ_SUM = 0, GQ_MIN, GQ_MAX, GQ_COUNT_STAR } gq_aggop;
typedef struct { gq_aggop op; int32_t expr; /* index into exprs[]; ignored for COUNT_STAR */ } gq_agg;

enum {
  GQ_F_UNIQUE_KEYS = 1u << 0,      /* gq_build_desc: caller asserts unique build keys; VERIFIED on device, never trusted */
  GQ_F_CHECK_DEPENDENT = 1u << 1,  /* gq_agg_desc: debug check of `ndependent`: every row compares its
                                      dependent key with the one stored for its group; a mismatch sets the sticky
                                      GQ_ERR_DEPENDENT_KEY instead of silently merging two groups */
  GQ_F_FINAL_MODE = 1u << 3,       /* gq_agg_desc: aggregation mode Final ("aggregation modes"): the input rows
                                      are INTERMEDIATE results — the output rows of earlier (Partial) aggregations over the
                                      same keys and aggregates, e.g. gathered from several streams or workers. SUM / MIN /
                                      MAX combine the partial values; a GQ_COUNT_STAR aggregate names through `expr` the
                                      expression that holds the partial counts and SUMS them. Mode Partial needs no flag:
                                      its output (without derived AVG columns) is the intermediate form */
  GQ_F_DENSE_KEYS = 1u << 2        /* gq_build_desc: the planner knows (column min/max statistics) that every build key
                                      lies in [key_min, key_max] and the range is not much larger than the row count:
                                      the table becomes a DIRECT-ADDRESS table — a membership bitmap plus a payload
                                      array indexed by key - key_min; no hashing, no probing, a probe costs one 8-byte
                                      load from an L2-resident bitmap (which also yields the key's rank among the build
                                      keys: the slot index of direct aggregation) ("the query planner should choose the
                                      operator implementation based on ... the expected input"). Requires
                                      GQ_F_UNIQUE_KEYS. VERIFIED on device: a key outside the range sets the sticky
                                      GQ_ERR_KEY_RANGE at once, a repeated key GQ_ERR_DUPLICATE_KEY at
                                      gq_hash_build_finish (fewer member keys than rows inserted) */
};
enum { GQ_MAX_PREDS = 16, GQ_MAX_TOKS = 32, GQ_MAX_EXPRS = 8, GQ_MAX_AGGS = 8, GQ_MAX_PROBES = 4, GQ_MAX_PAYLOAD = 3,
       GQ_MAX_KEYS = 2, GQ_MAX_COLS = 32, GQ_MAX_TOPK = 32, GQ_SIDE_SLOTS = 64 };

typedef struct gq_ctx gq_ctx;           /* device + stream + sticky error */
typedef struct gq_table gq_table;       /* join hash table (host handle; storage in caller's workspace) */
typedef struct gq_aggstate gq_aggstate; /* group-by hash table (host handle; storage in caller's workspace) */

/* ---- context ------------------------------------------------------------------------------------------------- */
/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream), 0 = legacy default stream. */
gq_status gq_create(gq_ctx** out, int device, void* cuda_stream);
/* gq_create allocates and gq_destroy frees a small device block (error word, merge table) and a pinned host word: like any
   cudaMalloc / cudaFree they must not run while a stream of the process is being captured into a CUDA graph. Every other
   call only enqueues work on the context's stream and can be captured. */
gq_status gq_destroy(gq_ctx*);
/* Blocks the HOST until the stream is idle (the pipeline boundary); returns the sticky device error. */
gq_status gq_sync(gq_ctx*);
/* Clears the sticky device error (enqueued on the stream). */
gq_status gq_clear_error(gq_ctx*);
const char* gq_status_str(gq_status);
int gq_last_cuda_error(gq_ctx*);                 /* last cudaError_t seen by this context */
const char* gq_last_message(gq_ctx*);            /* HOST string: last validation / compile diagnostic */
/* Number of kernels this context has launched since creation (bench.py's gpu_launches). */
int64_t gq_launch_count(gq_ctx*);

/* ---- FilterProject, standalone and materialising ----------------------- */
/* out_cols[e] : int64 column for expression e, capacity >= in->nrows. *d_out_count (DEVICE int64) += rows written,
 * so the caller zeroes it before the first batch. Output row order unspecified. */
gq_status gq_filter_project(gq_ctx*, const gq_batch* in, const gq_pred* preds, int32_t npred,
                            const gq_expr* exprs, int32_t nexpr, int64_t* const* out_cols, int64_t out_capacity,
                            int64_t* d_out_count);

/* ---- HashBuild ------------------------------------------------------------ */
typedef struct { const gq_table* table; int32_t key_col; } gq_probe_step;  /* key_col may name an earlier payload */
typedef struct {
  const gq_pred* preds; int32_t npred;
  const gq_probe_step* probes; int32_t nprobes;  /* chained joins: rows must match these tables before insertion */
  int32_t key_col;                               /* int64-widened key column (may be a payload of a probe step) */
  const int32_t* payload_cols; int32_t npayload; /* stored beside the key, handed to probers */
  uint32_t flags;                                /* GQ_F_UNIQUE_KEYS, GQ_F_DENSE_KEYS */
  int64_t key_min, key_max;                      /* GQ_F_DENSE_KEYS: inclusive key range (ignored otherwise) */
} gq_build_desc;
/* Open addressing, linear probing, 64-bit CAS; capacity = max_build_rows / load slots rounded up to a multiple of
 * 1024 (not to a power of two: slot = multiply-shift range reduction of the hash), load = 0.4 for tables that fit L2 and
 * 0.7 for larger ones; read in 32-byte (key-only) or 64-byte (key + payload) buckets. */
gq_status gq_hash_build_workspace(int64_t max_build_rows, int32_t npayload, size_t* bytes);
/* Workspace of a GQ_F_DENSE_KEYS table: header + 8 bytes per 32 keys of [key_min, key_max] (membership bits and rank
 * prefix) + one payload row per key of the range + one word per build row (the key of every rank). max_build_rows bounds
 * the rows inserted (exceeding it => GQ_ERR_CAPACITY at gq_hash_build_finish); <= 0 means "as many as the range has
 * keys". Such a table MUST be finished with gq_hash_build_finish before it is probed: that call computes the ranks. */
gq_status gq_hash_build_workspace_dense(int64_t key_min, int64_t key_max, int64_t max_build_rows, int32_t npayload, size_t* bytes);
/* *table == NULL: creates the table in d_workspace (enqueues its initialisation) and inserts the batch.
 * *table != NULL: inserts a further batch (same schema and desc; d_workspace/bytes/max_build_rows ignored). */
gq_status gq_hash_build(gq_ctx*, gq_table** table, void* d_workspace, size_t bytes, int64_t max_build_rows,
                        const gq_batch* in, const gq_build_desc* desc);
/* "noMoreInput": records an event on the building stream; probing contexts on OTHER streams wait on it (the
 * cross-pipeline synchronisation of PAPER.md:123). No host synchronisation. For a GQ_F_DENSE_KEYS table it first
 * enqueues the rank computation (two small kernels). */
gq_status gq_hash_build_finish(gq_ctx*, gq_table*);
/* *d_count (DEVICE int64) = rows inserted so far (enqueued copy). */
gq_status gq_table_count(gq_ctx*, const gq_table*, int64_t* d_count);
gq_status gq_table_destroy(gq_table*);           /* frees the host handle; the workspace stays the caller's */

/* ---- HashProbe, standalone and materialising inner join -------------------------- */
/* Output row = exprs (int64 each) over [probe columns ++ payloads of the probed tables]; every matching pair is
 * emitted (multiset semantics); unmatched probe rows are dropped. *d_out_count += rows written. */
gq_status gq_hash_probe(gq_ctx*, const gq_batch* probe, const gq_pred* preds, int32_t npred,
                        const gq_probe_step* probes, int32_t nprobes, const gq_expr* exprs, int32_t nexpr,
                        int64_t* const* out_cols, int64_t out_capacity, int64_t* d_out_count);

/* ---- HashAggregation, mode Single, streaming --------------------------------- */
typedef struct {
  const gq_pred* preds; int32_t npred;
  const gq_probe_step* probes; int32_t nprobes;
  const gq_expr* exprs; int32_t nexpr;
  const int32_t* key_cols; int32_t nkeys;        /* 0 = one global group; <= GQ_MAX_KEYS */
  int32_t ndependent;  /* trailing key columns functionally dependent on the leading ones: stored, not hashed.
                          Needed when the packed key tuple is wider than 64 bits. */
  const gq_agg* aggs; int32_t naggs;
  int64_t max_groups;  /* capacity bound (exceeding it => GQ_ERR_CAPACITY); <= 64 selects the low-cardinality path
                          (per-thread cells in shared memory) */
  uint32_t flags;      /* GQ_F_CHECK_DEPENDENT, GQ_F_FINAL_MODE */
} gq_agg_desc;
gq_status gq_hash_aggregate_workspace(int64_t max_groups, int32_t nkeys, int32_t naggs, size_t* bytes);
/* Plan-aware size: at least the size above; larger when the plan qualifies for DIRECT aggregation — the single hashed
 * group key is the key column of a probe step into a GQ_F_UNIQUE_KEYS table (and a dependent key, if any, is a payload
 * of that table), so a row's group is the table slot it matched and the aggregates live in an array indexed by that
 * slot (no second hash table; SURVEY §8(d) note on C3). gq_hash_aggregate takes that path when the workspace it is
 * given is at least this large; the probed table's workspace must then stay alive until the state is finished.
 * It also adds the record buffers of the RADIX-CLUSTERED path taken by high-cardinality states whose table is >= 256 MB
 * when the first batch has >= 16 Mi rows (32-byte records, sized for every row of that batch: e.g. 24 GB for C5): the
 * scan appends surviving rows per table partition and a second kernel applies them partition by partition. */
gq_status gq_hash_aggregate_workspace_for(const gq_batch* in, const gq_agg_desc* desc, size_t* bytes);
/* *state == NULL: creates the state in d_workspace and aggregates the batch; else aggregates a further batch. */
gq_status gq_hash_aggregate(gq_ctx*, gq_aggstate** state, void* d_workspace, size_t bytes, const gq_batch* in,
                            const gq_agg_desc* desc);
/* AVG derived in the finaliser: out = (double)agg[sum_agg] / (double)agg[count_agg] (IEEE-754 binary64). */
typedef struct { int32_t sum_agg; int32_t count_agg; } gq_avg;
/* Emits dense groups. out_key_cols[k] has the dtype of key column k; out_agg_cols[a] int64; out_avg_cols[j] double.
 * topk == 0: all groups, order unspecified, *d_out_ngroups = group count (capacity exceeded => GQ_ERR_CAPACITY).
 * topk  > 0: the topk groups with the largest aggregate `topk_agg`, ordered (aggregate desc, key tuple asc).
 * d_topk_scratch: gq_topk_scratch_bytes() bytes, needed only when topk > 0. */
size_t gq_topk_scratch_bytes(void);
gq_status gq_hash_aggregate_finish(gq_ctx*, gq_aggstate*, void* const* out_key_cols, int64_t* const* out_agg_cols,
                                   const gq_avg* avgs, int32_t navg, double* const* out_avg_cols,
                                   int64_t out_capacity, int32_t topk, int32_t topk_agg, void* d_topk_scratch,
                                   int64_t* d_out_ngroups);
gq_status gq_aggstate_destroy(gq_aggstate*);
/* Partial -> Final between two live states (e.g. one per stream, Fig. 3): folds every group of `src` into `dst`
 * (same keys and aggregates; direct-aggregation states must share their join table). `src` is left unchanged. Enqueued
 * on ctx's stream: the caller orders it after the work that filled `src` (same context, or gq_sync on the other). */
gq_status gq_aggstate_merge(gq_ctx*, gq_aggstate* dst, const gq_aggstate* src);
/* *d_count (DEVICE int64) = groups currently in the state (enqueued). */
gq_status gq_aggstate_count(gq_ctx*, const gq_aggstate*, int64_t* d_count);
/* Growth ("dynamic hash table expansion"): re-hashes a high-cardinality state into a larger table in a
 * new workspace of gq_hash_aggregate_workspace(new_max_groups, ...) bytes; stream-ordered, no host synchronisation. The
 * old workspace may be released once this call's work has completed. A planner needs no device round trip to decide:
 * the groups of a state never exceed the rows fed to it, so it grows the state when that bound passes max_groups
 * (or after reading gq_aggstate_count at a pipeline boundary). */
gq_status gq_aggstate_rehash(gq_ctx*, gq_aggstate*, void* d_new_workspace, size_t bytes, int64_t new_max_groups);

/* ---- OrderBy / TopN (PAPER.md:138 and Fig. 2: CudfOrderBy, TopN) ----------------------------- */
/* Sorts the rows of a batch by key columns: lexicographic with keys[0] most significant, ascending or descending per
 * key, signed comparison, ties broken by input row position (a STABLE sort: the result is unique). Writes the first
 * min(limit, nrows) rows (limit <= 0: all): d_out_index[i] (int64, may be NULL) = input row number of output row i, and,
 * when out_cols != NULL, out_cols[c][i] = column c of that row with the input column's dtype (an entry may be NULL).
 * nkeys == 0 keeps the input order. Method: LSD radix sort of (sortable key, row) pairs, one key column at a time;
 * radix passes over bytes in which all keys agree are skipped on the device; limit << nrows first selects the candidate
 * rows with a two-level radix select on keys[0]; up to 2048 rows are sorted by one CTA in one launch. Stream-ordered, no
 * host synchronisation. nrows <= 2^31. */
typedef struct { int32_t col; int32_t descending; } gq_sort_key;
gq_status gq_order_by_workspace(int64_t nrows, size_t* bytes);
gq_status gq_order_by(gq_ctx*, const gq_batch* in, const gq_sort_key* keys, int32_t nkeys, int64_t limit, void* d_workspace,
                      size_t bytes, int64_t* d_out_index, void* const* out_cols);
/* ---- Hash partitioning: the GPU side of PartitionedOutput ---------------
 * Groups the rows of a batch by DESTINATION so that every destination's rows form one contiguous, packed range of the
 * output columns ("cudf columns gathered into contiguous memory"), ready for an exchange: rows of
 * destination d are out rows [d_out_offsets[d], d_out_offsets[d + 1]); inside a destination rows keep their input order
 * (the result is unique). Whole rows move: every input column is written, with its dtype, to out_cols[c] (nrows
 * elements, 16-byte aligned, the caller's). d_out_row (optional, int64[nrows]) receives the input row number of every
 * output row; d_out_offsets is int64[nparts + 1]. The destination of a row depends on its key columns only:
 *     h = 0x9E3779B97F4A7C15;  for k in key_cols (in order): h = fmix64(h ^ (uint64)(int64)value_k);
 *     destination = ((h >> 32) * nparts) >> 32                       (fmix64 = MurmurHash3's 64-bit finaliser:
 *     x ^= x >> 33; x *= 0xff51afd7ed558ccd; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53; x ^= x >> 33)
 * so that every sender maps equal keys to the same destination. 1 <= nparts <= GQ_MAX_PARTITIONS, 1..8 key columns,
 * nrows <= 2^31. Stream-ordered, no host synchronisation; three launches (histogram, scan, scatter). */
enum { GQ_MAX_PARTITIONS = 256 };
gq_status gq_hash_partition_workspace(int32_t nparts, size_t* bytes);
gq_status gq_hash_partition(gq_ctx*, const gq_batch* in, const int32_t* key_cols, int32_t nkeys, int32_t nparts,
                            void* d_workspace, size_t bytes, void* const* out_cols, int64_t* d_out_row,
                            int64_t* d_out_offsets);

/* The same partitioning FUSED WITH ITS TRANSFER, in two phases (exchange "without requiring the transfer
 * to the host memory"; over NVLink the scatter's stores ARE the transfer - no packed send buffer, no separate
 * all-to-all):
 *   gq_hash_partition_count       histogram + scan; d_out_counts[d] (int64[nparts]) = rows this batch holds for
 *                                 destination d. The senders exchange their counts; receiver d lays the senders out one
 *                                 after the other, which gives every sender the row where its run starts in d's buffers.
 *   gq_hash_partition_scatter_to  the scatter of THE SAME batch, keys, nparts and workspace (it reuses the scanned
 *                                 histogram: call it after _count, on the same stream, with nothing in between that
 *                                 touches the workspace). Rows of destination d are written, in input order, to rows
 *                                 d_dst_row0[d], d_dst_row0[d] + 1, ... of d's own column buffers: d_dst_cols is a
 *                                 DEVICE array of nparts * ncols pointers, column c of destination d at [d * ncols + c],
 *                                 each 16-byte aligned and writable from this GPU - local memory, or another GPU's memory
 *                                 mapped into this process (peer access / IPC / symmetric memory); d_dst_row0 is a
 *                                 DEVICE int64[nparts]. A destination buffer holds < 2^32 rows.
 * The receiver may read its buffers once every sender's scatter has completed (an event / barrier of the caller's). */
gq_status gq_hash_partition_count(gq_ctx*, const gq_batch* in, const int32_t* key_cols, int32_t nkeys, int32_t nparts,
                                  void* d_workspace, size_t bytes, int64_t* d_out_counts);
gq_status gq_hash_partition_scatter_to(gq_ctx*, const gq_batch* in, const int32_t* key_cols, int32_t nkeys, int32_t nparts,
                                       void* d_workspace, size_t bytes, void* const* d_dst_cols,
                                       const int64_t* d_dst_row0);

/* Allocation-free variant of gq_order_by for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight
 * serving loops, harnesses that forbid it): same arguments, results and order, but the scratch lives in a file-scope
 * device array inside libgq.so (4.2 MB, held by every GPU that loads the library until the process exits), so the call
 * takes no workspace and makes no cudaMalloc / cudaFree / allocating library call. Limit: in->nrows <=
 * gq_order_by_static_max_rows() (131072); more rows => GQ_ERR_UNSUPPORTED with a message, nothing is launched. All calls on
 * one device share that array (it keeps the last call's contents; the call clears what it needs zeroed): calls that
 * OVERLAP on the GPU - two streams or two contexts of one device - race; serialise them. Inputs and outputs stay the
 * caller's. */
int64_t gq_order_by_static_max_rows(void);
gq_status gq_order_by_static(gq_ctx*, const gq_batch* in, const gq_sort_key* keys, int32_t nkeys, int64_t limit,
                             int64_t* d_out_index, void* const* out_cols);

/* ---- Fused pipeline: scan -> filter -> probe t1..tk -> project -> aggregate -> finalise ------- */
typedef struct {
  const gq_batch* in; gq_agg_desc agg;
  const gq_avg* avgs; int32_t navg;
  int32_t topk; int32_t topk_agg;
} gq_plan;
gq_status gq_pipeline_workspace(const gq_plan*, size_t* bytes);
/* One stream-ordered pass, no host synchronisation inside: state init, fused scan kernel, finaliser.
 * Key-less and low-cardinality plans (max_groups <= 64) without top-k run as ONE kernel: every CTA writes its partial
 * groups to the workspace and the last CTA to finish merges them and writes the result. The calls can be captured into
 * a CUDA graph. */
gq_status gq_pipeline(gq_ctx*, const gq_plan*, void* d_workspace, size_t bytes, void* const* out_key_cols,
                      int64_t* const* out_agg_cols, double* const* out_avg_cols, int64_t out_capacity,
                      int64_t* d_out_ngroups);
/* End-to-end variant with HOST input columns (plan->in->cols[].data are HOST pointers, pinned for full overlap):
 * the batch is cut into chunks of chunk_rows, each copied host->device into a double-buffered staging area inside
 * d_workspace while the previous chunk is aggregated (streaming of batches); results are copied back
 * into HOST output buffers and the call returns after they have landed. Probed tables stay device-resident. */
gq_status gq_pipeline_host_workspace(const gq_plan*, int64_t chunk_rows, size_t* bytes);
gq_status gq_pipeline_host(gq_ctx*, const gq_plan*, int64_t chunk_rows, void* d_workspace, size_t bytes,
                           void* const* h_out_key_cols, int64_t* const* h_out_agg_cols, double* const* h_out_avg_cols,
                           int64_t out_capacity, int64_t* h_out_ngroups);

/* ---- plan-time compilation ------------------------------------------------------------------------------------ */
/* Directory of the on-disk kernel cache (<hash>.cubin + <hash>.cu); default: $GQ_KERNEL_CACHE or ./_kcache beside
 * libgq.so. Plans are compiled on first use; these calls let a build step do it ahead of time, without a GPU. */
gq_status gq_set_kernel_cache_dir(const char* h_path);
/* Compiles (or finds in the cache) the fused kernel for the plan shape; needs no GPU. tables in probe steps may be
 * described by handles created with gq_table_describe (no device memory). */
gq_status gq_precompile_pipeline(const gq_plan*, char* h_msg, size_t msg_bytes);
gq_status gq_precompile_build(const gq_batch* in, const gq_build_desc*, char* h_msg, size_t msg_bytes);
/* The materialising kernel of gq_filter_project (nprobes == 0) / gq_hash_probe for this shape. */
gq_status gq_precompile_materialise(const gq_batch* in, const gq_pred* preds, int32_t npred, const gq_probe_step* probes,
                                    int32_t nprobes, const gq_expr* exprs, int32_t nexpr, char* h_msg, size_t msg_bytes);
/* Host-only table handle carrying just the schema (payload dtypes, flags) for precompilation. */
gq_status gq_table_describe(gq_table** out, const gq_dtype* payload_dtypes, int32_t npayload, uint32_t flags);   /* flags: GQ_F_UNIQUE_KEYS, GQ_F_DENSE_KEYS */

/* ---- measurement helper ---------------------------------------------------------------------------------------- */
/* Read-only streaming sum over `bytes` bytes (16-byte aligned, multiple of 16): the practical read roofline probe of
 * SURVEY §7.1 step 5. *d_out (DEVICE uint64) receives the wrapping sum of the 64-bit words. */
gq_status gq_read_probe(gq_ctx*, const void* d_data, size_t bytes, uint64_t* d_out);

/* ---- per-kernel timing (the operator-level breakdown the paper reports, Fig. 5/6) ----------------------- */
/* enable != 0: from now on every kernel (or small kernel group) this context launches is bracketed by a pair of CUDA
 * events on its stream (a few microseconds each; leave it off inside timed loops and CUDA-graph capture). */
gq_status gq_profile(gq_ctx*, int32_t enable);
/* Blocks until the stream is idle, then returns the number of entries recorded since the last read (<= max_entries):
 * h_ms[i] = device milliseconds of entry i, h_names = their names separated by '\n' (HOST buffers). -1 on error. */
int32_t gq_profile_read(gq_ctx*, char* h_names, size_t names_bytes, float* h_ms, int32_t max_entries);

/* ---- planner knobs --------------------------------------------------------------------------------------------- */
/* Process-wide thresholds a planner may override ("the query planner should choose the operator
 * implementation based on both the expected input and the available resources"). Names:
 *   "part_min_table_mb"  group-by tables at least this large take the radix-partitioned path (default 256)
 *   "part_min_rows"      ... when the first batch has at least this many rows (default 16 Mi)
 *   "hot_min_rows"       batches at least this large are sampled for heavy hitters (default 4 Mi)
 *   "psa_max_log2_partitions"  cap on the pass-A partitions of the partitioned shared-memory aggregation (default 14);
 *                        key ranges beyond it are resolved by sub-passes of pass B
 *   "psa_threads"        512 / 1024 threads per CTA in pass B (default 1024), 0 = default
 *   "psa_cluster"        2 (default): pass A of the partitioned shared-memory aggregation runs as thread-block clusters of
 *                        two CTAs that share the open record chunk of every partition through distributed shared
 *                        memory (half as many partly written record lines compete for L2); 1 = every CTA on its own
 *   "dpart_min_acc_mb"   direct aggregations whose accumulator array is at least this large cluster their updates by
 *                        slice of the array (records appended by the scan, applied slice by slice); default: never
 *                        (measured slower on C3), a planner may enable it for arrays far beyond L2
 * Unknown names return GQ_ERR_INVALID_ARG. A negative value restores the default. */
gq_status gq_set_option(const char* h_name, int64_t value);

#ifdef __cplusplus
}
#endif
#endif
