/* oracle.h — C interface of the CPU oracle.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this library.
 * The product path (paper_2606_24647_b200/) never includes, links or calls anything here, and this directory
 * includes nothing from the product: the descriptor types below are the oracle's own.
 *
 * What it computes: the plain definitions of SURVEY.md §8(c) — the operators the paper names (Filter, Project,
 * inner Join, HashAggregation; "inner join" :92; no nulls :59) evaluated row by
 * row, single-threaded, in the order the definition states. No blocking, fusion or reordering.
 */
#ifndef GQ_ORACLE_H
#define GQ_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { OCL_I8 = 1, OCL_I32 = 2, OCL_I64 = 3 };                                   /* column element types (signed) */
enum { OCL_LT = 0, OCL_LE, OCL_GT, OCL_GE, OCL_EQ, OCL_NE, OCL_RANGE_CO /* lo<=x<hi */, OCL_RANGE_CC /* lo<=x<=hi */ };
enum { OCL_X_COL = 0, OCL_X_CONST, OCL_X_ADD, OCL_X_SUB, OCL_X_MUL };             /* postfix tokens */
enum { OCL_SUM = 0, OCL_MIN, OCL_MAX, OCL_COUNT_STAR };

typedef struct { const void* data; int32_t dtype; } ocl_column;                  /* HOST pointer, no nulls */
typedef struct { const ocl_column* cols; int32_t ncols; int64_t nrows; } ocl_table;
typedef struct { int32_t col; int32_t op; int64_t lo, hi; } ocl_pred;             /* one-sided ops compare with lo */
typedef struct { int32_t op; int64_t arg; } ocl_tok;
typedef struct { const ocl_tok* toks; int32_t ntoks; } ocl_expr;
typedef struct { int32_t op; int32_t expr; } ocl_agg;
/* A probe step joins the current row with relation `build` on  row[key_col] == build.key  and appends that
 * relation's payload columns to the row (inner join: no match => row dropped; k matches => k rows). */
typedef struct { int32_t build; int32_t key_col; } ocl_probe;
/* A build relation: filter `in`, run its own probe steps (chained joins), keep (key, payloads) of surviving rows.
 * Column indices >= in.ncols name payload columns appended by this relation's earlier probe steps, in order. */
typedef struct {
  ocl_table in; const ocl_pred* preds; int32_t npred; const ocl_probe* probes; int32_t nprobes;
  int32_t key_col; const int32_t* payload_cols; int32_t npayload;
} ocl_build;
typedef struct {
  const ocl_build* builds; int32_t nbuilds;                /* evaluated in order; probes may only name earlier ones */
  ocl_table in; const ocl_pred* preds; int32_t npred; const ocl_probe* probes; int32_t nprobes;
  const ocl_expr* exprs; int32_t nexpr;
  const int32_t* key_cols; int32_t nkeys;                  /* group key tuple (0 keys => one global group) */
  const ocl_agg* aggs; int32_t naggs;
  int32_t topk; int32_t topk_agg;                          /* 0 = all groups sorted by key tuple ascending */
} ocl_query;

typedef struct ocl_result ocl_result;   /* owns its arrays; free with ocl_result_free */

/* Filter + join chain + grouped aggregation (+ top-k). Returns NULL on a malformed query. */
ocl_result* ocl_run_query(const ocl_query* q);
/* Filter + project only: output rows in input order, one int64 column per expression. */
ocl_result* ocl_filter_project(const ocl_table* in, const ocl_pred* preds, int32_t npred, const ocl_expr* exprs, int32_t nexpr);
/* Inner equi-join of two filtered tables as sorted (probe_row, build_row) pairs: hash-multimap version and the
 * brute-force double loop that checks it (column 0 = probe row index, column 1 = build row index). */
ocl_result* ocl_join_pairs(const ocl_table* build, const ocl_pred* bpreds, int32_t nbpred, int32_t bkey,
                           const ocl_table* probe, const ocl_pred* ppreds, int32_t nppred, int32_t pkey);
ocl_result* ocl_join_pairs_bruteforce(const ocl_table* build, const ocl_pred* bpreds, int32_t nbpred, int32_t bkey,
                                      const ocl_table* probe, const ocl_pred* ppreds, int32_t nppred, int32_t pkey);

/* ORDER BY ... LIMIT (PAPER.md:138 OrderBy / TopN): the definition written out — rows compared
 * lexicographically over the key columns (keys[0] first; signed values; descending keys compare reversed), ties keep
 * input order (std::stable_sort). Result: column 0 = input row numbers of the first min(limit, nrows) rows in order
 * (limit <= 0: all rows), then every input column gathered in that order (widened to int64). */
typedef struct { int32_t col; int32_t descending; } ocl_sort_key;
ocl_result* ocl_order_by(const ocl_table* in, const ocl_sort_key* keys, int32_t nkeys, int64_t limit);

/* Hash partitioning of a batch to nparts destinations (PAPER.md:160, :174 CudfPartitionedOutput):
 * destination(row) = the function include/gq.h defines over the key columns (restated in oracle.cpp, not shared);
 * rows are emitted destination by destination, in input order inside a destination. Result: column 0 = destination of
 * every output row, column 1 = its input row number, then every input column (widened to int64). */
ocl_result* ocl_hash_partition(const ocl_table* in, const int32_t* key_cols, int32_t nkeys, int32_t nparts);

int64_t ocl_result_nrows(const ocl_result*);              /* groups / output rows / pairs */
int32_t ocl_result_ncols(const ocl_result*);              /* keys then aggregates (query); exprs; 2 (pairs) */
const int64_t* ocl_result_col(const ocl_result*, int32_t c);
int64_t ocl_result_input_rows(const ocl_result*);         /* rows that survived filters and joins (fed to GROUP BY) */
int32_t ocl_result_overflow(const ocl_result*);           /* 1 if any expression value or running SUM left int64
                                                             range in the __int128 shadow evaluation (S6) */
double ocl_avg(int64_t sum, int64_t count);               /* derived AVG = (double)sum / (double)count (S7/§8(c).7) */
void ocl_result_free(ocl_result*);

#ifdef __cplusplus
}
#endif
#endif
