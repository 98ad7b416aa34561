/*
 * spmv_b200.h -- C ABI of the B200-native autotuned fp64 CSR SpMV library.
 *
 *      y = alpha * A * x + beta * y        A: CSR, fp64 values, int32 indices
 *
 * The operation and its boundary are those of BASELINE.json:north_star (a)
 * ("spmv_create / spmv_tune / spmv_apply / spmv_destroy, with arguments following
 * the paper's problem statement of matrix, vectors and scalars"); the paper states
 * the problem only as "sparse kernels vs cuSPARSE and CUSP" (sec. 3)
 * and the method as annotate -> generate variants -> run -> compare outputs with
 * the reference -> keep the fastest (sec. 2).
 * fixes the conventions below.
 *
 * General rules
 *   - C linkage, no exceptions or aborts cross this boundary; every call returns a
 *     spmv_status_t (except the string/getter helpers).
 *   - "d_" arguments are DEVICE pointers, "h_" arguments are HOST pointers.
 *   - `stream` arguments are a cudaStream_t passed as void* (NULL = legacy default
 *     stream).  spmv_apply / spmv_apply_batch are asynchronous and never
 *     synchronise; spmv_create, spmv_tune, spmv_select synchronise the stream they
 *     use.
 *   - The handle BORROWS d_row_ptr / d_col_idx / d_val: the caller keeps them alive
 *     and unmodified until spmv_destroy.  Converted formats and workspaces are OWNED
 *     by the handle (allocated through the spmv_allocator_t callbacks, or
 *     cudaMalloc/cudaFree when none is given).  x and y are caller-owned and must
 *     not alias each other or the matrix.
 *   - Limits: rows, cols, nnz <= 2^31-1 (int32 indices, BASELINE.json:configs[0]);
 *     rows == 0 and nnz == 0 are valid.
 *   - There is no CPU fallback: without a CUDA device every compute entry point
 *     returns SPMV_ERR_CUDA.
 *   - Concurrency: distinct handles are independent.  One handle may have several applies in
 *     flight on different streams.  Variants that own a workspace -- merge-path (tile carries)
 *     and row-split SELL (segment sums), one workspace per handle -- are ordered by the library:
 *     an spmv_apply on another stream than the handle's previous apply first makes its stream wait
 *     (on the device, through an event) for that apply.  Exceptions the caller orders: applies
 *     enqueued inside a stream capture, and replays of an spmv_graph_t next to other applies of the
 *     same handle.  spmv_apply itself may be called from several host threads.  spmv_cg allocates per call.
 *
 * Variant descriptors (spmv_select, tune reports, spmv_list_variants): "family:key<int>:..."
 *   families  csr_scalar (thread per row), csr_vector (w lanes per row), sell / sell_tma
 *             (SELL-C-sigma; _tma: matrix stream by cp.async.bulk + mbarrier ring), ell, merge
 *             (merge-path), bcsr3 (3x3 blocks), dia / dia_tma (diagonals, no column indices),
 *             dia_const (constant-coefficient stencil: no matrix values read), sell16 / sell16_tma (SELL with 16-bit
 *             delta-encoded column indices per slice: 10 bytes per entry, banded patterns whose slices span
 *             fewer than 65535 columns)
 *   keys      b threads per block | g grid: 0/absent exact cover, k = k waves of resident blocks |
 *             co shared-memory carve-out percent | u unroll (sell_tma/dia_tma: steps per stage) |
 *             r rows per thread | w lanes per (block) row | x x path: 0 ld.global.nc, 1 ld.global,
 *             2 (sell_tma, sell16_tma) the x window of a slice staged in shared memory (+ h = window half-width;
 *             gathers outside it go through L1), 3 (sell_tma, sell16_tma) the same with h >= the matrix bandwidth:
 *             every gather is a shared-memory read (sigma 1, even column count); 3 (bcsr3) the 3-vector of a
 *             block as an aligned 16-byte pair + one 8-byte load | c slice height |
 *             s sorting window sigma | l row-split length (rows longer than l become segments) |
 *             i merge items per thread (sell_tma/dia_tma: pipeline stages; bcsr3: i16 = 16-bit block columns
 *             relative to the block row, 74 instead of 76 bytes per block)
 *   "default" = csr_scalar:b256:r1:u1:x0, the fixed default variant.
 */
#ifndef SPMV_B200_H
#define SPMV_B200_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define SPMV_API __attribute__((visibility("default")))
#else
#define SPMV_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spmv_handle_s* spmv_handle_t;

typedef enum {
  SPMV_OK = 0,
  SPMV_ERR_INVALID_ARG = 1,     /* NULL pointer, negative size, unknown descriptor   */
  SPMV_ERR_INVALID_MATRIX = 2,  /* row_ptr not monotone / wrong ends, col out of range */
  SPMV_ERR_UNSUPPORTED = 3,     /* size over the int32 limits, variant not eligible  */
  SPMV_ERR_ALLOC = 4,
  SPMV_ERR_CUDA = 5,            /* text via spmv_last_error()                        */
  SPMV_ERR_VERIFY_FAILED = 6,   /* no candidate matched the reference result          */
  SPMV_ERR_INTERNAL = 7
} spmv_status_t;

/* Optional device allocator (e.g. the torch caching allocator). */
typedef struct {
  void* (*alloc)(size_t bytes, void* stream, void* ctx);
  void (*free)(void* ptr, void* ctx);
  void* ctx;
} spmv_allocator_t;

/* Matrix statistics, structure signature and the selected variant. */
typedef struct {
  int64_t rows, cols, nnz;
  int32_t min_row_len, max_row_len;
  double mean_row_len, var_row_len;
  int64_t len_hist[32];     /* [0]: empty rows; [b>=1]: rows with 2^(b-1) <= len < 2^b */
  int64_t bandwidth;        /* max |col - row| over stored entries                    */
  int32_t cols_sorted;      /* 1: every row strictly ascending (sorted, no duplicates) */
  int32_t block3_full;      /* 1: matrix is a union of dense, aligned 3x3 blocks       */
  int64_t n_blocks3;        /* number of 3x3 blocks touched (valid if cols_sorted)     */
  uint64_t sig_row_ptr;     /* order-independent 64-bit hashes of the structure        */
  uint64_t sig_col_idx;
  int32_t tuned;            /* 1 after a successful spmv_tune / cache hit              */
  int32_t sm_count;
  int64_t l2_bytes;
  int64_t format_bytes;     /* matrix bytes streamed per apply by the selected variant */
  int64_t owned_bytes;      /* device bytes currently owned by the handle              */
  char variant[128];        /* descriptor of the selected variant                      */
  char device_name[64];
} spmv_info_t;

/* Tuning options; zero-initialise for defaults. */
typedef struct {
  int32_t has_scalars;        /* 0: tune for alpha=1, beta=0; 1: use alpha/beta below */
  double alpha, beta;
  const double* d_x_probe;    /* cols  entries, device; NULL: tuner draws U[-1,1) from seed */
  const double* d_y0_probe;   /* rows  entries, device; NULL: idem                      */
  const double* d_y_ref;      /* optional externally computed reference result (device) */
  const double* d_scale;      /*   and its per-row tolerance denominators; both or none.
                                   When NULL the reference is the library's own unfused,
                                   stored-order, one-thread-per-row device kernel -- the
                                   "un-annotated program" of PAPER.md:19.                */
  double tolerance;           /* 0 -> 1e-12 (north_star)                                */
  int32_t warmup;             /* 0 -> 2 untimed launches per candidate                  */
  int32_t reps;               /* 0 -> 5 timed batches per candidate (median)            */
  double min_batch_ms;        /* 0 -> 0.5 ms per batch                                  */
  double time_budget_s;       /* 0 -> unlimited                                         */
  const char* variant_filter; /* comma-separated family prefixes, e.g. "csr_vector,sell"; NULL = all */
  int32_t n_carveouts;        /* 0 -> {-1 (driver default)}                             */
  int32_t carveouts[8];       /* shared-memory carve-out percentages, -1 = default      */
  int32_t use_cache;          /* 0 -> use the in-process cache; 2 -> bypass it           */
  const char* cache_path;     /* optional file persisted across processes.  A cached winner (in process or from
                                 this file) is a claim: it is adopted only after one launch of it has passed the same
                                 verification as every candidate; an entry that fails is dropped and the search runs */
  const char* fault_inject;   /* TEST ONLY: descriptor prefix of candidates whose output
                                 is perturbed before verification                       */
  uint64_t seed;
  int32_t flush_l2;           /* 1: overwrite a > L2-sized buffer before each timed launch */
  int32_t search;             /* 0: exhaustive (every eligible candidate, the paper's loop);
                                 1: feature-guided: only the families the structure
                                 statistics predict -- diagonal pattern -> dia*, dense 3x3 blocks -> bcsr3,
                                 skewed row lengths -> row-split sell + merge, otherwise sell_tma / sell /
                                 csr_vector -- plus sell_tma and csr_vector as the fallback.  Every candidate
                                 that is run is still verified before it may win. */
  void* stream;
} spmv_tune_opts_t;

typedef struct {
  char winner[128];
  double winner_us;            /* median time per apply of the winner                  */
  double default_us;           /* same protocol, the fixed default variant             */
  int32_t n_enumerated, n_pruned_structural, n_pruned_slow, n_rejected, n_timed;
  double tune_seconds;
  int32_t cache_hit;
  char runner_up[128];
  double runner_up_us;
  /* optional per-candidate log: "descriptor status time_us max_err_over_scale\n"; status in
   * {timed, timed1 (one batch only: > 25 % behind the leader), retimed (tie-break: within 2 % of the best, timed
   * again with 3x the batches; a tie within 0.5 % goes to the lexicographically smallest descriptor),
   * pruned_slow, pruned_format, rejected} */
  char* log_buf;
  size_t log_cap;
  size_t log_len;
} spmv_tune_report_t;

/* Build a handle: validates the CSR arrays on the device and gathers statistics.
 * Errors: INVALID_ARG (NULL out / negative size / NULL array with nnz > 0),
 * UNSUPPORTED (over int32 limits), INVALID_MATRIX, CUDA, ALLOC.  *out untouched on
 * failure. */
SPMV_API spmv_status_t spmv_create(spmv_handle_t* out, int64_t rows, int64_t cols, int64_t nnz,
                          const int32_t* d_row_ptr, const int32_t* d_col_idx,
                          const double* d_val, const spmv_allocator_t* alloc, void* stream);

/* The paper's loop: enumerate candidates (variant x launch config x
 * carve-out), run each on the actual matrix, compare its output with the reference
 * result, time the ones that match, keep the fastest, cache it per matrix signature. */
SPMV_API spmv_status_t spmv_tune(spmv_handle_t h, const spmv_tune_opts_t* opts, spmv_tune_report_t* report);

/* y = alpha*A*x + beta*y with the selected variant (the fixed default variant until
 * spmv_tune / spmv_select).  beta == 0: y is write-only (never read).  alpha == 0:
 * y = beta*y, A and x are not referenced.  Asynchronous on `stream`. */
SPMV_API spmv_status_t spmv_apply(spmv_handle_t h, double alpha, const double* d_x, double beta,
                         double* d_y, void* stream);

/* Same operation with HOST vectors (pinned memory overlaps; pageable memory works): copies x (and y when beta != 0) to
 * the device, applies, copies y back; synchronises `stream` before returning.  Where the selected variant has a
 * row-range form (see spmv_apply_rows) the call is a pipeline over chunks of rows on three internal streams --
 * upload of x as far as the chunk's rows reach (its rows + the matrix bandwidth) and of the chunk of y | kernel on the
 * chunk | download of the chunk of y -- bit-identical to the one-launch form.  Chunks hold ~3 MB of y (environment
 * variable SPMV_HOST_CHUNK_MB overrides, for experiments).  Zero-copy y: when h_y is pinned AND mapped host memory
 * (cudaHostAlloc / cudaHostRegister; 16-byte aligned) and the variant stores y one row per thread in row order (the
 * DIA families), the chunk kernels read and write h_y in place over PCIe instead of through a staging vector and
 * two copies (~8 MB chunks; SPMV_HOST_ZEROCOPY=0 turns it off); same kernels, same bits.  For a DIA-family variant
 * on a small system (x and y together <= 1 MB) with x mapped as well, the one kernel reads x and updates y in place:
 * one launch + one synchronise instead of three copies. */
SPMV_API spmv_status_t spmv_apply_host(spmv_handle_t h, double alpha, const double* h_x, double beta,
                              double* h_y, void* stream);

/* n host-vector applies (n DIFFERENT handles; BASELINE.json configs[4]: "four independent ... matrices ... applied
 * concurrently") as one call: every member's pipeline is enqueued first -- each runs on its handle's own internal
 * streams behind the work queued on `stream` when the call began, so the members' copies and kernels interleave --
 * then `stream` is synchronised once.  Results equal n spmv_apply_host calls bit for bit.
 * Errors: INVALID_ARG (NULL, a handle twice), ALLOC, CUDA. */
SPMV_API spmv_status_t spmv_apply_host_batch(int32_t n, const spmv_handle_t* hs, const double* alphas,
                                    const double* const* h_xs, const double* betas, double* const* h_ys,
                                    void* stream);

/* k back-to-back applies y <- alpha*A*x + beta*y of the selected variant captured into ONE CUDA graph (SURVEY.md
 * sec. 8(d): "a CUDA-graph replay of K applies may be reported as an additional, clearly labelled line"
 * lists the launch configuration among the tuned parameters -- for a launch-bound matrix the launch itself is the
 * cost).  Pointers, scalars and the variant are baked in: re-create the graph after spmv_select / spmv_tune /
 * spmv_update_values.  spmv_graph_launch replays it on `stream` (asynchronous).  Errors: INVALID_ARG, CUDA. */
typedef struct spmv_graph_s* spmv_graph_t;
SPMV_API spmv_status_t spmv_graph_create(spmv_handle_t h, double alpha, const double* d_x, double beta, double* d_y,
                                int32_t k, spmv_graph_t* out);
SPMV_API spmv_status_t spmv_graph_launch(spmv_graph_t g, void* stream);
SPMV_API spmv_status_t spmv_graph_destroy(spmv_graph_t g);

/* ---- Row-sharded apply: rows are independent, so A and y split into
 * nnz-balanced contiguous row blocks, one per GPU; before an apply each GPU needs the x entries its columns
 * reference and does not own.  The library provides the compute-side pieces; the transport between processes
 * is torch.distributed (NCCL over NVLink) in paper_1309_1894_b200/sharded.py.
 *
 * spmv_partition_rows: bounds[0..nparts] with bounds[0] = 0, bounds[nparts] = rows, interior bounds multiples
 *   of `align`, chosen so that part g holds about nnz/nparts stored entries (h_row_ptr is a HOST array).
 * spmv_external_columns: the sorted distinct columns referenced by the handle's matrix outside [own_lo, own_hi)
 *   -- the halo this shard must receive.  *count receives their number; at most cap are written to h_cols (HOST).
 *   Also reports, per row, whether it references an external column: [*int_lo, *int_hi) is the longest run of
 *   rows that do not (the interior, computable before the halo arrives).  Synchronises `stream`.
 * spmv_gather / spmv_scatter: dst[i] = src[idx[i]] / dst[idx[i]] = src[i] for i < n (device arrays, idx int32):
 *   packing the entries a peer needs, unpacking what arrived.  Asynchronous on `stream`.
 * spmv_apply_rows: spmv_apply restricted to rows [row_begin, row_end) (d_x, d_y: the whole vectors).  row_begin
 *   must be a multiple of *align_out = the selected variant's range alignment (query with row_begin = row_end);
 *   UNSUPPORTED when the variant has no row-range form (merge-path, row-split SELL, ELL, dia_win). */
SPMV_API spmv_status_t spmv_partition_rows(int64_t rows, const int32_t* h_row_ptr, int32_t nparts, int64_t align,
                                  int64_t* h_bounds);
SPMV_API spmv_status_t spmv_external_columns(spmv_handle_t h, int64_t own_lo, int64_t own_hi, int32_t* h_cols,
                                    int64_t cap, int64_t* count, int64_t* int_lo, int64_t* int_hi, void* stream);
SPMV_API spmv_status_t spmv_gather(int64_t n, const int32_t* d_idx, const double* d_src, double* d_dst, void* stream);
SPMV_API spmv_status_t spmv_scatter(int64_t n, const int32_t* d_idx, const double* d_src, double* d_dst, void* stream);
SPMV_API spmv_status_t spmv_apply_rows(spmv_handle_t h, double alpha, const double* d_x, double beta, double* d_y,
                              int64_t row_begin, int64_t row_end, int64_t* align_out, void* stream);

/* n independent applies, handle i on streams[i % nstreams] ("number of
 * asynchronous streams").  No synchronisation. */
SPMV_API spmv_status_t spmv_apply_batch(int32_t n, const spmv_handle_t* hs, const double* alphas,
                               const double* const* d_xs, const double* betas,
                               double* const* d_ys, void* const* streams, int32_t nstreams);

/* Times spmv_apply_batch over 1, 2, 4, ... <= max_streams of the caller's streams and
 * returns the fastest count; us_per_count[i] (may be NULL) receives the batch time for
 * the i-th count tried. */
SPMV_API spmv_status_t spmv_tune_batch(int32_t n, const spmv_handle_t* hs, const double* alphas,
                              const double* const* d_xs, const double* betas,
                              double* const* d_ys, void* const* streams, int32_t max_streams,
                              int32_t* best_nstreams, double* us_per_count);

/* ---- The product for callers that may not allocate device memory.
 *
 * Every other compute entry point obtains device memory at some stage: spmv_create / spmv_select / spmv_tune build
 * converted formats and workspaces through cudaMalloc (or the allocator callbacks), spmv_cg and spmv_jacobi take
 * three vectors per call.  Some users of the library cannot afford that at the place where they need y = alpha*A*x +
 * beta*y: a component living inside an application that has already handed all of the GPU's memory to its own pool
 * (cudaMalloc then fails, and the pool is not the library's to draw from); or a step of a latency-bound loop,
 * where cudaMalloc / cudaFree are unwelcome because they serialise against all work running on the device.
 *
 * spmv_merge_apply_noalloc is for them.  It runs the merge-path CSR kernels (north_star (c) "merge-path CSR for
 * skewed row lengths"; descriptor merge:b256:i7:x0) straight from the caller's CSR arrays: no handle, no conversion,
 * no cudaMalloc / cudaFree, no allocating library routine, on any call.  The scratch memory these kernels need (a
 * table of tile starts and one carry per tile, 16 bytes per tile of 1792 merge-path items) is a fixed 1 MiB + 256 B
 * array compiled into the library; each GPU that loads the library carries it until the process exits, whether or
 * not this entry point is ever called.
 *   Limit: rows + nnz <= spmv_merge_noalloc_max_path() = 117 440 512 (65 536 tiles).  Above it the call returns
 *     SPMV_ERR_UNSUPPORTED, spmv_last_error() says by how much, and nothing is launched.
 *   Arguments: device pointers; the CSR arrays, x (cols entries) and y (rows entries) are the caller's, as for
 *     spmv_create / spmv_apply, and must not alias.  The matrix is NOT validated (that would need a read-back): pass
 *     arrays that satisfy spmv_create's rules (monotone row_ptr with row_ptr[0] = 0 and row_ptr[rows] = nnz, columns
 *     in [0, cols)).  beta == 0: y is write-only.  alpha == 0: y = beta*y, the matrix and x are not referenced.
 *   Result: bit-identical to spmv_select(h, "merge:b256:i7:x0") + spmv_apply on the same arrays, and to itself on
 *     every repeat (no floating-point atomics).
 *   First call on a device: looks up the array's address on the CURRENT device (cudaGetSymbolAddress, once per
 *     device, remembered per device ordinal; ordinals 0..63).  That makes the driver load the library's device code
 *     if it has not yet, so make the first call on each device during set-up, before any stream capture begins
 *     and outside the part of the program that must not stall.  Later calls are three kernel launches on `stream`.
 *   Sharing: there is ONE array per GPU, used by every call on that GPU from any thread, and it keeps what the last
 *     call wrote.  A call never relies on those contents (each call first rewrites every word it later reads), so
 *     back-to-back calls on one stream need nothing in between.  Two calls whose kernels can overlap on the GPU --
 *     different streams without an event between them, or two host threads -- race on the array and produce
 *     garbage: order them.
 *   Asynchronous on `stream`; never synchronises.  Errors: INVALID_ARG (negative size, NULL array that is needed,
 *     d_x == d_y), UNSUPPORTED (over the limit above or over int32 sizes), CUDA. */
SPMV_API spmv_status_t spmv_merge_apply_noalloc(int64_t rows, int64_t cols, int64_t nnz, const int32_t* d_row_ptr,
                                       const int32_t* d_col_idx, const double* d_val, double alpha,
                                       const double* d_x, double beta, double* d_y, void* stream);
SPMV_API int64_t spmv_merge_noalloc_max_path(void);

/* Force a variant by descriptor ("default" = the fixed default).  Builds the format it
 * needs.  Errors: INVALID_ARG (unparsable), UNSUPPORTED (not eligible for this matrix). */
SPMV_API spmv_status_t spmv_select(spmv_handle_t h, const char* variant_descriptor, void* stream);

/* New values on the SAME sparsity pattern (row_ptr / col_idx unchanged; e.g. a time-dependent
 * coefficient): the handle now borrows d_val, the format of the selected variant is rebuilt from it
 * and the tuning result (a function of the structure signature) is kept.  If the selected variant
 * no longer applies to the new values (dia_const on coefficients that stopped being constant) the
 * handle falls back to the best remaining family it can build (dia_tma, else the default variant)
 * and *fell_back (may be NULL) is set to 1.  Synchronises `stream`. */
SPMV_API spmv_status_t spmv_update_values(spmv_handle_t h, const double* d_val, int32_t* fell_back, void* stream);

/* Solver loop around apply (the paper's ref [1], is about
 * iterative solvers): conjugate gradients for a symmetric positive definite A, with the selected
 * SpMV variant as the matrix product.
 *   d_b [rows] right-hand side (device, read only); d_x [rows] initial guess in, solution out (device).
 * Stops first when ||r_k|| <= tol * ||b|| (recurrence residual) or after max_iters iterations, or
 * when p.Ap <= 0 (A not positive definite: result->breakdown = 1).  Scalars stay on the device;
 * `check_every` iterations are replayed as one CUDA graph between host polls (plain launches when
 * `stream` is the legacy default stream, which cannot be captured, or no_graph != 0).
 * Workspace (3 vectors) comes from the handle's allocator for the duration of the call.
 * Synchronises `stream`.  Errors: INVALID_ARG (rows != cols, NULL), ALLOC, CUDA. */
typedef struct {
  double tol;            /* 0 -> 1e-10 */
  int32_t max_iters;     /* 0 -> 1000; negative -> 0 iterations (residual of the initial guess only) */
  int32_t check_every;   /* 0 -> 8 */
  int32_t no_graph;      /* 1: never use a CUDA graph */
  int32_t no_fused;      /* 1: never use the single cooperative kernel that runs the whole solve for small
                            systems (rows <= 262144, nnz <= 4 Mi): launch-bound otherwise */
  int32_t no_fused_dot;  /* 1: never fuse p.q into the SpMV kernel's epilogue (large systems; available for the
                            dia_const family): a dot kernel then makes a second pass over p and q */
  int32_t tune_loop;     /* 1: before solving, time a few iterations of the loop with each of the leaders of the
                            last spmv_tune of this handle and adopt the fastest (SURVEY 8(f) rank 3 "tune for the
                            loop rather than the single apply"); no-op when the handle was not tuned in this process */
} spmv_cg_opts_t;
typedef struct {
  int32_t iters, converged, breakdown;
  int32_t iterations_launched;   /* >= iters: iterations issued after convergence are device-side no-ops */
  int32_t graph_replays;
  int32_t fused;                 /* 1: the whole solve ran in the single cooperative kernel */
  int32_t fused_dot;             /* 1: p.q came out of the SpMV kernel's epilogue */
  int32_t kernels_per_iteration; /* launches per iteration (0 when fused) */
  char loop_variant[128];        /* the variant the loop ran with (differs from the apply winner after tune_loop) */
  double rel_residual;           /* sqrt(r.r) / ||b||  (sqrt(r.r) when b == 0) */
  double device_seconds;         /* CUDA events around the whole solve */
  double wall_seconds;
} spmv_cg_result_t;
SPMV_API spmv_status_t spmv_cg(spmv_handle_t h, const double* d_b, double* d_x, const spmv_cg_opts_t* opts,
                      spmv_cg_result_t* result, void* stream);

/* Second solver loop (SURVEY.md sec. 8(f) rank 3 names "CG / Jacobi using spmv_apply"): the weighted Jacobi
 * iteration  x_{k+1} = x_k + omega * D^-1 (b - A x_k)  for a square A with a non-zero diagonal (d_i = the sum of
 * the stored entries (i, i)), the selected SpMV variant as the product.  Per iteration: t = A x_k, then one fused
 * pass (residual, its norm, next iterate).  The stop test precedes the update: the call stops first when
 * ||b - A x_k|| <= tol * ||b||, or when k == max_iters; d_x then holds x_k and rel_residual ITS residual.
 *   d_b [rows] right-hand side (device, read only); d_x [rows] initial guess in, iterate out (device).
 * Scalars stay on the device; `check_every` (rounded up to even) iterations are replayed as one CUDA graph
 * between host polls.  A zero diagonal entry: result->zero_diagonal = 1, d_x untouched, SPMV_OK.
 * Workspace (3 vectors) comes from the handle's allocator for the duration of the call.  Synchronises `stream`.
 * Errors: INVALID_ARG (rows != cols, NULL), ALLOC, CUDA. */
typedef struct {
  double omega;          /* 0 -> 1.0 */
  double tol;            /* 0 -> 1e-10 */
  int32_t max_iters;     /* 0 -> 1000; negative -> 0 iterations (residual of the initial guess only) */
  int32_t check_every;   /* 0 -> 8 */
  int32_t no_graph;      /* 1: never use a CUDA graph */
  int32_t no_fused;      /* 1: never fuse the step into the product kernel (available for the dia_const family: product,
                            residual, update and norm partials in one pass; the iterates are bit-identical either way) */
} spmv_jacobi_opts_t;
typedef struct {
  int32_t iters, converged, zero_diagonal;
  int32_t iterations_launched;   /* > iters: the pass that meets the stop rule, and passes issued after it, update nothing */
  int32_t graph_replays;
  int32_t kernels_per_iteration;
  int32_t fused_step;            /* 1: the step ran inside the product kernel */
  double rel_residual;           /* ||b - A x|| / ||b|| of the returned x  (the norm itself when b == 0) */
  double device_seconds;         /* CUDA events around the whole call */
  double wall_seconds;
} spmv_jacobi_result_t;
SPMV_API spmv_status_t spmv_jacobi(spmv_handle_t h, const double* d_b, double* d_x, const spmv_jacobi_opts_t* opts,
                          spmv_jacobi_result_t* result, void* stream);

/* Writes the newline-separated descriptors of every candidate the tuner would
 * enumerate for this matrix (after structural pruning) into buf; *len = bytes needed. */
SPMV_API spmv_status_t spmv_list_variants(spmv_handle_t h, char* buf, size_t cap, size_t* len);

SPMV_API spmv_status_t spmv_get_info(spmv_handle_t h, spmv_info_t* out);

/* Inspection (tests): copy an owned array of the selected variant's format to the host.
 * name in {"slice_ptr","sval","scol","scol16","sbase","perm","brow_ptr","bcol","bval","tile_row","dia_val",
 * "dia_mask","dia_mask_small","dia_off","dia_coef"};
 * *bytes receives the array size; copies min(cap, size) bytes when h_buf != NULL. */
SPMV_API spmv_status_t spmv_format_download(spmv_handle_t h, const char* name, void* h_buf,
                                   size_t cap, size_t* bytes, void* stream);

/* Errors: INVALID_ARG on NULL or on a handle that was already destroyed. */
SPMV_API spmv_status_t spmv_destroy(spmv_handle_t h);

/* Measured ceilings with the library's own kernels, for the bench report:
 * kind 0: device copy GB/s (read+write bytes) and 1: read-only streaming sum GB/s, `bytes` per launch,
 * launches back to back over rotating windows (cold);
 * 2: empty-kernel launch latency in microseconds, 3: random 8-byte gathers out of a vector of
 * `bytes` bytes, in giga-gathers per second (the ceiling of the x path when columns are
 * unstructured), 4: the value loads of the bcsr3 kernel alone (records of 27 3x3 blocks in the block-row layout,
 * 16 lanes per record, no x / index / FMA; GB/s, median batch): what the layout's load pattern allows. */
SPMV_API spmv_status_t spmv_measure_ceiling(int32_t kind, size_t bytes, int32_t reps, void* stream,
                                   double* result);

SPMV_API const char* spmv_status_string(spmv_status_t s);
SPMV_API const char* spmv_last_error(void);   /* thread-local text of the last CUDA/internal error */
SPMV_API const char* spmv_version(void);
SPMV_API void spmv_clear_cache(void);          /* drops the in-process tuning cache */

#ifdef __cplusplus
}
#endif
#endif /* SPMV_B200_H */
