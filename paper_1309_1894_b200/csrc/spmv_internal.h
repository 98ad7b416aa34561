// Internal declarations shared by the translation units of libspmv_b200.so.
// Nothing here is shared with oracle/ (independent paths).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include <string>
#include <vector>

#include "../../include/spmv_b200.h"

namespace spmv {

// ---------------------------------------------------------------- formats
struct CsrView {
  int64_t rows = 0, cols = 0, nnz = 0;
  const int32_t* row_ptr = nullptr;
  const int32_t* col_idx = nullptr;
  const double* val = nullptr;
};

// SELL-C-sigma (ELL is the one-slice case).  Storage is slice-column-major:
//   entry (row r of slice s, position j) at  slice_ptr[s] + j*C + r.
// Padding carries col = -1 and is never multiplied (reading A7).
struct SellFormat {
  int C = 0;                 // rows per slice (multiple of 128; ELL: padded row count)
  int logC = -1;             // log2(C), or -1 when there is a single slice (ELL)
  int sigma = 1;             // sorting window (1: no permutation)
  int64_t nslices = 0;
  int64_t padded = 0;        // stored entries including padding
  int64_t* slice_ptr = nullptr;   // [nslices+1]
  double* val = nullptr;          // [padded]
  int32_t* col = nullptr;         // [padded]  (null in the 16-bit form)
  // 16-bit delta-encoded column indices: col = sbase[slice] + col16, col16 == 0xFFFF
  // marks padding; built only when every slice spans fewer than 65535 columns.  10 bytes per entry.
  uint16_t* col16 = nullptr;      // [padded]
  int32_t* sbase = nullptr;       // [nslices] smallest column of the slice
  int32_t* perm = nullptr;        // [nslices*C] sell row -> original row (or -1); null if sigma==1
  bool is_ell = false;
  // Row splitting (split = L > 0): a row longer than L is cut into ceil(len/L) segments of at most L
  // entries; every segment is a "virtual row" of the SELL structure, so one heavy row can no longer
  // stretch a slice.  perm[p] >= 0: original row (written with the epilogue); -1: padding row;
  // <= -2: the virtual row is a segment, its plain sum goes to part[-(perm[p]+2)] and
  // sell_split_fixup adds the segments of each split row in a fixed order.
  int split = 0;
  int64_t vrows = 0;              // virtual rows (== rows when split == 0)
  int64_t nparts = 0;             // segments of split rows
  int64_t nsplit = 0;             // rows that were split
  double* part = nullptr;         // [nparts] workspace, rewritten by every apply
  int32_t* srow = nullptr;        // [nsplit] original row of split row i
  int32_t* sptr = nullptr;        // [nsplit+1] its segments are part[sptr[i] .. sptr[i+1])
};

// 3x3 BCSR, values transposed per block row:
//   element k (= 3*r + c) of block j of block row b at  9*brow_ptr[b] + k*nb_b + j.
struct BcsrFormat {
  int64_t brows = 0, nblocks = 0;
  int32_t* brow_ptr = nullptr;   // [brows+1]
  int32_t* bcol = nullptr;       // [nblocks] block column
  uint16_t* bcol16 = nullptr;    // [nblocks] 16-bit form (variant key i16): bcol - block row + 32768; built on demand
  double* bval = nullptr;        // [9*nblocks]
  double fill = 0.0;             // nnz / (9*nblocks)
};

// DIA (stencil-aware): nd <= 32 diagonals, diagonal-major values, no column
// indices; mask[row] bit d says whether entry (row, row + off[d]) is stored.
struct DiaFormat {
  int nd = 0;
  int off[32] = {0};             // ascending; entries past nd repeat the last one
  int C = 0, logC = 0;           // slice height (128, 256 or 512)
  int64_t ld = 0;                // rows rounded up to a multiple of C
  double* val = nullptr;         // [nd * ld], slice-major: ((row / C) * nd + d) * C + row % C
  unsigned* mask = nullptr;      // [ld]
  // constant-coefficient detection: is_const when every stored entry of each
  // diagonal holds the same bit pattern; coef[d] is that value.  dia_const then reads no matrix values.
  bool is_const = false;
  double coef[32] = {0};
  void* mask_small = nullptr;    // is_const && nd <= 16: the mask words narrowed to mask_elem bytes per row
  int mask_elem = 4;
  // x windows for the dia_win kernels (kernels_dia_win.cu): groups of near-consecutive offsets share one
  // contiguous window of x per slice
  int ng = 0, win_total = 0;     // groups; total window entries per slice
  int g_lo[32] = {0};            // window start relative to the slice's first row (even)
  int g_len[32] = {0};           // window length (even)
  int g_dst[32] = {0};           // offset of the window inside the stage's window area
  int d_xoff[32] = {0};          // per diagonal: index of x[s*C + off[d]] inside the window area
};

// Merge-path plan: tile t covers merge-path diagonals [t*tile_items, (t+1)*tile_items);
// tile_row[t] = number of row-end items consumed before that diagonal.
struct MergePlan {
  int tile_items = 0;
  int64_t ntiles = 0;
  int32_t* tile_row = nullptr;   // [ntiles+1]
  int32_t* carry_row = nullptr;  // [ntiles]
  double* carry_val = nullptr;   // [ntiles]
};

// ---------------------------------------------------------------- variants
enum Family { FAM_CSR_SCALAR = 0, FAM_CSR_VECTOR, FAM_SELL, FAM_ELL, FAM_MERGE, FAM_BCSR3, FAM_SELL_TMA, FAM_DIA, FAM_DIA_TMA, FAM_DIA_CONST, FAM_DIA_WIN, FAM_DIA_CWIN, FAM_SELL16, FAM_SELL16_TMA, FAM_COUNT };

struct Variant {
  int fam = FAM_CSR_SCALAR;
  int block = 256;   // b: threads per block                       (PAPER.md:23 knob 1)
  int grid = 0;      // g: 0 exact cover, k>0: k * SMs * resident blocks, grid-stride (knob 2)
  int carve = -1;    // co: shared-memory carve-out percent, -1 default         (knob 4)
  int U = 1;         // u: unroll factor (sell_tma: steps per stage)             (knob 5)
  int R = 1;         // r: rows per thread (csr_scalar, sell)
  int W = 1;         // w: lanes per row (csr_vector), lanes per block row (bcsr3)
  int X = 0;         // x: 0 read-only path (ld.global.nc), 1 plain ld.global, 2 window staged in shared memory
  int H = 0;         // h: half-width of the shared-memory x window around the slice's rows (x2 only)
  int C = 0;         // c: SELL slice height
  int S = 1;         // s: SELL sorting window sigma
  int I = 0;         // i: merge-path items per thread (sell_tma: pipeline stages)
  int L = 0;         // l: SELL row-split length (0: rows are not split)
};

std::string variant_to_string(const Variant& v);
bool variant_from_string(const char* s, Variant* out);
Variant default_variant();

struct ApplyArgs {
  double alpha, beta;
  const double* x;
  double* y;
  cudaStream_t stream;
};

struct DeviceProps {
  int sm_count = 0;
  int64_t l2_bytes = 0;
  char name[64] = {0};
};

// ---------------------------------------------------------------- launch plans
// Everything a launch needs, resolved ONCE (spmv_select / spmv_tune / per tuner candidate): kernel, grid,
// block, dynamic shared memory, and the marshalled argument block.  spmv_apply copies the block, patches
// alpha / x / beta / y (and the few alignment-dependent arguments) and launches: no map lookups, no
// occupancy queries, no attribute calls and no locks on the apply path.
struct KernelCall {
  const void* fn = nullptr;
  unsigned grid = 0, block = 0, smem = 0;
  bool pdl = false;              // programmatic dependent launch (the kernel executes griddepcontrol.wait)
  int nargs = 0, used = 0;
  int off[20] = {0};
  int i_alpha = -1, i_x = -1, i_beta = -1, i_y = -1;
  // arguments that depend on the vectors' alignment: kind 1: int = (y 16-byte aligned), 2: int = (x 16-byte
  // aligned), 3: int64 = flag_val if x is 16-byte aligned else 0
  int flag_idx[2] = {-1, -1}, flag_kind[2] = {0, 0};
  int64_t flag_val = 0;
  // row-range launches (spmv_apply_host pipelines chunks of rows): element offsets added to x / y when the
  // pointers are patched, and the rows (slices, block rows) one block covers, to size a range's grid
  int64_t x_off = 0, y_off = 0, per_block = 0;
  alignas(16) unsigned char store[1280];
  template <typename T>
  void set(int i, const T& v) { memcpy(store + off[i], &v, sizeof(T)); }
  template <typename T>
  T get(int i) const { T v; memcpy(&v, store + off[i], sizeof(T)); return v; }
  template <typename T>
  int add(const T& v) {
    used = (int)((used + alignof(T) - 1) / alignof(T) * alignof(T));
    memcpy(store + used, &v, sizeof(T));
    off[nargs] = used;
    used += (int)sizeof(T);
    return nargs++;
  }
  void add_alpha() { i_alpha = add(0.0); }
  void add_beta() { i_beta = add(0.0); }
  void add_x() { i_x = add((const double*)nullptr); }
  void add_y() { i_y = add((double*)nullptr); }
  void add_flag(int kind, int64_t val = 0) {
    const int slot = flag_idx[0] < 0 ? 0 : 1;
    flag_kind[slot] = kind;
    flag_val = val;
    flag_idx[slot] = kind == 3 ? add((int64_t)0) : add((int)0);
  }
};
// how (whether) a plan can be re-aimed at a range of rows: which arguments shift (variants.cu: plan_for_rows)
enum RangeKind { RANGE_NONE = 0, RANGE_CSR, RANGE_BCSR, RANGE_SELL, RANGE_SELL_TMA, RANGE_DIA, RANGE_DIA_TMA, RANGE_DIA_CONST };
struct LaunchPlan {
  int range_kind = RANGE_NONE;
  int range_align = 1;           // range boundaries are multiples of this many rows
  int range_elem = 0;            // kind-specific (DIA: diagonals; dia_const: bytes per mask word)
  int n = 0;                     // kernel launches per apply (0: nothing to do)
  KernelCall k[2];               // [1]: the ordered fix-up of merge-path / row-split SELL
  bool has_alt = false;          // alt replaces k[0] when x or y is not 16-byte aligned (dia_const pairs)
  KernelCall alt;
};
cudaError_t run_plan(const LaunchPlan& p, const ApplyArgs& a);
cudaError_t run_call(const KernelCall& c, const ApplyArgs& a);
// the plan's kernel call re-aimed at rows [a, b) (a a multiple of range_align; b too, or b == rows); the x / y
// pointers passed at run time stay those of the WHOLE vectors.  false: this plan has no range form.
bool plan_for_rows(const LaunchPlan& p, int64_t rows, int64_t cols, int64_t a, int64_t b, bool aligned, KernelCall* out);
// grid for "g waves of resident blocks" (Variant::grid > 0), capped at the exact cover; sets nothing
cudaError_t resolve_grid(int g, const void* fn, int block, size_t smem, int sm_count, int64_t exact, unsigned* grid);
// cudaFuncAttributeMaxDynamicSharedMemorySize (per device and function: set at every plan build)
cudaError_t allow_smem(const void* fn, size_t smem);

// Per-family entry points (kernels_*.cu).  `supported` checks template-parameter
// availability only; structural eligibility is decided by the tuner / select.  `plan` fills the
// launch plan for a built format.
bool csr_scalar_supported(const Variant&);
cudaError_t csr_scalar_plan(const Variant&, const CsrView&, int sm_count, LaunchPlan*);
bool csr_vector_supported(const Variant&);
cudaError_t csr_vector_plan(const Variant&, const CsrView&, int sm_count, LaunchPlan*);
bool sell_supported(const Variant&);
cudaError_t sell_plan(const Variant&, int64_t rows, const SellFormat&, int sm_count, LaunchPlan*);
bool sell_tma_supported(const Variant&);
cudaError_t sell_tma_plan(const Variant&, int64_t rows, int64_t cols, const SellFormat&, int sm_count, LaunchPlan*);
// adds the segment sums of split rows in a fixed order (after a SELL kernel ran on a split format)
void sell_split_fixup_call(const SellFormat&, KernelCall*);
bool merge_supported(const Variant&);
cudaError_t merge_plan(const Variant&, const CsrView&, const MergePlan&, LaunchPlan*);
bool bcsr_supported(const Variant&);
cudaError_t bcsr_plan(const Variant&, const BcsrFormat&, int sm_count, LaunchPlan*);
bool dia_supported(const Variant&);
cudaError_t dia_plan(const Variant&, int64_t rows, const DiaFormat&, int sm_count, LaunchPlan*);
bool dia_const_supported(const Variant&);
cudaError_t dia_const_plan(const Variant&, int64_t rows, int64_t cols, const DiaFormat&, LaunchPlan*);
// y = alpha*A*x + beta*y AND part[b] = block b's share of sum_i x_i*y_i (square matrix); *n_part = blocks
cudaError_t dia_const_dot_plan(const Variant&, int64_t rows, int64_t cols, const DiaFormat&, double* part,
                               int* n_part, LaunchPlan*);
// one weighted-Jacobi step fused into the constant-coefficient stencil product: x_next = x + omega * (b - A x) / d (d =
// the coefficient of the offset-0 diagonal; the caller guarantees every row stores it, else *done is set) and
// part[block] = the block's share of ||b - A x||^2; a no-op once *done != 0.  blocks: how many partials it writes
int dia_const_jacobi_blocks(const Variant&, int64_t rows);
cudaError_t dia_const_jacobi_launch(const Variant&, int64_t rows, int64_t cols, const DiaFormat&, double omega,
                                    const double* x, double* x_next, const double* b, double* part,
                                    const int* done, cudaStream_t s);
bool dia_win_supported(const Variant&);
bool dia_win_fits(const Variant&, const DiaFormat&);
cudaError_t dia_win_plan(const Variant&, int64_t rows, int64_t cols, const DiaFormat&, int sm_count, LaunchPlan*);
void dia_compute_windows(DiaFormat& f);
bool dia_tma_supported(const Variant&);
cudaError_t dia_tma_plan(const Variant&, int64_t rows, int64_t cols, const DiaFormat&, int sm_count, LaunchPlan*);

// Launch through cudaLaunchKernelExC; pdl = true marks the launch as a programmatic dependent launch
// (cudaLaunchAttributeProgrammaticStreamSerialization): the kernel may start while the previous kernel of
// the stream drains, and MUST execute griddepcontrol.wait (device_utils.cuh: pdl_wait) before it touches
// anything a previous kernel may write or still read.
inline cudaError_t launch_kernel_pdl(const void* k, unsigned grid, unsigned block, size_t smem, cudaStream_t s,
                                     void** args, bool pdl = true) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid, 1, 1);
  cfg.blockDim = dim3(block, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelExC(&cfg, k, args);
}

// y = beta*y (or 0): the alpha == 0 path (reading A2)
cudaError_t scale_y_launch(int64_t rows, double beta, double* y, cudaStream_t s);

// ---------------------------------------------------------------- allocator
struct Allocator {
  spmv_allocator_t cb{};
  bool has_cb = false;
  int64_t owned = 0;
  void* alloc(size_t bytes, cudaStream_t s);
  void free(void* p, size_t bytes);
};

// ---------------------------------------------------------------- converters / stats (convert.cu)
struct RawStats {   // filled on the device, copied back once
  unsigned long long bad_row_ptr, bad_col;
  unsigned long long sum_len, sum_len_sq;
  unsigned long long hist[32];
  unsigned long long sig_row_ptr, sig_col_idx;
  unsigned long long unsorted_rows;     // rows whose columns are not strictly ascending
  unsigned long long block3_bad;        // block rows violating the dense aligned 3x3 pattern
  unsigned long long n_blocks3;
  long long bandwidth;
  int min_len, max_len;
};
cudaError_t compute_stats(const CsrView& A, RawStats* h_out, cudaStream_t s);

spmv_status_t build_sell(const CsrView& A, int C, int sigma, bool ell, int split, Allocator& al,
                         cudaStream_t s, SellFormat* out);
// replaces f.col by (sbase, col16); UNSUPPORTED (f left as it was) when a slice spans 65535 columns or more
spmv_status_t sell_narrow_indices(SellFormat& f, Allocator& al, cudaStream_t s);
void free_sell(SellFormat& f, Allocator& al);
spmv_status_t build_bcsr3(const CsrView& A, Allocator& al, cudaStream_t s, BcsrFormat* out);
void free_bcsr3(BcsrFormat& f, Allocator& al);
// bcol16 from bcol (UNSUPPORTED when some |bcol - block row| >= 32768); drop one of the two index arrays
spmv_status_t bcsr3_narrow_indices(BcsrFormat& f, Allocator& al, cudaStream_t s);
void bcsr3_drop_indices(BcsrFormat& f, Allocator& al, bool drop16);
spmv_status_t build_dia(const CsrView& A, int C, Allocator& al, cudaStream_t s, DiaFormat* out);
void free_dia(DiaFormat& f, Allocator& al);
spmv_status_t build_merge_plan(const CsrView& A, int tile_items, Allocator& al, cudaStream_t s,
                               MergePlan* out);
void free_merge_plan(MergePlan& p, Allocator& al);

// ---------------------------------------------------------------- verification kernels (verify.cu)
struct VerifyResult {
  unsigned long long n_fail;
  long long first_fail;
  double max_ratio;
};
// reference: unfused, stored-order, one thread per row; also emits scale
cudaError_t reference_launch(const CsrView& A, double alpha, const double* x, double beta,
                             double* y, double* scale, cudaStream_t s);
cudaError_t compare_launch(int64_t rows, const double* y_test, const double* y_ref,
                           const double* scale, double tol, VerifyResult* d_result, cudaStream_t s);
cudaError_t fill_uniform_launch(double* p, int64_t n, uint64_t seed, cudaStream_t s);
cudaError_t perturb_launch(double* y, int64_t rows, cudaStream_t s);
cudaError_t flush_l2_launch(double* buf, int64_t n, cudaStream_t s);

// error text
void set_last_error(const char* fmt, ...);
const char* last_error_text();
#define SPMV_CUDA_TRY(expr)                                                        \
  do {                                                                             \
    cudaError_t _e = (expr);                                                       \
    if (_e != cudaSuccess) {                                                       \
      spmv::set_last_error("%s:%d %s -> %s", __FILE__, __LINE__, #expr, cudaGetErrorString(_e)); \
      return SPMV_ERR_CUDA;                                                        \
    }                                                                              \
  } while (0)

}  // namespace spmv
