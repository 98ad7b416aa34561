// Compute-side pieces of the row-sharded apply (include/spmv_b200.h):
// nnz-balanced row partition, the set of external columns of a shard (its halo), pack / unpack kernels and
// the row-range apply that lets a shard work on its interior rows while the halo is in flight.
#include <algorithm>
#include <vector>

#include "handle.h"

namespace spmv {

// flags[c] = 1 for every referenced column outside [lo, hi); ext_row[r] = 1 when row r references one
__global__ void ext_flag_kernel(int64_t rows, const int* __restrict__ rp, const int* __restrict__ ci, int lo, int hi,
                                unsigned char* __restrict__ flags, unsigned char* __restrict__ ext_row) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= rows) return;
  bool any = false;
  for (unsigned k = (unsigned)rp[r]; k < (unsigned)rp[r + 1]; ++k) {
    const int c = ci[k];
    if (c < lo || c >= hi) { flags[c] = 1; any = true; }     // benign race: every writer stores 1
  }
  ext_row[r] = any ? 1 : 0;
}

__global__ void gather_kernel(int64_t n, const int* __restrict__ idx, const double* __restrict__ src,
                              double* __restrict__ dst) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = src[idx[i]];
}
__global__ void scatter_kernel(int64_t n, const int* __restrict__ idx, const double* __restrict__ src,
                               double* __restrict__ dst) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[idx[i]] = src[i];
}

}  // namespace spmv

using namespace spmv;

extern "C" {

spmv_status_t spmv_partition_rows(int64_t rows, const int32_t* h_row_ptr, int32_t nparts, int64_t align,
                                  int64_t* h_bounds) {
  if (rows < 0 || !h_row_ptr || nparts < 1 || align < 1 || !h_bounds) return SPMV_ERR_INVALID_ARG;
  const int64_t nnz = h_row_ptr[rows];
  h_bounds[0] = 0;
  for (int g = 1; g < nparts; ++g) {
    // first row r with row_ptr[r] >= g * nnz / nparts, rounded to the nearest multiple of align, monotone
    const int64_t target = (int64_t)((__int128)nnz * g / nparts);
    int64_t r = std::lower_bound(h_row_ptr, h_row_ptr + rows + 1, target,
                                 [](int32_t a, int64_t t) { return (int64_t)a < t; }) - h_row_ptr;
    r = (r + align / 2) / align * align;
    r = std::min(r, rows);
    h_bounds[g] = std::max(r, h_bounds[g - 1]);
  }
  h_bounds[nparts] = rows;
  return SPMV_OK;
}

spmv_status_t spmv_external_columns(spmv_handle_t h, int64_t own_lo, int64_t own_hi, int32_t* h_cols, int64_t cap,
                                    int64_t* count, int64_t* int_lo, int64_t* int_hi, void* stream) {
  if (!handle_alive(h) || !count || own_lo < 0 || own_hi < own_lo || own_hi > h->A.cols) return SPMV_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const int64_t rows = h->A.rows, cols = h->A.cols;
  *count = 0;
  if (int_lo) *int_lo = 0;
  if (int_hi) *int_hi = rows;
  if (rows == 0 || cols == 0) return SPMV_OK;
  const size_t bytes = (size_t)cols + (size_t)rows;
  unsigned char* d = (unsigned char*)h->al.alloc(bytes, s);
  if (!d) return SPMV_ERR_ALLOC;
  std::vector<unsigned char> host(bytes);
  cudaError_t e = cudaMemsetAsync(d, 0, bytes, s);
  if (e == cudaSuccess) {
    ext_flag_kernel<<<(unsigned)((rows + 255) / 256), 256, 0, s>>>(rows, h->A.row_ptr, h->A.col_idx, (int)own_lo,
                                                                 (int)own_hi, d, d + cols);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(host.data(), d, bytes, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  h->al.free(d, bytes);
  if (e != cudaSuccess) { set_last_error("spmv_external_columns: %s", cudaGetErrorString(e)); return SPMV_ERR_CUDA; }
  int64_t n = 0;
  for (int64_t c = 0; c < cols; ++c)
    if (host[c]) { if (h_cols && n < cap) h_cols[n] = (int32_t)c; ++n; }
  *count = n;
  // longest run of rows without external columns
  int64_t best_a = 0, best_b = 0, a = 0;
  const unsigned char* er = host.data() + cols;
  for (int64_t r = 0; r <= rows; ++r) {
    if (r == rows || er[r]) {
      if (r - a > best_b - best_a) { best_a = a; best_b = r; }
      a = r + 1;
    }
  }
  if (int_lo) *int_lo = best_a;
  if (int_hi) *int_hi = best_b;
  return SPMV_OK;
}

spmv_status_t spmv_gather(int64_t n, const int32_t* d_idx, const double* d_src, double* d_dst, void* stream) {
  if (n < 0 || (n > 0 && (!d_idx || !d_src || !d_dst))) return SPMV_ERR_INVALID_ARG;
  if (n == 0) return SPMV_OK;
  gather_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(n, d_idx, d_src, d_dst);
  SPMV_CUDA_TRY(cudaGetLastError());
  return SPMV_OK;
}
spmv_status_t spmv_scatter(int64_t n, const int32_t* d_idx, const double* d_src, double* d_dst, void* stream) {
  if (n < 0 || (n > 0 && (!d_idx || !d_src || !d_dst))) return SPMV_ERR_INVALID_ARG;
  if (n == 0) return SPMV_OK;
  scatter_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(n, d_idx, d_src, d_dst);
  SPMV_CUDA_TRY(cudaGetLastError());
  return SPMV_OK;
}

spmv_status_t spmv_apply_rows(spmv_handle_t h, double alpha, const double* d_x, double beta, double* d_y,
                              int64_t row_begin, int64_t row_end, int64_t* align_out, void* stream) {
  if (!h || h->magic != kHandleMagic) return SPMV_ERR_INVALID_ARG;
  if (align_out) *align_out = h->plan.range_kind == RANGE_NONE ? 0 : h->plan.range_align;
  if (row_begin < 0 || row_end < row_begin || row_end > h->A.rows) return SPMV_ERR_INVALID_ARG;
  if (row_begin == row_end) return SPMV_OK;
  if (!d_y || (h->A.cols > 0 && !d_x && alpha != 0.0)) return SPMV_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  if (alpha == 0.0) {                                   // reading A2, on the range
    cudaError_t e = scale_y_launch(row_end - row_begin, beta, d_y + row_begin, s);
    return e == cudaSuccess ? SPMV_OK : SPMV_ERR_CUDA;
  }
  if (row_begin == 0 && row_end == h->A.rows) return spmv_apply(h, alpha, d_x, beta, d_y, stream);
  KernelCall kc;
  const bool aligned = (((uintptr_t)d_x | (uintptr_t)d_y) & 15) == 0;
  if (!plan_for_rows(h->plan, h->A.rows, h->A.cols, row_begin, row_end, aligned, &kc)) {
    set_last_error("spmv_apply_rows: the selected variant has no row-range form, or the range is not aligned");
    return SPMV_ERR_UNSUPPORTED;
  }
  ApplyArgs a{alpha, beta, d_x, d_y, s};
  cudaError_t e = run_call(kc, a);
  if (e != cudaSuccess) { set_last_error("spmv_apply_rows: %s", cudaGetErrorString(e)); return SPMV_ERR_CUDA; }
  return SPMV_OK;
}

}  // extern "C"
