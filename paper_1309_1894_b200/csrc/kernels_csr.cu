// CSR kernels:
//   csr_scalar<R,U,X>: one thread per row, R rows per thread interleaved, unroll U.
//                      <1,1,0> with 256 threads is the fixed DEFAULT variant (reading A17):
//                      the literal CUDA form of the serial row loop the paper's flow starts
//                      from.
//   csr_vector<W,U,X>: W lanes per row (W in 2..32), __shfl_xor butterfly, unroll U.
// Tuning knobs of PAPER.md:23: threads/block (runtime), blocks/grid (exact or grid-stride),
// unroll (template), L1/shared carve-out (function attribute set by the caller).
#include "device_utils.cuh"
#include "spmv_internal.h"

namespace spmv {

template <int R, int U, int X>
__global__ void __launch_bounds__(1024)
csr_scalar_kernel(int rows, const int* __restrict__ rp, const int* __restrict__ ci,
                  const double* __restrict__ va, double alpha, const double* __restrict__ x,
                  double beta, double* __restrict__ y) {
  const int64_t G = (int64_t)gridDim.x * blockDim.x;
  for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < rows; g += G * R) {
    // unsigned: k + U can pass 2^31 - 1 when nnz is near the int32 limit (positions stay below 2^32)
    unsigned k[R], e[R];
    double s[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      int64_t row = g + (int64_t)r * G;
      bool ok = row < rows;
      k[r] = ok ? (unsigned)__ldg(rp + row) : 0u;
      e[r] = ok ? (unsigned)__ldg(rp + row + 1) : 0u;
      s[r] = 0.0;
    }
    bool more = true;
    while (more) {
      more = false;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        double v[U];
        int c[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {          // all loads first
          bool ok = k[r] + u < e[r];
          v[u] = ok ? __ldg(va + k[r] + u) : 0.0;
          c[u] = ok ? __ldg(ci + k[r] + u) : -1;
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
          if (c[u] >= 0) s[r] = fma(v[u], ldx<X>(x, c[u]), s[r]);
        k[r] += U;
        more |= k[r] < e[r];
      }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      int64_t row = g + (int64_t)r * G;
      if (row < rows) store_y(y, row, alpha, s[r], beta);
    }
  }
}

template <int W, int U, int X>
__global__ void __launch_bounds__(1024)
csr_vector_kernel(int rows, const int* __restrict__ rp, const int* __restrict__ ci,
                  const double* __restrict__ va, double alpha, const double* __restrict__ x,
                  double beta, double* __restrict__ y) {
  const int lane = threadIdx.x & (W - 1);
  const int64_t nsub = ((int64_t)gridDim.x * blockDim.x) / W;
  const int64_t sub0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / W;
  // warp-uniform trip count: the shuffles below need every lane of the warp
  const int64_t warp_first = sub0 - (threadIdx.x & 31) / W;
  for (int64_t base = warp_first; base < rows; base += nsub) {
    const int64_t row = base + (threadIdx.x & 31) / W;
    const bool ok = row < rows;
    const unsigned start = ok ? (unsigned)__ldg(rp + row) : 0u;     // unsigned: k + u*W may pass 2^31 - 1
    const unsigned end = ok ? (unsigned)__ldg(rp + row + 1) : 0u;
    double s = 0.0;
    for (unsigned k = start + lane; k < end; k += W * U) {
      double v[U];
      int c[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const unsigned kk = k + u * W;
        bool in = kk < end;
        v[u] = in ? __ldg(va + kk) : 0.0;
        c[u] = in ? __ldg(ci + kk) : -1;
      }
#pragma unroll
      for (int u = 0; u < U; ++u)
        if (c[u] >= 0) s = fma(v[u], ldx<X>(x, c[u]), s);
    }
    s = butterfly_sum<W>(s);
    if (ok && lane == 0) store_y(y, row, alpha, s, beta);
  }
}

__global__ void scale_y_kernel(int64_t rows, double beta, double* __restrict__ y) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < rows) y[i] = (beta == 0.0) ? 0.0 : beta * y[i];
}

cudaError_t scale_y_launch(int64_t rows, double beta, double* y, cudaStream_t s) {
  if (rows == 0) return cudaSuccess;
  scale_y_kernel<<<(unsigned)((rows + 255) / 256), 256, 0, s>>>(rows, beta, y);
  return cudaGetLastError();
}

// ------------------------------------------------------------------ dispatch tables
typedef void (*csr_kernel_t)(int, const int*, const int*, const double*, double, const double*,
                             double, double*);

template <int X>
static csr_kernel_t scalar_pick_ru(int R, int U) {
#define P(r, u) if (R == r && U == u) return csr_scalar_kernel<r, u, X>;
  P(1, 1) P(1, 2) P(1, 4) P(2, 1) P(2, 2) P(2, 4) P(4, 1) P(4, 2)
#undef P
  return nullptr;
}
static csr_kernel_t scalar_pick(const Variant& v) {
  return v.X == 0 ? scalar_pick_ru<0>(v.R, v.U) : v.X == 1 ? scalar_pick_ru<1>(v.R, v.U) : nullptr;
}

template <int X>
static csr_kernel_t vector_pick_wu(int W, int U) {
#define P(w, u) if (W == w && U == u) return csr_vector_kernel<w, u, X>;
  P(2, 1) P(2, 2) P(2, 4) P(4, 1) P(4, 2) P(4, 4) P(8, 1) P(8, 2) P(8, 4)
  P(16, 1) P(16, 2) P(16, 4) P(32, 1) P(32, 2) P(32, 4)
#undef P
  return nullptr;
}
static csr_kernel_t vector_pick(const Variant& v) {
  return v.X == 0 ? vector_pick_wu<0>(v.W, v.U) : v.X == 1 ? vector_pick_wu<1>(v.W, v.U) : nullptr;
}

static bool block_ok(int b) { return b >= 32 && b <= 1024 && (b % 32) == 0; }

bool csr_scalar_supported(const Variant& v) { return block_ok(v.block) && scalar_pick(v) != nullptr; }
static void csr_args(KernelCall& c, const CsrView& A) {
  c.add((int)A.rows); c.add(A.row_ptr); c.add(A.col_idx); c.add(A.val);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
}
cudaError_t csr_scalar_plan(const Variant& v, const CsrView& A, int sm_count, LaunchPlan* out) {
  csr_kernel_t k = scalar_pick(v);
  if (!k) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (A.rows == 0) return cudaSuccess;
  KernelCall& c = out->k[0];
  c.fn = (const void*)k;
  c.block = v.block;
  const int64_t exact = (A.rows + (int64_t)v.block * v.R - 1) / ((int64_t)v.block * v.R);
  cudaError_t e = resolve_grid(v.grid, c.fn, v.block, 0, sm_count, exact, &c.grid);
  if (e != cudaSuccess) return e;
  csr_args(c, A);
  c.per_block = (int64_t)v.block * v.R;
  out->n = 1;
  out->range_kind = RANGE_CSR;
  return cudaSuccess;
}

bool csr_vector_supported(const Variant& v) { return block_ok(v.block) && vector_pick(v) != nullptr; }
cudaError_t csr_vector_plan(const Variant& v, const CsrView& A, int sm_count, LaunchPlan* out) {
  csr_kernel_t k = vector_pick(v);
  if (!k) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (A.rows == 0) return cudaSuccess;
  KernelCall& c = out->k[0];
  c.fn = (const void*)k;
  c.block = v.block;
  const int64_t rows_per_block = v.block / v.W;
  const int64_t exact = (A.rows + rows_per_block - 1) / rows_per_block;
  cudaError_t e = resolve_grid(v.grid, c.fn, v.block, 0, sm_count, exact, &c.grid);
  if (e != cudaSuccess) return e;
  csr_args(c, A);
  c.per_block = rows_per_block;
  out->n = 1;
  out->range_kind = RANGE_CSR;
  return cudaSuccess;
}

}  // namespace spmv
