// Tuner support kernels: the in-library reference program, the output comparison, probe
// vectors, fault injection, L2 flush and the measured ceilings.
//
// the un-annotated program "acts as a reference implementation that can be
// compiled and executed to obtain reference results"; every variant's outputs are compared
// with those before its timing counts.  reference_kernel is that program on the device:
// one thread per row, stored order, unfused multiply and add -- no tuning of any kind.
#include <math.h>

#include <algorithm>

#include "device_utils.cuh"
#include "spmv_internal.h"

namespace spmv {

__global__ void reference_kernel(int64_t rows, const int* __restrict__ rp, const int* __restrict__ ci,
                                 const double* __restrict__ va, double alpha, const double* __restrict__ x,
                                 double beta, double* __restrict__ y, double* __restrict__ scale) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= rows) return;
  double s = 0.0, a = 0.0;
  if (alpha != 0.0) {
    for (int k = rp[i]; k < rp[i + 1]; ++k) {
      const double t = __dmul_rn(va[k], x[ci[k]]);
      s = __dadd_rn(s, t);
      a = __dadd_rn(a, fabs(t));
    }
  }
  if (beta == 0.0) {
    y[i] = __dmul_rn(alpha, s);
    scale[i] = __dmul_rn(fabs(alpha), a);
  } else {
    const double by = __dmul_rn(beta, y[i]);
    y[i] = __dadd_rn(__dmul_rn(alpha, s), by);
    scale[i] = __dadd_rn(__dmul_rn(fabs(alpha), a), fabs(by));
  }
}

cudaError_t reference_launch(const CsrView& A, double alpha, const double* x, double beta, double* y,
                             double* scale, cudaStream_t s) {
  if (A.rows == 0) return cudaSuccess;
  reference_kernel<<<(unsigned)((A.rows + 127) / 128), 128, 0, s>>>(A.rows, A.row_ptr, A.col_idx, A.val, alpha, x,
                                                                 beta, y, scale);
  return cudaGetLastError();
}

// Acceptance rule: |y - ref| <= tol*scale; scale == 0 -> equal values;
// NaN matches NaN; +-Inf matches the same infinity.
__global__ void compare_kernel(int64_t rows, const double* __restrict__ yt, const double* __restrict__ yr,
                               const double* __restrict__ scale, double tol, VerifyResult* __restrict__ res) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= rows) return;
  const double t = yt[i], r = yr[i], sc = scale[i];
  bool ok;
  double ratio = 0.0;
  if (isnan(r)) ok = isnan(t);
  else if (isinf(r)) ok = (t == r);
  else if (isnan(t) || isinf(t)) ok = false;
  else if (sc == 0.0 || isnan(sc)) ok = (t == r);
  else if (isinf(sc)) ok = true;
  else {
    const double d = fabs(t - r);
    ratio = d / sc;
    ok = d <= tol * sc;
  }
  if (ratio > 0.0) atomicMax(reinterpret_cast<unsigned long long*>(&res->max_ratio), (unsigned long long)__double_as_longlong(ratio));
  if (!ok) {
    atomicAdd(&res->n_fail, 1ull);
    atomicMin(&res->first_fail, (long long)i);
  }
}

cudaError_t compare_launch(int64_t rows, const double* y_test, const double* y_ref, const double* scale, double tol,
                           VerifyResult* d_result, cudaStream_t s) {
  VerifyResult init;
  init.n_fail = 0;
  init.first_fail = 0x7fffffffffffffffll;
  init.max_ratio = 0.0;
  cudaError_t e = cudaMemcpyAsync(d_result, &init, sizeof(init), cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess || rows == 0) return e;
  compare_kernel<<<(unsigned)((rows + 255) / 256), 256, 0, s>>>(rows, y_test, y_ref, scale, tol, d_result);
  return cudaGetLastError();
}

// Probe vectors: U[-1,1) from a counter hash (the tuner's own; not the test generators').
__global__ void fill_uniform_kernel(double* __restrict__ p, int64_t n, unsigned long long seed) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  unsigned long long z = (unsigned long long)i * 0x9E3779B97F4A7C15ull + seed * 0xD1B54A32D192ED03ull + 0x2545F4914F6CDD1Dull;
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
  z ^= z >> 27; z *= 0x94D049BB133111EBull;
  z ^= z >> 31;
  p[i] = (double)(z >> 11) * (2.0 / 9007199254740992.0) - 1.0;
}
cudaError_t fill_uniform_launch(double* p, int64_t n, uint64_t seed, cudaStream_t s) {
  if (n == 0) return cudaSuccess;
  fill_uniform_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(p, n, seed);
  return cudaGetLastError();
}

// TEST-ONLY fault injection: perturb one output element.
__global__ void perturb_kernel(double* y, int64_t rows) {
  const int64_t i = rows / 2;
  y[i] = y[i] * 1.001 + 1.0;
}
cudaError_t perturb_launch(double* y, int64_t rows, cudaStream_t s) {
  if (rows == 0) return cudaSuccess;
  perturb_kernel<<<1, 1, 0, s>>>(y, rows);
  return cudaGetLastError();
}

__global__ void flush_kernel(double* __restrict__ buf, int64_t n) {
  const int64_t G = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += G) buf[i] = (double)i;
}
cudaError_t flush_l2_launch(double* buf, int64_t n, cudaStream_t s) {
  flush_kernel<<<148 * 8, 256, 0, s>>>(buf, n);
  return cudaGetLastError();
}

// ------------------------------------------------------------------ measured ceilings
__global__ void ceiling_copy_kernel(const double2* __restrict__ src, double2* __restrict__ dst, int64_t n) {
  const int64_t G = (int64_t)gridDim.x * blockDim.x;
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (; i + 3 * G < n; i += 4 * G) {
    double2 a = src[i], b = src[i + G], c = src[i + 2 * G], d = src[i + 3 * G];
    dst[i] = a; dst[i + G] = b; dst[i + 2 * G] = c; dst[i + 3 * G] = d;
  }
  for (; i < n; i += G) dst[i] = src[i];
}
__global__ void ceiling_read_kernel(const double2* __restrict__ src, int64_t n, double* __restrict__ out) {
  const int64_t G = (int64_t)gridDim.x * blockDim.x;
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double s = 0.0;
  for (; i + 3 * G < n; i += 4 * G) {
    double2 a = src[i], b = src[i + G], c = src[i + 2 * G], d = src[i + 3 * G];
    s += (a.x + a.y) + (b.x + b.y) + (c.x + c.y) + (d.x + d.y);
  }
  for (; i < n; i += G) s += src[i].x + src[i].y;
  if (s == 1.2345e300) out[0] = s;   // keeps the loads alive without a write stream
}
__global__ void ceiling_empty_kernel() {}
// Random 8-byte gathers out of an L2-resident vector: the ceiling of the x path for matrices
// with unstructured columns (cfg3).  The index stream is precomputed (counter hash) and read
// coalesced, 8 gathers in flight per thread.
__global__ void ceiling_index_kernel(int* __restrict__ idx, int64_t n, int64_t nx) {
  const int64_t G = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += G) {
    unsigned long long z = (unsigned long long)i * 0x9E3779B97F4A7C15ull;
    z ^= z >> 29; z *= 0xBF58476D1CE4E5B9ull; z ^= z >> 32;
    idx[i] = (int)__umul64hi(z, (unsigned long long)nx);
  }
}
__global__ void ceiling_gather_kernel(const double* __restrict__ x, const int* __restrict__ idx, int64_t n,
                                      double* __restrict__ out) {
  const int64_t G = (int64_t)gridDim.x * blockDim.x;
  double s = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += 8 * G) {
    int c[8];
    double v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) c[u] = (i + u * G < n) ? __ldcs(idx + i + u * G) : 0;
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = __ldg(x + c[u]);
#pragma unroll
    for (int u = 0; u < 8; ++u) s += v[u];
  }
  if (s == 1.2345e300) out[0] = s;
}

// The VALUE loads of bcsr3_kernel<16, 2, ...> and nothing else (no block columns, no x, no FMA chain, no y): `nrec`
// records of 9 * nb doubles, element k of block j of record r at r * 9 * nb + k * nb + j; 16 lanes per record, lane l
// reads blocks l and l + 16 of each of the nine element streams -- runs of nb doubles that start at any 8-byte
// boundary.  Answers: is the block-row layout's load pattern (many short unaligned runs through LSU) what keeps the
// bcsr3 winner below the one-stream read ceiling, or is it the rest of the kernel?
__global__ void __launch_bounds__(512)
ceiling_blockrow_kernel(const double* __restrict__ src, int64_t nrec, int nb, double* __restrict__ out) {
  constexpr int T = 16, U = 2;
  const int lane = threadIdx.x & (T - 1);
  const int64_t nsub = ((int64_t)gridDim.x * blockDim.x) / T;
  double s = 0.0;
  for (int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / T; r < nrec; r += nsub) {
    const double* pv = src + r * 9 * (int64_t)nb;
    for (int j = lane; j < nb; j += T * U) {
      double v[U][9];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int jj = j + u * T;
#pragma unroll
        for (int k = 0; k < 9; ++k) v[u][k] = jj < nb ? ld_stream(pv + (int64_t)k * nb + jj) : 0.0;
      }
#pragma unroll
      for (int u = 0; u < U; ++u)
#pragma unroll
        for (int k = 0; k < 9; ++k) s += v[u][k];
    }
  }
  if (s == 1.2345e300) out[0] = s;
}

}  // namespace spmv

extern "C" spmv_status_t spmv_measure_ceiling(int32_t kind, size_t bytes, int32_t reps, void* stream, double* result) {
  using namespace spmv;
  if (!result || reps <= 0) return SPMV_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  cudaEvent_t e0, e1;
  SPMV_CUDA_TRY(cudaEventCreate(&e0));
  SPMV_CUDA_TRY(cudaEventCreate(&e1));
  float ms = 0.f;
  if (kind == 2) {
    for (int i = 0; i < 10; ++i) ceiling_empty_kernel<<<1, 32, 0, s>>>();
    SPMV_CUDA_TRY(cudaEventRecord(e0, s));
    for (int i = 0; i < reps; ++i) ceiling_empty_kernel<<<1, 32, 0, s>>>();
    SPMV_CUDA_TRY(cudaEventRecord(e1, s));
    SPMV_CUDA_TRY(cudaEventSynchronize(e1));
    SPMV_CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
    *result = (double)ms * 1e3 / reps;
  } else if (kind == 0 || kind == 1) {
    // `bytes` per launch; the launches of a batch run back to back (as the applies in bench.py do) and
    // rotate over windows of a buffer of >= 768 MB so that every launch streams from HBM, not from L2
    const int64_t n = (int64_t)(bytes / 16);
    if (n <= 0) return SPMV_ERR_INVALID_ARG;
    const int64_t nwin = std::max<int64_t>(1, ((int64_t)768 << 20) / (n * 16) + 1);
    double2 *a = nullptr, *b = nullptr;
    double* o = nullptr;
    SPMV_CUDA_TRY(cudaMalloc(&a, nwin * n * 16));
    if (kind == 0) SPMV_CUDA_TRY(cudaMalloc(&b, nwin * n * 16));
    SPMV_CUDA_TRY(cudaMalloc(&o, 8));
    SPMV_CUDA_TRY(cudaMemsetAsync(a, 0, nwin * n * 16, s));
    const int grid = 148 * 8, block = 256;
    const int K = (int)std::max<int64_t>(4, std::min<int64_t>(64, ((int64_t)2 << 30) / (n * 16)));
    double best = 0.0;
    int64_t w = 0;
    for (int i = 0; i < reps + 2; ++i) {
      SPMV_CUDA_TRY(cudaEventRecord(e0, s));
      for (int k = 0; k < K; ++k, w = (w + 1) % nwin) {
        if (kind == 0) ceiling_copy_kernel<<<grid, block, 0, s>>>(a + w * n, b + w * n, n);
        else ceiling_read_kernel<<<grid, block, 0, s>>>(a + w * n, n, o);
      }
      SPMV_CUDA_TRY(cudaEventRecord(e1, s));
      SPMV_CUDA_TRY(cudaEventSynchronize(e1));
      SPMV_CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
      const double gbs = (kind == 0 ? 2.0 : 1.0) * (double)K * (double)n * 16.0 / ((double)ms * 1e6);
      if (i >= 2 && gbs > best) best = gbs;
    }
    *result = best;
    cudaFree(a);
    if (b) cudaFree(b);
    cudaFree(o);
  } else if (kind == 3) {
    // bytes = size of the gathered vector; 64 M gathers per timed launch, indices precomputed and
    // streamed (4 bytes per gather, as a SpMV kernel streams its column indices)
    const int64_t nx = (int64_t)(bytes / 8), n = (int64_t)1 << 26;
    if (nx <= 0 || nx > 0x7fffffff) return SPMV_ERR_INVALID_ARG;
    double *xv = nullptr, *o = nullptr;
    int* idx = nullptr;
    SPMV_CUDA_TRY(cudaMalloc(&xv, nx * 8));
    SPMV_CUDA_TRY(cudaMalloc(&idx, n * 4));
    SPMV_CUDA_TRY(cudaMalloc(&o, 8));
    SPMV_CUDA_TRY(cudaMemsetAsync(xv, 0, nx * 8, s));
    ceiling_index_kernel<<<148 * 8, 512, 0, s>>>(idx, n, nx);
    double best = 0.0;
    for (int i = 0; i < reps + 2; ++i) {
      SPMV_CUDA_TRY(cudaEventRecord(e0, s));
      ceiling_gather_kernel<<<148 * 8, 512, 0, s>>>(xv, idx, n, o);
      SPMV_CUDA_TRY(cudaEventRecord(e1, s));
      SPMV_CUDA_TRY(cudaEventSynchronize(e1));
      SPMV_CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
      const double gps = (double)n / ((double)ms * 1e6);     // giga-gathers per second
      if (i >= 2 && gps > best) best = gps;
    }
    *result = best;
    cudaFree(xv);
    cudaFree(idx);
    cudaFree(o);
  } else if (kind == 4) {
    // `bytes` per launch as records of 27 blocks (cfg4's interior block rows: 1944 B each), launches back to back
    // over rotating windows of a >= 768 MB buffer like kinds 0 / 1; MEDIAN batch (the protocol of the applies)
    const int nb = 27;
    const int64_t nrec = (int64_t)(bytes / (72 * nb)), n = nrec * 9 * nb;
    if (nrec <= 0) return SPMV_ERR_INVALID_ARG;
    const int64_t nwin = std::max<int64_t>(1, ((int64_t)768 << 20) / (n * 8) + 1);
    double *a = nullptr, *o = nullptr;
    SPMV_CUDA_TRY(cudaMalloc(&a, nwin * n * 8));
    SPMV_CUDA_TRY(cudaMalloc(&o, 8));
    SPMV_CUDA_TRY(cudaMemsetAsync(a, 0, nwin * n * 8, s));
    const int K = (int)std::max<int64_t>(4, std::min<int64_t>(64, ((int64_t)2 << 30) / (n * 8)));
    std::vector<double> all;
    int64_t w = 0;
    for (int i = 0; i < reps + 2; ++i) {
      SPMV_CUDA_TRY(cudaEventRecord(e0, s));
      for (int k = 0; k < K; ++k, w = (w + 1) % nwin)
        ceiling_blockrow_kernel<<<148 * 8 * 8, 128, 0, s>>>(a + w * n, nrec, nb, o);
      SPMV_CUDA_TRY(cudaEventRecord(e1, s));
      SPMV_CUDA_TRY(cudaEventSynchronize(e1));
      SPMV_CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
      if (i >= 2) all.push_back((double)K * (double)n * 8.0 / ((double)ms * 1e6));
    }
    std::sort(all.begin(), all.end());
    *result = all[all.size() / 2];
    cudaFree(a);
    cudaFree(o);
  } else {
    return SPMV_ERR_INVALID_ARG;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return SPMV_OK;
}
