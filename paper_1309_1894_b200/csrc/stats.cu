// Ingest: validation + statistics + structure signature.
// Integer-only work; every reduction is an integer atomic, so results are order-independent.
#include "spmv_internal.h"

namespace spmv {

__device__ __forceinline__ unsigned long long mix2(unsigned long long a, unsigned long long b) {
  unsigned long long z = a * 0x9E3779B97F4A7C15ull + b + 0x7F4A7C159E3779B9ull;
  z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
  z ^= z >> 27; z *= 0x94D049BB133111EBull;
  z ^= z >> 31;
  return z;
}

template <typename T, typename Op>
__device__ __forceinline__ T warp_reduce(T v, Op op) {
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) v = op(v, __shfl_xor_sync(0xffffffffu, v, d));
  return v;
}

__global__ void stats_rows_kernel(int64_t rows, int64_t cols, int64_t nnz, const int* __restrict__ rp,
                                  const int* __restrict__ ci, RawStats* __restrict__ st) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool ok = i < rows;
  __shared__ unsigned int s_hist[32];           // per-block histogram: 32 global atomics per block, not one per row
  if (threadIdx.x < 32) s_hist[threadIdx.x] = 0;
  __syncthreads();
  unsigned long long bad_rp = 0, bad_col = 0, len_u = 0, len_sq = 0, sig_rp = 0, sig_ci = 0, unsorted = 0;
  long long bw = 0;
  int len = 0, mn = 0x7fffffff, mx = 0;
  if (i == 0) {
    if (rp[0] != 0 || (int64_t)rp[rows] != nnz) bad_rp = 1;
    sig_rp += mix2((unsigned long long)rows, (unsigned long long)(unsigned)rp[rows]);
  }
  if (ok) {
    const int a = rp[i], b = rp[i + 1];
    sig_rp += mix2((unsigned long long)i, (unsigned long long)(unsigned)a);
    if (a < 0 || b < a || (int64_t)b > nnz) {
      bad_rp += 1;
    } else {
      len = b - a;
      mn = mx = len;
      len_u = (unsigned long long)len;
      len_sq = len_u * len_u;
      int prev = -1;
      bool sorted = true;
      for (int k = a; k < b; ++k) {
        const int c = ci[k];
        sig_ci += mix2((unsigned long long)k, (unsigned long long)(unsigned)c);
        if (c < 0 || (int64_t)c >= cols) bad_col += 1;
        long long d = (long long)c - (long long)i;
        if (d < 0) d = -d;
        if (d > bw) bw = d;
        if (c <= prev) sorted = false;
        prev = c;
      }
      if (!sorted) unsorted = 1;
      int bin = len == 0 ? 0 : (32 - __clz(len));     // 2^(bin-1) <= len < 2^bin
      if (bin > 31) bin = 31;
      atomicAdd(&s_hist[bin], 1u);
    }
  }
  __syncthreads();
  if (threadIdx.x < 32 && s_hist[threadIdx.x]) atomicAdd(&st->hist[threadIdx.x], (unsigned long long)s_hist[threadIdx.x]);
  auto add = [](unsigned long long x, unsigned long long y) { return x + y; };
  bad_rp = warp_reduce(bad_rp, add);
  bad_col = warp_reduce(bad_col, add);
  len_u = warp_reduce(len_u, add);
  len_sq = warp_reduce(len_sq, add);
  sig_rp = warp_reduce(sig_rp, add);
  sig_ci = warp_reduce(sig_ci, add);
  unsorted = warp_reduce(unsorted, add);
  bw = warp_reduce(bw, [](long long x, long long y) { return x > y ? x : y; });
  mn = warp_reduce(ok ? mn : 0x7fffffff, [](int x, int y) { return x < y ? x : y; });
  mx = warp_reduce(mx, [](int x, int y) { return x > y ? x : y; });
  if ((threadIdx.x & 31) == 0) {
    if (bad_rp) atomicAdd(&st->bad_row_ptr, bad_rp);
    if (bad_col) atomicAdd(&st->bad_col, bad_col);
    atomicAdd(&st->sum_len, len_u);
    atomicAdd(&st->sum_len_sq, len_sq);
    atomicAdd(&st->sig_row_ptr, sig_rp);
    atomicAdd(&st->sig_col_idx, sig_ci);
    if (unsorted) atomicAdd(&st->unsorted_rows, unsorted);
    atomicMax(&st->bandwidth, bw);
    atomicMin(&st->min_len, mn);
    atomicMax(&st->max_len, mx);
  }
}

// Dense aligned 3x3 block pattern: the three rows of a block row hold the same columns,
// and those come as aligned triples (3c, 3c+1, 3c+2).
__global__ void stats_block3_kernel(int64_t brows, const int* __restrict__ rp, const int* __restrict__ ci,
                                    RawStats* __restrict__ st) {
  const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= brows) return;
  const int a0 = rp[3 * b], a1 = rp[3 * b + 1], a2 = rp[3 * b + 2], a3 = rp[3 * b + 3];
  const int L = a1 - a0;
  bool good = (a2 - a1 == L) && (a3 - a2 == L) && (L % 3 == 0);
  if (good) {
    for (int j = 0; j < L; j += 3) {
      const int c = ci[a0 + j];
      good = good && (c % 3 == 0) && ci[a0 + j + 1] == c + 1 && ci[a0 + j + 2] == c + 2;
      if (j > 0) good = good && (c > ci[a0 + j - 1]);
    }
    for (int j = 0; j < L && good; ++j) good = (ci[a1 + j] == ci[a0 + j]) && (ci[a2 + j] == ci[a0 + j]);
  }
  if (!good) atomicAdd(&st->block3_bad, 1ull);
  else if (L) atomicAdd(&st->n_blocks3, (unsigned long long)(L / 3));
}

cudaError_t compute_stats(const CsrView& A, RawStats* h_out, cudaStream_t s) {
  RawStats* d = nullptr;
  cudaError_t e = cudaMalloc(&d, sizeof(RawStats));
  if (e != cudaSuccess) return e;
  RawStats init{};
  init.min_len = 0x7fffffff;
  e = cudaMemcpyAsync(d, &init, sizeof(init), cudaMemcpyHostToDevice, s);
  if (e == cudaSuccess) {
    // row_ptr must be readable even for rows == 0 (one entry)
    int64_t n = A.rows > 0 ? A.rows : 1;
    stats_rows_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(A.rows, A.cols, A.nnz, A.row_ptr, A.col_idx, d);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(h_out, d, sizeof(RawStats), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  // the block check walks the column lists, so it runs only on a validated matrix
  if (e == cudaSuccess && h_out->bad_row_ptr == 0 && h_out->bad_col == 0 && A.rows > 0 && A.rows % 3 == 0 &&
      A.cols % 3 == 0 && h_out->unsorted_rows == 0) {
    int64_t brows = A.rows / 3;
    stats_block3_kernel<<<(unsigned)((brows + 255) / 256), 256, 0, s>>>(brows, A.row_ptr, A.col_idx, d);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_out, d, sizeof(RawStats), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  } else if (e == cudaSuccess) {
    h_out->block3_bad = 1;
  }
  cudaFree(d);
  return e;
}

}  // namespace spmv
