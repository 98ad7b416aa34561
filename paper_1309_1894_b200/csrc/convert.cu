// On-device format converters (north_star (b)):
// CSR -> SELL-C-sigma, CSR -> ELL (one-slice SELL), CSR -> 3x3 BCSR.
// Integer work and copies only; hand-written sort (bitonic per sigma-window) and scan.
#include <algorithm>

#include "spmv_internal.h"

namespace spmv {

// ------------------------------------------------------------------ single-block inclusive scan
// In place over a[1..n]; a[0] must already hold 0.  Off the apply path.
template <typename T>
__global__ void scan_inclusive_kernel(T* __restrict__ a, int64_t n) {
  __shared__ T s_w[32];
  __shared__ T s_carry;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  if (tid == 0) s_carry = 0;
  __syncthreads();
  for (int64_t base = 1; base <= n; base += blockDim.x) {
    const int64_t i = base + tid;
    T v = i <= n ? a[i] : 0;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      T u = __shfl_up_sync(0xffffffffu, v, d);
      if (lane >= d) v += u;
    }
    if (lane == 31) s_w[w] = v;
    __syncthreads();
    if (w == 0) {
      T x = lane < (blockDim.x >> 5) ? s_w[lane] : 0;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        T u = __shfl_up_sync(0xffffffffu, x, d);
        if (lane >= d) x += u;
      }
      s_w[lane] = x;
    }
    __syncthreads();
    const T carry = s_carry;
    v += carry + (w > 0 ? s_w[w - 1] : 0);
    if (i <= n) a[i] = v;
    __syncthreads();
    if (tid == blockDim.x - 1) s_carry = v;
    __syncthreads();
  }
}

// ---- multi-block form: tiles of 1024 entries scanned in place, the tile totals scanned by the single-block
// kernel above, then added back.  In place over a[1..n]; a[0] must already hold 0.
template <typename T>
__global__ void __launch_bounds__(1024) scan_tiles_kernel(T* __restrict__ a, int64_t n, T* __restrict__ totals) {
  __shared__ T s_w[32];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int64_t i = 1 + (int64_t)blockIdx.x * 1024 + tid;
  T v = i <= n ? a[i] : 0;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    T u = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += u;
  }
  if (lane == 31) s_w[w] = v;
  __syncthreads();
  if (w == 0) {
    T x = s_w[lane];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      T u = __shfl_up_sync(0xffffffffu, x, d);
      if (lane >= d) x += u;
    }
    s_w[lane] = x;
  }
  __syncthreads();
  v += w > 0 ? s_w[w - 1] : 0;
  if (i <= n) a[i] = v;
  if (tid == 1023) totals[blockIdx.x + 1] = v;      // totals[0] = 0 is set by the caller's memset
}
template <typename T>
__global__ void scan_add_kernel(T* __restrict__ a, int64_t n, const T* __restrict__ totals) {
  const int64_t i = 1 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= n) a[i] += totals[(i - 1) >> 10];       // inclusive totals of the tiles before this one
}
template <typename T>
static spmv_status_t scan_inclusive(T* a, int64_t n, Allocator& al, cudaStream_t s) {
  if (n <= 0) return SPMV_OK;
  const int64_t ntiles = (n + 1023) / 1024;
  if (ntiles <= 4) {
    scan_inclusive_kernel<T><<<1, 1024, 0, s>>>(a, n);
    SPMV_CUDA_TRY(cudaGetLastError());
    return SPMV_OK;
  }
  T* totals = (T*)al.alloc(sizeof(T) * (ntiles + 1), s);
  if (!totals) return SPMV_ERR_ALLOC;
  cudaError_t e = cudaMemsetAsync(totals, 0, sizeof(T), s);
  if (e == cudaSuccess) {
    scan_tiles_kernel<T><<<(unsigned)ntiles, 1024, 0, s>>>(a, n, totals);
    scan_inclusive_kernel<T><<<1, 1024, 0, s>>>(totals, ntiles);
    scan_add_kernel<T><<<(unsigned)((n + 255) / 256), 256, 0, s>>>(a, n, totals);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);      // totals is freed below
  al.free(totals, sizeof(T) * (ntiles + 1));
  if (e != cudaSuccess) { set_last_error("scan: %s", cudaGetErrorString(e)); return SPMV_ERR_CUDA; }
  return SPMV_OK;
}

// ------------------------------------------------------------------ SELL-C-sigma
// perm[p] = original row stored at SELL position p (or -1).  Within each window of sigma
// positions, rows are ordered by descending length, ties by ascending row (stable).
__global__ void sell_sort_kernel(int64_t rows, int64_t rows_padded, int sigma, const int* __restrict__ rp,
                                 int* __restrict__ perm) {
  extern __shared__ unsigned long long s_key[];
  const int64_t w0 = (int64_t)blockIdx.x * sigma;
  for (int j = threadIdx.x; j < sigma; j += blockDim.x) {
    const int64_t r = w0 + j;
    unsigned long long key = ~0ull;
    if (r < rows) {
      const unsigned len = (unsigned)(rp[r + 1] - rp[r]);
      key = ((unsigned long long)(0x7fffffffu - len) << 32) | (unsigned)j;
    }
    s_key[j] = key;
  }
  __syncthreads();
  for (int k = 2; k <= sigma; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = threadIdx.x; i < sigma; i += blockDim.x) {
        const int p = i ^ j;
        if (p > i) {
          const unsigned long long a = s_key[i], b = s_key[p];
          const bool up = (i & k) == 0;
          if ((a > b) == up) { s_key[i] = b; s_key[p] = a; }
        }
      }
      __syncthreads();
    }
  }
  for (int j = threadIdx.x; j < sigma; j += blockDim.x) {
    const int64_t p = w0 + j;
    if (p < rows_padded) {
      const unsigned long long key = s_key[j];
      perm[p] = key == ~0ull ? -1 : (int)(w0 + (key & 0xffffffffu));
    }
  }
}

// slice_ptr[s+1] = C * max row length in slice s (scanned afterwards)
__global__ void sell_width_kernel(int64_t rows, int64_t nslices, int C, const int* __restrict__ rp,
                                  const int* __restrict__ perm, int64_t* __restrict__ slice_ptr) {
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (warp >= nslices) return;
  int mx = 0;
  for (int j = lane; j < C; j += 32) {
    const int64_t p = warp * C + j;
    const int64_t r = perm ? perm[p] : (p < rows ? p : -1);
    if (r >= 0) mx = max(mx, rp[r + 1] - rp[r]);
  }
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, d));
  if (lane == 0) {
    slice_ptr[warp + 1] = (int64_t)mx * C;
    if (warp == 0) slice_ptr[0] = 0;
  }
}

__global__ void sell_fill_kernel(int64_t rows, int64_t rows_padded, int C, int logC, const int* __restrict__ rp,
                                 const int* __restrict__ ci, const double* __restrict__ va,
                                 const int* __restrict__ perm, const int64_t* __restrict__ slice_ptr,
                                 double* __restrict__ sval, int* __restrict__ scol) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= rows_padded) return;
  const int64_t s = logC >= 0 ? (p >> logC) : 0;
  const int off = (int)(p - s * C);
  const int64_t base = slice_ptr[s];
  const int w = (int)((slice_ptr[s + 1] - base) / C);
  const int64_t r = perm ? perm[p] : (p < rows ? p : -1);
  const int a = r >= 0 ? rp[r] : 0;
  const int len = r >= 0 ? rp[r + 1] - a : 0;
  for (int j = 0; j < w; ++j) {
    const int64_t q = base + (int64_t)j * C + off;
    if (j < len) {
      sval[q] = va[a + j];
      scol[q] = ci[a + j];
    } else {
      sval[q] = 0.0;
      scol[q] = -1;       // padding marker: skipped by the kernel, never multiplied (A7)
    }
  }
}

// ---- row splitting (SellFormat::split): virtual rows
// pass 1: per row, number of virtual rows / partial-sum slots / split flag (scanned afterwards)
__global__ void split_count_kernel(int64_t rows, int L, const int* __restrict__ rp, int* __restrict__ vstart,
                                   int* __restrict__ pstart, int* __restrict__ sidx) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r == 0) { vstart[0] = 0; pstart[0] = 0; sidx[0] = 0; }
  if (r >= rows) return;
  const int len = rp[r + 1] - rp[r];
  const bool split = len > L;
  const int nseg = split ? (len + L - 1) / L : 1;
  vstart[r + 1] = nseg;
  pstart[r + 1] = split ? nseg : 0;
  sidx[r + 1] = split ? 1 : 0;
}
// pass 2: virtual row pointers and targets (original row, or -(2+slot) for a segment)
__global__ void split_fill_kernel(int64_t rows, int64_t vrows, int nnz, int L, const int* __restrict__ rp,
                                  const int* __restrict__ vstart, const int* __restrict__ pstart,
                                  const int* __restrict__ sidx, int* __restrict__ vrp, int* __restrict__ vtarget,
                                  int* __restrict__ srow, int* __restrict__ sptr) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r == 0) { vrp[vrows] = nnz; sptr[sidx[rows]] = pstart[rows]; }
  if (r >= rows) return;
  const int a = rp[r], len = rp[r + 1] - a, v0 = vstart[r];
  if (len <= L) {
    vrp[v0] = a;
    vtarget[v0] = (int)r;
    return;
  }
  const int nseg = vstart[r + 1] - v0, p0 = pstart[r];
  for (int sgm = 0; sgm < nseg; ++sgm) {
    vrp[v0 + sgm] = a + sgm * L;
    vtarget[v0 + sgm] = -(2 + p0 + sgm);
  }
  srow[sidx[r]] = (int)r;
  sptr[sidx[r]] = p0;
}
__global__ void split_compose_kernel(int64_t rows_padded, const int* __restrict__ vtarget, int* __restrict__ perm) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= rows_padded) return;
  const int v = perm[p];
  perm[p] = v >= 0 ? vtarget[v] : -1;
}

// ---- 16-bit delta-encoded column indices
// one warp per slice: smallest and largest stored column; bad[0] counts slices spanning >= 65535 columns
__global__ void sell_span_kernel(int64_t nslices, const int64_t* __restrict__ slice_ptr, const int* __restrict__ scol,
                                 int* __restrict__ sbase, unsigned* __restrict__ bad) {
  const int64_t s = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (s >= nslices) return;
  int lo = 0x7fffffff, hi = -1;
  for (int64_t q = slice_ptr[s] + lane; q < slice_ptr[s + 1]; q += 32) {
    const int c = scol[q];
    if (c >= 0) { lo = min(lo, c); hi = max(hi, c); }
  }
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, d));
    hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, d));
  }
  if (lane == 0) {
    sbase[s] = hi < 0 ? 0 : lo;
    if (hi >= 0 && hi - lo >= 0xFFFF) atomicAdd(bad, 1u);
  }
}
__global__ void sell_narrow_kernel(int64_t nslices, const int64_t* __restrict__ slice_ptr, const int* __restrict__ scol,
                                   const int* __restrict__ sbase, unsigned short* __restrict__ col16) {
  const int64_t s = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (s >= nslices) return;
  const int base = sbase[s];
  for (int64_t q = slice_ptr[s] + lane; q < slice_ptr[s + 1]; q += 32) {
    const int c = scol[q];
    col16[q] = c < 0 ? (unsigned short)0xFFFFu : (unsigned short)(c - base);
  }
}

spmv_status_t sell_narrow_indices(SellFormat& f, Allocator& al, cudaStream_t s) {
  if (f.col16 || !f.col || f.split) return SPMV_ERR_UNSUPPORTED;
  int32_t* sbase = (int32_t*)al.alloc(sizeof(int32_t) * (f.nslices + 1), s);      // [nslices] + the bad-slice counter
  if (!sbase) return SPMV_ERR_ALLOC;
  unsigned* bad = (unsigned*)(sbase + f.nslices);
  unsigned h_bad = 1;
  const unsigned grid = (unsigned)((f.nslices * 32 + 255) / 256);
  cudaError_t e = cudaMemsetAsync(bad, 0, sizeof(unsigned), s);
  if (e == cudaSuccess) {
    sell_span_kernel<<<grid, 256, 0, s>>>(f.nslices, f.slice_ptr, f.col, sbase, bad);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h_bad, bad, sizeof(unsigned), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess || h_bad) {
    al.free(sbase, sizeof(int32_t) * (f.nslices + 1));
    if (e != cudaSuccess) { set_last_error("sell_narrow_indices: %s", cudaGetErrorString(e)); return SPMV_ERR_CUDA; }
    set_last_error("sell16: %u slices span 65535 columns or more", h_bad);
    return SPMV_ERR_UNSUPPORTED;
  }
  uint16_t* c16 = (uint16_t*)al.alloc(sizeof(uint16_t) * f.padded, s);
  if (!c16) { al.free(sbase, sizeof(int32_t) * (f.nslices + 1)); return SPMV_ERR_ALLOC; }
  sell_narrow_kernel<<<grid, 256, 0, s>>>(f.nslices, f.slice_ptr, f.col, sbase, c16);
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) {
    al.free(sbase, sizeof(int32_t) * (f.nslices + 1));
    al.free(c16, sizeof(uint16_t) * f.padded);
    set_last_error("sell_narrow_indices: %s", cudaGetErrorString(e));
    return SPMV_ERR_CUDA;
  }
  al.free(f.col, sizeof(int32_t) * f.padded);
  f.col = nullptr;
  f.col16 = c16;
  f.sbase = sbase;
  return SPMV_OK;
}

void free_sell(SellFormat& f, Allocator& al) {
  if (f.col16) al.free(f.col16, sizeof(uint16_t) * f.padded);
  if (f.sbase) al.free(f.sbase, sizeof(int32_t) * (f.nslices + 1));
  if (f.slice_ptr) al.free(f.slice_ptr, sizeof(int64_t) * (f.nslices + 1));
  if (f.val) al.free(f.val, sizeof(double) * f.padded);
  if (f.col) al.free(f.col, sizeof(int32_t) * f.padded);
  if (f.perm) al.free(f.perm, sizeof(int32_t) * f.nslices * f.C);
  if (f.part) al.free(f.part, sizeof(double) * std::max<int64_t>(f.nparts, 1));
  if (f.srow) al.free(f.srow, sizeof(int32_t) * std::max<int64_t>(f.nsplit, 1));
  if (f.sptr) al.free(f.sptr, sizeof(int32_t) * (f.nsplit + 1));
  f = SellFormat();
}

spmv_status_t build_sell(const CsrView& A0, int C, int sigma, bool ell, int split, Allocator& al, cudaStream_t s,
                         SellFormat* out) {
  SellFormat f;
  // every error return below frees what was built so far (the converters are all-or-nothing)
  struct Guard { SellFormat& f; Allocator& al; bool keep; ~Guard() { if (!keep) free_sell(f, al); } } guard{f, al, false};
  f.is_ell = ell;
  CsrView A = A0;
  f.vrows = A0.rows;
  // temporaries of the split pre-pass, released on every exit path
  int *vstart = nullptr, *pstart = nullptr, *sidx = nullptr, *vrp = nullptr, *vtarget = nullptr;
  const int64_t rows0 = A0.rows;
  int64_t vrows_alloc = 0;
  struct Tmp {
    Allocator& al; int*& a; int*& b; int*& c; int*& d; int*& e; const int64_t& n; int64_t& v;
    ~Tmp() {
      if (a) al.free(a, sizeof(int) * (n + 1));
      if (b) al.free(b, sizeof(int) * (n + 1));
      if (c) al.free(c, sizeof(int) * (n + 1));
      if (d) al.free(d, sizeof(int) * (v + 1));
      if (e) al.free(e, sizeof(int) * std::max<int64_t>(v, 1));
    }
  } tmp{al, vstart, pstart, sidx, vrp, vtarget, rows0, vrows_alloc};
  if (split > 0 && !ell && sigma > 1 && rows0 > 0) {
    f.split = split;
    vstart = (int*)al.alloc(sizeof(int) * (rows0 + 1), s);
    pstart = (int*)al.alloc(sizeof(int) * (rows0 + 1), s);
    sidx = (int*)al.alloc(sizeof(int) * (rows0 + 1), s);
    if (!vstart || !pstart || !sidx) return SPMV_ERR_ALLOC;
    const unsigned g = (unsigned)((rows0 + 255) / 256);
    split_count_kernel<<<g, 256, 0, s>>>(rows0, split, A0.row_ptr, vstart, pstart, sidx);
    SPMV_CUDA_TRY(cudaGetLastError());
    for (int* arr : {vstart, pstart, sidx}) {
      spmv_status_t sst = scan_inclusive<int>(arr, rows0, al, s);
      if (sst != SPMV_OK) return sst;
    }
    int tot[3] = {0, 0, 0};
    SPMV_CUDA_TRY(cudaMemcpyAsync(&tot[0], vstart + rows0, sizeof(int), cudaMemcpyDeviceToHost, s));
    SPMV_CUDA_TRY(cudaMemcpyAsync(&tot[1], pstart + rows0, sizeof(int), cudaMemcpyDeviceToHost, s));
    SPMV_CUDA_TRY(cudaMemcpyAsync(&tot[2], sidx + rows0, sizeof(int), cudaMemcpyDeviceToHost, s));
    SPMV_CUDA_TRY(cudaStreamSynchronize(s));
    f.vrows = tot[0];
    f.nparts = tot[1];
    f.nsplit = tot[2];
    vrows_alloc = f.vrows;
    vrp = (int*)al.alloc(sizeof(int) * (f.vrows + 1), s);
    vtarget = (int*)al.alloc(sizeof(int) * std::max<int64_t>(f.vrows, 1), s);
    f.part = (double*)al.alloc(sizeof(double) * std::max<int64_t>(f.nparts, 1), s);
    f.srow = (int32_t*)al.alloc(sizeof(int32_t) * std::max<int64_t>(f.nsplit, 1), s);
    f.sptr = (int32_t*)al.alloc(sizeof(int32_t) * (f.nsplit + 1), s);
    if (!vrp || !vtarget || !f.part || !f.srow || !f.sptr) return SPMV_ERR_ALLOC;
    split_fill_kernel<<<g, 256, 0, s>>>(rows0, f.vrows, (int)A0.nnz, split, A0.row_ptr, vstart, pstart, sidx, vrp,
                                        vtarget, f.srow, f.sptr);
    SPMV_CUDA_TRY(cudaGetLastError());
    A.rows = f.vrows;
    A.row_ptr = vrp;
  }
  if (ell) {
    int64_t padded_rows = ((A.rows + 127) / 128) * 128;
    if (padded_rows == 0) padded_rows = 128;
    if (padded_rows > 0x7fffff80) return SPMV_ERR_UNSUPPORTED;
    f.C = (int)padded_rows;
    f.logC = -1;
    f.sigma = 1;
    f.nslices = 1;
  } else {
    f.C = C;
    f.logC = 0;
    while ((1 << f.logC) < C) ++f.logC;
    f.sigma = sigma;
    f.nslices = (A.rows + C - 1) / C;
    if (f.nslices == 0) f.nslices = 1;
  }
  const int64_t rows_padded = f.nslices * f.C;
  f.slice_ptr = (int64_t*)al.alloc(sizeof(int64_t) * (f.nslices + 1), s);
  if (!f.slice_ptr) return SPMV_ERR_ALLOC;
  if (f.sigma > 1) {
    f.perm = (int32_t*)al.alloc(sizeof(int32_t) * rows_padded, s);
    if (!f.perm) return SPMV_ERR_ALLOC;
    const int64_t nwin = (rows_padded + f.sigma - 1) / f.sigma;
    const size_t smem = sizeof(unsigned long long) * f.sigma;
    if (smem > 48 * 1024)
      SPMV_CUDA_TRY(cudaFuncSetAttribute((const void*)sell_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    sell_sort_kernel<<<(unsigned)nwin, std::min(1024, std::max(32, f.sigma / 2)), smem, s>>>(A.rows, rows_padded, f.sigma,
                                                                                          A.row_ptr, f.perm);
    SPMV_CUDA_TRY(cudaGetLastError());
  }
  sell_width_kernel<<<(unsigned)((f.nslices * 32 + 255) / 256), 256, 0, s>>>(A.rows, f.nslices, f.C, A.row_ptr, f.perm,
                                                                         f.slice_ptr);
  SPMV_CUDA_TRY(cudaGetLastError());
  {
    spmv_status_t sst = scan_inclusive<int64_t>(f.slice_ptr, f.nslices, al, s);
    if (sst != SPMV_OK) return sst;
  }
  int64_t total = 0;
  SPMV_CUDA_TRY(cudaMemcpyAsync(&total, f.slice_ptr + f.nslices, sizeof(int64_t), cudaMemcpyDeviceToHost, s));
  SPMV_CUDA_TRY(cudaStreamSynchronize(s));
  f.padded = total;
  const int64_t n_alloc = total > 0 ? total : 2;
  f.val = (double*)al.alloc(sizeof(double) * n_alloc, s);
  f.col = (int32_t*)al.alloc(sizeof(int32_t) * n_alloc, s);
  f.padded = n_alloc;
  if (!f.val || !f.col) return SPMV_ERR_ALLOC;
  if (total > 0) {
    sell_fill_kernel<<<(unsigned)((rows_padded + 127) / 128), 128, 0, s>>>(A.rows, rows_padded, f.C, f.logC, A.row_ptr,
                                                                        A.col_idx, A.val, f.perm, f.slice_ptr, f.val,
                                                                        f.col);
    SPMV_CUDA_TRY(cudaGetLastError());
  }
  if (f.split) {
    split_compose_kernel<<<(unsigned)((rows_padded + 255) / 256), 256, 0, s>>>(rows_padded, vtarget, f.perm);
    SPMV_CUDA_TRY(cudaGetLastError());
  }
  SPMV_CUDA_TRY(cudaStreamSynchronize(s));
  guard.keep = true;
  *out = f;
  return SPMV_OK;
}

// ------------------------------------------------------------------ 3x3 BCSR
// Three-way merge over the block columns (col/3) of the three rows of a block row.
// FILL = false: count unique block columns; FILL = true: write bcol and scatter values.
template <bool FILL>
__global__ void bcsr3_merge_kernel(int64_t brows, const int* __restrict__ rp, const int* __restrict__ ci,
                                   const double* __restrict__ va, int* __restrict__ brow_ptr,
                                   int* __restrict__ bcol, double* __restrict__ bval) {
  const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= brows) return;
  int p[3], e[3];
#pragma unroll
  for (int r = 0; r < 3; ++r) { p[r] = rp[3 * b + r]; e[r] = rp[3 * b + r + 1]; }
  const int start = FILL ? brow_ptr[b] : 0;
  const int nb = FILL ? brow_ptr[b + 1] - start : 0;
  int count = 0;
  while (true) {
    int bc = 0x7fffffff;
#pragma unroll
    for (int r = 0; r < 3; ++r)
      if (p[r] < e[r]) bc = min(bc, ci[p[r]] / 3);
    if (bc == 0x7fffffff) break;
#pragma unroll
    for (int r = 0; r < 3; ++r) {
      while (p[r] < e[r] && ci[p[r]] / 3 == bc) {
        if (FILL) bval[9 * (int64_t)start + (int64_t)(3 * r + ci[p[r]] % 3) * nb + count] = va[p[r]];
        ++p[r];
      }
    }
    if (FILL) bcol[start + count] = bc;
    ++count;
  }
  if (!FILL) {
    brow_ptr[b + 1] = count;
    if (b == 0) brow_ptr[0] = 0;
  }
}

// 16-bit block columns (the BCSR counterpart of sell16): a block row of a banded matrix
// references block columns near its own index, so bcol - block row + 32768 fits 16 bits: 74 B per block, not 76
__global__ void bcsr3_narrow_kernel(int64_t brows, const int* __restrict__ bp, const int* __restrict__ bcol,
                                    unsigned short* __restrict__ bcol16, int* __restrict__ bad) {
  const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= brows) return;
  for (int k = bp[b]; k < bp[b + 1]; ++k) {
    const int64_t d = (int64_t)bcol[k] - b + 32768;
    if (d < 0 || d > 65535) { *bad = 1; bcol16[k] = 0; }
    else bcol16[k] = (unsigned short)d;
  }
}

// bytes of the bcol16 allocation: the indices, padded to 4 bytes, then the converter's flag word
static size_t bcol16_bytes(int64_t nblocks) { return (((size_t)std::max<int64_t>(nblocks, 1) * 2 + 3) & ~(size_t)3) + sizeof(int); }

spmv_status_t bcsr3_narrow_indices(BcsrFormat& f, Allocator& al, cudaStream_t s) {
  if (f.bcol16) return SPMV_OK;
  if (!f.bcol) return SPMV_ERR_INTERNAL;
  const size_t bytes = bcol16_bytes(f.nblocks);
  uint16_t* c16 = (uint16_t*)al.alloc(bytes, s);
  if (!c16) return SPMV_ERR_ALLOC;
  struct Guard { uint16_t* p; size_t n; Allocator& al; bool keep; ~Guard() { if (!keep) al.free(p, n); } } guard{c16, bytes, al, false};
  int* d_bad = (int*)((char*)c16 + bytes - sizeof(int));
  SPMV_CUDA_TRY(cudaMemsetAsync(d_bad, 0, sizeof(int), s));
  bcsr3_narrow_kernel<<<(unsigned)((f.brows + 127) / 128), 128, 0, s>>>(f.brows, f.brow_ptr, f.bcol, c16, d_bad);
  SPMV_CUDA_TRY(cudaGetLastError());
  int bad = 0;
  SPMV_CUDA_TRY(cudaMemcpyAsync(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost, s));
  SPMV_CUDA_TRY(cudaStreamSynchronize(s));
  if (bad) { set_last_error("bcsr3 i16: a block column is 32768 or more block rows away from its block row"); return SPMV_ERR_UNSUPPORTED; }
  guard.keep = true;
  f.bcol16 = c16;
  return SPMV_OK;
}

void bcsr3_drop_indices(BcsrFormat& f, Allocator& al, bool drop16) {
  if (drop16 && f.bcol16) { al.free(f.bcol16, bcol16_bytes(f.nblocks)); f.bcol16 = nullptr; }
  if (!drop16 && f.bcol && f.bcol16) { al.free(f.bcol, sizeof(int32_t) * std::max<int64_t>(f.nblocks, 1)); f.bcol = nullptr; }
}

void free_bcsr3(BcsrFormat& f, Allocator& al) {
  if (f.brow_ptr) al.free(f.brow_ptr, sizeof(int32_t) * (f.brows + 1));
  if (f.bcol16) al.free(f.bcol16, bcol16_bytes(f.nblocks));
  if (f.bcol) al.free(f.bcol, sizeof(int32_t) * std::max<int64_t>(f.nblocks, 1));
  if (f.bval) al.free(f.bval, sizeof(double) * 9 * std::max<int64_t>(f.nblocks, 1));
  f = BcsrFormat();
}

spmv_status_t build_bcsr3(const CsrView& A, Allocator& al, cudaStream_t s, BcsrFormat* out) {
  if (A.rows % 3 || A.cols % 3 || A.rows == 0) return SPMV_ERR_UNSUPPORTED;
  BcsrFormat f;
  struct Guard { BcsrFormat& f; Allocator& al; bool keep; ~Guard() { if (!keep) free_bcsr3(f, al); } } guard{f, al, false};
  f.brows = A.rows / 3;
  f.brow_ptr = (int32_t*)al.alloc(sizeof(int32_t) * (f.brows + 1), s);
  if (!f.brow_ptr) return SPMV_ERR_ALLOC;
  const unsigned grid = (unsigned)((f.brows + 127) / 128);
  bcsr3_merge_kernel<false><<<grid, 128, 0, s>>>(f.brows, A.row_ptr, A.col_idx, A.val, f.brow_ptr, nullptr, nullptr);
  SPMV_CUDA_TRY(cudaGetLastError());
  {
    spmv_status_t sst = scan_inclusive<int>(f.brow_ptr, f.brows, al, s);
    if (sst != SPMV_OK) return sst;
  }
  int total = 0;
  SPMV_CUDA_TRY(cudaMemcpyAsync(&total, f.brow_ptr + f.brows, sizeof(int), cudaMemcpyDeviceToHost, s));
  SPMV_CUDA_TRY(cudaStreamSynchronize(s));
  f.nblocks = total;
  const int64_t n_alloc = std::max<int64_t>(f.nblocks, 1);
  f.bcol = (int32_t*)al.alloc(sizeof(int32_t) * n_alloc, s);
  f.bval = (double*)al.alloc(sizeof(double) * 9 * n_alloc, s);
  if (!f.bcol || !f.bval) return SPMV_ERR_ALLOC;
  SPMV_CUDA_TRY(cudaMemsetAsync(f.bval, 0, sizeof(double) * 9 * n_alloc, s));
  bcsr3_merge_kernel<true><<<grid, 128, 0, s>>>(f.brows, A.row_ptr, A.col_idx, A.val, f.brow_ptr, f.bcol, f.bval);
  SPMV_CUDA_TRY(cudaGetLastError());
  SPMV_CUDA_TRY(cudaStreamSynchronize(s));
  f.fill = f.nblocks ? (double)A.nnz / (9.0 * (double)f.nblocks) : 1.0;
  guard.keep = true;
  *out = f;
  return SPMV_OK;
}

}  // namespace spmv
