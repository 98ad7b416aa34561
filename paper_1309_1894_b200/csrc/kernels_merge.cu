// Merge-path CSR kernel (north_star (c): "merge-path CSR for
// skewed row lengths").  Restates the published merge-path decomposition: the list of row
// ends (row_ptr[1..rows]) is merged with the list of non-zero indices 0..nnz-1; the merged
// path of rows+nnz items is cut into equal tiles (one per thread block, precomputed once per
// matrix in MergePlan::tile_row) and, inside a tile, into equal per-thread pieces.
//
// Determinism (reading A20): no floating-point atomics.  Partial sums that cross thread
// boundaries are combined by a fixed-shape segmented scan; partial sums that cross tile
// boundaries go to (carry_row, carry_val) and are added in tile order by merge_fixup_kernel.
#include <limits.h>

#include <mutex>

#include "device_utils.cuh"
#include "spmv_internal.h"

namespace spmv {

template <int B, int I>
struct MergeSmem {
  static constexpr int TI = B * I;
  static constexpr size_t bytes = sizeof(double) * TI * 2 + sizeof(int) * (TI + 2) +
                                  sizeof(int) * B + sizeof(double) * B + 32 * (sizeof(int) + sizeof(double)) + 16;
};

template <int B, int I, int X>
__global__ void __launch_bounds__(B)
merge_kernel(int rows, int nnz, const int* __restrict__ rp, const int* __restrict__ ci,
             const double* __restrict__ va, const int* __restrict__ tile_row,
             int* __restrict__ carry_row, double* __restrict__ carry_val, double alpha,
             const double* __restrict__ x, double beta, double* __restrict__ y) {
  constexpr int TI = B * I;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* s_prod = reinterpret_cast<double*>(smem_raw);
  double* s_rowsum = s_prod + TI;
  double* s_cval = s_rowsum + TI;
  double* s_wval = s_cval + B;
  int* s_rowend = reinterpret_cast<int*>(s_wval + 32);
  int* s_ckey = s_rowend + TI + 2;
  int* s_wkey = s_ckey + B;

  const int t = blockIdx.x;
  const int tid = threadIdx.x;
  const int64_t P = (int64_t)rows + nnz;
  const int64_t d0 = (int64_t)t * TI;
  const int64_t d1 = (d0 + TI < P) ? d0 + TI : P;
  const int i0 = __ldg(tile_row + t), i1 = __ldg(tile_row + t + 1);
  const int k0 = (int)(d0 - i0), k1 = (int)(d1 - i1);
  const int nrows_t = i1 - i0;       // rows finished inside this tile
  const int nk = k1 - k0;            // non-zeros consumed inside this tile
  const int tile_len = (int)(d1 - d0);

  // stage row ends (one extra: the row the tile ends inside) and the products
  for (int j = tid; j <= nrows_t; j += B) {
    int r = i0 + j;
    s_rowend[j] = (r < rows) ? __ldg(rp + r + 1) : INT_MAX;
  }
  {
    double v[I];
    int c[I];
#pragma unroll
    for (int u = 0; u < I; ++u) {
      int k = tid + u * B;
      bool in = k < nk;
      v[u] = in ? ld_stream(va + k0 + k) : 0.0;
      c[u] = in ? ld_stream(ci + k0 + k) : -1;
    }
#pragma unroll
    for (int u = 0; u < I; ++u) {
      int k = tid + u * B;
      if (c[u] >= 0) s_prod[k] = v[u] * ldx<X>(x, c[u]);
    }
  }
  __syncthreads();

  // per-thread start on the tile-local merge path
  int ld = tid * I;
  if (ld > tile_len) ld = tile_len;
  int lo = ld - nk > 0 ? ld - nk : 0;
  int hi = ld < nrows_t ? ld : nrows_t;
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (s_rowend[mid] - k0 <= ld - mid - 1) lo = mid + 1; else hi = mid;
  }
  int i = lo, k = ld - lo;
  double s = 0.0;
  int end = ld + I < tile_len ? ld + I : tile_len;
  for (int it = ld; it < end; ++it) {
    if (k < nk && k + k0 < s_rowend[i]) {
      s += s_prod[k];
      ++k;
    } else {
      s_rowsum[i] = s;      // row i0+i ends here; carry-ins are added below
      s = 0.0;
      ++i;
    }
  }

  // segmented inclusive scan of (key = local row the thread ended in, val = open partial sum)
  const int lane = tid & 31, w = tid >> 5;
  int key = i;
  double val = s;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    int kk = __shfl_up_sync(0xffffffffu, key, d);
    double vv = __shfl_up_sync(0xffffffffu, val, d);
    if (lane >= d && kk == key) val += vv;
  }
  if (lane == 31) { s_wkey[w] = key; s_wval[w] = val; }
  __syncthreads();
  if (w == 0) {
    constexpr int NW = B / 32;
    int wk = lane < NW ? s_wkey[lane] : INT_MAX;
    double wv = lane < NW ? s_wval[lane] : 0.0;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      int kk = __shfl_up_sync(0xffffffffu, wk, d);
      double vv = __shfl_up_sync(0xffffffffu, wv, d);
      if (lane >= d && kk == wk) wv += vv;
    }
    if (lane < NW) s_wval[lane] = wv;
  }
  __syncthreads();
  if (w > 0 && s_wkey[w - 1] == key) val += s_wval[w - 1];
  s_ckey[tid] = key;
  s_cval[tid] = val;
  __syncthreads();
  const bool seg_last = (tid == B - 1) || (s_ckey[tid + 1] != key);
  if (seg_last) {
    if (key < nrows_t) {
      s_rowsum[key] += val;              // finished by the next thread of this tile
    } else if (tid == B - 1) {           // the row the tile ends inside
      int row_start = (i1 < rows) ? __ldg(rp + i1) : nnz;
      int from = row_start > k0 ? row_start : k0;
      bool open = (i1 < rows) && (k1 > from);
      carry_row[t] = open ? i1 : -1;
      carry_val[t] = open ? val : 0.0;
    }
  }
  __syncthreads();
  for (int j = tid; j < nrows_t; j += B) store_y(y, i0 + j, alpha, s_rowsum[j], beta);
}

// Adds the tile carry-outs in tile order: one thread per run of equal carry_row.
__global__ void merge_fixup_kernel(int64_t ntiles, const int* __restrict__ carry_row,
                                   const double* __restrict__ carry_val, double alpha,
                                   double* __restrict__ y) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ntiles) return;
  int r = carry_row[t];
  if (r < 0) return;
  if (t > 0 && carry_row[t - 1] == r) return;    // not a run head
  double s = carry_val[t];
  for (int64_t u = t + 1; u < ntiles && carry_row[u] == r; ++u) s += carry_val[u];
  y[r] = fma(alpha, s, y[r]);
}

// One thread per tile boundary: diagonal search on the global row_ptr (done once per matrix).
__global__ void merge_partition_kernel(int rows, int nnz, const int* __restrict__ rp, int tile_items,
                                       int64_t ntiles, int* __restrict__ tile_row) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t > ntiles) return;
  int64_t P = (int64_t)rows + nnz;
  int64_t d = t * tile_items;
  if (d > P) d = P;
  int64_t lo = d - nnz > 0 ? d - nnz : 0;
  int64_t hi = d < rows ? d : rows;
  while (lo < hi) {
    int64_t mid = (lo + hi) >> 1;
    if ((int64_t)__ldg(rp + mid + 1) <= d - mid - 1) lo = mid + 1; else hi = mid;
  }
  tile_row[t] = (int)lo;
}

typedef void (*merge_kernel_t)(int, int, const int*, const int*, const double*, const int*, int*, double*,
                               double, const double*, double, double*);

struct MergeEntry { int B, I, X; merge_kernel_t k; size_t smem; };
#define ME(b, i) {b, i, 0, merge_kernel<b, i, 0>, MergeSmem<b, i>::bytes}, {b, i, 1, merge_kernel<b, i, 1>, MergeSmem<b, i>::bytes}
static const MergeEntry g_merge[] = {ME(128, 5), ME(128, 7), ME(128, 11), ME(256, 5), ME(256, 7), ME(256, 11),
                                     ME(512, 5), ME(512, 7)};
#undef ME

static const MergeEntry* merge_pick(const Variant& v) {
  for (const auto& e : g_merge)
    if (e.B == v.block && e.I == v.I && e.X == v.X) return &e;
  return nullptr;
}

bool merge_supported(const Variant& v) { return merge_pick(v) != nullptr; }
cudaError_t merge_plan(const Variant& v, const CsrView& A, const MergePlan& p, LaunchPlan* out) {
  const MergeEntry* e = merge_pick(v);
  if (!e || p.tile_items != v.block * v.I) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (A.rows == 0) return cudaSuccess;
  KernelCall& c = out->k[0];
  c.fn = (const void*)e->k;
  c.grid = (unsigned)p.ntiles;
  c.block = e->B;
  c.smem = (unsigned)e->smem;
  cudaError_t err = allow_smem(c.fn, c.smem);
  if (err != cudaSuccess) return err;
  c.add((int)A.rows); c.add((int)A.nnz); c.add(A.row_ptr); c.add(A.col_idx); c.add(A.val);
  c.add((const int*)p.tile_row); c.add(p.carry_row); c.add(p.carry_val);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
  KernelCall& f = out->k[1];
  f.fn = (const void*)merge_fixup_kernel;
  f.grid = (unsigned)((p.ntiles + 255) / 256);
  f.block = 256;
  f.add((int64_t)p.ntiles); f.add((const int*)p.carry_row); f.add((const double*)p.carry_val);
  f.add_alpha(); f.add_y();
  out->n = 2;
  return cudaSuccess;
}

spmv_status_t build_merge_plan(const CsrView& A, int tile_items, Allocator& al, cudaStream_t s,
                               MergePlan* out) {
  MergePlan p;
  p.tile_items = tile_items;
  int64_t P = A.rows + A.nnz;
  p.ntiles = (P + tile_items - 1) / tile_items;
  if (p.ntiles == 0) p.ntiles = 1;
  p.tile_row = (int32_t*)al.alloc(sizeof(int32_t) * (p.ntiles + 1), s);
  p.carry_row = (int32_t*)al.alloc(sizeof(int32_t) * p.ntiles, s);
  p.carry_val = (double*)al.alloc(sizeof(double) * p.ntiles, s);
  if (!p.tile_row || !p.carry_row || !p.carry_val) {
    free_merge_plan(p, al);
    return SPMV_ERR_ALLOC;
  }
  merge_partition_kernel<<<(unsigned)((p.ntiles + 1 + 255) / 256), 256, 0, s>>>((int)A.rows, (int)A.nnz, A.row_ptr,
                                                                           tile_items, p.ntiles, p.tile_row);
  SPMV_CUDA_TRY(cudaGetLastError());
  *out = p;
  return SPMV_OK;
}

void free_merge_plan(MergePlan& p, Allocator& al) {
  if (p.tile_row) al.free(p.tile_row, sizeof(int32_t) * (p.ntiles + 1));
  if (p.carry_row) al.free(p.carry_row, sizeof(int32_t) * p.ntiles);
  if (p.carry_val) al.free(p.carry_val, sizeof(double) * p.ntiles);
  p = MergePlan();
}

}  // namespace spmv

// ---------------------------------------------------------------------------------------------------------
// spmv_merge_apply_noalloc (include/spmv_b200.h): the merge-path product above for callers that cannot
// allocate device memory.  Same three kernels as the handle path (merge_partition_kernel, merge_kernel<256,7,0>,
// merge_fixup_kernel), same tile size, hence the same bits as spmv_select("merge:b256:i7:x0") + spmv_apply; the
// only difference is where the tile table and the tile carries live: not in buffers a handle obtained from
// cudaMalloc (build_merge_plan), but in the file-scope array below, which is part of the library image and is
// placed on every GPU that loads the library, for as long as the process runs.
//
// Layout of the array for kNoAllocMaxTiles tiles T:   [0, 8T) carry_val (double) | [8T, 12T) carry_row (int) |
// [12T, 16T + 4) tile_row (int, T + 1 entries).  1 MiB + 256 B in all.
//
// Nothing in it has to start at zero: a call reads only words the same call wrote earlier on the same stream
// (the partition kernel writes tile_row[0..ntiles], every tile of merge_kernel writes its own carry_row /
// carry_val, and the fix-up reads those ntiles entries only), so what an earlier call -- possibly with more
// tiles -- left behind is never looked at.
namespace spmv {

constexpr int kNoAllocBlock = 256, kNoAllocItems = 7;
constexpr int kNoAllocTileItems = kNoAllocBlock * kNoAllocItems;        // 1792 merge-path items per tile
constexpr int64_t kNoAllocMaxTiles = 65536;
constexpr int64_t kNoAllocMaxPath = kNoAllocMaxTiles * kNoAllocTileItems;  // rows + nnz <= 117 440 512
constexpr size_t kNoAllocBytes = (size_t)((16 * kNoAllocMaxTiles + 4 + 255) / 256 * 256);

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

// In host code `g_noalloc_scratch` is only a stand-in the runtime uses to look the array up: its value is not a
// device address and must never reach a kernel.  The address on a given GPU comes from cudaGetSymbolAddress,
// asked once per device with that device current, and is kept here.
constexpr int kNoAllocMaxDevices = 64;
static std::mutex g_noalloc_mu;
static unsigned char* g_noalloc_addr[kNoAllocMaxDevices] = {nullptr};

static spmv_status_t noalloc_scratch_for_current_device(unsigned char** out) {
  int dev = -1;
  SPMV_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoAllocMaxDevices) {
    set_last_error("spmv_merge_apply_noalloc: device ordinal %d is outside the %d this entry point keeps track of",
                   dev, kNoAllocMaxDevices);
    return SPMV_ERR_UNSUPPORTED;
  }
  std::lock_guard<std::mutex> lk(g_noalloc_mu);
  if (!g_noalloc_addr[dev]) {
    unsigned char* p = nullptr;
    SPMV_CUDA_TRY(cudaGetSymbolAddress((void**)&p, g_noalloc_scratch));
    if (!p) {
      set_last_error("spmv_merge_apply_noalloc: cudaGetSymbolAddress returned a null address on device %d", dev);
      return SPMV_ERR_CUDA;
    }
    g_noalloc_addr[dev] = p;
  }
  *out = g_noalloc_addr[dev];
  return SPMV_OK;
}

}  // namespace spmv

extern "C" {

int64_t spmv_merge_noalloc_max_path(void) { return spmv::kNoAllocMaxPath; }

spmv_status_t spmv_merge_apply_noalloc(int64_t rows, int64_t cols, int64_t nnz, const int32_t* d_row_ptr,
                                       const int32_t* d_col_idx, const double* d_val, double alpha,
                                       const double* d_x, double beta, double* d_y, void* stream) {
  using namespace spmv;
  if (rows < 0 || cols < 0 || nnz < 0) return SPMV_ERR_INVALID_ARG;
  if (rows > 0 && (!d_row_ptr || !d_y)) return SPMV_ERR_INVALID_ARG;
  if (nnz > 0 && (!d_col_idx || !d_val)) return SPMV_ERR_INVALID_ARG;
  if (rows > 0x7fffffffll || cols > 0x7fffffffll || nnz > 0x7fffffffll) {
    set_last_error("spmv_merge_apply_noalloc: sizes over the int32 index range");
    return SPMV_ERR_UNSUPPORTED;
  }
  const int64_t path = rows + nnz;
  if (path > kNoAllocMaxPath) {
    set_last_error("spmv_merge_apply_noalloc: rows + nnz = %lld is over the limit of %lld that the built-in "
                   "scratch array (%zu bytes) can serve; use spmv_create / spmv_select / spmv_apply instead",
                   (long long)path, (long long)kNoAllocMaxPath, kNoAllocBytes);
    return SPMV_ERR_UNSUPPORTED;
  }
  cudaStream_t s = (cudaStream_t)stream;
  if (rows == 0) return SPMV_OK;
  if (alpha == 0.0) {                                // y = beta*y: A, x and the scratch are not touched
    cudaError_t e = scale_y_launch(rows, beta, d_y, s);
    if (e != cudaSuccess) { set_last_error("scale kernel: %s", cudaGetErrorString(e)); return SPMV_ERR_CUDA; }
    return SPMV_OK;
  }
  if (cols > 0 && nnz > 0 && !d_x) return SPMV_ERR_INVALID_ARG;
  if (d_x == d_y) return SPMV_ERR_INVALID_ARG;       // x and y must not alias

  unsigned char* base = nullptr;
  spmv_status_t st = noalloc_scratch_for_current_device(&base);
  if (st != SPMV_OK) return st;
  int64_t ntiles = (path + kNoAllocTileItems - 1) / kNoAllocTileItems;
  if (ntiles == 0) ntiles = 1;
  double* carry_val = reinterpret_cast<double*>(base);
  int32_t* carry_row = reinterpret_cast<int32_t*>(base + 8 * kNoAllocMaxTiles);
  int32_t* tile_row = reinterpret_cast<int32_t*>(base + 12 * kNoAllocMaxTiles);

  merge_partition_kernel<<<(unsigned)((ntiles + 1 + 255) / 256), 256, 0, s>>>((int)rows, (int)nnz, d_row_ptr,
                                                                          kNoAllocTileItems, ntiles, tile_row);
  SPMV_CUDA_TRY(cudaGetLastError());
  constexpr size_t smem = MergeSmem<kNoAllocBlock, kNoAllocItems>::bytes;
  static_assert(smem <= 48 * 1024, "needs no opt-in shared memory attribute");
  merge_kernel<kNoAllocBlock, kNoAllocItems, 0><<<(unsigned)ntiles, kNoAllocBlock, smem, s>>>(
      (int)rows, (int)nnz, d_row_ptr, d_col_idx, d_val, tile_row, carry_row, carry_val, alpha, d_x, beta, d_y);
  SPMV_CUDA_TRY(cudaGetLastError());
  merge_fixup_kernel<<<(unsigned)((ntiles + 255) / 256), 256, 0, s>>>(ntiles, carry_row, carry_val, alpha, d_y);
  SPMV_CUDA_TRY(cudaGetLastError());
  return SPMV_OK;
}

}  // extern "C"
