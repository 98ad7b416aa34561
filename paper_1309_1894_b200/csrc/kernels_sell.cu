// SELL-C-sigma / ELL kernel (north_star (c): "SELL-C-sigma
// with coalesced 128-bit vectorised loads of values and column indices").
//
// Row-vectorised layout (SURVEY "SELL layout" option 1): entry (slice s, position j, row r)
// lives at slice_ptr[s] + j*C + r; a thread owns R ADJACENT rows, so one step is one
// R*8-byte load of values and one R*4-byte load of column indices (R=2: double2 + int2,
// R=4: 2 x double2 + int4), fully coalesced across the warp, with no width padding.
// Padding entries have col = -1 and are skipped, never multiplied (reading A7), so a
// NaN/Inf in x cannot leak into a row that CSR would leave clean.
//
// 16-bit form (sell16, SURVEY sec. 8(f) rank 1 "16-bit delta-encoded column indices inside SELL slices"):
// the column of an entry is sbase[slice] + a 16-bit delta (0xFFFF = padding), 10 bytes per stored entry
// instead of 12, for banded matrices that DIA refuses (more than 32 diagonals, fill below one half).
#include <algorithm>

#include "device_utils.cuh"
#include "spmv_internal.h"

namespace spmv {

__device__ __forceinline__ unsigned short ld_stream_u16(const unsigned short* p) {
  unsigned short v;
  asm volatile("ld.global.nc.L1::no_allocate.u16 %0, [%1];" : "=h"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ unsigned ld_stream_u32(const void* p) {     // 4-byte aligned
  unsigned v;
  asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ uint2 ld_stream_u32x2(const void* p) {      // 8-byte aligned
  uint2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ int col_of_delta(unsigned d, int base) { return d == 0xFFFFu ? -1 : base + (int)d; }

template <int R>
struct VecLoad;
template <>
struct VecLoad<1> {
  static __device__ __forceinline__ void load(const double* pv, const int* pc, int, double* v, int* c) {
    v[0] = ld_stream(pv);
    c[0] = ld_stream(pc);
  }
  static __device__ __forceinline__ void load(const double* pv, const unsigned short* pc, int base, double* v, int* c) {
    v[0] = ld_stream(pv);
    c[0] = col_of_delta(ld_stream_u16(pc), base);
  }
};
template <>
struct VecLoad<2> {
  static __device__ __forceinline__ void load(const double* pv, const int* pc, int, double* v, int* c) {
    double2 a = ld_stream2(pv);
    int2 b = ld_stream2(pc);
    v[0] = a.x; v[1] = a.y; c[0] = b.x; c[1] = b.y;
  }
  static __device__ __forceinline__ void load(const double* pv, const unsigned short* pc, int base, double* v, int* c) {
    double2 a = ld_stream2(pv);
    const unsigned b = ld_stream_u32(pc);
    v[0] = a.x; v[1] = a.y;
    c[0] = col_of_delta(b & 0xFFFFu, base); c[1] = col_of_delta(b >> 16, base);
  }
};
template <>
struct VecLoad<4> {
  static __device__ __forceinline__ void load(const double* pv, const int* pc, int, double* v, int* c) {
    double2 a0 = ld_stream2(pv);
    double2 a1 = ld_stream2(pv + 2);
    int4 b = ld_stream4(pc);
    v[0] = a0.x; v[1] = a0.y; v[2] = a1.x; v[3] = a1.y;
    c[0] = b.x; c[1] = b.y; c[2] = b.z; c[3] = b.w;
  }
  static __device__ __forceinline__ void load(const double* pv, const unsigned short* pc, int base, double* v, int* c) {
    double2 a0 = ld_stream2(pv);
    double2 a1 = ld_stream2(pv + 2);
    const uint2 b = ld_stream_u32x2(pc);
    v[0] = a0.x; v[1] = a0.y; v[2] = a1.x; v[3] = a1.y;
    c[0] = col_of_delta(b.x & 0xFFFFu, base); c[1] = col_of_delta(b.x >> 16, base);
    c[2] = col_of_delta(b.y & 0xFFFFu, base); c[3] = col_of_delta(b.y >> 16, base);
  }
};

// heavier instantiations trade occupancy for registers (loads in flight per thread)
constexpr int sell_max_block(int R, int U) { return R * U >= 16 ? 256 : 512; }

// IT = int: 32-bit column indices; IT = unsigned short: 16-bit deltas against sbase[slice]
template <int R, int U, int PERM, int X, typename IT>
__global__ void __launch_bounds__(sell_max_block(R, U))
sell_kernel(int64_t rows, int64_t rows_padded, int C, int logC,
            const int64_t* __restrict__ slice_ptr, const double* __restrict__ sval,
            const IT* __restrict__ scol, const int* __restrict__ sbase, const int* __restrict__ perm,
            double* __restrict__ part, double alpha, const double* __restrict__ x, double beta,
            double* __restrict__ y) {
  // Programmatic dependent launch: the next kernel of the stream may start now; this one reads the format
  // (immutable, owned by the handle) at once and waits for the previous kernel only before it touches x or y.
  pdl_launch_dependents();
  bool waited = false;
  const int64_t G = (int64_t)gridDim.x * blockDim.x;
  for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g * R < rows_padded; g += G) {
    const int64_t r0 = g * R;
    const int64_t s = logC >= 0 ? (r0 >> logC) : 0;
    const int off = (int)(r0 - s * C);
    const int64_t base = __ldg(slice_ptr + s);
    const int w = (int)((__ldg(slice_ptr + s + 1) - base) / C);
    const int cbase = sizeof(IT) == 2 ? __ldg(sbase + s) : 0;
    const double* pv = sval + base + off;
    const IT* pc = scol + base + off;
    double acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = 0.0;
    // destination rows and (beta != 0) the old y values are fetched up front so that their
    // latency overlaps the matrix stream instead of trailing it
    int64_t orow[R];
    double yold[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int64_t row = r0 + r;
      if (PERM) orow[r] = __ldg(perm + row);
      else orow[r] = row < rows ? row : -1;
    }
    if (!waited) { pdl_wait(); waited = true; }
#pragma unroll
    for (int r = 0; r < R; ++r) yold[r] = (beta != 0.0 && orow[r] >= 0) ? y[orow[r]] : 0.0;
    // U steps per trip, every load of the trip issued before the first use; steps beyond
    // the slice width are predicated off (warp-uniform), so U >= w streams a short row in
    // one batch
    for (int j = 0; j < w; j += U) {
      double v[U][R];
      int c[U][R];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        // steps past the slice width re-read the last valid step (in bounds, L2-resident) and
        // are masked afterwards: unconditional loads let the compiler batch all U of them
        const int jj = min(j + u, w - 1);
        VecLoad<R>::load(pv + (int64_t)jj * C, pc + (int64_t)jj * C, cbase, v[u], c[u]);
      }
#pragma unroll
      for (int u = 0; u < U; ++u)
        if (j + u >= w) {
#pragma unroll
          for (int r = 0; r < R; ++r) c[u][r] = -1;
        }
      phase_fence();
      double xv[U][R];
#pragma unroll
      for (int u = 0; u < U; ++u)
#pragma unroll
        for (int r = 0; r < R; ++r) xv[u][r] = ldx<X>(x, max(c[u][r], 0));   // padding reads x[0], masked below
      phase_fence();
#pragma unroll
      for (int u = 0; u < U; ++u)
#pragma unroll
        for (int r = 0; r < R; ++r)
          acc[r] = c[u][r] >= 0 ? fma(v[u][r], xv[u][r], acc[r]) : acc[r];
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (orow[r] >= 0) y[orow[r]] = (beta == 0.0) ? alpha * acc[r] : fma(alpha, acc[r], beta * yold[r]);
      else if (PERM && orow[r] < -1) part[-(orow[r] + 2)] = acc[r];   // segment of a split row
    }
  }
  if (!waited) pdl_wait();
}

// W lanes per split row: lane-strided sums over its segments, then the fixed butterfly over the W lanes -- the
// order depends only on the format, so results are bit-identical across runs (reading A20).  W = 8: a split
// row has ceil(len / l) segments, a handful on the power-law matrix (a full warp per row left 3/4 of the lanes
// idle and took 23 us for 105 K rows; profiles/r02_cfg3_sell_split_ncu_full.md).
constexpr int kFixW = 8;
__global__ void sell_split_fixup_kernel(int64_t nsplit, const int* __restrict__ srow, const int* __restrict__ sptr,
                                        const double* __restrict__ part, double alpha, double beta,
                                        double* __restrict__ y) {
  pdl_launch_dependents();
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / kFixW;
  const int lane = threadIdx.x & (kFixW - 1);
  const bool live = w < nsplit;                      // every lane stays for the shuffles
  const int a = live ? __ldg(sptr + w) : 0, b = live ? __ldg(sptr + w + 1) : 0;
  const int row = live ? __ldg(srow + w) : 0;
  pdl_wait();                                       // part[] is the previous kernel's output
  double s = 0.0;
  for (int k = a + lane; k < b; k += kFixW) s += part[k];
  s = butterfly_sum<kFixW>(s);
  if (live && lane == 0) store_y(y, row, alpha, s, beta);
}

void sell_split_fixup_call(const SellFormat& f, KernelCall* c) {
  *c = KernelCall();
  c->fn = (const void*)sell_split_fixup_kernel;
  c->grid = (unsigned)((f.nsplit * kFixW + 255) / 256);
  c->block = 256;
  c->pdl = true;
  c->add((int64_t)f.nsplit); c->add((const int*)f.srow); c->add((const int*)f.sptr); c->add((const double*)f.part);
  c->add_alpha(); c->add_beta(); c->add_y();
}

template <int PERM, int X, typename IT>
static const void* pick_ru(int R, int U) {
#define P(r, u) if (R == r && U == u) return (const void*)sell_kernel<r, u, PERM, X, IT>;
  P(1, 1) P(1, 2) P(1, 4) P(1, 8) P(2, 1) P(2, 2) P(2, 4) P(2, 8) P(4, 1) P(4, 2) P(4, 4) P(4, 8)
#undef P
  return nullptr;
}
template <typename IT>
static const void* pick_it(const Variant& v, bool perm) {
  if (v.X == 0) return perm ? pick_ru<1, 0, IT>(v.R, v.U) : pick_ru<0, 0, IT>(v.R, v.U);
  if (v.X == 1) return perm ? pick_ru<1, 1, IT>(v.R, v.U) : pick_ru<0, 1, IT>(v.R, v.U);
  return nullptr;
}
static const void* pick(const Variant& v, bool perm) {
  return v.fam == FAM_SELL16 ? pick_it<unsigned short>(v, perm) : pick_it<int>(v, perm);
}

bool sell_supported(const Variant& v) {
  if (pick(v, false) == nullptr) return false;
  if (v.block < 32 || v.block > sell_max_block(v.R, v.U) || v.block % 32) return false;
  if (v.fam == FAM_SELL || v.fam == FAM_SELL16) {
    if (v.C < 128 || v.C > 4096 || (v.C & (v.C - 1))) return false;   // power of two, multiple of 32*Rmax
    if (v.S < 1) return false;
    if (v.S > 1 && (v.S % v.C != 0 || v.S > 8192 || (v.S & (v.S - 1)))) return false;
  }
  return true;
}
cudaError_t sell_plan(const Variant& v, int64_t rows, const SellFormat& f, int sm_count, LaunchPlan* out) {
  const bool perm = f.perm != nullptr;
  const void* k = pick(v, perm);
  if (!k || (v.fam == FAM_SELL16) != (f.col16 != nullptr)) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (rows == 0) return cudaSuccess;
  KernelCall& c = out->k[0];
  c.fn = k;
  c.block = v.block;
  c.pdl = true;
  const int64_t rows_padded = f.nslices * (int64_t)f.C;
  const int64_t threads = (rows_padded + v.R - 1) / v.R;
  const int64_t exact = (threads + v.block - 1) / v.block;
  cudaError_t e = resolve_grid(v.grid, c.fn, v.block, 0, sm_count, exact, &c.grid);
  if (e != cudaSuccess) return e;
  c.add(rows); c.add(rows_padded); c.add(f.C); c.add(f.logC); c.add((const int64_t*)f.slice_ptr);
  c.add((const double*)f.val); c.add(f.col16 ? (const void*)f.col16 : (const void*)f.col); c.add((const int*)f.sbase);
  c.add((const int*)f.perm); c.add(f.part);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
  c.per_block = (int64_t)v.block * v.R;
  out->n = 1;
  if (f.split && f.nsplit > 0) { sell_split_fixup_call(f, &out->k[1]); out->n = 2; }
  else if (!f.is_ell && !f.split) {       // slices [s0, s1): the rows of a sorting window stay inside it
    out->range_kind = RANGE_SELL;
    out->range_align = std::max(f.C, f.sigma);
    out->range_elem = f.C;
  }
  return cudaSuccess;
}

}  // namespace spmv
