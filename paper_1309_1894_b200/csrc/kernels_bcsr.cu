// 3x3 BCSR kernel (north_star (c) "3x3 BCSR").
//
// T lanes share a block row; lane l takes blocks l, l+T, ...  The values of a block row
// are stored TRANSPOSED inside the block row (element k of block j at 9*start + k*nb + j),
// a library-owned layout, so that each of the 9 value loads is contiguous across lanes
// instead of striding by 72 bytes.  One int32 block column per 9 values: 8.44 B/nnz
// instead of CSR's 12 (8.22 B/nnz with the 16-bit block columns of variant key i16).  x is read as the 3-vector x[3*bc .. 3*bc+2]: three 8-byte loads (X = 0, 1), or -- X = 3 --
// one aligned 16-byte pair plus one 8-byte load (the pair starts at 3*bc for an even block column, at 3*bc + 1
// for an odd one): a third fewer L1 requests on the x path, which is where this kernel's L1TEX time goes
// (each lane of a warp touches another line of x).  X = 3 needs a 16-byte aligned x; otherwise it runs as X = 0.
#include "device_utils.cuh"
#include "spmv_internal.h"

namespace spmv {

__device__ __forceinline__ int ld_bcol(const int* p, int) { return ld_stream(p); }
// 16-bit form (variant key i16): block column = stored delta - 32768 + the block row's index in the whole matrix.
// Measured on cfg4 (74 instead of 76 B per block): with three 8-byte x loads (x0) 281.5 us against 288.7 us for 32-bit
// block columns and 286 us for the 32-bit x3 form (the round-2 winner until then); with the pair loads of x3 it loses
// (312 vs 286 us; loading the index as its aligned 32-bit word: 320 us).  The tuner's measurement decides per matrix.
__device__ __forceinline__ int ld_bcol(const unsigned short* p, int br_global) {
  unsigned short v;
  asm volatile("ld.global.nc.L1::no_allocate.u16 %0, [%1];" : "=h"(v) : "l"(p));
  return (int)v - 32768 + br_global;
}

// br0: index of the range's first block row in the whole matrix (row-range launches; 0 otherwise)
template <int T, int U, int X, typename IT>
__global__ void __launch_bounds__(X == 3 ? 1024 : 512)
bcsr3_kernel(int brows, const int* __restrict__ bp, const IT* __restrict__ bcol,
             const double* __restrict__ bval, double alpha, const double* __restrict__ x,
             double beta, double* __restrict__ y, int br0) {
  const int lane = threadIdx.x & (T - 1);
  const bool xpair = (reinterpret_cast<uintptr_t>(x) & 15) == 0;
  const int sub_in_warp = (threadIdx.x & 31) / T;
  const int64_t nsub = ((int64_t)gridDim.x * blockDim.x) / T;
  const int64_t warp_first = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / T - sub_in_warp;
  for (int64_t base = warp_first; base < brows; base += nsub) {
    const int64_t br = base + sub_in_warp;
    const bool ok = br < brows;
    const int start = ok ? __ldg(bp + br) : 0;
    const int nb = ok ? __ldg(bp + br + 1) - start : 0;
    const double* pv = bval + 9 * (int64_t)start;
    const IT* pc = bcol + start;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int j = lane; j < nb; j += T * U) {
      double v[U][9];
      int c[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int jj = j + u * T;
        const bool in = jj < nb;
        c[u] = in ? ld_bcol(pc + jj, (int)br + br0) : -1;
#pragma unroll
        for (int k = 0; k < 9; ++k) v[u][k] = in ? ld_stream(pv + (int64_t)k * nb + jj) : 0.0;
      }
      if constexpr (X == 3) {
        // pair loads: per-block branches (measured on cfg4: 286 us; with the loads of both blocks hoisted above the
        // FMAs as in the other branch the kernel needs 70 registers and takes 310 us, 297 us when held to 64)
#pragma unroll
        for (int u = 0; u < U; ++u) {
          if (c[u] >= 0) {
            const double* px = x + 3 * (int64_t)c[u];
            double x0, x1, x2;
            if (xpair) {
              const int p = c[u] & 1;
              const double2 a = __ldg(reinterpret_cast<const double2*>(px + p));
              const double b = __ldg(px + (p ? 0 : 2));
              x0 = p ? b : a.x; x1 = p ? a.x : a.y; x2 = p ? a.y : b;
            } else {
              x0 = ldx<0>(px, 0); x1 = ldx<0>(px, 1); x2 = ldx<0>(px, 2);
            }
            s0 = fma(v[u][0], x0, fma(v[u][1], x1, fma(v[u][2], x2, s0)));
            s1 = fma(v[u][3], x0, fma(v[u][4], x1, fma(v[u][5], x2, s1)));
            s2 = fma(v[u][6], x0, fma(v[u][7], x1, fma(v[u][8], x2, s2)));
          }
        }
      } else {
        // every x load of the trip is issued before the first FMA (measured on cfg4, x0: 306.0 -> 288.7 us; with 16-bit
        // block columns 296.6 -> 281.5 us).  A lane past the end of the block row reads block column 0 and is never
        // multiplied: its sums are selected, not its products zeroed, so a non-finite x[0..2] cannot leak into the row.
        double xx[U][3];
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const double* px = x + 3 * (int64_t)max(c[u], 0);
          xx[u][0] = ldx<X>(px, 0); xx[u][1] = ldx<X>(px, 1); xx[u][2] = ldx<X>(px, 2);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const double t0 = fma(v[u][0], xx[u][0], fma(v[u][1], xx[u][1], fma(v[u][2], xx[u][2], s0)));
          const double t1 = fma(v[u][3], xx[u][0], fma(v[u][4], xx[u][1], fma(v[u][5], xx[u][2], s1)));
          const double t2 = fma(v[u][6], xx[u][0], fma(v[u][7], xx[u][1], fma(v[u][8], xx[u][2], s2)));
          const bool on = c[u] >= 0;
          s0 = on ? t0 : s0; s1 = on ? t1 : s1; s2 = on ? t2 : s2;
        }
      }
    }
    s0 = butterfly_sum<T>(s0);
    s1 = butterfly_sum<T>(s1);
    s2 = butterfly_sum<T>(s2);
    // after the butterfly every lane holds the three sums: lanes 0..2 store one row each (one store instruction,
    // 24 contiguous bytes per block row)
    if (ok && lane < 3) store_y(y, 3 * br + lane, alpha, lane == 0 ? s0 : lane == 1 ? s1 : s2, beta);
  }
}

template <int X, typename IT>
static const void* pick_tu(int T, int U) {
#define P(t, u) if (T == t && U == u) return (const void*)bcsr3_kernel<t, u, X, IT>;
  P(4, 1) P(4, 2) P(8, 1) P(8, 2) P(16, 1) P(16, 2) P(32, 1) P(32, 2)
#undef P
  return nullptr;
}
template <typename IT>
static const void* pick_x(const Variant& v) {
  return v.X == 0 ? pick_tu<0, IT>(v.W, v.U) : v.X == 1 ? pick_tu<1, IT>(v.W, v.U) : v.X == 3 ? pick_tu<3, IT>(v.W, v.U) : nullptr;
}
static const void* pick(const Variant& v) {
  return v.I == 16 ? pick_x<unsigned short>(v) : v.I == 0 ? pick_x<int>(v) : nullptr;
}

bool bcsr_supported(const Variant& v) {
  return v.block >= 32 && v.block <= (v.X == 3 ? 1024 : 512) && v.block % 32 == 0 && pick(v) != nullptr;
}
cudaError_t bcsr_plan(const Variant& v, const BcsrFormat& f, int sm_count, LaunchPlan* out) {
  const void* k = pick(v);
  if (!k || (v.I == 16 ? !f.bcol16 : !f.bcol)) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (f.brows == 0) return cudaSuccess;
  KernelCall& c = out->k[0];
  c.fn = k;
  c.block = v.block;
  const int64_t per_block = v.block / v.W;
  const int64_t exact = (f.brows + per_block - 1) / per_block;
  cudaError_t e = resolve_grid(v.grid, c.fn, v.block, 0, sm_count, exact, &c.grid);
  if (e != cudaSuccess) return e;
  c.add((int)f.brows); c.add((const int*)f.brow_ptr);
  c.add(v.I == 16 ? (const void*)f.bcol16 : (const void*)f.bcol); c.add((const double*)f.bval);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
  c.add((int)0);                 // argument 8: br0, set by plan_for_rows
  c.per_block = per_block;       // block rows
  out->n = 1;
  out->range_kind = RANGE_BCSR;
  out->range_align = 3;
  return cudaSuccess;
}

}  // namespace spmv
