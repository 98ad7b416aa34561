// Device-side load helpers for sm_100a.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace spmv {

// x gather: X == 0 -> read-only path (ld.global.nc, allocates in L1), X == 1 -> plain ld.global
template <int X>
__device__ __forceinline__ double ldx(const double* __restrict__ x, int c) {
  if (X == 0) return __ldg(x + c);
  double v;
  asm volatile("ld.global.f64 %0, [%1];" : "=d"(v) : "l"(x + c));
  return v;
}

// Streaming loads of matrix data: read once, keep them out of L1 so that x stays there.
__device__ __forceinline__ double ld_stream(const double* p) {
  double v;
  asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ int ld_stream(const int* p) {
  int v;
  asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ double2 ld_stream2(const double* p) {   // 16-byte aligned
  double2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ int2 ld_stream2(const int* p) {         // 8-byte aligned
  int2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.s32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ int4 ld_stream4(const int* p) {         // 16-byte aligned
  int4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}

// Compiler-level fence: keeps the phases of an unrolled trip (all matrix loads | all x
// gathers | all FMAs) in that order in the generated code.  Warps issue in order, so a
// dependent use placed between two loads would delay every load behind it.
__device__ __forceinline__ void phase_fence() { asm volatile("" ::: "memory"); }

// Programmatic dependent launch (sm_90+): launch_dependents lets the next kernel of the stream begin its
// prologue while this grid is still running; wait blocks until every prerequisite grid has completed and its
// memory is visible.  Both are no-ops for a kernel launched without the attribute.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// BLAS-style epilogue (reading A1): y is not read when beta == 0.
__device__ __forceinline__ void store_y(double* __restrict__ y, int64_t i, double alpha, double s, double beta) {
  y[i] = (beta == 0.0) ? alpha * s : fma(alpha, s, beta * y[i]);
}

template <int W>
__device__ __forceinline__ double butterfly_sum(double s) {
#pragma unroll
  for (int d = W / 2; d >= 1; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d, W);
  return s;
}

}  // namespace spmv
