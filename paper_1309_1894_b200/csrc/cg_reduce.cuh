// Deterministic grid-wide sums for the solver loop (solver.cu) and for SpMV kernels with a fused dot
// product (kernels_dia.cu): every block writes ONE partial; the block that arrives last adds the partials in
// index order with a fixed-shape tree, so the result does not depend on which block that is.  No
// floating-point atomics (reading A20: bit-identical across runs).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace spmv {

// Arrival counter of one grid-wide reduction, two levels: thousands of blocks adding to ONE address serialise
// in L2 (~2 ns each: measured 25 us for 8192 blocks); 64 sub-counters take the arrivals in parallel and the
// block that completes a sub-counter arrives at the top.  All zero before and after every use.
struct GridCounter {
  unsigned sub[64];
  unsigned top;
};

struct CgState {
  double rr, rr_prev, bb, pq;
  int iters, done, converged, breakdown;
  int x_pending;                  // 1: r was advanced with alpha, x += alpha p is still to be done
  GridCounter cnt_pq, cnt_rr;
};

// true in exactly one block: the last of the grid to arrive (call from thread 0 only)
__device__ __forceinline__ bool grid_arrive_last(GridCounter* c) {
  const unsigned j = blockIdx.x & 63u;
  const unsigned in_group = (gridDim.x + 63u - j) >> 6;                 // blocks b with (b & 63) == j
  const unsigned groups = gridDim.x < 64u ? gridDim.x : 64u;
  __threadfence();                                   // this block's results are visible before it is counted
  if (atomicAdd(&c->sub[j], 1u) != in_group - 1) return false;
  c->sub[j] = 0u;
  __threadfence();
  if (atomicAdd(&c->top, 1u) != groups - 1) return false;
  c->top = 0u;
  __threadfence();
  return true;
}

// sum over the block (any blockDim.x that is a multiple of 32, <= 1024); fixed shape; result in every thread
__device__ __forceinline__ double block_sum_fixed(double v, double* s_warp /* [33] */) {
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  const int w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __syncthreads();                                   // s_warp may still be read from a previous call
  if ((threadIdx.x & 31) == 0) s_warp[w] = v;
  __syncthreads();
  if (w == 0) {
    double t = (int)(threadIdx.x & 31) < nw ? s_warp[threadIdx.x & 31] : 0.0;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) t += __shfl_xor_sync(0xffffffffu, t, d);
    if (threadIdx.x == 0) s_warp[32] = t;
  }
  __syncthreads();
  return s_warp[32];
}

// Block-level partial -> part[blockIdx.x]; returns true in the LAST block to arrive, with *total = the sum of
// all gridDim.x partials in index order.  The counter is reset for the next use.
__device__ __forceinline__ bool grid_sum_last_block(double block_partial, double* __restrict__ part,
                                                    GridCounter* __restrict__ counter, double* s_warp, double* total) {
  __shared__ int s_last;
  if (threadIdx.x == 0) {
    part[blockIdx.x] = block_partial;
    s_last = grid_arrive_last(counter);
  }
  __syncthreads();
  if (!s_last) return false;
  __threadfence();
  double v = 0.0;
  for (unsigned i = threadIdx.x; i < gridDim.x; i += blockDim.x) v += __ldcg(part + i);
  *total = block_sum_fixed(v, s_warp);
  return true;
}

}  // namespace spmv
