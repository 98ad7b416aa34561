// Solver loop around apply (the paper's ref [1], is about
// iterative solvers): conjugate gradients with the tuned SpMV variant as its matrix product.
//
//   r0 = b - A x0, p0 = r0, rr = r0.r0;  per iteration:  q = A p;  alpha = rr / p.q;
//   x += alpha p;  r -= alpha q;  rr' = r.r;  beta = rr'/rr;  p = r + beta p.
//
// No host round trip inside the loop: alpha, beta, rr, the iteration count and the "done" flag live
// in device memory, kernels turn into no-ops once done is set, and `check_every` iterations are
// captured in ONE CUDA graph that is replayed until the host sees done.  Vector updates are fused
// (x and r update + r.r partials in one pass; p update reads the new partials), reductions are
// two-level with a fixed shape (per-block partials, then every block re-adds the partials in the same
// order), so the iterates are bit-identical across runs (reading A20).  No atomics.
#include <cooperative_groups.h>
#include <math.h>
#include <string.h>

#include <algorithm>
#include <chrono>

#include "cg_reduce.cuh"
#include "handle.h"

namespace spmv {

constexpr int kCgBlock = 256;

__device__ __forceinline__ double cg_block_sum(double v, double* s_red) {
  const int tid = threadIdx.x;
  s_red[tid] = v;
  __syncthreads();
#pragma unroll
  for (int d = kCgBlock / 2; d >= 1; d >>= 1) {
    if (tid < d) s_red[tid] += s_red[tid + d];
    __syncthreads();
  }
  const double out = s_red[0];
  __syncthreads();
  return out;
}
// every block adds the nb partials in the same fixed order -> the same value in every block
__device__ __forceinline__ double cg_sum_partials(const double* __restrict__ part, int nb, double* s_red) {
  double v = 0.0;
  for (int i = threadIdx.x; i < nb; i += kCgBlock) v += part[i];
  return cg_block_sum(v, s_red);
}

// Large systems: three or four kernels per iteration, every reduction finished by the last block to arrive
// (cg_reduce.cuh), so no kernel exists only to add partials and no block re-adds them:
//   q = A p, then st->pq = p.q: cg_dot_kernel, or -- when the SpMV kernel has the fused dot and wrote its block
//                                partials -- the one-block cg_pq_kernel (no second pass over p and q)
//   cg_update_kernel : x += alpha p, r -= alpha q, r.r; its last block also advances the scalars
//   cg_pupdate_kernel: p = r + beta p
__global__ void __launch_bounds__(kCgBlock)
cg_init_kernel(int64_t n, const double* __restrict__ b, const double* __restrict__ q, double* __restrict__ r,
               double* __restrict__ p, double* __restrict__ part_rr, double* __restrict__ part_bb,
               CgState* __restrict__ st, double tol, int max_iters) {
  __shared__ double s_warp[33];
  double rr = 0.0, bb = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * kCgBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kCgBlock) {
    const double bi = b[i], ri = bi - q[i];
    r[i] = ri;
    p[i] = ri;
    rr = fma(ri, ri, rr);
    bb = fma(bi, bi, bb);
  }
  rr = block_sum_fixed(rr, s_warp);
  bb = block_sum_fixed(bb, s_warp);
  if (threadIdx.x == 0) part_bb[blockIdx.x] = bb;      // published by the fence inside grid_sum_last_block
  double rr_all = 0.0;
  if (grid_sum_last_block(rr, part_rr, &st->cnt_rr, s_warp, &rr_all)) {
    double v = 0.0;
    for (unsigned i = threadIdx.x; i < gridDim.x; i += blockDim.x) v += __ldcg(part_bb + i);
    const double bb_all = block_sum_fixed(v, s_warp);
    if (threadIdx.x == 0) {
      st->rr = rr_all; st->rr_prev = rr_all; st->bb = bb_all; st->pq = 0.0;
      st->iters = 0; st->breakdown = 0;
      st->converged = sqrt(rr_all) <= tol * sqrt(bb_all);
      st->done = st->converged || max_iters <= 0;
    }
  }
}

__global__ void __launch_bounds__(kCgBlock)
cg_dot_kernel(int64_t n, const double* __restrict__ p, const double* __restrict__ q, double* __restrict__ part,
              CgState* __restrict__ st) {
  __shared__ double s_warp[33];
  if (st->done) return;
  double s = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * kCgBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kCgBlock)
    s = fma(p[i], q[i], s);
  s = block_sum_fixed(s, s_warp);
  double all = 0.0;
  if (grid_sum_last_block(s, part, &st->cnt_pq, s_warp, &all) && threadIdx.x == 0) st->pq = all;
}

// st->pq = sum of the SpMV kernel's block partials (fused dot), one block, index order
__global__ void __launch_bounds__(1024)
cg_pq_kernel(int n_part, const double* __restrict__ part, CgState* __restrict__ st) {
  __shared__ double s_warp[33];
  if (st->done) return;
  double v = 0.0;
  for (int i = threadIdx.x; i < n_part; i += blockDim.x) v += part[i];
  v = block_sum_fixed(v, s_warp);
  if (threadIdx.x == 0) st->pq = v;
}

// r -= alpha q and the new r.r; alpha = rr / p.q.  The last block to arrive advances the scalars: every other
// block has read the old ones by then.  x += alpha p is left to cg_pupdate_kernel, which reads p anyway
// (p is then read once per iteration instead of twice).
__global__ void __launch_bounds__(kCgBlock)
cg_update_kernel(int64_t n, CgState* __restrict__ st, double* __restrict__ r, const double* __restrict__ q,
                 double* __restrict__ part_rr, double tol, int max_iters) {
  __shared__ double s_warp[33];
  if (st->done) {                                         // no step this iteration: nothing for cg_pupdate_kernel either
    if (blockIdx.x == 0 && threadIdx.x == 0) st->x_pending = 0;
    return;
  }
  const double pq = st->pq;
  const double alpha = pq > 0.0 ? st->rr / pq : 0.0;      // pq <= 0: not SPD; the loop stops below
  double rr = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * kCgBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kCgBlock) {
    const double ri = fma(-alpha, q[i], r[i]);
    r[i] = ri;
    rr = fma(ri, ri, rr);
  }
  rr = block_sum_fixed(rr, s_warp);
  double rr_new = 0.0;
  if (grid_sum_last_block(rr, part_rr, &st->cnt_rr, s_warp, &rr_new) && threadIdx.x == 0) {
    if (!(pq > 0.0)) { st->breakdown = 1; st->done = 1; st->x_pending = 0; return; }
    st->rr_prev = st->rr;
    st->rr = rr_new;
    st->iters += 1;
    st->x_pending = 1;
    st->converged = sqrt(rr_new) <= tol * sqrt(st->bb);
    st->done = st->converged || st->iters >= max_iters;
  }
}

// x += alpha p (alpha = rr_old / p.q, the step cg_update_kernel took) and, unless the loop just finished,
// p = r + beta p with beta = rr_new / rr_old
__global__ void __launch_bounds__(kCgBlock)
cg_pupdate_kernel(int64_t n, const CgState* __restrict__ st, double* __restrict__ x, const double* __restrict__ r,
                  double* __restrict__ p) {
  if (!st->x_pending) return;
  const double alpha = st->rr_prev / st->pq;
  const double beta = st->rr / st->rr_prev;
  const bool more = !st->done;
  for (int64_t i = (int64_t)blockIdx.x * kCgBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kCgBlock) {
    const double pi = p[i];
    x[i] = fma(alpha, pi, x[i]);
    if (more) p[i] = fma(beta, pi, r[i]);
  }
}

// ------------------------------------------------------------------ small systems: the whole solve in ONE kernel
// When every row fits in one resident grid the loop is launch-bound (five graph nodes per iteration cost
// ~3 us each on a 4096-row system).  This cooperative kernel runs all iterations with three grid-wide
// barriers per iteration and no launch in between: q = A p straight from the caller's CSR arrays (thread
// per row, the matrix is cache-resident at this size) with the p.q partial fused into the same pass, then
// the x/r update with the r.r partial, then the p update.  Same recurrence, same stop rule, fixed
// reduction shape (deterministic); every block derives the scalars from the partials in the same order.
__global__ void __launch_bounds__(kCgBlock)
cg_fused_kernel(int64_t n, const int* __restrict__ rp, const int* __restrict__ ci, const double* __restrict__ va,
                const double* __restrict__ b, double* __restrict__ x, double* __restrict__ r,
                double* __restrict__ p, double* __restrict__ q, double* __restrict__ part_a,
                double* __restrict__ part_b, CgState* __restrict__ st, double tol, int max_iters) {
  namespace cg = cooperative_groups;
  cg::grid_group grid = cg::this_grid();
  __shared__ double s_red[kCgBlock];
  const int nb = gridDim.x;
  const int64_t G = (int64_t)nb * kCgBlock, t0 = (int64_t)blockIdx.x * kCgBlock + threadIdx.x;
  auto row_dot = [&](int64_t i, const double* __restrict__ v) {
    double s = 0.0;
    for (int k = rp[i]; k < rp[i + 1]; ++k) s = fma(va[k], v[ci[k]], s);
    return s;
  };
  // r0 = b - A x0, p0 = r0
  double a = 0.0, c = 0.0;
  for (int64_t i = t0; i < n; i += G) {
    const double bi = b[i], ri = bi - row_dot(i, x);
    r[i] = ri; p[i] = ri;
    a = fma(ri, ri, a);
    c = fma(bi, bi, c);
  }
  a = cg_block_sum(a, s_red);
  c = cg_block_sum(c, s_red);
  if (threadIdx.x == 0) { part_a[blockIdx.x] = a; part_b[blockIdx.x] = c; }
  grid.sync();
  double rr = cg_sum_partials(part_a, nb, s_red);
  const double bb = cg_sum_partials(part_b, nb, s_red);
  const double stop = tol * sqrt(bb);
  int k = 0, breakdown = 0;
  grid.sync();                                   // part_a / part_b are reused below
  while (!(sqrt(rr) <= stop) && k < max_iters) {
    double pq = 0.0;
    for (int64_t i = t0; i < n; i += G) {        // q = A p, fused with the p.q partial
      const double qi = row_dot(i, p);
      q[i] = qi;
      pq = fma(p[i], qi, pq);
    }
    pq = cg_block_sum(pq, s_red);
    if (threadIdx.x == 0) part_a[blockIdx.x] = pq;
    grid.sync();
    pq = cg_sum_partials(part_a, nb, s_red);
    if (!(pq > 0.0)) { breakdown = 1; break; }   // uniform across the grid: every block sees the same pq
    const double alpha = rr / pq;
    double rn = 0.0;
    for (int64_t i = t0; i < n; i += G) {
      x[i] = fma(alpha, p[i], x[i]);
      const double ri = fma(-alpha, q[i], r[i]);
      r[i] = ri;
      rn = fma(ri, ri, rn);
    }
    rn = cg_block_sum(rn, s_red);
    if (threadIdx.x == 0) part_b[blockIdx.x] = rn;
    grid.sync();
    rn = cg_sum_partials(part_b, nb, s_red);
    const double beta = rn / rr;
    rr = rn;
    for (int64_t i = t0; i < n; i += G) p[i] = fma(beta, p[i], r[i]);
    ++k;
    grid.sync();                                 // p complete before the next product
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    st->rr = rr; st->rr_prev = rr; st->bb = bb; st->pq = 0.0;
    st->iters = k; st->breakdown = breakdown;
    st->converged = sqrt(rr) <= stop;
    st->done = 1;
  }
}

}  // namespace spmv

using namespace spmv;

extern "C" spmv_status_t spmv_cg(spmv_handle_t h, const double* d_b, double* d_x, const spmv_cg_opts_t* opts,
                                 spmv_cg_result_t* result, void* stream) {
  if (!handle_alive(h) || !result) return SPMV_ERR_INVALID_ARG;
  if (h->A.rows != h->A.cols) { set_last_error("spmv_cg needs a square matrix"); return SPMV_ERR_INVALID_ARG; }
  const int64_t n = h->A.rows;
  if (n > 0 && (!d_b || !d_x)) return SPMV_ERR_INVALID_ARG;
  spmv_cg_opts_t o{};
  if (opts) o = *opts;
  const double tol = o.tol > 0 ? o.tol : 1e-10;
  const int max_iters = o.max_iters > 0 ? o.max_iters : (o.max_iters < 0 ? 0 : 1000);
  const int check_every = o.check_every > 0 ? o.check_every : 8;
  const bool use_graph = o.no_graph == 0;
  cudaStream_t s = (cudaStream_t)stream;
  memset(result, 0, sizeof(*result));
  if (n == 0) { result->converged = 1; return SPMV_OK; }

  // Tune for the loop: the single-apply ranking is measured cold, the loop runs with its
  // five vectors resident in L2 and a dot product attached to the product.  Each leader of the last spmv_tune
  // runs a few iterations of THIS loop on a scratch solution vector; the fastest is adopted.
  if (o.tune_loop && h->leaders.size() > 1) {
    double* xs = (double*)h->al.alloc(sizeof(double) * (size_t)n, s);
    if (!xs) return SPMV_ERR_ALLOC;
    spmv_cg_opts_t po = o;
    po.tune_loop = 0; po.tol = 1e-300; po.max_iters = 24; po.check_every = 8;
    std::string best;
    double best_s = 1e300;
    const std::vector<std::string> leaders = h->leaders;
    const Variant incoming = h->sel;                         // what the caller had selected (the apply winner)
    const bool incoming_tuned = h->tuned;
    for (const std::string& d : leaders) {
      Variant v;
      std::string why;
      if (!variant_from_string(d.c_str(), &v) || !variant_eligible(h, v, &why) || adopt_variant(h, v, s) != SPMV_OK) continue;
      spmv_cg_result_t pr;
      double t = 1e300;
      for (int rep = 0; rep < 2; ++rep) {                    // the second run is the measurement
        if (cudaMemsetAsync(xs, 0, sizeof(double) * (size_t)n, s) != cudaSuccess) break;
        if (spmv_cg(h, d_b, xs, &po, &pr, stream) != SPMV_OK) break;
        if (rep == 1 && pr.iters > 0) t = pr.device_seconds / pr.iters;
      }
      if (t < best_s) { best_s = t; best = d; }
    }
    cudaStreamSynchronize(s);
    h->al.free(xs, sizeof(double) * (size_t)n);
    // no probe produced a time (b == 0, breakdown, a failed probe): back to the caller's selection, not to
    // whichever leader happened to be probed last
    Variant v = incoming;
    if (!best.empty() && !variant_from_string(best.c_str(), &v)) v = incoming;
    spmv_status_t st = adopt_variant(h, v, s);
    if (st != SPMV_OK && !best.empty()) st = adopt_variant(h, incoming, s);
    if (st != SPMV_OK) return st;
    h->tuned = incoming_tuned;
    h->leaders = leaders;
  }

  // small systems: one cooperative kernel for the whole solve (see cg_fused_kernel)
  int fused_blocks = 0;
  if (o.no_fused == 0 && n <= 262144 && h->A.nnz <= 4 * 1024 * 1024) {
    int occ = 0, coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->device);
    if (coop && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void*)cg_fused_kernel, kCgBlock, 0) == cudaSuccess && occ > 0)
      fused_blocks = (int)std::min<int64_t>((n + kCgBlock - 1) / kCgBlock, (int64_t)h->dev.sm_count * occ);
  }
  // one wave of fat blocks, grid-stride: the fence + arrival at the tail of a reducing kernel is paid per block,
  // and with the five vectors mostly L2-resident an exact grid measured slower for the p/x update too
  const int nb = fused_blocks > 0 ? fused_blocks
                                  : (int)std::min<int64_t>((n + kCgBlock - 1) / kCgBlock, (int64_t)h->dev.sm_count * 8);
  // partial arrays: one slot per block of whichever kernel writes them (the SpMV kernel with the fused dot
  // runs an exact grid of >= 32 rows per block)
  const size_t npart = std::max<size_t>((size_t)nb, (size_t)((n + 31) / 32));    // (fused: nb is the cooperative grid)
  const size_t ns = ((size_t)n + 15) & ~(size_t)15;          // 128-byte stride: every vector 16-byte aligned (pair loads)
  const size_t ws_bytes = sizeof(double) * (3 * ns + 3 * npart) + sizeof(CgState);
  double* ws = (double*)h->al.alloc(ws_bytes, s);
  if (!ws) return SPMV_ERR_ALLOC;
  double *r = ws, *p = r + ns, *q = p + ns, *part_rr = q + ns, *part_bb = part_rr + npart, *part_pq = part_bb + npart;
  CgState* st = (CgState*)(part_pq + npart);
  if (cudaMemsetAsync(st, 0, sizeof(CgState), s) != cudaSuccess) { h->al.free(ws, ws_bytes); return SPMV_ERR_CUDA; }
  // q = A p with p.q fused into the SpMV kernel's epilogue where the selected family has that form
  LaunchPlan dot_plan;
  int n_dot_part = 0;
  const bool fused_dot = o.no_fused_dot == 0 && fused_blocks == 0 &&
                         build_dot_plan(h, part_pq, &n_dot_part, &dot_plan) == SPMV_OK && (size_t)n_dot_part <= npart;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t gexec = nullptr;
  auto cleanup = [&]() {
    if (gexec) cudaGraphExecDestroy(gexec);
    if (graph) cudaGraphDestroy(graph);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaStreamSynchronize(s);
    h->al.free(ws, ws_bytes);
  };
  auto fail = [&](spmv_status_t code) { cleanup(); return code; };
  auto iteration = [&]() -> spmv_status_t {
    ApplyArgs a{1.0, 0.0, p, q, s};
    spmv_status_t st1 = launch_plan(fused_dot ? dot_plan : h->plan, a);      // q = A p  [+ st->pq = p.q]
    if (st1 != SPMV_OK) return st1;
    if (fused_dot) cg_pq_kernel<<<1, 1024, 0, s>>>(n_dot_part, part_pq, st);
    else cg_dot_kernel<<<nb, kCgBlock, 0, s>>>(n, p, q, part_pq, st);
    cg_update_kernel<<<nb, kCgBlock, 0, s>>>(n, st, r, q, part_rr, tol, max_iters);
    cg_pupdate_kernel<<<nb, kCgBlock, 0, s>>>(n, st, d_x, r, p);     // (measured: programmatic dependent launches gain nothing here)
    return cudaGetLastError() == cudaSuccess ? SPMV_OK : SPMV_ERR_CUDA;
  };
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return fail(SPMV_ERR_CUDA);
  const auto t0 = std::chrono::steady_clock::now();
  cudaEventRecord(e0, s);
  CgState hs{};
  int launched = 0, graph_replays = 0;
  if (fused_blocks > 0) {
    int64_t n_arg = n;
    const int *rp = h->A.row_ptr, *ci = h->A.col_idx;
    const double *va = h->A.val, *bb = d_b;
    double tol_arg = tol;
    int mi = max_iters;
    void* args[] = {&n_arg, &rp, &ci, &va, &bb, &d_x, &r, &p, &q, &part_rr, &part_bb, &st, &tol_arg, &mi};
    if (cudaLaunchCooperativeKernel((const void*)cg_fused_kernel, dim3(fused_blocks), dim3(kCgBlock), args, 0, s) != cudaSuccess) {
      set_last_error("spmv_cg: cooperative launch failed: %s", cudaGetErrorString(cudaGetLastError()));
      return fail(SPMV_ERR_CUDA);
    }
    if (cudaMemcpyAsync(&hs, st, sizeof(hs), cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess)
      return fail(SPMV_ERR_CUDA);
    launched = hs.iters;
  } else {
  {
    ApplyArgs a{1.0, 0.0, d_x, q, s};
    spmv_status_t st1 = launch_plan(h->plan, a);                       // q = A x0
    if (st1 != SPMV_OK) return fail(st1);
  }
  cg_init_kernel<<<nb, kCgBlock, 0, s>>>(n, d_b, q, r, p, part_rr, part_bb, st, tol, max_iters);
  if (cudaGetLastError() != cudaSuccess) return fail(SPMV_ERR_CUDA);
  auto poll = [&]() -> bool {
    return cudaMemcpyAsync(&hs, st, sizeof(hs), cudaMemcpyDeviceToHost, s) == cudaSuccess &&
           cudaStreamSynchronize(s) == cudaSuccess;
  };
  if (!poll()) return fail(SPMV_ERR_CUDA);
  if (!hs.done) {
    // the first iteration runs un-captured: it settles function attributes and occupancy caches
    spmv_status_t st1 = iteration();
    if (st1 != SPMV_OK) return fail(st1);
    ++launched;
    if (use_graph && max_iters > 1) {
      // the legacy default stream cannot be captured: plain launches then
      if (s != nullptr && cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
        for (int k = 0; k < check_every && st1 == SPMV_OK; ++k) st1 = iteration();
        cudaError_t ce = cudaStreamEndCapture(s, &graph);
        if (st1 != SPMV_OK || ce != cudaSuccess || !graph) { set_last_error("spmv_cg: graph capture failed"); return fail(SPMV_ERR_CUDA); }
        if (cudaGraphInstantiate(&gexec, graph, 0) != cudaSuccess) return fail(SPMV_ERR_CUDA);
      } else {
        cudaGetLastError();
      }
    }
    for (;;) {
      if (!poll()) return fail(SPMV_ERR_CUDA);
      if (hs.done || launched >= max_iters + check_every) break;
      if (gexec) {
        if (cudaGraphLaunch(gexec, s) != cudaSuccess) return fail(SPMV_ERR_CUDA);
        ++graph_replays;
      } else {
        for (int k = 0; k < check_every; ++k) { st1 = iteration(); if (st1 != SPMV_OK) return fail(st1); }
      }
      launched += check_every;
    }
  }
  }
  cudaEventRecord(e1, s);
  cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  result->iters = hs.iters;
  result->converged = hs.converged;
  result->breakdown = hs.breakdown;
  result->rel_residual = hs.bb > 0.0 ? sqrt(hs.rr) / sqrt(hs.bb) : sqrt(hs.rr);
  result->device_seconds = (double)ms * 1e-3;
  result->wall_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
  result->iterations_launched = launched;
  result->graph_replays = graph_replays;
  strncpy(result->loop_variant, variant_to_string(h->sel).c_str(), sizeof(result->loop_variant) - 1);
  result->fused = fused_blocks > 0;
  result->fused_dot = fused_dot ? 1 : 0;
  result->kernels_per_iteration = fused_blocks > 0 ? 0 : 4 + (h->plan.n > 1 ? h->plan.n - 1 : 0);
  cleanup();
  return SPMV_OK;
}
