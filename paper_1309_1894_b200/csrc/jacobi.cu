// Solver loop around apply, second form (SURVEY.md sec. 8(f) rank 3 names "CG / Jacobi using spmv_apply"): the
// weighted Jacobi iteration  x_{k+1} = x_k + omega * D^-1 (b - A x_k)  with the selected SpMV variant as the
// matrix product.  Two kernels per iteration: t = A x_k (the variant's own launch plan), then ONE fused pass that
// forms r_k = b - t, its squared norm (block partials, finished by the last block to arrive: cg_reduce.cuh) and the
// next iterate (for a constant-coefficient stencil variant the product joins that pass: dia_const_jacobi_kernel reads
// mask, x, b, d and writes the next iterate -- ONE pass over the vectors per iteration, plus a one-block finishing
// kernel).  The stop test belongs BEFORE the update (textbook order, and the oracle's): the pass therefore
// writes x_{k+1} into the OTHER of two buffers, and the block that finishes the norm decides whether the step
// counts -- when it does not, the result simply stays in the buffer the step read.  Iteration j reads buffer j & 1,
// so a CUDA graph of an even number of iterations can be replayed; scalars live on the device, kernels are no-ops
// once `done` is set (the products keep running on stale data, harmlessly).  Deterministic: fixed reduction
// shapes, no floating-point atomics.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <chrono>

#include "cg_reduce.cuh"
#include "device_utils.cuh"
#include "handle.h"

namespace spmv {

constexpr int kJacBlock = 256;

struct JacobiState {
  double rr, bb;
  int iters, done, converged, zero_diag;
  GridCounter cnt;
};

// d_i = sum of the stored entries (i, i) of row i in stored order (duplicates sum, reading A8)
__global__ void __launch_bounds__(kJacBlock)
jacobi_diag_kernel(int64_t n, const int* __restrict__ rp, const int* __restrict__ ci, const double* __restrict__ va,
                   double* __restrict__ d, JacobiState* __restrict__ st) {
  const int64_t i = (int64_t)blockIdx.x * kJacBlock + threadIdx.x;
  if (i >= n) return;
  double s = 0.0;
  for (int k = rp[i]; k < rp[i + 1]; ++k)
    if (ci[k] == (int)i) s += va[k];
  d[i] = s;
  if (s == 0.0) st->zero_diag = 1;                 // every writer stores the same value
}

__global__ void __launch_bounds__(kJacBlock)
jacobi_init_kernel(int64_t n, const double* __restrict__ b, double* __restrict__ part, JacobiState* __restrict__ st) {
  __shared__ double s_warp[33];
  double bb = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * kJacBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kJacBlock)
    bb = fma(b[i], b[i], bb);
  bb = block_sum_fixed(bb, s_warp);
  double all = 0.0;
  if (grid_sum_last_block(bb, part, &st->cnt, s_warp, &all) && threadIdx.x == 0) {
    st->bb = all; st->rr = 0.0; st->iters = 0; st->converged = 0;
    st->done = st->zero_diag;
  }
}

// r = b - t, ||r||^2, x_next = x_cur + omega * (r / d); the last block to arrive applies the stop rule
__global__ void __launch_bounds__(kJacBlock)
jacobi_step_kernel(int64_t n, const double* __restrict__ b, const double* __restrict__ t, const double* __restrict__ d,
                   const double* __restrict__ x_cur, double* __restrict__ x_next, double omega,
                   double* __restrict__ part, JacobiState* __restrict__ st, double tol, int max_iters) {
  __shared__ double s_warp[33];
  if (st->done) return;
  double rr = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * kJacBlock + threadIdx.x; i < n; i += (int64_t)gridDim.x * kJacBlock) {
    const double ri = b[i] - t[i];
    rr = fma(ri, ri, rr);
    x_next[i] = fma(omega, ri / d[i], x_cur[i]);
  }
  rr = block_sum_fixed(rr, s_warp);
  double all = 0.0;
  if (grid_sum_last_block(rr, part, &st->cnt, s_warp, &all) && threadIdx.x == 0) {
    st->rr = all;
    const int conv = sqrt(all) <= tol * sqrt(st->bb);
    if (conv || st->iters >= max_iters) { st->converged = conv; st->done = 1; }   // x_next is not adopted
    else st->iters += 1;
  }
}

// Finishing kernel of the FUSED step (constant-coefficient stencils: the product, the residual, the update and the
// block partials of ||r||^2 all come out of dia_const_jacobi_kernel): one block adds the partials in index order and
// applies the stop rule -- the same rule as jacobi_step_kernel's last block.
__global__ void __launch_bounds__(1024)
jacobi_finish_kernel(int n_part, const double* __restrict__ part, JacobiState* __restrict__ st, double tol, int max_iters) {
  __shared__ double s_warp[33];
  pdl_launch_dependents();                         // the next step's kernel may load its mask words meanwhile
  pdl_wait();                                      // the partials are the previous kernel's output
  if (st->done) return;
  double v = 0.0;
  for (int i = threadIdx.x; i < n_part; i += blockDim.x) v += part[i];
  v = block_sum_fixed(v, s_warp);
  if (threadIdx.x == 0) {
    st->rr = v;
    const int conv = sqrt(v) <= tol * sqrt(st->bb);
    if (conv || st->iters >= max_iters) { st->converged = conv; st->done = 1; }
    else st->iters += 1;
  }
}

}  // namespace spmv

using namespace spmv;

extern "C" spmv_status_t spmv_jacobi(spmv_handle_t h, const double* d_b, double* d_x, const spmv_jacobi_opts_t* opts,
                                     spmv_jacobi_result_t* result, void* stream) {
  if (!handle_alive(h) || !result) return SPMV_ERR_INVALID_ARG;
  if (h->A.rows != h->A.cols) { set_last_error("spmv_jacobi needs a square matrix"); return SPMV_ERR_INVALID_ARG; }
  const int64_t n = h->A.rows;
  if (n > 0 && (!d_b || !d_x)) return SPMV_ERR_INVALID_ARG;
  spmv_jacobi_opts_t o{};
  if (opts) o = *opts;
  const double omega = o.omega != 0.0 ? o.omega : 1.0;
  const double tol = o.tol > 0 ? o.tol : 1e-10;
  const int max_iters = o.max_iters > 0 ? o.max_iters : (o.max_iters < 0 ? 0 : 1000);
  const int check_every = std::max(2, ((o.check_every > 0 ? o.check_every : 8) + 1) / 2 * 2);    // even: buffer parity
  const bool use_graph = o.no_graph == 0;
  cudaStream_t s = (cudaStream_t)stream;
  memset(result, 0, sizeof(*result));
  if (n == 0) { result->converged = 1; return SPMV_OK; }

  const int nb = (int)std::min<int64_t>((n + kJacBlock - 1) / kJacBlock, (int64_t)h->dev.sm_count * 8);
  // constant-coefficient stencil selected: the whole step is ONE pass (product, residual, update, norm partials)
  const DiaFormat* fused_f = nullptr;
  if (o.no_fused == 0 && h->sel.fam == FAM_DIA_CONST && h->sel.X == 0) {
    auto it = h->dias.find(h->sel.C);
    if (it != h->dias.end() && it->second.is_const) fused_f = &it->second;
  }
  const int n_fpart = fused_f ? dia_const_jacobi_blocks(h->sel, n) : 0;
  const size_t npart = (size_t)std::max(nb, n_fpart);
  const size_t ns = ((size_t)n + 15) & ~(size_t)15;          // 128-byte stride: every vector 16-byte aligned (pair loads)
  const size_t ws_bytes = sizeof(double) * (3 * ns + npart) + sizeof(JacobiState);
  double* ws = (double*)h->al.alloc(ws_bytes, s);
  if (!ws) return SPMV_ERR_ALLOC;
  double *d = ws, *t = d + ns, *x1 = t + ns, *part = x1 + ns;
  JacobiState* st = (JacobiState*)(part + npart);
  double* buf[2] = {d_x, x1};
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
  if (cudaMemsetAsync(st, 0, sizeof(JacobiState), s) != cudaSuccess) return fail(SPMV_ERR_CUDA);
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return fail(SPMV_ERR_CUDA);
  const auto t0 = std::chrono::steady_clock::now();
  cudaEventRecord(e0, s);
  jacobi_diag_kernel<<<(unsigned)((n + kJacBlock - 1) / kJacBlock), kJacBlock, 0, s>>>(n, h->A.row_ptr, h->A.col_idx, h->A.val, d, st);
  jacobi_init_kernel<<<nb, kJacBlock, 0, s>>>(n, d_b, part, st);
  if (cudaGetLastError() != cudaSuccess) return fail(SPMV_ERR_CUDA);
  int launched = 0, graph_replays = 0;
  auto iteration = [&]() -> spmv_status_t {                 // iteration j reads buffer j & 1
    const double* xc = buf[launched & 1];
    double* xn = buf[(launched + 1) & 1];
    if (fused_f) {
      if (dia_const_jacobi_launch(h->sel, n, n, *fused_f, omega, xc, xn, d_b, part, &st->done, s) != cudaSuccess) return SPMV_ERR_CUDA;
      int np_arg = n_fpart, mi = max_iters;
      const double* part_c = part;
      double tol_arg = tol;
      JacobiState* st_arg = st;
      void* fargs[] = {&np_arg, &part_c, &st_arg, &tol_arg, &mi};
      ++launched;
      return launch_kernel_pdl((const void*)jacobi_finish_kernel, 1, 1024, 0, s, fargs, true) == cudaSuccess ? SPMV_OK : SPMV_ERR_CUDA;
    }
    ApplyArgs a{1.0, 0.0, xc, t, s};
    spmv_status_t st1 = launch_plan(h->plan, a);            // t = A x_k
    if (st1 != SPMV_OK) return st1;
    jacobi_step_kernel<<<nb, kJacBlock, 0, s>>>(n, d_b, t, d, xc, xn, omega, part, st, tol, max_iters);
    ++launched;
    return cudaGetLastError() == cudaSuccess ? SPMV_OK : SPMV_ERR_CUDA;
  };
  JacobiState hs{};
  auto poll = [&]() -> bool {
    return cudaMemcpyAsync(&hs, st, sizeof(hs), cudaMemcpyDeviceToHost, s) == cudaSuccess &&
           cudaStreamSynchronize(s) == cudaSuccess;
  };
  // two iterations run un-captured (every kernel of the loop has then been loaded and launched once)
  spmv_status_t st1 = iteration();
  if (st1 == SPMV_OK) st1 = iteration();
  if (st1 != SPMV_OK) return fail(st1);
  if (use_graph && max_iters > 2 && s != nullptr &&                 // the legacy default stream cannot be captured
      cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
    const int before = launched;
    for (int k = 0; k < check_every && st1 == SPMV_OK; ++k) st1 = iteration();
    launched = before;                                              // captured, not run
    cudaError_t ce = cudaStreamEndCapture(s, &graph);
    if (st1 != SPMV_OK || ce != cudaSuccess || !graph) { set_last_error("spmv_jacobi: graph capture failed"); return fail(SPMV_ERR_CUDA); }
    if (cudaGraphInstantiate(&gexec, graph, 0) != cudaSuccess) return fail(SPMV_ERR_CUDA);
  } else {
    cudaGetLastError();
  }
  for (;;) {
    if (!poll()) return fail(SPMV_ERR_CUDA);
    if (hs.done || launched >= max_iters + 1 + check_every) break;
    if (gexec) {
      if (cudaGraphLaunch(gexec, s) != cudaSuccess) return fail(SPMV_ERR_CUDA);
      ++graph_replays;
      launched += check_every;
    } else {
      for (int k = 0; k < check_every; ++k) { st1 = iteration(); if (st1 != SPMV_OK) return fail(st1); }
    }
  }
  // the iterate x_iters sits in buffer iters & 1
  if (!hs.zero_diag && (hs.iters & 1))
    if (cudaMemcpyAsync(d_x, x1, sizeof(double) * (size_t)n, cudaMemcpyDeviceToDevice, s) != cudaSuccess) return fail(SPMV_ERR_CUDA);
  cudaEventRecord(e1, s);
  cudaEventSynchronize(e1);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  result->iters = hs.iters;
  result->converged = hs.converged;
  result->zero_diagonal = hs.zero_diag;
  result->rel_residual = hs.bb > 0.0 ? sqrt(hs.rr) / sqrt(hs.bb) : sqrt(hs.rr);
  result->device_seconds = (double)ms * 1e-3;
  result->wall_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
  result->iterations_launched = launched;
  result->graph_replays = graph_replays;
  result->kernels_per_iteration = fused_f ? 2 : 1 + h->plan.n;
  result->fused_step = fused_f ? 1 : 0;
  cleanup();
  return SPMV_OK;
}
