// SELL-C-sigma with the matrix stream moved by the TMA engine (sm_100a):
// cp.async.bulk (1-D bulk copy, SASS UBLKCP) + mbarrier producer/consumer ring.
//
// Why: SpMV on short rows is latency-bound when the bytes in flight depend on how many
// loads each warp has issued (warps issue in order and ptxas sinks loads next to their
// uses).  A slice of the SELL format is one contiguous run of values and one of column
// indices, so ONE elected producer thread can keep STAGES x (J*C*12) bytes per CTA in
// flight with two bulk copies per stage, independent of what the consumer warps do.
// Consumers read values/indices from shared memory (conflict-free: consecutive threads,
// consecutive addresses), gather x through L1 and accumulate in registers.
//
// x path: X == 0 gathers x through the read-only/L1 path; X == 2 STAGES THE
// X WINDOW IN SHARED MEMORY: once per slice the producer bulk-copies the contiguous run
// x[lo, lo + C + 2H) around the slice's own rows (lo = s*C - H, clipped) into one of two window buffers
// (their own full/empty barriers, independent of the stage ring: the window of slice s+1 arrives while
// slice s is consumed), and a gather whose column falls inside the window is a shared-memory read; the
// others (far diagonals of a 3D stencil, unstructured columns) still go through L1.  H is the variant's
// `h` parameter: 72 / 136 for the near diagonals of a stencil, or the matrix bandwidth for a banded matrix
// (every gather of the slice is then a shared-memory read: a warp's 32 scattered columns cost ~3 bank
// conflict wavefronts instead of up to 32 L1 wavefronts -- the L1 data pipe is what bounds the L1 path on
// the banded bench matrix, profiles/r02_banded_sell16_tma_ncu_full.md).
//
// Layout and padding semantics are those of kernels_sell.cu (same SellFormat).
// Work split: CTA b owns slices b, b+gridDim, ...; a slice wider than J steps is streamed
// as ceil(w/J) stages.  Deterministic: each row is summed by one thread in stored order.
#include <algorithm>

#include "device_utils.cuh"
#include "spmv_internal.h"
#include "tma_utils.cuh"

namespace spmv {

using tma::bar_arrive;
using tma::bar_expect_tx;
using tma::bar_init;
using tma::bar_wait;
using tma::bulk_g2s;

__device__ __forceinline__ int tma_col_of_delta(unsigned d, int base) { return d == 0xFFFFu ? -1 : base + (int)d; }

template <int R>
struct SmemVec;
template <>
struct SmemVec<1> {
  static __device__ __forceinline__ void load(const double* pv, const int* pc, int, double* v, int* c) { v[0] = *pv; c[0] = *pc; }
  static __device__ __forceinline__ void load(const double* pv, const unsigned short* pc, int base, double* v, int* c) {
    v[0] = *pv; c[0] = tma_col_of_delta(*pc, base);
  }
};
template <>
struct SmemVec<2> {
  static __device__ __forceinline__ void load(const double* pv, const int* pc, int, double* v, int* c) {
    double2 a = *reinterpret_cast<const double2*>(pv);
    int2 b = *reinterpret_cast<const int2*>(pc);
    v[0] = a.x; v[1] = a.y; c[0] = b.x; c[1] = b.y;
  }
  static __device__ __forceinline__ void load(const double* pv, const unsigned short* pc, int base, double* v, int* c) {
    double2 a = *reinterpret_cast<const double2*>(pv);
    const unsigned b = *reinterpret_cast<const unsigned*>(pc);
    v[0] = a.x; v[1] = a.y;
    c[0] = tma_col_of_delta(b & 0xFFFFu, base); c[1] = tma_col_of_delta(b >> 16, base);
  }
};

// blockDim.x = C/R consumer threads + 32 (warp C/R/32 is the producer warp)
// IT = int: 32-bit column indices; IT = unsigned short: 16-bit deltas against sbase[slice] (sell16_tma)
template <int R, int STAGES, int J, int PERM, int X, typename IT>
__global__ void __launch_bounds__(512 + 32)
sell_tma_kernel(int64_t rows, int64_t nslices, int C, const int64_t* __restrict__ slice_ptr,
                const double* __restrict__ sval, const IT* __restrict__ scol, const int* __restrict__ sbase,
                const int* __restrict__ perm, double* __restrict__ part, double alpha,
                const double* __restrict__ x, double beta, double* __restrict__ y, int64_t cols, int H) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int nconsumers = C / R;
  const int WIN = X >= 2 ? C + 2 * H : 0;                                    // x window entries per stage
  double* s_val = reinterpret_cast<double*>(smem_raw);                       // [STAGES][J*C]
  double* s_x = s_val + (size_t)STAGES * J * C;                              // [2][WIN]: one window per slice, double-buffered
  IT* s_col = reinterpret_cast<IT*>(s_x + (size_t)2 * WIN);                  // [STAGES][J*C]
  uint64_t* full = reinterpret_cast<uint64_t*>(s_col + (size_t)STAGES * J * C);   // J*C*sizeof(IT) is a multiple of 256
  uint64_t* empty = full + STAGES;
  uint64_t* wfull = empty + STAGES;                                          // [2]
  uint64_t* wempty = wfull + 2;                                              // [2]
  const int tid = threadIdx.x;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) {
      bar_init(&full[s], 1);
      bar_init(&empty[s], nconsumers / 32);
    }
    if (X >= 2) {
      bar_init(&wfull[0], 1); bar_init(&wfull[1], 1);
      bar_init(&wempty[0], nconsumers / 32); bar_init(&wempty[1], nconsumers / 32);
    }
    tma::bar_init_fence();
  }
  __syncthreads();

  if (tid >= nconsumers) {
    // ---------------- producer warp: one elected lane streams the slices
    if (tid == nconsumers) {
      uint32_t stage = 0, phase = 0, wk = 0;
      for (int64_t s = blockIdx.x; s < nslices; s += gridDim.x) {
        const int64_t base = __ldg(slice_ptr + s);
        const int w = (int)((__ldg(slice_ptr + s + 1) - base) / C);
        if (X >= 2 && w > 0) {     // this slice's window [lo, lo + n) of x, lo even (16-byte aligned source), n even
          const uint32_t wb = wk & 1u, wph = (wk >> 1) & 1u;
          ++wk;
          bar_wait(&wempty[wb], wph ^ 1);
          tma::fence_proxy_async();
          const int64_t lo = max((int64_t)0, s * C - H) & ~(int64_t)1;
          const int64_t n = min((int64_t)WIN, cols - lo) & ~(int64_t)1;
          const uint32_t xb = n > 0 ? (uint32_t)n * sizeof(double) : 0u;
          bar_expect_tx(&wfull[wb], xb);                     // no bytes (unaligned x: cols = 0): a plain arrive
          if (xb) bulk_g2s(s_x + (size_t)wb * WIN, x + lo, xb, &wfull[wb]);
        }
        for (int j0 = 0; j0 < w; j0 += J) {
          const int nj = min(J, w - j0);
          bar_wait(&empty[stage], phase ^ 1);
          // The consumers read this stage through the generic proxy; the refill is an async-proxy
          // write.  Without this cross-proxy fence the refill was observed (B200, full-size
          // cfg5, sorted slices) to land under reads that had been ordered before the arrive.
          tma::fence_proxy_async();
          const uint32_t vb = (uint32_t)nj * C * sizeof(double), cb = (uint32_t)nj * C * sizeof(IT);
          bar_expect_tx(&full[stage], vb + cb);
          bulk_g2s(s_val + (size_t)stage * J * C, sval + base + (int64_t)j0 * C, vb, &full[stage]);
          bulk_g2s(s_col + (size_t)stage * J * C, scol + base + (int64_t)j0 * C, cb, &full[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
    return;
  }

  // ---------------- consumers: thread t owns rows [t*R, t*R+R) of the current slice
  uint32_t stage = 0, phase = 0, wk = 0;
  const int lane = tid & 31;
  for (int64_t s = blockIdx.x; s < nslices; s += gridDim.x) {
    const int64_t base = __ldg(slice_ptr + s);
    const int w = (int)((__ldg(slice_ptr + s + 1) - base) / C);
    // X == 2: this slice's x window (the producer's arithmetic, repeated)
    const uint32_t wb = wk & 1u;
    const int64_t wlo = X >= 2 ? (max((int64_t)0, s * C - H) & ~(int64_t)1) : 0;
    const int64_t wn = X >= 2 ? (min((int64_t)WIN, cols - wlo) & ~(int64_t)1) : 0;
    const double* xs = s_x + (size_t)wb * WIN;
    if (X >= 2 && w > 0) {
      bar_wait(&wfull[wb], (wk >> 1) & 1u);
      ++wk;
    }
    const int64_t r0 = s * C + (int64_t)tid * R;
    const int cbase = sizeof(IT) == 2 ? __ldg(sbase + s) : 0;
    int64_t orow[R];
    double yold[R], acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int64_t row = r0 + r;
      if (PERM) orow[r] = __ldg(perm + row);
      else orow[r] = row < rows ? row : -1;
      acc[r] = 0.0;
    }
#pragma unroll
    for (int r = 0; r < R; ++r) yold[r] = (beta != 0.0 && orow[r] >= 0) ? y[orow[r]] : 0.0;
    for (int j0 = 0; j0 < w; j0 += J) {
      const int nj = min(J, w - j0);
      bar_wait(&full[stage], phase);
      const double* pv = s_val + (size_t)stage * J * C + tid * R;
      const IT* pc = s_col + (size_t)stage * J * C + tid * R;
      double v[J][R];
      int c[J][R];
#pragma unroll
      for (int j = 0; j < J; ++j) {
        SmemVec<R>::load(pv + j * C, pc + j * C, cbase, v[j], c[j]);
        if (j >= nj) {          // beyond this stage's steps: stale shared memory, masked off
#pragma unroll
          for (int r = 0; r < R; ++r) c[j][r] = -1;
        }
      }
      double xv[J][R];
      // The stage is now in registers: hand it back to the producer before the x gathers.
      // The fence orders every lane's shared-memory reads before the arrive.
      asm volatile("fence.acq_rel.cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) bar_arrive(&empty[stage]);
      if (X == 3) {
        // the window covers every column the slice references (h >= bandwidth, rows in natural order, checked on
        // the host): every gather is a shared-memory read, no range test and no L1 path
        const int wl = (int)wlo;
#pragma unroll
        for (int j = 0; j < J; ++j)
#pragma unroll
          for (int r = 0; r < R; ++r) xv[j][r] = xs[c[j][r] < 0 ? 0 : c[j][r] - wl];
      } else if (X == 2) {
        // gathers inside the slice's window are shared-memory reads
#pragma unroll
        for (int j = 0; j < J; ++j)
#pragma unroll
          for (int r = 0; r < R; ++r) {
            const int cc = max(c[j][r], 0);
            const int64_t d = (int64_t)cc - wlo;
            xv[j][r] = (d >= 0 && d < wn) ? xs[d] : ldx<0>(x, cc);
          }
      } else {
#pragma unroll
        for (int j = 0; j < J; ++j)
#pragma unroll
          for (int r = 0; r < R; ++r) xv[j][r] = ldx<X>(x, max(c[j][r], 0));
      }
#pragma unroll
      for (int j = 0; j < J; ++j)
#pragma unroll
        for (int r = 0; r < R; ++r) acc[r] = c[j][r] >= 0 ? fma(v[j][r], xv[j][r], acc[r]) : acc[r];
      if (++stage == STAGES) { stage = 0; phase ^= 1; }
    }
    if (X >= 2 && w > 0) {       // every window read of this warp is done: the buffer may be refilled
      asm volatile("fence.acq_rel.cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) bar_arrive(&wempty[wb]);
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (orow[r] >= 0) y[orow[r]] = (beta == 0.0) ? alpha * acc[r] : fma(alpha, acc[r], beta * yold[r]);
      else if (PERM && orow[r] < -1) part[-(orow[r] + 2)] = acc[r];   // segment of a split row
    }
  }
}

struct TmaEntry { int R, STAGES, J, X, I16; const void* k[2]; };
#define TE(r, st, j) {r, st, j, 0, 0, {(const void*)sell_tma_kernel<r, st, j, 0, 0, int>, (const void*)sell_tma_kernel<r, st, j, 1, 0, int>}}
#define TX(r, st, j) {r, st, j, 2, 0, {(const void*)sell_tma_kernel<r, st, j, 0, 2, int>, (const void*)sell_tma_kernel<r, st, j, 1, 2, int>}}
#define TS(r, st, j) {r, st, j, 0, 1, {(const void*)sell_tma_kernel<r, st, j, 0, 0, unsigned short>, (const void*)sell_tma_kernel<r, st, j, 1, 0, unsigned short>}}
static const TmaEntry g_tma[] = {TE(1, 2, 8), TE(1, 3, 8), TE(1, 4, 8), TE(1, 3, 4), TE(1, 4, 4), TE(1, 6, 4),
                                 TE(2, 2, 8), TE(2, 3, 8), TE(2, 4, 8), TE(2, 3, 4), TE(2, 4, 4), TE(2, 6, 4),
                                 TE(1, 3, 16), TE(2, 3, 16), TE(1, 2, 16), TE(2, 2, 16),
                                 TX(1, 2, 8), TX(1, 3, 8), TX(1, 4, 8), TX(1, 3, 4), TX(1, 4, 4), TX(2, 2, 8), TX(2, 3, 8),
                                 TX(2, 3, 4), TX(2, 4, 4), TX(1, 2, 16), TX(1, 3, 16), TX(2, 2, 16), TX(1, 6, 4), TX(2, 4, 8),
                                 TS(1, 2, 8), TS(1, 3, 4), TS(1, 3, 8), TS(1, 4, 8), TS(1, 4, 4), TS(1, 6, 4), TS(1, 2, 16), TS(1, 3, 16),
                                 TS(2, 3, 8), TS(2, 4, 8), TS(2, 4, 4), TS(2, 6, 4), TS(2, 2, 16), TS(2, 3, 16)};
#undef TS
#undef TX
#undef TE
#define TX3(r, st, j) {r, st, j, 3, 0, {(const void*)sell_tma_kernel<r, st, j, 0, 3, int>, nullptr}}, \
                      {r, st, j, 3, 1, {(const void*)sell_tma_kernel<r, st, j, 0, 3, unsigned short>, nullptr}}
static const TmaEntry g_tma_full[] = {TX3(1, 2, 8), TX3(1, 3, 8), TX3(1, 4, 8), TX3(1, 3, 4), TX3(1, 4, 4), TX3(1, 6, 4),
                                      TX3(2, 3, 8), TX3(2, 4, 8), TX3(2, 4, 4), TX3(1, 2, 16), TX3(1, 3, 16)};
#undef TX3
#define TSX(r, st, j) {r, st, j, 2, 1, {(const void*)sell_tma_kernel<r, st, j, 0, 2, unsigned short>, (const void*)sell_tma_kernel<r, st, j, 1, 2, unsigned short>}}
static const TmaEntry g_tma16x[] = {TSX(1, 2, 8), TSX(1, 3, 8), TSX(1, 4, 8), TSX(1, 3, 4), TSX(1, 4, 4), TSX(1, 6, 4),
                                    TSX(2, 3, 8), TSX(2, 4, 8), TSX(2, 4, 4)};
#undef TSX

static const TmaEntry* tma_pick(const Variant& v) {
  const int i16 = v.fam == FAM_SELL16_TMA ? 1 : 0;
  for (const auto& e : g_tma)
    if (e.R == v.R && e.STAGES == v.I && e.J == v.U && e.X == v.X && e.I16 == i16) return &e;
  for (const auto& e : g_tma16x)
    if (e.R == v.R && e.STAGES == v.I && e.J == v.U && e.X == v.X && e.I16 == i16) return &e;
  for (const auto& e : g_tma_full)
    if (e.R == v.R && e.STAGES == v.I && e.J == v.U && e.X == v.X && e.I16 == i16) return &e;
  return nullptr;
}
static int tma_win(const Variant& v) { return v.X >= 2 ? v.C + 2 * v.H : 0; }
static size_t tma_smem(const Variant& v) {
  const size_t entry = v.fam == FAM_SELL16_TMA ? 10 : 12;
  return (size_t)v.I * v.U * v.C * entry + (size_t)2 * tma_win(v) * 8 + (2 * v.I + 4) * 8 + 128;
}

bool sell_tma_supported(const Variant& v) {
  if (!tma_pick(v)) return false;
  if (v.C < 128 || v.C > 1024 || (v.C & (v.C - 1))) return false;
  if (v.S < 1 || (v.S > 1 && (v.S % v.C != 0 || v.S > 8192 || (v.S & (v.S - 1))))) return false;
  const int consumers = v.C / v.R;
  if (consumers < 32 || consumers > 512 || v.block != consumers + 32) return false;
  if (v.X >= 2 ? (v.H < 8 || v.H > 4096 || v.H % 8) : v.H != 0) return false;
  return tma_smem(v) <= 200 * 1024;
}
cudaError_t sell_tma_plan(const Variant& v, int64_t rows, int64_t cols, const SellFormat& f, int sm_count,
                          LaunchPlan* out) {
  const TmaEntry* e = tma_pick(v);
  if (!e || f.C != v.C || (v.fam == FAM_SELL16_TMA) != (f.col16 != nullptr)) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (rows == 0) return cudaSuccess;
  KernelCall& c = out->k[0];
  c.fn = e->k[f.perm ? 1 : 0];
  if (!c.fn) return cudaErrorInvalidValue;       // x3 exists for natural row order only
  c.block = v.block;
  c.smem = (unsigned)tma_smem(v);
  cudaError_t err = allow_smem(c.fn, c.smem);
  if (err != cudaSuccess) return err;
  // persistent: g (default 1) waves of resident CTAs, never more CTAs than slices
  err = resolve_grid(v.grid > 0 ? v.grid : 1, c.fn, v.block, c.smem, sm_count, f.nslices, &c.grid);
  if (err != cudaSuccess) return err;
  c.add(rows); c.add((int64_t)f.nslices); c.add(f.C); c.add((const int64_t*)f.slice_ptr); c.add((const double*)f.val);
  c.add(f.col16 ? (const void*)f.col16 : (const void*)f.col); c.add((const int*)f.sbase); c.add((const int*)f.perm);
  c.add(f.part);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
  // x window bulk copies need a 16-byte aligned x; otherwise the window is empty (cols = 0: every gather
  // goes through L1) -- same results, the variant just loses its point
  if (v.X == 2) c.add_flag(3, cols); else c.add(cols);
  if (v.X == 3) {          // the window copies need a 16-byte aligned x: otherwise the x0 kernel of the same shape runs
    Variant v0 = v; v0.X = 0; v0.H = 0;
    LaunchPlan p0;
    err = sell_tma_plan(v0, rows, cols, f, sm_count, &p0);
    if (err != cudaSuccess) return err;
    out->alt = p0.k[0];
    out->has_alt = true;
  }
  c.add((int)v.H);
  c.per_block = 1;               // slices per CTA trip; the grid is capped at the persistent size
  out->n = 1;
  if (f.split && f.nsplit > 0) { sell_split_fixup_call(f, &out->k[1]); out->n = 2; }
  else if (v.X < 2) {
    out->range_kind = RANGE_SELL_TMA;
    out->range_align = std::max(f.C, f.sigma);
    out->range_elem = f.C;
  }
  return cudaSuccess;
}

}  // namespace spmv
