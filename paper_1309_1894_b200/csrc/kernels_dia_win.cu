// DIA with EVERYTHING staged in shared memory by the TMA engine: values, mask words, old y and the
// x WINDOWS of the slice (SURVEY.md sec. 8(a) row a10 (ii) "x staged in shared memory", applied to the
// stencil-aware format of sec. 8(f) rank 1).
//
// Why: in dia / dia_tma / dia_const every x[row + off[d]] is an LDG through L1.  A warp-wide 8-byte load
// of 32 consecutive (unaligned) entries is 2-3 L1 wavefronts and multi-wavefront loads replay at ~2
// cycles per wavefront (B300_MICROARCH.md, "L1tex wavefront queue"): 27 diagonals cost ~150 L1 cycles
// per 32 rows, 7 diagonals of the constant-coefficient kernel were ~all of its 16 us of active time.
// Diagonals come in GROUPS of near-consecutive offsets (a 27-point stencil: 9 groups of 3; a 7-point
// one: -n^2, -n, {-1,0,1}, n, n^2), and one contiguous window x[s*C + lo_g, s*C + lo_g + len_g) serves
// every diagonal of its group for all C rows of slice s.  One elected producer thread brings, per slice,
// one bulk copy per group plus values / masks / old y; consumers only read shared memory (conflict-free:
// consecutive threads, consecutive addresses) and write y.  No L1 wavefronts on the load side at all.
//
// Entries absent from the CSR matrix are never multiplied (mask bit, reading A7).  Window parts outside
// [0, cols) are not copied (and never referenced by a set mask bit); if cols is odd its last entry cannot
// be part of a 16-byte copy and is read with a plain load.  Deterministic: a row is summed by one thread
// in ascending-offset order -- bit-identical to dia / dia_const.
#include <algorithm>

#include "device_utils.cuh"
#include "spmv_internal.h"
#include "tma_utils.cuh"

namespace spmv {

struct DiaWinMeta {
  int off[32];     // diagonal offsets (ascending)
  int xoff[32];    // element index inside the stage's window area of x[s*C + off[d]]  (row 0 of the slice)
  double coef[32]; // constant coefficients (CONST kernels)
  int g_lo[32];    // per group: window start relative to s*C (even)
  int g_len[32];   // per group: window length in entries (even)
  int g_dst[32];   // per group: element offset of the window inside the window area
  int ng, win_total;
};

// blockDim.x = C/R consumers + 32 (producer warp).  One stage = one whole slice.
template <int R, int STAGES, int CONST>
__global__ void __launch_bounds__(512 + 32)
dia_win_kernel(int64_t rows, int64_t cols, int64_t nslices, int C, int nd, DiaWinMeta meta,
               const double* __restrict__ dval, const unsigned* __restrict__ mask, double alpha,
               const double* __restrict__ x, double beta, double* __restrict__ y, int y_bulk, int x_bulk) {
  extern __shared__ __align__(128) unsigned char win_smem[];
  const int nconsumers = C / R;
  const int vals_d = CONST ? 0 : nd * C;                         // doubles
  const int stage_d = vals_d + C + meta.win_total + C / 2;       // vals | old y | windows | masks (u32)
  double* s_stage = reinterpret_cast<double*>(win_smem);
  uint64_t* full = reinterpret_cast<uint64_t*>(s_stage + (size_t)STAGES * stage_d);
  uint64_t* empty = full + STAGES;
  int* s_off = reinterpret_cast<int*>(empty + STAGES);           // [32] offsets
  int* s_xoff = s_off + 32;                                      // [32] window indices
  double* s_coef = reinterpret_cast<double*>(s_xoff + 32);       // [32]
  const int tid = threadIdx.x;
  if (tid < 32) { s_off[tid] = meta.off[tid]; s_xoff[tid] = meta.xoff[tid]; s_coef[tid] = meta.coef[tid]; }
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) {
      tma::bar_init(&full[s], 1);
      tma::bar_init(&empty[s], nconsumers / 32);
    }
    tma::bar_init_fence();
  }
  __syncthreads();
  const bool want_y = beta != 0.0 && y_bulk;
  const int64_t cols_even = cols & ~(int64_t)1;

  if (tid >= nconsumers) {
    if (tid == nconsumers) {
      uint32_t stage = 0, phase = 0;
      for (int64_t s = blockIdx.x; s < nslices; s += gridDim.x) {
        double* st = s_stage + (size_t)stage * stage_d;
        const bool ybulk = want_y && (s + 1) * C <= rows;
        tma::bar_wait(&empty[stage], phase ^ 1);
        tma::fence_proxy_async();
        // byte count first (the copies below must add up to exactly this)
        uint32_t bytes = (uint32_t)vals_d * 8u + (uint32_t)C * 4u + (ybulk ? (uint32_t)C * 8u : 0u);
        if (x_bulk) {
          for (int g = 0; g < meta.ng; ++g) {
            const int64_t gs = s * C + meta.g_lo[g], ge = gs + meta.g_len[g];
            const int64_t cs = gs > 0 ? gs : 0, ce = ge < cols_even ? ge : cols_even;
            if (ce > cs) bytes += (uint32_t)(ce - cs) * 8u;
          }
        }
        tma::bar_expect_tx(&full[stage], bytes);
        if (!CONST) tma::bulk_g2s(st, dval + s * nd * C, (uint32_t)vals_d * 8u, &full[stage]);
        if (ybulk) tma::bulk_g2s(st + vals_d, y + s * C, (uint32_t)C * 8u, &full[stage]);
        tma::bulk_g2s(st + vals_d + C + meta.win_total, mask + s * C, (uint32_t)C * 4u, &full[stage]);
        if (x_bulk) {
          for (int g = 0; g < meta.ng; ++g) {
            const int64_t gs = s * C + meta.g_lo[g], ge = gs + meta.g_len[g];
            const int64_t cs = gs > 0 ? gs : 0, ce = ge < cols_even ? ge : cols_even;
            if (ce > cs)
              tma::bulk_g2s(st + vals_d + C + meta.g_dst[g] + (cs - gs), x + cs, (uint32_t)(ce - cs) * 8u, &full[stage]);
          }
        }
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
    }
    return;
  }

  uint32_t stage = 0, phase = 0;
  const int lane = tid & 31;
  for (int64_t s = blockIdx.x; s < nslices; s += gridDim.x) {
    const double* st = s_stage + (size_t)stage * stage_d;
    const double* s_val = st;
    const double* s_y = st + vals_d;
    const double* s_win = st + vals_d + C;
    const unsigned* s_mask = reinterpret_cast<const unsigned*>(st + vals_d + C + meta.win_total);
    const bool ybulk = want_y && (s + 1) * C <= rows;
    const int i0 = tid * R;
    const int64_t r0 = s * C + i0;
    double yold[R], acc[R];
    unsigned m[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { acc[r] = 0.0; yold[r] = 0.0; }
    if (beta != 0.0 && !ybulk) {
#pragma unroll
      for (int r = 0; r < R; ++r) yold[r] = r0 + r < rows ? y[r0 + r] : 0.0;
    }
    tma::bar_wait(&full[stage], phase);
#pragma unroll
    for (int r = 0; r < R; ++r) {
      m[r] = s_mask[i0 + r];
      if (ybulk) yold[r] = s_y[i0 + r];
    }
#pragma unroll 4
    for (int d = 0; d < nd; ++d) {
      const int o = s_off[d], xo = s_xoff[d];
      const double c = CONST ? s_coef[d] : 0.0;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        if ((m[r] >> d) & 1u) {
          const int64_t xi = r0 + r + o;                 // in [0, cols) because the entry is stored
          const double xv = (x_bulk && xi < cols_even) ? s_win[xo + i0 + r] : __ldg(x + xi);
          const double v = CONST ? c : s_val[d * C + i0 + r];
          acc[r] = fma(v, xv, acc[r]);
        }
      }
    }
    // every lane has read what it needs from the stage: hand it back
    asm volatile("fence.acq_rel.cta;" ::: "memory");
    __syncwarp();
    if (lane == 0) tma::bar_arrive(&empty[stage]);
#pragma unroll
    for (int r = 0; r < R; ++r)
      if (r0 + r < rows) y[r0 + r] = (beta == 0.0) ? alpha * acc[r] : fma(alpha, acc[r], beta * yold[r]);
    if (++stage == STAGES) { stage = 0; phase ^= 1; }
  }
}

typedef void (*dia_win_kernel_t)(int64_t, int64_t, int64_t, int, int, DiaWinMeta, const double*, const unsigned*, double,
                                 const double*, double, double*, int, int);
struct DiaWinEntry { int R, STAGES, CONST; dia_win_kernel_t k; };
#define WE(r, st) {r, st, 0, dia_win_kernel<r, st, 0>}, {r, st, 1, dia_win_kernel<r, st, 1>}
static const DiaWinEntry g_dia_win[] = {WE(1, 2), WE(1, 3), WE(1, 4), WE(2, 2), WE(2, 3), WE(2, 4)};
#undef WE

static const DiaWinEntry* dia_win_pick(const Variant& v) {
  const int cst = v.fam == FAM_DIA_CWIN ? 1 : 0;
  if (v.X != 0) return nullptr;
  for (const auto& e : g_dia_win)
    if (e.R == v.R && e.STAGES == v.I && e.CONST == cst) return &e;
  return nullptr;
}

bool dia_win_supported(const Variant& v) {
  if (!dia_win_pick(v)) return false;
  if (!(v.C == 128 || v.C == 256 || v.C == 512)) return false;
  const int consumers = v.C / v.R;
  return consumers >= 32 && consumers <= 512 && v.block == consumers + 32;
}
static size_t dia_win_smem(const Variant& v, const DiaFormat& f) {
  const size_t vals_d = v.fam == FAM_DIA_CWIN ? 0 : (size_t)f.nd * f.C;
  const size_t stage_d = vals_d + f.C + f.win_total + f.C / 2;
  return (size_t)v.I * stage_d * 8 + 2 * (size_t)v.I * 8 + 32 * 4 * 2 + 32 * 8 + 128;
}
bool dia_win_fits(const Variant& v, const DiaFormat& f) { return dia_win_smem(v, f) <= 200 * 1024; }

cudaError_t dia_win_plan(const Variant& v, int64_t rows, int64_t cols, const DiaFormat& f, int sm_count,
                         LaunchPlan* out) {
  const DiaWinEntry* e = dia_win_pick(v);
  if (!e || f.C != v.C || (e->CONST && !f.is_const)) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (rows == 0) return cudaSuccess;
  KernelCall& c = out->k[0];
  const size_t smem = dia_win_smem(v, f);
  if (smem > 200 * 1024) return cudaErrorInvalidValue;
  c.fn = (const void*)e->k;
  c.block = v.block;
  c.smem = (unsigned)smem;
  cudaError_t err = allow_smem(c.fn, c.smem);
  if (err != cudaSuccess) return err;
  const int64_t nslices = f.ld / f.C;
  err = resolve_grid(v.grid > 0 ? v.grid : 1, c.fn, v.block, c.smem, sm_count, nslices, &c.grid);   // persistent
  if (err != cudaSuccess) return err;
  DiaWinMeta m;
  for (int i = 0; i < 32; ++i) {
    m.off[i] = f.off[i]; m.xoff[i] = f.d_xoff[i]; m.coef[i] = f.coef[i];
    m.g_lo[i] = f.g_lo[i]; m.g_len[i] = f.g_len[i]; m.g_dst[i] = f.g_dst[i];
  }
  m.ng = f.ng;
  m.win_total = f.win_total;
  c.add(rows); c.add(cols); c.add(nslices); c.add(f.C); c.add(f.nd); c.add(m);
  c.add((const double*)f.val); c.add((const unsigned*)f.mask);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
  c.add_flag(1);                 // y_bulk
  c.add_flag(2);                 // x_bulk
  out->n = 1;
  return cudaSuccess;
}

// Offset groups for a slice height C (host; called by build_dia): consecutive offsets whose spread stays
// within 8 entries share one window [lo, lo + len), lo and len even so that every copy is 16-byte aligned.
void dia_compute_windows(DiaFormat& f) {
  int g = 0, dst = 0;
  int d = 0;
  while (d < f.nd) {
    int e = d;
    while (e + 1 < f.nd && f.off[e + 1] - f.off[d] <= 8) ++e;
    const int lo = f.off[d] & ~1;                            // floor to even (two's complement, also for negatives)
    int len = f.C + (f.off[e] - lo);                         // covers rows 0..C-1 for every offset of the group
    len = (len + 1) & ~1;
    f.g_lo[g] = lo; f.g_len[g] = len; f.g_dst[g] = dst;
    for (int k = d; k <= e; ++k) f.d_xoff[k] = dst + (f.off[k] - lo);
    dst += len;
    ++g;
    d = e + 1;
  }
  f.ng = g;
  f.win_total = dst;                                         // even: every g_len is even
  for (int k = f.nd; k < 32; ++k) f.d_xoff[k] = f.d_xoff[f.nd - 1];
}

}  // namespace spmv
