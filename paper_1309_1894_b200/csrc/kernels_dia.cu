// Stencil-aware DIA format: converter and kernel (the paper's own GPU
// work is "stencil-aware" / "stencil-based", PAPER.md:33 ref [1], PAPER.md:39 ref [2]).
//
// A matrix whose stored entries lie on nd <= 32 diagonals (col - row in a small set) is stored
// WITHOUT column indices, slice-major (slices of C rows, C in {128, 256, 512}):
//     dval[((row / C) * nd + d) * C + row % C] = value of entry (row, row + off[d])
//     mask[row] bit d                          = 1 iff that entry is stored in the CSR matrix
// so the values of consecutive diagonals of one slice are one contiguous run (one bulk copy).
// 8 bytes per non-zero instead of CSR's 12 (plus 4 bytes per row for the mask).  Entries that are
// absent from the CSR matrix (Dirichlet-truncated neighbours) are never multiplied (reading A7): the
// mask bit predicates both the x load and the FMA, so NaN/Inf in x reaches exactly the rows CSR
// semantics say.  x[row + off] is a shifted contiguous stream: coalesced, no gather.
// Deterministic: one thread sums a row over the diagonals in ascending-offset order.
#include <string.h>

#include <algorithm>

#include "cg_reduce.cuh"
#include "device_utils.cuh"
#include "spmv_internal.h"
#include "tma_utils.cuh"

namespace spmv {

struct DiaOffsets { int off[32]; };

template <int R>
struct DiaVec;
template <>
struct DiaVec<1> {
  static __device__ __forceinline__ void load(const double* p, double* v) { v[0] = ld_stream(p); }
};
template <>
struct DiaVec<2> {
  static __device__ __forceinline__ void load(const double* p, double* v) {
    double2 a = ld_stream2(p);
    v[0] = a.x; v[1] = a.y;
  }
};
template <>
struct DiaVec<4> {
  static __device__ __forceinline__ void load(const double* p, double* v) {
    double2 a = ld_stream2(p), b = ld_stream2(p + 2);
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
  }
};

// thread owns R adjacent rows of one slice; U diagonals per trip, all loads of a trip issued before the FMAs
template <int R, int U, int X>
__global__ void __launch_bounds__(512)
dia_kernel(int64_t rows, int64_t ld, int C, int logC, int nd, DiaOffsets offs, const double* __restrict__ dval,
           const unsigned* __restrict__ mask, double alpha, const double* __restrict__ x, double beta,
           double* __restrict__ y) {
  const int64_t G = (int64_t)gridDim.x * blockDim.x;
  for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g * R < ld; g += G) {
    const int64_t r0 = g * R;
    const int64_t sl = r0 >> logC;
    const double* pv = dval + sl * nd * C + (r0 - (sl << logC));      // diagonal d of this slice at pv + d*C
    unsigned m[R];
    double acc[R], yold[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      m[r] = r0 + r < rows ? __ldg(mask + r0 + r) : 0u;
      acc[r] = 0.0;
    }
#pragma unroll
    for (int r = 0; r < R; ++r) yold[r] = (beta != 0.0 && r0 + r < rows) ? y[r0 + r] : 0.0;
    for (int d0 = 0; d0 < nd; d0 += U) {
      double v[U][R], xv[U][R];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int d = min(d0 + u, nd - 1);          // past-the-end trips re-read the last diagonal, masked below
        DiaVec<R>::load(pv + (int64_t)d * C, v[u]);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int d = d0 + u;
        const int o = offs.off[min(d, nd - 1)];
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const bool on = d < nd && ((m[r] >> d) & 1u);
          xv[u][r] = on ? ldx<X>(x, (int)(r0 + r) + o) : 0.0;   // absent entries are never loaded (A7)
        }
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int d = d0 + u;
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const bool on = d < nd && ((m[r] >> d) & 1u);
          acc[r] = on ? fma(v[u][r], xv[u][r], acc[r]) : acc[r];
        }
      }
    }
#pragma unroll
    for (int r = 0; r < R; ++r)
      if (r0 + r < rows) y[r0 + r] = (beta == 0.0) ? alpha * acc[r] : fma(alpha, acc[r], beta * yold[r]);
  }
}

typedef void (*dia_kernel_t)(int64_t, int64_t, int, int, int, DiaOffsets, const double*, const unsigned*, double,
                             const double*, double, double*);

template <int X>
static dia_kernel_t dia_pick_ru(int R, int U) {
#define P(r, u) if (R == r && U == u) return dia_kernel<r, u, X>;
  P(1, 1) P(1, 2) P(1, 4) P(1, 8) P(2, 1) P(2, 2) P(2, 4) P(2, 8) P(4, 2) P(4, 4)
#undef P
  return nullptr;
}
static dia_kernel_t dia_pick(const Variant& v) {
  return v.X == 0 ? dia_pick_ru<0>(v.R, v.U) : v.X == 1 ? dia_pick_ru<1>(v.R, v.U) : nullptr;
}
static bool dia_c_ok(int C) { return C == 128 || C == 256 || C == 512; }

bool dia_supported(const Variant& v) {
  return v.block >= 32 && v.block <= 512 && v.block % 32 == 0 && dia_c_ok(v.C) && dia_pick(v) != nullptr;
}
static DiaOffsets dia_offsets(const DiaFormat& f) {
  DiaOffsets o;
  for (int i = 0; i < 32; ++i) o.off[i] = f.off[i];
  return o;
}

cudaError_t dia_plan(const Variant& v, int64_t rows, const DiaFormat& f, int sm_count, LaunchPlan* out) {
  dia_kernel_t k = dia_pick(v);
  if (!k || f.C != v.C) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (rows == 0) return cudaSuccess;
  KernelCall& c = out->k[0];
  c.fn = (const void*)k;
  c.block = v.block;
  const int64_t threads = (f.ld + v.R - 1) / v.R;
  const int64_t exact = (threads + v.block - 1) / v.block;
  cudaError_t e = resolve_grid(v.grid, c.fn, v.block, 0, sm_count, exact, &c.grid);
  if (e != cudaSuccess) return e;
  c.add(rows); c.add((int64_t)f.ld); c.add(f.C); c.add(f.logC); c.add(f.nd); c.add(dia_offsets(f));
  c.add((const double*)f.val); c.add((const unsigned*)f.mask);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
  c.per_block = (int64_t)v.block * v.R;
  out->n = 1;
  out->range_kind = RANGE_DIA;
  out->range_align = f.C;
  out->range_elem = f.nd;
  return cudaSuccess;
}

// ------------------------------------------------------------------ constant-coefficient stencil
// When every stored entry of a diagonal carries the same value (a constant-coefficient stencil such as
// cfg2's diag 6 / off -1), the values need not be streamed at all: the kernel reads the mask word
// (which entries exist near the boundary), x and y only.  Same summation order as dia_kernel, and the
// coefficients are the stored bit patterns, so the result equals dia_kernel's bit for bit.
//
// Shape (round 2; measured on cfg2 with a stand-alone probe of the same stencil, not kept): one trip per thread over an EXACT grid
// -- the hardware block scheduler keeps every SM's load queue full, a persistent grid-stride loop with
// software pipelining (round 1: 124 registers, 21 us) does not -- a thread owns R adjacent rows and reads
// x[r0 + off .. r0 + off + R) as aligned 16-byte pairs; for an odd offset the pair is taken one element
// to the left and the missing right neighbour comes from the next lane by shuffle (lane 31 loads it).
// The mask is stored in the narrowest type that holds nd bits (1 byte per row for nd <= 8).  The kernel
// is a programmatic dependent launch: it signals its own dependents at once, loads its mask words
// (immutable, owned by the handle) and only then waits for the previous kernel of the stream, so the
// launch latency and the first memory round trip of apply k+1 overlap the tail of apply k.
struct DiaCoefs { double c[32]; };

template <int X>
__device__ __forceinline__ double2 ldx2(const double* __restrict__ x, int i) {     // 16-byte aligned
  if (X == 0) return __ldg(reinterpret_cast<const double2*>(x + i));
  double2 v;
  asm volatile("ld.global.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(x + i));
  return v;
}

// x indices are relative to the x pointer the kernel was given and valid in [xlo, xhi] (the whole vector:
// [0, cols - 1]; a row range [a, b) launched by spmv_apply_host: x + a, [-a, cols - 1 - a]).
// R > 1 (needs cols % 2 == 0, xlo even and a 16-byte aligned x): e[r] = x[b + r], r < R, b even, as aligned pairs.
// A pair lies either completely inside [xlo, xhi] or completely outside; an outside pair is read at a clamped
// (still aligned) index and never multiplied (its mask bits are off: such entries cannot be stored).
template <int R, int X>
__device__ __forceinline__ void dia_load_pairs(const double* __restrict__ x, int b, int xlo, int xhi, double (&e)[R]) {
#pragma unroll
  for (int r = 0; r < R; r += 2) {
    const double2 p = ldx2<X>(x, min(max(b + r, xlo), xhi - 1));
    e[r] = p.x; e[r + 1] = p.y;
  }
}

template <typename MT> struct DiaMaskVec;
template <> struct DiaMaskVec<unsigned char> { typedef uchar2 V2; typedef uchar4 V4; };
template <> struct DiaMaskVec<unsigned short> { typedef ushort2 V2; typedef ushort4 V4; };
template <> struct DiaMaskVec<unsigned> { typedef uint2 V2; typedef uint4 V4; };

// ND > 0: exactly ND diagonals, fully unrolled, no run-time diagonal count (5-, 7-, 9-, 27-point stencils);
// ND == 0: any nd <= 32, chunks of 8 with warp-uniform guards.  Registers decide this kernel's speed (one
// memory round trip per thread: occupancy IS the memory-level parallelism; measured 21 us at 59 registers,
// 12.7 us at 23 on cfg2), hence the exact instantiations and the min-blocks launch bound.
constexpr int dia_const_min_blocks(int R, int ND) { return (ND == 0 || ND > 9) ? (R == 4 ? 1 : 2) : (R == 1 ? 4 : R == 2 ? 2 : 1); }

// DOT (R == 1 only; the solver loop, solver.cu): the kernel also writes its block's share of sum_i x_i * y_i
// (square matrix) to dot_part[blockIdx.x]; the caller adds the gridDim.x partials in index order.  No
// arrival counter here: a fence + atomic at the tail of 8192 short blocks costs more than the dot pass saved.
// TRI (R == 2 only): the diagonals come in runs (o - 1, o, o + 1) with o even around every "base" offset -- the
// natural ordering of a 5-, 7- or 27-point stencil on a grid of even extent: diagonal d with d % 3 == tri_phase is
// the centre of a run, its left and right neighbours are NOT loaded: x[r0 + o - 1 .. ] and x[r0 + o + 1 .. ] are
// assembled from the centre's aligned pair and one shuffle (the previous lane's second element, the next lane's
// first); lanes 0 and 31 load their missing element in the load phase, so it stays one memory round trip.
// Centres: every diagonal whose two neighbours in the list are at distance 1 (tri_mask, checked on the host).
// BZ: beta == 0 (y is write-only).  Instruction count decides a kernel this short (ncu: 6.6 M warp instructions
// took 15.5 us, 4.4 M took 11.9 us, same memory requests), so the two cases are separate instantiations chosen by
// a uniform branch at kernel entry instead of predicated code, and the R > 1 forms require rows % R == 0 (the plan
// falls back to R = 1 otherwise) so that a thread's rows are all live or all dead.
// DOT == 2 (R == 1, BZ, square matrix; the Jacobi loop, jacobi.cu): the whole weighted-Jacobi step in this kernel.
// alpha carries omega, y is the NEXT iterate: r_i = jb[i] - (A x)_i, y[i] = x[i] + omega * r_i / jd, and the block's
// share of sum_i r_i^2 goes to dot_part[blockIdx.x] (added in index order by the caller's finishing kernel).  jd is
// the coefficient of the offset-0 diagonal: with constant coefficients every row that stores its diagonal entry has
// that value, and the caller has established on the device that every row does (else it never lets this kernel run).
template <int R, int ND, int X, typename MT, int DOT, unsigned TRI, bool BZ>
__device__ __forceinline__ void
dia_const_body(int rows, int xlo, int xhi, int nd_rt, const DiaOffsets& offs, const DiaCoefs& coefs, const MT* __restrict__ mask,
               double alpha, const double* __restrict__ x, double beta, double* __restrict__ y,
               double* __restrict__ dot_part = nullptr, const double* __restrict__ jb = nullptr, double jd = 1.0,
               const int* __restrict__ jdone = nullptr) {
  constexpr int NDC = ND == 0 ? 8 : (ND % 9 == 0 ? 9 : (ND <= 8 ? ND : 8));     // diagonals per chunk
  constexpr int DMAX = ND == 0 ? 32 : ND;
  const int nd = ND == 0 ? nd_rt : ND;
  // 32-bit indices: build_dia admits the pattern only when rows + cols < 2^31.  Exact grid, one trip per
  // thread.  Lanes past the end stay for the shuffles (R > 1) on the virtual rows after the last one: their
  // x indices are clamped, their mask words exist (the mask array is padded to a multiple of the slice
  // height >= 32*R), nothing is stored.
  const int r0 = (blockIdx.x * blockDim.x + threadIdx.x) * R;
  const int lane = threadIdx.x & 31;
  (void)lane;
  if (R == 1 && DOT == 0 && r0 >= rows) return;
  unsigned m[R];
  if constexpr (R == 2) {
    const typename DiaMaskVec<MT>::V2 mm = *reinterpret_cast<const typename DiaMaskVec<MT>::V2*>(mask + r0);
    m[0] = mm.x; m[1] = mm.y;
  } else if constexpr (R == 4) {
    const typename DiaMaskVec<MT>::V4 mm = *reinterpret_cast<const typename DiaMaskVec<MT>::V4*>(mask + r0);
    m[0] = mm.x; m[1] = mm.y; m[2] = mm.z; m[3] = mm.w;
  } else {
    m[0] = mask[r0];
  }
  pdl_wait();                                                // x and y may be the previous kernel's output
  if constexpr (DOT == 2) {
    if (*jdone) return;                                      // the loop has stopped (uniform; written by the finishing kernel)
  }
  const bool live = r0 < rows;                               // R > 1: rows % R == 0, so all R rows or none
  double yold[R], acc[R];
#pragma unroll
  for (int r = 0; r < R; ++r) { yold[r] = 0.0; acc[r] = 0.0; }
  double jbi = 0.0;                                          // Jacobi step: right-hand side of this row,
  if constexpr (DOT == 2) {                                  // loaded in the same round trip as x
    if (live) jbi = jb[r0];
  }
  if constexpr (!BZ) {
    if (live) {
      if constexpr (R > 1) {
#pragma unroll
        for (int r = 0; r < R; r += 2) {
          const double2 p = *reinterpret_cast<const double2*>(y + r0 + r);
          yold[r] = p.x; yold[r + 1] = p.y;
        }
      } else {
        yold[0] = y[r0];
      }
    }
  }
  // statically unrolled over the chunks so that the by-value offset / coefficient parameters are never
  // indexed dynamically
#pragma unroll
  for (int d0 = 0; d0 < DMAX; d0 += NDC) {
    if (ND == 0 && d0 >= nd) break;
    double xv[NDC][R];
#pragma unroll
    for (int u = 0; u < NDC; ++u) {
      const int d = d0 + u;
      if (d < DMAX && (ND != 0 || d < nd)) {                 // warp-uniform
        const int o = offs.off[d < 32 ? d : 31];
        if constexpr (R == 1) {
          xv[u][0] = ldx<X>(x, min(max(r0 + o, xlo), xhi));
        } else if constexpr (R == 2 && TRI != 0) {
          if ((TRI >> (d & 31)) & 1u) {                        // centre of a run: its pair serves three diagonals
            dia_load_pairs<R, X>(x, r0 + o, xlo, xhi, xv[u]);
          } else if (d + 1 < DMAX && ((TRI >> ((d + 1) & 31)) & 1u)) {   // left neighbour: lane 0 loads x[r0 + o]
            xv[u][0] = lane == 0 ? ldx<X>(x, min(max(r0 + o, xlo), xhi)) : 0.0;
          } else if (d >= 1 && ((TRI >> ((d - 1) & 31)) & 1u)) {         // right neighbour: lane 31 loads x[r0 + o + 1]
            xv[u][1] = lane == 31 ? ldx<X>(x, min(max(r0 + o + 1, xlo), xhi)) : 0.0;
          } else {                                             // outside the runs every offset is even (host-checked):
            dia_load_pairs<R, X>(x, r0 + o, xlo, xhi, xv[u]);  // a run-time parity test compiles to both paths, predicated
          }
        } else {
          // warp-uniform on the offset's parity (r0 is even): an even offset is R/2 aligned 16-byte pairs; an odd
          // one is R 8-byte loads.  (Taking the odd run from the pair one element to the left plus a shuffle
          // from the next lane puts a dependent exchange between the loads of consecutive diagonals and a
          // second round trip for lane 31: measured 15.6 us against 11.4 us for one row per thread.)
          if ((o & 1) == 0) {
            dia_load_pairs<R, X>(x, r0 + o, xlo, xhi, xv[u]);
          } else {
#pragma unroll
            for (int r = 0; r < R; ++r) xv[u][r] = ldx<X>(x, min(max(r0 + o + r, xlo), xhi));
          }
        }
      }
    }
    if constexpr (R == 2 && TRI != 0) {
      // second phase, after every load of the chunk has been issued: the neighbours of each centre
#pragma unroll
      for (int u = 0; u < NDC; ++u) {
        const int d = d0 + u;
        if (d < DMAX && ((TRI >> (d & 31)) & 1u)) {
          const double up = __shfl_up_sync(0xffffffffu, xv[u][1], 1);       // previous lane's x[r0 - 1 + o]
          const double dn = __shfl_down_sync(0xffffffffu, xv[u][0], 1);     // next lane's x[r0 + 2 + o]
          if (u >= 1) { xv[u - 1][0] = lane == 0 ? xv[u - 1][0] : up; xv[u - 1][1] = xv[u][0]; }
          if (u + 1 < NDC) { xv[u + 1][1] = lane == 31 ? xv[u + 1][1] : dn; xv[u + 1][0] = xv[u][1]; }
        }
      }
    }
#pragma unroll
    for (int u = 0; u < NDC; ++u) {
      const int d = d0 + u;
      if (d < DMAX && (ND != 0 || d < nd)) {
        const double c = coefs.c[d < 32 ? d : 31];
#pragma unroll
        for (int r = 0; r < R; ++r) acc[r] = ((m[r] >> d) & 1u) ? fma(c, xv[u][r], acc[r]) : acc[r];
      }
    }
  }
  double out[R];
#pragma unroll
  for (int r = 0; r < R; ++r) out[r] = BZ ? alpha * acc[r] : fma(alpha, acc[r], beta * yold[r]);
  if constexpr (DOT == 2) {
    __shared__ double s_warp[33];
    double rr = 0.0;
    if (live) {
      const double ri = jbi - acc[0];
      y[r0] = fma(alpha, ri / jd, ldx<X>(x, r0));
      rr = ri * ri;
    }
    const double mine = block_sum_fixed(rr, s_warp);
    if (threadIdx.x == 0) dot_part[blockIdx.x] = mine;
    return;
  }
  if constexpr (DOT == 1) {
    __shared__ double s_warp[33];
    if (live) y[r0] = out[0];
    const double mine = block_sum_fixed(live ? ldx<X>(x, r0) * out[0] : 0.0, s_warp);
    if (threadIdx.x == 0) dot_part[blockIdx.x] = mine;
    return;
  }
  if (!live) return;
  if constexpr (R > 1) {
#pragma unroll
    for (int r = 0; r < R; r += 2) *reinterpret_cast<double2*>(y + r0 + r) = make_double2(out[r], out[r + 1]);
  } else {
    y[r0] = out[0];
  }
}

// kernel entry: launch_dependents, then the beta == 0 / beta != 0 instantiation of the body
#define DIA_CONST_ENTRY(R_, ND_, X_, MT_, DOT_, TRI_, ...)                                                         \
  pdl_launch_dependents();                                                                                        \
  if (beta == 0.0) dia_const_body<R_, ND_, X_, MT_, DOT_, TRI_, true>(rows, xlo, xhi, nd_rt, offs, coefs, mask, alpha, x, beta, y, ##__VA_ARGS__); \
  else dia_const_body<R_, ND_, X_, MT_, DOT_, TRI_, false>(rows, xlo, xhi, nd_rt, offs, coefs, mask, alpha, x, beta, y, ##__VA_ARGS__)

template <int R, int ND, int X, typename MT>
__global__ void __launch_bounds__(512, dia_const_min_blocks(R, ND))
dia_const_kernel(int rows, int xlo, int xhi, int nd_rt, const __grid_constant__ DiaOffsets offs,
                 const __grid_constant__ DiaCoefs coefs, const MT* __restrict__ mask, double alpha,
                 const double* __restrict__ x, double beta, double* __restrict__ y) {
  DIA_CONST_ENTRY(R, ND, X, MT, 0, 0u);
}

// centres of the (o - 1, o, o + 1) runs of a 5-, 7- or 27-point stencil in natural ordering (0: no such form)
constexpr unsigned dia_tri_mask(int ND) {
  return ND == 5 ? 0x4u : ND == 7 ? 0x8u : ND == 27 ? 0x2492492u : 0u;     // d = 2 | d = 3 | d = 1, 4, ..., 25
}
// two rows per thread, the +-1 neighbours shuffled out of the centre pair (TRI): 5 loads instead of 7 on cfg2
template <int ND, int X, typename MT>
__global__ void __launch_bounds__(256, ND <= 9 ? 6 : 3)
dia_const_kernel_r2t(int rows, int xlo, int xhi, int nd_rt, const __grid_constant__ DiaOffsets offs,
                     const __grid_constant__ DiaCoefs coefs, const MT* __restrict__ mask, double alpha,
                     const double* __restrict__ x, double beta, double* __restrict__ y) {
  DIA_CONST_ENTRY(2, ND, X, MT, 0, dia_tri_mask(ND));
}
template <int X, typename MT>
static const void* dia_const_pick_tri(int nd) {
  switch (nd) {
    case 5: return (const void*)dia_const_kernel_r2t<5, X, MT>;
    case 7: return (const void*)dia_const_kernel_r2t<7, X, MT>;
    case 27: return (const void*)dia_const_kernel_r2t<27, X, MT>;
    default: return nullptr;
  }
}
// host check of the run structure the TRI kernels assume
static bool dia_tri_ok(const DiaFormat& f) {
  const unsigned m = f.nd == 5 ? dia_tri_mask(5) : f.nd == 7 ? dia_tri_mask(7) : f.nd == 27 ? dia_tri_mask(27) : 0u;
  if (!m) return false;
  for (int c = 0; c < f.nd; ++c) {
    if ((m >> c) & 1u) {
      if (c < 1 || c + 1 >= f.nd || (f.off[c] & 1) || f.off[c - 1] != f.off[c] - 1 || f.off[c + 1] != f.off[c] + 1) return false;
    } else {
      const bool neighbour = (c + 1 < f.nd && ((m >> (c + 1)) & 1u)) || (c >= 1 && ((m >> (c - 1)) & 1u));
      if (!neighbour && (f.off[c] & 1)) return false;        // every diagonal outside the runs is read as aligned pairs
    }
  }
  return true;
}

// two rows per thread on a small stencil, blocks of at most 256 threads: 40 registers, 1536 threads per SM
template <int ND, int X, typename MT>
__global__ void __launch_bounds__(256, 6)
dia_const_kernel_r2(int rows, int xlo, int xhi, int nd_rt, const __grid_constant__ DiaOffsets offs,
                    const __grid_constant__ DiaCoefs coefs, const MT* __restrict__ mask, double alpha,
                    const double* __restrict__ x, double beta, double* __restrict__ y) {
  DIA_CONST_ENTRY(2, ND, X, MT, 0, 0u);
}

// one row per thread with the fused dot product (the solver loop)
template <int ND, typename MT>
__global__ void __launch_bounds__(512, 2)
dia_const_dot_kernel(int rows, int xlo, int xhi, int nd_rt, const __grid_constant__ DiaOffsets offs,
                     const __grid_constant__ DiaCoefs coefs, const MT* __restrict__ mask, double alpha,
                     const double* __restrict__ x, double beta, double* __restrict__ y, double* __restrict__ dot_part) {
  DIA_CONST_ENTRY(1, ND, 0, MT, 1, 0u, dot_part);
}
// the weighted-Jacobi step fused into the stencil product (jacobi.cu); a no-op once *done is set
template <int ND, typename MT>
__global__ void __launch_bounds__(512, 2)
dia_const_jacobi_kernel(int rows, int xhi, int nd_rt, const __grid_constant__ DiaOffsets offs,
                        const __grid_constant__ DiaCoefs coefs, const MT* __restrict__ mask, double omega,
                        const double* __restrict__ x, double* __restrict__ x_next, const double* __restrict__ b,
                        double d, double* __restrict__ part, const int* __restrict__ done) {
  pdl_launch_dependents();
  dia_const_body<1, ND, 0, MT, 2, 0u, true>(rows, 0, xhi, nd_rt, offs, coefs, mask, omega, x, 0.0, x_next, part, b, d, done);
}
template <typename MT>
static cudaError_t dia_const_jacobi_launch_mt(const DiaFormat& f, int block, int rows, int cols, const MT* mask, double omega,
                                              const double* x, double* x_next, const double* b, double d,
                                              double* part, const int* done, cudaStream_t s) {
  DiaCoefs co;
  for (int i = 0; i < 32; ++i) co.c[i] = f.coef[i];
  const DiaOffsets of = dia_offsets(f);
  const unsigned grid = (unsigned)((rows + block - 1) / block);
  const void* fn = f.nd == 5 ? (const void*)dia_const_jacobi_kernel<5, MT> : f.nd == 7 ? (const void*)dia_const_jacobi_kernel<7, MT>
                 : f.nd == 27 ? (const void*)dia_const_jacobi_kernel<27, MT> : (const void*)dia_const_jacobi_kernel<0, MT>;
  int xhi = cols - 1, nd = f.nd;
  void* args[] = {&rows, &xhi, &nd, (void*)&of, (void*)&co, &mask, &omega, &x, &x_next, &b, &d, &part, &done};
  return launch_kernel_pdl(fn, grid, (unsigned)block, 0, s, args, true);      // programmatic dependent launch
}
int dia_const_jacobi_blocks(const Variant& v, int64_t rows) {
  const int block = std::min(std::max(v.block, 32), 512);
  return (int)((rows + block - 1) / block);
}
cudaError_t dia_const_jacobi_launch(const Variant& v, int64_t rows, int64_t cols, const DiaFormat& f, double omega,
                                    const double* x, double* x_next, const double* b, double* part,
                                    const int* done, cudaStream_t s) {
  if (!f.is_const || rows != cols || rows == 0) return cudaErrorInvalidValue;
  double d = 1.0;                                  // (no offset-0 diagonal: every row lacks it, the caller's `done` is set)
  for (int i = 0; i < f.nd; ++i)
    if (f.off[i] == 0) d = f.coef[i];
  const int block = std::min(std::max(v.block, 32), 512);
  const int me = f.mask_small ? f.mask_elem : 4;
  if (me == 1) return dia_const_jacobi_launch_mt<unsigned char>(f, block, (int)rows, (int)cols, (const unsigned char*)f.mask_small, omega, x, x_next, b, d, part, done, s);
  if (me == 2) return dia_const_jacobi_launch_mt<unsigned short>(f, block, (int)rows, (int)cols, (const unsigned short*)f.mask_small, omega, x, x_next, b, d, part, done, s);
  return dia_const_jacobi_launch_mt<unsigned>(f, block, (int)rows, (int)cols, (const unsigned*)f.mask, omega, x, x_next, b, d, part, done, s);
}

template <typename MT>
static const void* dia_const_dot_pick_nd(int nd) {
  switch (nd) {
    case 5: return (const void*)dia_const_dot_kernel<5, MT>;
    case 7: return (const void*)dia_const_dot_kernel<7, MT>;
    case 27: return (const void*)dia_const_dot_kernel<27, MT>;
    default: return (const void*)dia_const_dot_kernel<0, MT>;
  }
}

template <int R, int X, typename MT>
static const void* dia_const_pick_nd(int nd, int block) {
  if constexpr (R == 2) {
    if (block <= 256) switch (nd) {               // 40 registers under __launch_bounds__(256, 6)
      case 3: return (const void*)dia_const_kernel_r2<3, X, MT>;
      case 5: return (const void*)dia_const_kernel_r2<5, X, MT>;
      case 7: return (const void*)dia_const_kernel_r2<7, X, MT>;
      case 9: return (const void*)dia_const_kernel_r2<9, X, MT>;
      default: break;
    }
  }
  switch (nd) {
    case 3: return (const void*)dia_const_kernel<R, 3, X, MT>;
    case 5: return (const void*)dia_const_kernel<R, 5, X, MT>;
    case 7: return (const void*)dia_const_kernel<R, 7, X, MT>;
    case 9: return (const void*)dia_const_kernel<R, 9, X, MT>;
    case 27: return (const void*)dia_const_kernel<R, 27, X, MT>;
    default: return (const void*)dia_const_kernel<R, 0, X, MT>;
  }
}
template <int R, int X>
static const void* dia_const_pick_mt(int mask_elem, int nd, int block) {
  return mask_elem == 1 ? dia_const_pick_nd<R, X, unsigned char>(nd, block)
       : mask_elem == 2 ? dia_const_pick_nd<R, X, unsigned short>(nd, block) : dia_const_pick_nd<R, X, unsigned>(nd, block);
}
static const void* dia_const_pick(int R, int X, int mask_elem, int nd, int block = 512) {
#define P(r, xx) if (R == r && X == xx) return dia_const_pick_mt<r, xx>(mask_elem, nd, block);
  P(1, 0) P(2, 0) P(4, 0) P(1, 1) P(2, 1) P(4, 1)
#undef P
  return nullptr;
}
bool dia_const_supported(const Variant& v) {      // exact grid only (no g key): one trip per thread
  return v.block >= 32 && v.block <= 512 && v.block % 32 == 0 && v.grid == 0 && dia_c_ok(v.C) &&
         dia_const_pick(v.R, v.X, 4, 0) != nullptr;
}
static void dia_const_call(KernelCall& c, int R, const Variant& v, int64_t rows, int64_t cols, const DiaFormat& f) {
  c = KernelCall();
  c.fn = dia_const_pick(R, v.X, f.mask_small ? f.mask_elem : 4, f.nd, v.block);
  if (R == 2 && v.block <= 256 && dia_tri_ok(f)) {     // (o - 1, o, o + 1) runs: the neighbours come out of the centre pair
    const int me = f.mask_small ? f.mask_elem : 4;
    const void* t = v.X == 0 ? (me == 1 ? dia_const_pick_tri<0, unsigned char>(f.nd) : me == 2 ? dia_const_pick_tri<0, unsigned short>(f.nd) : dia_const_pick_tri<0, unsigned>(f.nd))
                             : (me == 1 ? dia_const_pick_tri<1, unsigned char>(f.nd) : me == 2 ? dia_const_pick_tri<1, unsigned short>(f.nd) : dia_const_pick_tri<1, unsigned>(f.nd));
    if (t) c.fn = t;
  }
  c.block = v.block;
  const int64_t threads = (rows + R - 1) / R;
  c.grid = (unsigned)((threads + v.block - 1) / v.block);
  c.pdl = true;
  DiaCoefs co;
  for (int i = 0; i < 32; ++i) co.c[i] = f.coef[i];
  c.add((int)rows); c.add((int)0); c.add((int)cols - 1); c.add(f.nd); c.add(dia_offsets(f)); c.add(co);
  c.add(f.mask_small ? (const void*)f.mask_small : (const void*)f.mask);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
  c.per_block = (int64_t)v.block * R;
}
cudaError_t dia_const_dot_plan(const Variant& v, int64_t rows, int64_t cols, const DiaFormat& f, double* part,
                               int* n_part, LaunchPlan* out) {
  if (!f.is_const || rows != cols || rows == 0) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  KernelCall& c = out->k[0];
  const int me = f.mask_small ? f.mask_elem : 4;
  c.fn = me == 1 ? dia_const_dot_pick_nd<unsigned char>(f.nd)
       : me == 2 ? dia_const_dot_pick_nd<unsigned short>(f.nd) : dia_const_dot_pick_nd<unsigned>(f.nd);
  c.block = v.block;
  c.grid = (unsigned)((rows + v.block - 1) / v.block);
  c.pdl = true;
  DiaCoefs co;
  for (int i = 0; i < 32; ++i) co.c[i] = f.coef[i];
  c.add((int)rows); c.add((int)0); c.add((int)cols - 1); c.add(f.nd); c.add(dia_offsets(f)); c.add(co);
  c.add(f.mask_small ? (const void*)f.mask_small : (const void*)f.mask);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
  c.add(part);
  *n_part = (int)c.grid;
  out->n = 1;
  return cudaSuccess;
}

cudaError_t dia_const_plan(const Variant& v, int64_t rows, int64_t cols, const DiaFormat& f, LaunchPlan* out) {
  if (!f.is_const || !dia_const_pick(v.R, v.X, 4, 0)) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (rows == 0) return cudaSuccess;
  // 16-byte pair accesses need an even column count (a pair is then never half inside [0, cols)) and aligned
  // vectors: the one-row-per-thread instantiation is the alternative taken per apply when x or y is not
  const int R = (cols % 2 == 0 && rows % v.R == 0) ? v.R : 1;
  dia_const_call(out->k[0], R, v, rows, cols, f);
  if (R > 1) { dia_const_call(out->alt, 1, v, rows, cols, f); out->has_alt = true; }
  out->n = 1;
  out->range_kind = RANGE_DIA_CONST;
  out->range_align = f.C;
  out->range_elem = f.mask_small ? f.mask_elem : 4;
  return cudaSuccess;
}

// ------------------------------------------------------------------ DIA with the value stream on the TMA engine
// Same producer/consumer ring as kernels_sell_tma.cu: the values of J diagonals of one slice are ONE
// contiguous run (slice-major layout), so a stage is a single cp.async.bulk.  The x addresses do not
// depend on loaded data (row + offset), so the consumers issue their x loads BEFORE waiting for the stage.
// blockDim.x = C/R consumer threads + 32 (the last warp is the producer warp).
// With the first stage of a slice the producer also brings the slice's mask words and (beta != 0, Y_BULK)
// its old y values, so a consumer never waits on a dependent global load: the x loads are issued
// unpredicated (index clamped into [0, cols), never multiplied when the mask bit is off -- reading A7)
// before the stage wait, everything else arrives through the ring.
template <int R, int STAGES, int J, int X>
__global__ void __launch_bounds__(512 + 32)
dia_tma_kernel(int64_t rows, int64_t xlo, int64_t xhi, int64_t nslices, int C, int nd, DiaOffsets offs,
               const double* __restrict__ dval, const unsigned* __restrict__ mask, double alpha,
               const double* __restrict__ x, double beta, double* __restrict__ y, int y_bulk) {
  extern __shared__ __align__(128) unsigned char dia_smem[];
  const int nconsumers = C / R;
  double* s_val = reinterpret_cast<double*>(dia_smem);                                  // [STAGES][J*C]
  double* s_y = s_val + (size_t)STAGES * J * C;                                         // [STAGES][C]
  unsigned* s_mask = reinterpret_cast<unsigned*>(s_y + (size_t)STAGES * C);             // [STAGES][C]
  uint64_t* full = reinterpret_cast<uint64_t*>(s_mask + (size_t)STAGES * C);
  uint64_t* empty = full + STAGES;
  const int tid = threadIdx.x;
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

  if (tid >= nconsumers) {
    if (tid == nconsumers) {      // one elected lane streams the slices
      uint32_t stage = 0, phase = 0;
      for (int64_t s = blockIdx.x; s < nslices; s += gridDim.x) {
        const double* src = dval + s * nd * C;
        const bool ybulk = want_y && (s + 1) * C <= rows;
        for (int d0 = 0; d0 < nd; d0 += J) {
          const int nj = min(J, nd - d0);
          tma::bar_wait(&empty[stage], phase ^ 1);
          // generic-proxy reads of the previous occupant are ordered before this async-proxy refill
          tma::fence_proxy_async();
          const uint32_t vb = (uint32_t)nj * C * sizeof(double);
          const uint32_t mb = d0 == 0 ? (uint32_t)C * sizeof(unsigned) : 0u;
          const uint32_t yb = (d0 == 0 && ybulk) ? (uint32_t)C * sizeof(double) : 0u;
          tma::bar_expect_tx(&full[stage], vb + mb + yb);
          tma::bulk_g2s(s_val + (size_t)stage * J * C, src + (int64_t)d0 * C, vb, &full[stage]);
          if (mb) tma::bulk_g2s(s_mask + (size_t)stage * C, mask + s * C, mb, &full[stage]);
          if (yb) tma::bulk_g2s(s_y + (size_t)stage * C, y + s * C, yb, &full[stage]);
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
    return;
  }

  uint32_t stage = 0, phase = 0;
  const int lane = tid & 31;
  const int xmin = (int)xlo, xmax = (int)xhi;      // valid x indices relative to the x pointer given
  for (int64_t s = blockIdx.x; s < nslices; s += gridDim.x) {
    const int64_t r0 = s * C + (int64_t)tid * R;
    const bool ybulk = want_y && (s + 1) * C <= rows;
    unsigned m[R];
    double acc[R], yold[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { acc[r] = 0.0; yold[r] = 0.0; m[r] = 0u; }
    if (beta != 0.0 && !ybulk) {
#pragma unroll
      for (int r = 0; r < R; ++r) yold[r] = r0 + r < rows ? y[r0 + r] : 0.0;
    }
    for (int d0 = 0; d0 < nd; d0 += J) {
      double xv[J][R];
#pragma unroll
      for (int j = 0; j < J; ++j) {
        const int o = offs.off[min(d0 + j, nd - 1)];
#pragma unroll
        for (int r = 0; r < R; ++r) xv[j][r] = ldx<X>(x, min(max((int)(r0 + r) + o, xmin), xmax));
      }
      tma::bar_wait(&full[stage], phase);
      if (d0 == 0) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
          m[r] = s_mask[(size_t)stage * C + tid * R + r];
          if (ybulk) yold[r] = s_y[(size_t)stage * C + tid * R + r];
        }
      }
      const double* pv = s_val + (size_t)stage * J * C + tid * R;
      double v[J][R];
#pragma unroll
      for (int j = 0; j < J; ++j) {
        if (R == 2) {
          const double2 a = *reinterpret_cast<const double2*>(pv + j * C);
          v[j][0] = a.x; v[j][R - 1] = a.y;
        } else {
          v[j][0] = pv[j * C];
        }
      }
      // the stage is in registers: hand it back before the FMAs
      asm volatile("fence.acq_rel.cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) tma::bar_arrive(&empty[stage]);
#pragma unroll
      for (int j = 0; j < J; ++j) {
        const int d = d0 + j;
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const bool on = d < nd && ((m[r] >> d) & 1u);     // absent entries / stale shared memory: never multiplied
          acc[r] = on ? fma(v[j][r], xv[j][r], acc[r]) : acc[r];
        }
      }
      if (++stage == STAGES) { stage = 0; phase ^= 1; }
    }
#pragma unroll
    for (int r = 0; r < R; ++r)
      if (r0 + r < rows) y[r0 + r] = (beta == 0.0) ? alpha * acc[r] : fma(alpha, acc[r], beta * yold[r]);
  }
}

typedef void (*dia_tma_kernel_t)(int64_t, int64_t, int64_t, int64_t, int, int, DiaOffsets, const double*, const unsigned*, double,
                                 const double*, double, double*, int);
struct DiaTmaEntry { int R, STAGES, J; dia_tma_kernel_t k; };
#define DE(r, st, j) {r, st, j, dia_tma_kernel<r, st, j, 0>}
#define DE_J(j) DE(1, 2, j), DE(1, 3, j), DE(1, 4, j), DE(2, 2, j), DE(2, 3, j), DE(2, 4, j)
static const DiaTmaEntry g_dia_tma[] = {DE_J(4), DE_J(7), DE_J(8), DE_J(9), DE_J(14)};
#undef DE_J
#undef DE

static const DiaTmaEntry* dia_tma_pick(const Variant& v) {
  if (v.X != 0) return nullptr;
  for (const auto& e : g_dia_tma)
    if (e.R == v.R && e.STAGES == v.I && e.J == v.U) return &e;
  return nullptr;
}
static size_t dia_tma_smem(const Variant& v) { return (size_t)v.I * (v.U + 1) * v.C * 8 + (size_t)v.I * v.C * 4 + 2 * v.I * 8 + 128; }

bool dia_tma_supported(const Variant& v) {
  if (!dia_tma_pick(v) || !dia_c_ok(v.C)) return false;
  const int consumers = v.C / v.R;
  if (consumers < 32 || consumers > 512 || v.block != consumers + 32) return false;
  return dia_tma_smem(v) <= 200 * 1024;
}
cudaError_t dia_tma_plan(const Variant& v, int64_t rows, int64_t cols, const DiaFormat& f, int sm_count,
                         LaunchPlan* out) {
  const DiaTmaEntry* e = dia_tma_pick(v);
  if (!e || f.C != v.C) return cudaErrorInvalidValue;
  *out = LaunchPlan();
  if (rows == 0) return cudaSuccess;
  KernelCall& c = out->k[0];
  c.fn = (const void*)e->k;
  c.block = v.block;
  c.smem = (unsigned)dia_tma_smem(v);
  cudaError_t err = allow_smem(c.fn, c.smem);
  if (err != cudaSuccess) return err;
  const int64_t nslices = f.ld / f.C;
  err = resolve_grid(v.grid > 0 ? v.grid : 1, c.fn, v.block, c.smem, sm_count, nslices, &c.grid);   // persistent
  if (err != cudaSuccess) return err;
  c.add(rows); c.add((int64_t)0); c.add(cols - 1); c.add(nslices); c.add(f.C); c.add(f.nd); c.add(dia_offsets(f));
  c.add((const double*)f.val); c.add((const unsigned*)f.mask);
  c.add_alpha(); c.add_x(); c.add_beta(); c.add_y();
  c.add_flag(1);                 // y_bulk: cp.async.bulk needs 16-byte aligned global addresses
  c.per_block = f.C;             // one slice per CTA trip; the grid is capped at the persistent size
  out->n = 1;
  out->range_kind = RANGE_DIA_TMA;
  out->range_align = f.C;
  out->range_elem = f.nd;
  return cudaSuccess;
}

// ------------------------------------------------------------------ converter
// pass 1: flag every occupied diagonal (benign write race: all writers store 1)
__global__ void dia_flag_kernel(int64_t rows, const int* __restrict__ rp, const int* __restrict__ ci,
                                unsigned char* __restrict__ flags) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= rows) return;
  for (int k = rp[r]; k < rp[r + 1]; ++k) flags[(int64_t)ci[k] - r + rows] = 1;
}
// pass 2: collect up to 64 flagged diagonals (unordered; sorted on the host)
__global__ void dia_collect_kernel(int64_t n, int64_t rows, const unsigned char* __restrict__ flags,
                                   int* __restrict__ count, int* __restrict__ list) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n || !flags[i]) return;
  const int pos = atomicAdd(count, 1);
  if (pos < 64) list[pos] = (int)(i - rows);
}
// pass 3: scatter values diagonal-major and build the masks
__global__ void dia_fill_kernel(int64_t rows, int64_t ld, int C, int nd, DiaOffsets offs, const int* __restrict__ rp,
                                const int* __restrict__ ci, const double* __restrict__ va,
                                double* __restrict__ dval, unsigned* __restrict__ mask) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= ld) return;
  unsigned m = 0;
  if (r < rows) {
    for (int k = rp[r]; k < rp[r + 1]; ++k) {
      const int o = (int)((int64_t)ci[k] - r);
      int lo = 0, hi = nd - 1;
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (offs.off[mid] < o) lo = mid + 1; else hi = mid;
      }
      dval[((r / C) * nd + lo) * C + r % C] = va[k];     // slice-major: (slice, diagonal, row in slice)
      m |= 1u << lo;
    }
  }
  mask[r] = m;
}

// constant-coefficient detection: the first thread to reach a diagonal stores its value as the
// reference (ref[32+d]); then every stored value is compared with the reference bit for bit
__global__ void dia_ref_first_kernel(int64_t rows, int C, int nd, const double* __restrict__ dval,
                                     const unsigned* __restrict__ mask, unsigned long long* __restrict__ ref,
                                     unsigned* __restrict__ seen) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= rows) return;
  const unsigned m = mask[r];
  for (int d = 0; d < nd; ++d)
    if (((m >> d) & 1u) && *(volatile unsigned*)&seen[d] == 0u && atomicCAS(&seen[d], 0u, 1u) == 0u)   // plain test first: no atomic storm
      ref[32 + d] = (unsigned long long)__double_as_longlong(dval[((r / C) * nd + d) * C + r % C]);
}
__global__ void dia_cmp_kernel(int64_t rows, int C, int nd, const double* __restrict__ dval,
                               const unsigned* __restrict__ mask, const unsigned long long* __restrict__ ref,
                               unsigned* __restrict__ mismatch) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= rows) return;
  const unsigned m = mask[r];
  bool bad = false;
  for (int d = 0; d < nd; ++d)
    if ((m >> d) & 1u)
      bad |= (unsigned long long)__double_as_longlong(dval[((r / C) * nd + d) * C + r % C]) != ref[32 + d];
  if (bad) atomicAdd(mismatch, 1u);
}

// narrow copy of the mask words for dia_const (1 byte per row when nd <= 8, 2 when nd <= 16)
template <typename MT>
__global__ void dia_mask_narrow_kernel(int64_t ld, const unsigned* __restrict__ mask, MT* __restrict__ out) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r < ld) out[r] = (MT)mask[r];
}

void free_dia(DiaFormat& f, Allocator& al) {
  if (f.mask_small) al.free(f.mask_small, (size_t)f.mask_elem * std::max<int64_t>(f.ld, 1));
  if (f.val) al.free(f.val, sizeof(double) * std::max<int64_t>((int64_t)f.nd * f.ld, 1));
  if (f.mask) al.free(f.mask, sizeof(unsigned) * std::max<int64_t>(f.ld, 1));
  f = DiaFormat();
}

// UNSUPPORTED when the pattern has more than 32 diagonals or is less than half full.
spmv_status_t build_dia(const CsrView& A, int C, Allocator& al, cudaStream_t s, DiaFormat* out) {
  if (!dia_c_ok(C)) return SPMV_ERR_UNSUPPORTED;
  if (A.rows == 0 || A.nnz == 0 || A.rows + A.cols > 0x7ffffff0ll) return SPMV_ERR_UNSUPPORTED;
  DiaFormat f;
  const int64_t nflag = A.rows + A.cols + 1;
  unsigned char* flags = (unsigned char*)al.alloc(nflag, s);
  int* d_cnt = (int*)al.alloc(sizeof(int) * 65, s);
  if (!flags || !d_cnt) {
    if (flags) al.free(flags, nflag);
    if (d_cnt) al.free(d_cnt, sizeof(int) * 65);
    return SPMV_ERR_ALLOC;
  }
  auto drop_tmp = [&]() { al.free(flags, nflag); al.free(d_cnt, sizeof(int) * 65); };
  int h_cnt[65];
  cudaError_t e = cudaMemsetAsync(flags, 0, nflag, s);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_cnt, 0, sizeof(int) * 65, s);
  if (e == cudaSuccess) {
    dia_flag_kernel<<<(unsigned)((A.rows + 255) / 256), 256, 0, s>>>(A.rows, A.row_ptr, A.col_idx, flags);
    dia_collect_kernel<<<(unsigned)((nflag + 255) / 256), 256, 0, s>>>(nflag, A.rows, flags, d_cnt, d_cnt + 1);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(h_cnt, d_cnt, sizeof(int) * 65, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  drop_tmp();
  if (e != cudaSuccess) { set_last_error("build_dia: %s", cudaGetErrorString(e)); return SPMV_ERR_CUDA; }
  const int nd = h_cnt[0];
  if (nd < 1 || nd > 32) { set_last_error("DIA: %d diagonals (limit 32)", nd); return SPMV_ERR_UNSUPPORTED; }
  if ((double)A.nnz < 0.5 * (double)nd * (double)A.rows) {
    set_last_error("DIA: fill %.3f below 0.5", (double)A.nnz / ((double)nd * (double)A.rows));
    return SPMV_ERR_UNSUPPORTED;
  }
  std::sort(h_cnt + 1, h_cnt + 1 + nd);
  f.nd = nd;
  for (int i = 0; i < 32; ++i) f.off[i] = h_cnt[1 + std::min(i, nd - 1)];
  f.C = C;
  f.logC = C == 128 ? 7 : C == 256 ? 8 : 9;
  f.ld = ((A.rows + C - 1) / C) * C;
  dia_compute_windows(f);
  struct Guard { DiaFormat& f; Allocator& al; bool keep; ~Guard() { if (!keep) free_dia(f, al); } } guard{f, al, false};
  f.val = (double*)al.alloc(sizeof(double) * nd * f.ld, s);
  f.mask = (unsigned*)al.alloc(sizeof(unsigned) * f.ld, s);
  if (!f.val || !f.mask) return SPMV_ERR_ALLOC;
  SPMV_CUDA_TRY(cudaMemsetAsync(f.val, 0, sizeof(double) * nd * f.ld, s));
  DiaOffsets o;
  for (int i = 0; i < 32; ++i) o.off[i] = f.off[i];
  dia_fill_kernel<<<(unsigned)((f.ld + 255) / 256), 256, 0, s>>>(A.rows, f.ld, C, nd, o, A.row_ptr, A.col_idx, A.val,
                                                             f.val, f.mask);
  SPMV_CUDA_TRY(cudaGetLastError());
  // constant-coefficient detection
  {
    const size_t wbytes = sizeof(unsigned long long) * 64 + sizeof(unsigned) * 40;
    unsigned long long* d_ref = (unsigned long long*)al.alloc(wbytes, s);
    if (!d_ref) return SPMV_ERR_ALLOC;
    unsigned* d_seen = (unsigned*)(d_ref + 64);
    unsigned* d_mis = d_seen + 32;
    cudaError_t e2 = cudaMemsetAsync(d_ref, 0, wbytes, s);
    const unsigned g = (unsigned)((A.rows + 255) / 256);
    if (e2 == cudaSuccess) {
      dia_ref_first_kernel<<<g, 256, 0, s>>>(A.rows, C, nd, f.val, f.mask, d_ref, d_seen);
      dia_cmp_kernel<<<g, 256, 0, s>>>(A.rows, C, nd, f.val, f.mask, d_ref, d_mis);
      e2 = cudaGetLastError();
    }
    unsigned long long h_ref[64];
    unsigned h_mis = 1;
    if (e2 == cudaSuccess) e2 = cudaMemcpyAsync(h_ref, d_ref, sizeof(h_ref), cudaMemcpyDeviceToHost, s);
    if (e2 == cudaSuccess) e2 = cudaMemcpyAsync(&h_mis, d_mis, sizeof(unsigned), cudaMemcpyDeviceToHost, s);
    if (e2 == cudaSuccess) e2 = cudaStreamSynchronize(s);
    al.free(d_ref, wbytes);
    if (e2 != cudaSuccess) { set_last_error("build_dia: %s", cudaGetErrorString(e2)); return SPMV_ERR_CUDA; }
    f.is_const = h_mis == 0;
    for (int d = 0; d < 32; ++d) {
      const unsigned long long bits = h_ref[32 + std::min(d, nd - 1)];
      memcpy(&f.coef[d], &bits, sizeof(double));
    }
    if (f.is_const && nd <= 16) {
      f.mask_elem = nd <= 8 ? 1 : 2;
      f.mask_small = al.alloc((size_t)f.mask_elem * f.ld, s);
      if (!f.mask_small) return SPMV_ERR_ALLOC;
      const unsigned gm = (unsigned)((f.ld + 255) / 256);
      if (f.mask_elem == 1) dia_mask_narrow_kernel<unsigned char><<<gm, 256, 0, s>>>(f.ld, f.mask, (unsigned char*)f.mask_small);
      else dia_mask_narrow_kernel<unsigned short><<<gm, 256, 0, s>>>(f.ld, f.mask, (unsigned short*)f.mask_small);
      cudaError_t e3 = cudaGetLastError();
      if (e3 != cudaSuccess) { set_last_error("build_dia: %s", cudaGetErrorString(e3)); return SPMV_ERR_CUDA; }
    }
  }
  SPMV_CUDA_TRY(cudaStreamSynchronize(s));
  guard.keep = true;
  *out = f;
  return SPMV_OK;
}

}  // namespace spmv
