// Variant descriptors, eligibility, format management and launch dispatch.
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "handle.h"

namespace spmv {

// ------------------------------------------------------------------ error text
static thread_local char g_err[512] = "";
void set_last_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
const char* last_error_text() { return g_err; }

// ------------------------------------------------------------------ allocator
void* Allocator::alloc(size_t bytes, cudaStream_t s) {
  if (bytes == 0) bytes = 8;
  void* p = nullptr;
  if (has_cb) {
    p = cb.alloc(bytes, (void*)s, cb.ctx);
  } else if (cudaMalloc(&p, bytes) != cudaSuccess) {
    cudaGetLastError();
    p = nullptr;
  }
  if (p) owned += (int64_t)bytes;
  else set_last_error("device allocation of %zu bytes failed", bytes);
  return p;
}
void Allocator::free(void* p, size_t bytes) {
  if (!p) return;
  if (bytes == 0) bytes = 8;
  if (has_cb) cb.free(p, cb.ctx);
  else cudaFree(p);
  owned -= (int64_t)bytes;
}

// ------------------------------------------------------------------ descriptors
static const char* kFamName[FAM_COUNT] = {"csr_scalar", "csr_vector", "sell", "ell", "merge", "bcsr3", "sell_tma", "dia", "dia_tma", "dia_const", "dia_win", "dia_cwin", "sell16", "sell16_tma"};

Variant default_variant() { return Variant(); }   // csr_scalar:b256:r1:u1:x0 (reading A17)

std::string variant_to_string(const Variant& v) {
  char buf[160];
  int n = snprintf(buf, sizeof(buf), "%s:b%d", kFamName[v.fam], v.block);
  auto add = [&](const char* k, int val) { n += snprintf(buf + n, sizeof(buf) - n, ":%s%d", k, val); };
  switch (v.fam) {
    case FAM_CSR_SCALAR: add("r", v.R); add("u", v.U); break;
    case FAM_CSR_VECTOR: add("w", v.W); add("u", v.U); break;
    case FAM_SELL16:
    case FAM_SELL: add("c", v.C); add("s", v.S); if (v.L > 0) add("l", v.L); add("r", v.R); add("u", v.U); break;
    case FAM_ELL: add("r", v.R); add("u", v.U); break;
    case FAM_MERGE: add("i", v.I); break;
    case FAM_BCSR3: add("w", v.W); add("u", v.U); if (v.I == 16) add("i", 16); break;
    case FAM_DIA: add("c", v.C); add("r", v.R); add("u", v.U); break;
    case FAM_DIA_TMA: add("c", v.C); add("r", v.R); add("u", v.U); add("i", v.I); break;
    case FAM_DIA_CONST: add("r", v.R); break;
    case FAM_DIA_WIN:
    case FAM_DIA_CWIN: add("c", v.C); add("r", v.R); add("i", v.I); break;
    case FAM_SELL16_TMA:
    case FAM_SELL_TMA: add("c", v.C); add("s", v.S); if (v.L > 0) add("l", v.L); add("r", v.R); add("u", v.U); add("i", v.I); break;
  }
  add("x", v.X);
  if (v.X == 2 || (v.X == 3 && (v.fam == FAM_SELL_TMA || v.fam == FAM_SELL16_TMA))) add("h", v.H);
  if (v.grid > 0) add("g", v.grid);
  if (v.carve >= 0) add("co", v.carve);
  return std::string(buf);
}

bool variant_from_string(const char* s, Variant* out) {
  if (!s) return false;
  Variant v;
  if (!strcmp(s, "default")) { *out = v; return true; }
  char tmp[160];
  strncpy(tmp, s, sizeof(tmp) - 1);
  tmp[sizeof(tmp) - 1] = 0;
  char* save = nullptr;
  char* tok = strtok_r(tmp, ":", &save);
  if (!tok) return false;
  int fam = -1;
  for (int f = 0; f < FAM_COUNT; ++f)
    if (!strcmp(tok, kFamName[f])) fam = f;
  if (fam < 0) return false;
  v.fam = fam;
  if (fam == FAM_MERGE) v.I = 7;
  if (fam == FAM_SELL || fam == FAM_SELL16) { v.C = 128; v.S = 1; }
  if (fam == FAM_SELL_TMA || fam == FAM_SELL16_TMA) { v.C = 256; v.S = 1; v.U = 8; v.I = 3; v.block = 288; }
  if (fam == FAM_CSR_VECTOR || fam == FAM_BCSR3) v.W = 8;
  if (fam == FAM_DIA || fam == FAM_DIA_CONST) v.C = 128;
  if (fam == FAM_DIA_TMA) { v.C = 256; v.U = 8; v.I = 3; v.block = 288; }
  if (fam == FAM_DIA_WIN || fam == FAM_DIA_CWIN) { v.C = 256; v.I = 2; v.block = 288; }
  while ((tok = strtok_r(nullptr, ":", &save))) {
    char* end = nullptr;
    if (!strncmp(tok, "co", 2)) { v.carve = (int)strtol(tok + 2, &end, 10); }
    else {
      const int val = (int)strtol(tok + 1, &end, 10);
      switch (tok[0]) {
        case 'b': v.block = val; break;
        case 'g': v.grid = val; break;
        case 'u': v.U = val; break;
        case 'r': v.R = val; break;
        case 'w': v.W = val; break;
        case 'x': v.X = val; break;
        case 'c': v.C = val; break;
        case 's': v.S = val; break;
        case 'i': v.I = val; break;
        case 'l': v.L = val; break;
        case 'h': v.H = val; break;
        default: return false;
      }
    }
    if (!end || *end != 0) return false;
  }
  if (v.X == 2 && v.H == 0) v.H = 136;
  *out = v;
  return true;
}

static bool template_supported(const Variant& v) {
  switch (v.fam) {
    case FAM_CSR_SCALAR: return csr_scalar_supported(v);
    case FAM_CSR_VECTOR: return csr_vector_supported(v);
    case FAM_SELL:
    case FAM_SELL16:
    case FAM_ELL: return sell_supported(v);
    case FAM_MERGE: return merge_supported(v);
    case FAM_BCSR3: return bcsr_supported(v);
    case FAM_SELL16_TMA:
    case FAM_SELL_TMA: return sell_tma_supported(v);
    case FAM_DIA: return dia_supported(v);
    case FAM_DIA_TMA: return dia_tma_supported(v);
    case FAM_DIA_CONST: return dia_const_supported(v);
    case FAM_DIA_WIN:
    case FAM_DIA_CWIN: return dia_win_supported(v);
  }
  return false;
}

bool variant_eligible(const spmv_handle_s* h, const Variant& v, std::string* why) {
  auto no = [&](const char* m) { if (why) *why = m; return false; };
  if (v.grid < 0 || v.grid > 64 || v.carve < -1 || v.carve > 100) return no("bad grid/carve-out");
  if (!template_supported(v)) return no("no such template instantiation");
  const spmv_info_t& in = h->info;
  if (v.fam == FAM_ELL) {
    // eligibility rule of SURVEY 8(a) a3: width*rows <= 1.5*nnz
    if ((double)in.max_row_len * (double)in.rows > 1.5 * (double)in.nnz + 1024.0) return no("ELL padding > 1.5x");
  }
  if (v.fam == FAM_BCSR3) {
    if (in.rows % 3 || in.cols % 3 || in.rows == 0) return no("rows/cols not multiples of 3");
    if (!in.cols_sorted) return no("BCSR needs sorted unique columns");
    if (!in.block3_full) return no("3x3 block fill < 1.0 (zero fill would multiply x; reading A7)");
    // i16: |block column - block row| <= (|col - row| + 2) / 3 must stay below 32768
    if (v.I == 16 && (in.bandwidth + 2) / 3 >= 32768) return no("bcsr3 i16: block columns up to 32768 block rows away: 16-bit deltas do not fit");
  }
  if ((v.fam == FAM_DIA_CONST || v.fam == FAM_DIA_CWIN) && h->dia_state == 2)
    return no("coefficients are not constant along the diagonals");
  if (v.fam == FAM_DIA || v.fam == FAM_DIA_TMA || v.fam == FAM_DIA_CONST || v.fam == FAM_DIA_WIN || v.fam == FAM_DIA_CWIN) {
    if (!in.cols_sorted) return no("DIA needs sorted unique columns");
    if (in.max_row_len > 32 || in.nnz == 0) return no("more than 32 entries in a row: more than 32 diagonals");
    if (h->dia_state < 0) return no("pattern is not a set of at most 32 (half-full) diagonals");
  }
  if (is_sell16(v)) {
    // a slice of C rows inside a sorting window of S rows touches columns within bandwidth of its rows
    if (v.L != 0) return no("sell16 has no row splitting");
    if (2 * in.bandwidth + std::max(v.C, v.S) >= 0xFFFF && in.rows > 0)
      return no("column span of a slice can reach 65535: 16-bit deltas do not fit");
  }
  if ((v.fam == FAM_SELL_TMA || v.fam == FAM_SELL16_TMA) && v.X == 3) {
    // x3: every gather of a slice comes out of the shared-memory window, with no fallback path in the kernel
    if (v.S != 1 || v.L != 0) return no("x3 needs the rows of a slice in natural order (s1, no splitting)");
    if (v.H < in.bandwidth) return no("x3 needs a window half-width h >= the matrix bandwidth");
    if ((in.cols & 1) || (v.H & 1) || (v.C & 1)) return no("x3 needs an even column count, h and c (16-byte aligned windows)");
  }
  if (v.L != 0) {
    if (v.fam != FAM_SELL && v.fam != FAM_SELL_TMA) return no("row splitting is a SELL option");
    if (v.L < 4 || v.L > 65536) return no("split length out of range");
    if (v.S <= 1) return no("row splitting needs a sorting window (s > 1)");
  }
  if (v.fam == FAM_MERGE) {      // the merge path has rows + nnz items and is indexed with int32
    if (in.rows + in.nnz > 0x7ffffff0ll) return no("rows+nnz over int32");
  }
  return true;
}

// ------------------------------------------------------------------ formats
spmv_status_t ensure_format(spmv_handle_s* h, const Variant& v, cudaStream_t s) {
  switch (v.fam) {
    case FAM_SELL16:
    case FAM_SELL16_TMA:
    case FAM_SELL_TMA:
    case FAM_SELL: {
      auto key = sell_key(v);
      if (h->sells.count(key)) return SPMV_OK;
      SellFormat f;
      spmv_status_t st = build_sell(h->A, v.C, v.S, false, v.L, h->al, s, &f);
      if (st != SPMV_OK) return st;
      if ((double)f.padded > 2.0 * (double)h->A.nnz + 65536.0) {   // too padded to be a candidate
        free_sell(f, h->al);
        set_last_error("SELL c%d s%d: padding over 2x nnz", v.C, v.S);
        return SPMV_ERR_UNSUPPORTED;
      }
      if (is_sell16(v)) {
        st = sell_narrow_indices(f, h->al, s);
        if (st != SPMV_OK) { free_sell(f, h->al); return st; }
      }
      h->sells[key] = f;
      return SPMV_OK;
    }
    case FAM_ELL: {
      if (h->has_ell) return SPMV_OK;
      spmv_status_t st = build_sell(h->A, 0, 1, true, 0, h->al, s, &h->ell);
      if (st == SPMV_OK) h->has_ell = true;
      return st;
    }
    case FAM_BCSR3: {
      if (h->has_bcsr && !h->bcsr.bcol) {          // only the 16-bit indices were kept: rebuild for either form
        cudaDeviceSynchronize();
        free_bcsr3(h->bcsr, h->al);
        h->has_bcsr = false;
        if (h->sel.fam == FAM_BCSR3) reset_to_default(h);   // its plan pointed into the format just freed
      }
      if (!h->has_bcsr) {
        spmv_status_t st = build_bcsr3(h->A, h->al, s, &h->bcsr);
        if (st != SPMV_OK) return st;
        h->has_bcsr = true;
      }
      return v.I == 16 ? bcsr3_narrow_indices(h->bcsr, h->al, s) : SPMV_OK;
    }
    case FAM_DIA_WIN:
    case FAM_DIA_CWIN:
    case FAM_DIA_CONST:
    case FAM_DIA_TMA:
    case FAM_DIA: {
      const bool need_const = v.fam == FAM_DIA_CONST || v.fam == FAM_DIA_CWIN;
      const bool is_win = v.fam == FAM_DIA_WIN || v.fam == FAM_DIA_CWIN;
      if (h->dias.count(v.C)) {
        if (need_const && !h->dias[v.C].is_const) return SPMV_ERR_UNSUPPORTED;
        if (is_win && !dia_win_fits(v, h->dias[v.C])) { set_last_error("dia_win: a slice does not fit in shared memory"); return SPMV_ERR_UNSUPPORTED; }
        return SPMV_OK;
      }
      if (h->dia_state < 0) return SPMV_ERR_UNSUPPORTED;
      DiaFormat f;
      spmv_status_t st = build_dia(h->A, v.C, h->al, s, &f);
      if (st == SPMV_OK) {
        h->dias[v.C] = f;
        h->dia_state = f.is_const ? 1 : 2;       // 2: diagonal pattern, but values vary along the diagonals
        if (need_const && !f.is_const) return SPMV_ERR_UNSUPPORTED;
        if (is_win && !dia_win_fits(v, f)) { set_last_error("dia_win: a slice does not fit in shared memory"); return SPMV_ERR_UNSUPPORTED; }
      }
      else if (st == SPMV_ERR_UNSUPPORTED) h->dia_state = -1;
      return st;
    }
    case FAM_MERGE: {
      const int ti = v.block * v.I;
      if (h->plans.count(ti)) return SPMV_OK;
      MergePlan p;
      spmv_status_t st = build_merge_plan(h->A, ti, h->al, s, &p);
      if (st != SPMV_OK) return st;
      SPMV_CUDA_TRY(cudaStreamSynchronize(s));
      h->plans[ti] = p;
      return SPMV_OK;
    }
    default: return SPMV_OK;
  }
}

void release_formats_except(spmv_handle_s* h, const Variant& keep) {
  // An apply launched on ANY stream may still be reading a format that is about to be freed (and a
  // stream-ordered allocator behind the callbacks would recycle the memory at once): wait for the device
  // before the first free.  Slow path only (select / tune / update_values / destroy).
  const bool keeps_sell = is_sell_family(keep);
  const bool keeps_dia = keep.fam == FAM_DIA || keep.fam == FAM_DIA_TMA || keep.fam == FAM_DIA_CONST ||
                         keep.fam == FAM_DIA_WIN || keep.fam == FAM_DIA_CWIN;
  size_t n_free = (h->has_ell && keep.fam != FAM_ELL) + (h->has_bcsr && (keep.fam != FAM_BCSR3 || h->bcsr.bcol16));
  for (const auto& kv : h->sells) n_free += !(keeps_sell && kv.first == sell_key(keep));
  for (const auto& kv : h->dias) n_free += !(keeps_dia && kv.first == keep.C);
  for (const auto& kv : h->plans) n_free += !(keep.fam == FAM_MERGE && kv.first == keep.block * keep.I);
  if (n_free) cudaDeviceSynchronize();
  for (auto it = h->sells.begin(); it != h->sells.end();) {
    if (keeps_sell && it->first == sell_key(keep)) { ++it; continue; }
    free_sell(it->second, h->al);
    it = h->sells.erase(it);
  }
  if (h->has_ell && keep.fam != FAM_ELL) { free_sell(h->ell, h->al); h->has_ell = false; }
  if (h->has_bcsr && keep.fam != FAM_BCSR3) { free_bcsr3(h->bcsr, h->al); h->has_bcsr = false; }
  else if (h->has_bcsr) bcsr3_drop_indices(h->bcsr, h->al, keep.I != 16);        // the index array the kept variant does not read
  for (auto it = h->dias.begin(); it != h->dias.end();) {
    if ((keep.fam == FAM_DIA || keep.fam == FAM_DIA_TMA || keep.fam == FAM_DIA_CONST || keep.fam == FAM_DIA_WIN ||
         keep.fam == FAM_DIA_CWIN) && it->first == keep.C) { ++it; continue; }
    free_dia(it->second, h->al);
    it = h->dias.erase(it);
  }
  for (auto it = h->plans.begin(); it != h->plans.end();) {
    if (keep.fam == FAM_MERGE && it->first == keep.block * keep.I) { ++it; continue; }
    free_merge_plan(it->second, h->al);
    it = h->plans.erase(it);
  }
}

void release_all_formats(spmv_handle_s* h) {
  Variant none;   // csr_scalar keeps nothing
  release_formats_except(h, none);
}

int64_t variant_format_bytes(const spmv_handle_s* h, const Variant& v) {
  const CsrView& A = h->A;
  const int64_t csr = A.nnz * 12 + (A.rows + 1) * 4;
  switch (v.fam) {
    case FAM_SELL16:
    case FAM_SELL16_TMA:
    case FAM_SELL_TMA:
    case FAM_SELL: {
      auto it = h->sells.find(sell_key(v));
      if (it == h->sells.end()) return 0;
      const SellFormat& f = it->second;
      return f.padded * (f.col16 ? 10 : 12) + (f.nslices + 1) * 8 + (f.col16 ? f.nslices * 4 : 0) +
             (f.perm ? f.nslices * (int64_t)f.C * 4 : 0) + f.nparts * 16 + f.nsplit * 8;
    }
    case FAM_ELL: return h->has_ell ? h->ell.padded * 12 + 16 : 0;
    case FAM_BCSR3: return h->has_bcsr ? h->bcsr.nblocks * (v.I == 16 ? 74 : 76) + (h->bcsr.brows + 1) * 4 : 0;
    case FAM_DIA_CWIN:
    case FAM_DIA_CONST: {
      auto it = h->dias.find(v.C);
      if (it == h->dias.end()) return 0;                 // the mask words are all that is read of the matrix
      return A.rows * (v.fam == FAM_DIA_CONST && it->second.mask_small ? it->second.mask_elem : 4);
    }
    case FAM_DIA_WIN:
    case FAM_DIA_TMA:
    case FAM_DIA: {
      auto it = h->dias.find(v.C);
      return it == h->dias.end() ? 0 : (int64_t)it->second.nd * it->second.ld * 8 + it->second.ld * 4;
    }
    case FAM_MERGE: {
      auto it = h->plans.find(v.block * v.I);
      return csr + (it == h->plans.end() ? 0 : it->second.ntiles * 16 + 4);
    }
    default: return csr;
  }
}

// ------------------------------------------------------------------ launch plans
cudaError_t resolve_grid(int g, const void* fn, int block, size_t smem, int sm_count, int64_t exact, unsigned* grid) {
  int64_t n = exact;
  if (g > 0) {
    int occ = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, block, smem);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    n = std::min<int64_t>(exact, (int64_t)g * sm_count * occ);
  }
  if (n < 1) n = 1;
  if (n > 0x7fffffffll) return cudaErrorInvalidConfiguration;
  *grid = (unsigned)n;
  return cudaSuccess;
}

cudaError_t allow_smem(const void* fn, size_t smem) {
  if (smem <= 48 * 1024) return cudaSuccess;
  return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

cudaError_t run_call(const KernelCall& c, const ApplyArgs& a0) {
  ApplyArgs a = a0;
  a.x = a0.x ? a0.x + c.x_off : a0.x;
  a.y = a0.y ? a0.y + c.y_off : a0.y;
  // private copy of the argument block: concurrent applies of one handle never share mutable state
  alignas(16) unsigned char buf[sizeof(c.store)];
  memcpy(buf, c.store, (size_t)c.used);
  if (c.i_alpha >= 0) memcpy(buf + c.off[c.i_alpha], &a.alpha, sizeof(double));
  if (c.i_beta >= 0) memcpy(buf + c.off[c.i_beta], &a.beta, sizeof(double));
  if (c.i_x >= 0) memcpy(buf + c.off[c.i_x], &a.x, sizeof(void*));
  if (c.i_y >= 0) memcpy(buf + c.off[c.i_y], &a.y, sizeof(void*));
  for (int f = 0; f < 2; ++f) {
    if (c.flag_idx[f] < 0) continue;
    if (c.flag_kind[f] == 3) {
      const int64_t v = ((uintptr_t)a.x & 15) == 0 ? c.flag_val : 0;
      memcpy(buf + c.off[c.flag_idx[f]], &v, sizeof(v));
    } else {
      const int v = (((uintptr_t)(c.flag_kind[f] == 1 ? (const void*)a.y : (const void*)a.x)) & 15) == 0;
      memcpy(buf + c.off[c.flag_idx[f]], &v, sizeof(v));
    }
  }
  void* argp[20];
  for (int i = 0; i < c.nargs; ++i) argp[i] = buf + c.off[i];
  return launch_kernel_pdl(c.fn, c.grid, c.block, c.smem, a.stream, argp, c.pdl);
}

cudaError_t run_plan(const LaunchPlan& p, const ApplyArgs& a) {
  if (p.n == 0) return cudaSuccess;
  const bool aligned = p.has_alt ? ((((uintptr_t)a.x | (uintptr_t)a.y) & 15) == 0) : true;
  cudaError_t e = run_call(aligned ? p.k[0] : p.alt, a);
  if (e == cudaSuccess && p.n > 1) e = run_call(p.k[1], a);
  return e;
}

// The plan's kernel re-aimed at rows [a, b): counts shrink, the format pointers move to the first row (slice,
// block row) of the range, x / y get element offsets, the grid covers the range.  Argument positions are those
// the families' *_plan functions build (kernels_*.cu).
bool plan_for_rows(const LaunchPlan& p, int64_t rows, int64_t cols, int64_t a, int64_t b, bool aligned, KernelCall* out) {
  if (p.n != 1 || p.range_kind == RANGE_NONE || a < 0 || b > rows || a >= b || a % p.range_align) return false;
  if (b != rows && b % p.range_align) return false;
  KernelCall c = (p.has_alt && !aligned) ? p.alt : p.k[0];
  int64_t units = b - a;
  auto shift = [&](int i, int64_t bytes) {
    const char* ptr = c.get<const char*>(i);
    if (ptr) c.set(i, ptr + bytes);
  };
  switch (p.range_kind) {
    case RANGE_CSR:                      // rows, row_ptr (absolute positions: col_idx / val stay)
      c.set(0, (int)(b - a));
      shift(1, 4 * a);
      c.y_off = a;
      break;
    case RANGE_BCSR:                     // block rows, brow_ptr
      c.set(0, (int)((b - a) / 3));
      shift(1, 4 * (a / 3));
      c.set(8, (int)(a / 3));            // br0: the 16-bit block columns are relative to the block row's own index
      c.y_off = a;
      units = (b - a) / 3;
      break;
    case RANGE_SELL:
    case RANGE_SELL_TMA: {               // slices [s0, s1)
      const int C = p.range_elem;
      const int64_t s0 = a / C, s1 = (b + C - 1) / C;
      const bool tma = p.range_kind == RANGE_SELL_TMA;
      const int i_sp = tma ? 3 : 4, i_sbase = tma ? 6 : 7, i_perm = tma ? 7 : 8;
      const bool perm = c.get<const int*>(i_perm) != nullptr;
      c.set(0, (int64_t)(b - a));                                    // rows of the range (no permutation: row < rows)
      c.set(1, tma ? (int64_t)(s1 - s0) : (int64_t)(s1 - s0) * C);   // slices | padded rows
      shift(i_sp, 8 * s0);
      shift(i_sbase, 4 * s0);
      shift(i_perm, 4 * s0 * C);
      c.y_off = perm ? 0 : a;                                        // perm holds absolute rows
      units = tma ? (s1 - s0) : (s1 - s0) * C;
      break;
    }
    case RANGE_DIA: {                    // rows, ld, dval, mask
      const int C = p.range_align, nd = p.range_elem;
      const int64_t ld = (b - a + C - 1) / C * C;
      c.set(0, (int64_t)(b - a));
      c.set(1, ld);
      shift(6, 8 * (a / C) * nd * C);
      shift(7, 4 * a);
      c.x_off = a; c.y_off = a;
      units = ld;
      break;
    }
    case RANGE_DIA_TMA: {                // rows, xlo, xhi, nslices, dval, mask
      const int C = p.range_align, nd = p.range_elem;
      const int64_t ns = (b - a + C - 1) / C;
      c.set(0, (int64_t)(b - a));
      c.set(1, (int64_t)-a);
      c.set(2, (int64_t)(cols - 1 - a));
      c.set(3, ns);
      shift(7, 8 * (a / C) * nd * C);
      shift(8, 4 * a);
      c.x_off = a; c.y_off = a;
      units = ns * C;
      break;
    }
    case RANGE_DIA_CONST:                // rows, xlo, xhi, mask (range_elem bytes per word)
      c.set(0, (int)(b - a));
      c.set(1, (int)-a);
      c.set(2, (int)(cols - 1 - a));
      shift(6, (int64_t)p.range_elem * a);
      c.x_off = a; c.y_off = a;
      break;
    default: return false;
  }
  const int64_t g = (units + c.per_block - 1) / std::max<int64_t>(c.per_block, 1);
  c.grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(g, c.grid));
  *out = c;
  return true;
}

// Resolves everything a launch of `v` on this handle needs (the format must exist).  The carve-out
// ("size of L1 cache") is a per-function, per-process attribute: it is (re)set here, at select /
// tune time, never on the apply path; two handles that select the SAME kernel with DIFFERENT co values share
// the one set last.
spmv_status_t build_plan(spmv_handle_s* h, const Variant& v, LaunchPlan* out) {
  cudaError_t e = cudaErrorInvalidValue;
  const int sms = h->dev.sm_count;
  switch (v.fam) {
    case FAM_CSR_SCALAR: e = csr_scalar_plan(v, h->A, sms, out); break;
    case FAM_CSR_VECTOR: e = csr_vector_plan(v, h->A, sms, out); break;
    case FAM_SELL:
    case FAM_SELL16:
    case FAM_SELL16_TMA:
    case FAM_SELL_TMA: {
      auto it = h->sells.find(sell_key(v));
      if (it == h->sells.end()) return SPMV_ERR_INTERNAL;
      e = (v.fam == FAM_SELL || v.fam == FAM_SELL16) ? sell_plan(v, h->A.rows, it->second, sms, out)
                            : sell_tma_plan(v, h->A.rows, h->A.cols, it->second, sms, out);
      break;
    }
    case FAM_ELL:
      if (!h->has_ell) return SPMV_ERR_INTERNAL;
      e = sell_plan(v, h->A.rows, h->ell, sms, out);
      break;
    case FAM_MERGE: {
      auto it = h->plans.find(v.block * v.I);
      if (it == h->plans.end()) return SPMV_ERR_INTERNAL;
      e = merge_plan(v, h->A, it->second, out);
      break;
    }
    case FAM_BCSR3:
      if (!h->has_bcsr) return SPMV_ERR_INTERNAL;
      e = bcsr_plan(v, h->bcsr, sms, out);
      break;
    case FAM_DIA:
    case FAM_DIA_TMA:
    case FAM_DIA_CONST:
    case FAM_DIA_WIN:
    case FAM_DIA_CWIN: {
      auto it = h->dias.find(v.C);
      if (it == h->dias.end()) return SPMV_ERR_INTERNAL;
      const DiaFormat& f = it->second;
      e = v.fam == FAM_DIA ? dia_plan(v, h->A.rows, f, sms, out)
        : v.fam == FAM_DIA_TMA ? dia_tma_plan(v, h->A.rows, h->A.cols, f, sms, out)
        : v.fam == FAM_DIA_CONST ? dia_const_plan(v, h->A.rows, h->A.cols, f, out)
                                 : dia_win_plan(v, h->A.rows, h->A.cols, f, sms, out);
      break;
    }
  }
  if (e == cudaSuccess && out->n > 0) {
    e = cudaFuncSetAttribute(out->k[0].fn, cudaFuncAttributePreferredSharedMemoryCarveout, v.carve);
    if (e == cudaSuccess && out->has_alt)
      e = cudaFuncSetAttribute(out->alt.fn, cudaFuncAttributePreferredSharedMemoryCarveout, v.carve);
  }
  if (e != cudaSuccess) {
    cudaGetLastError();
    set_last_error("cannot prepare the launch of %s: %s", variant_to_string(v).c_str(), cudaGetErrorString(e));
    return SPMV_ERR_CUDA;
  }
  return SPMV_OK;
}

spmv_status_t build_dot_plan(spmv_handle_s* h, double* part, int* n_part, LaunchPlan* out) {
  const Variant& v = h->sel;
  if (v.fam != FAM_DIA_CONST || v.X != 0) return SPMV_ERR_UNSUPPORTED;
  auto it = h->dias.find(v.C);
  if (it == h->dias.end()) return SPMV_ERR_UNSUPPORTED;
  cudaError_t e = dia_const_dot_plan(v, h->A.rows, h->A.cols, it->second, part, n_part, out);
  if (e != cudaSuccess) { cudaGetLastError(); return SPMV_ERR_UNSUPPORTED; }
  return SPMV_OK;
}

spmv_status_t launch_plan(const LaunchPlan& p, const ApplyArgs& a) {
  cudaError_t e = run_plan(p, a);
  if (e != cudaSuccess) {
    set_last_error("kernel launch failed: %s", cudaGetErrorString(e));
    return SPMV_ERR_CUDA;
  }
  return SPMV_OK;
}

}  // namespace spmv
