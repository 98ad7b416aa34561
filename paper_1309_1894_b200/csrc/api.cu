// C ABI entry points (include/spmv_b200.h) except spmv_tune / spmv_tune_batch (tuner.cu)
// and spmv_measure_ceiling (verify.cu).
#include <math.h>
#include <stdlib.h>
#include <stdint.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <set>
#include <string>

#include "handle.h"

namespace spmv {
const char* last_error_text();

static std::mutex g_live_mu;
static std::set<void*> g_live;

bool handle_alive(spmv_handle_t h) {
  if (!h) return false;
  std::lock_guard<std::mutex> lk(g_live_mu);
  return g_live.count((void*)h) && h->magic == kHandleMagic;
}

static void refresh_info(spmv_handle_s* h) {
  h->info.tuned = h->tuned ? 1 : 0;
  h->info.format_bytes = variant_format_bytes(h, h->sel);
  h->info.owned_bytes = h->al.owned;
  std::string d = variant_to_string(h->sel);
  strncpy(h->info.variant, d.c_str(), sizeof(h->info.variant) - 1);
}
void handle_refresh_info(spmv_handle_s* h) { refresh_info(h); }

// Does the format the SELECTED variant's launch plan points into still exist?  (The plan holds raw device
// pointers into it; error paths of select / tune / update_values may have released it.)
bool selected_format_alive(const spmv_handle_s* h) {
  const Variant& v = h->sel;
  switch (v.fam) {
    case FAM_CSR_SCALAR: case FAM_CSR_VECTOR: return true;          // caller-owned CSR arrays only
    case FAM_SELL: case FAM_SELL_TMA: case FAM_SELL16: case FAM_SELL16_TMA: return h->sells.count(sell_key(v)) != 0;
    case FAM_ELL: return h->has_ell;
    case FAM_MERGE: return h->plans.count(v.block * v.I) != 0;
    case FAM_BCSR3: return h->has_bcsr && (v.I == 16 ? h->bcsr.bcol16 != nullptr : h->bcsr.bcol != nullptr);
    case FAM_DIA: case FAM_DIA_TMA: case FAM_DIA_CONST: case FAM_DIA_WIN: case FAM_DIA_CWIN: return h->dias.count(v.C) != 0;
    default: return false;
  }
}

// The fixed default variant reads the caller's CSR arrays only, so its plan needs no allocation and can never
// point at freed memory: where a selection's format has been (or may have been) released, the handle goes here.
void reset_to_default(spmv_handle_s* h) {
  const Variant d = default_variant();
  LaunchPlan p;
  if (build_plan(h, d, &p) != SPMV_OK) p = LaunchPlan();
  h->sel = d;
  h->plan = p;
  h->tuned = false;
  h->leaders.clear();
  refresh_info(h);
}
void repair_selection_after_failure(spmv_handle_s* h) {
  if (!selected_format_alive(h)) reset_to_default(h);
}

spmv_status_t adopt_variant(spmv_handle_s* h, const Variant& v, cudaStream_t s) {
  spmv_status_t st = ensure_format(h, v, s);
  if (st != SPMV_OK) { repair_selection_after_failure(h); return st; }
  LaunchPlan p;
  st = build_plan(h, v, &p);
  if (st != SPMV_OK) { repair_selection_after_failure(h); return st; }
  h->sel = v;
  h->plan = p;
  release_formats_except(h, v);
  refresh_info(h);
  return SPMV_OK;
}

}  // namespace spmv

using namespace spmv;

extern "C" {

const char* spmv_status_string(spmv_status_t s) {
  switch (s) {
    case SPMV_OK: return "SPMV_OK";
    case SPMV_ERR_INVALID_ARG: return "SPMV_ERR_INVALID_ARG";
    case SPMV_ERR_INVALID_MATRIX: return "SPMV_ERR_INVALID_MATRIX";
    case SPMV_ERR_UNSUPPORTED: return "SPMV_ERR_UNSUPPORTED";
    case SPMV_ERR_ALLOC: return "SPMV_ERR_ALLOC";
    case SPMV_ERR_CUDA: return "SPMV_ERR_CUDA";
    case SPMV_ERR_VERIFY_FAILED: return "SPMV_ERR_VERIFY_FAILED";
    case SPMV_ERR_INTERNAL: return "SPMV_ERR_INTERNAL";
  }
  return "SPMV_ERR_UNKNOWN";
}
const char* spmv_last_error(void) { return last_error_text(); }
const char* spmv_version(void) { return kVersion; }

spmv_status_t spmv_create(spmv_handle_t* out, int64_t rows, int64_t cols, int64_t nnz, const int32_t* d_row_ptr,
                          const int32_t* d_col_idx, const double* d_val, const spmv_allocator_t* alloc,
                          void* stream) {
  if (!out || rows < 0 || cols < 0 || nnz < 0 || !d_row_ptr) return SPMV_ERR_INVALID_ARG;
  if (nnz > 0 && (!d_col_idx || !d_val)) return SPMV_ERR_INVALID_ARG;
  if (alloc && (!alloc->alloc || !alloc->free)) return SPMV_ERR_INVALID_ARG;
  if (rows > 0x7fffffffll || cols > 0x7fffffffll || nnz > 0x7fffffffll) return SPMV_ERR_UNSUPPORTED;
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0;
  SPMV_CUDA_TRY(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  SPMV_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));

  spmv_handle_s* h = new (std::nothrow) spmv_handle_s();
  if (!h) return SPMV_ERR_ALLOC;
  h->magic = kHandleMagic;
  h->device = dev;
  h->A.rows = rows; h->A.cols = cols; h->A.nnz = nnz;
  h->A.row_ptr = d_row_ptr; h->A.col_idx = d_col_idx; h->A.val = d_val;
  if (alloc) { h->al.cb = *alloc; h->al.has_cb = true; }
  h->dev.sm_count = prop.multiProcessorCount;
  h->dev.l2_bytes = prop.l2CacheSize;
  strncpy(h->dev.name, prop.name, sizeof(h->dev.name) - 1);

  RawStats rs;
  cudaError_t e = compute_stats(h->A, &rs, s);
  if (e != cudaSuccess) {
    set_last_error("spmv_create: statistics pass failed: %s", cudaGetErrorString(e));
    delete h;
    return SPMV_ERR_CUDA;
  }
  if (rs.bad_row_ptr || rs.bad_col) {
    set_last_error("spmv_create: invalid CSR (%llu bad row_ptr entries, %llu columns out of range)",
                   rs.bad_row_ptr, rs.bad_col);
    delete h;
    return SPMV_ERR_INVALID_MATRIX;
  }
  spmv_info_t& in = h->info;
  in.rows = rows; in.cols = cols; in.nnz = nnz;
  in.min_row_len = rows ? rs.min_len : 0;
  in.max_row_len = rs.max_len;
  in.mean_row_len = rows ? (double)rs.sum_len / (double)rows : 0.0;
  in.var_row_len = rows ? (double)rs.sum_len_sq / (double)rows - in.mean_row_len * in.mean_row_len : 0.0;
  if (in.var_row_len < 0) in.var_row_len = 0;
  for (int b = 0; b < 32; ++b) in.len_hist[b] = (int64_t)rs.hist[b];
  in.bandwidth = rs.bandwidth;
  in.cols_sorted = rs.unsorted_rows == 0;
  in.block3_full = (rs.block3_bad == 0 && rows > 0 && rows % 3 == 0 && cols % 3 == 0) ? 1 : 0;
  in.n_blocks3 = in.block3_full ? (int64_t)rs.n_blocks3 : 0;
  in.sig_row_ptr = rs.sig_row_ptr;
  in.sig_col_idx = rs.sig_col_idx;
  in.sm_count = h->dev.sm_count;
  in.l2_bytes = h->dev.l2_bytes;
  strncpy(in.device_name, h->dev.name, sizeof(in.device_name) - 1);
  if (adopt_variant(h, default_variant(), s) != SPMV_OK) { delete h; return SPMV_ERR_CUDA; }
  {
    std::lock_guard<std::mutex> lk(g_live_mu);
    g_live.insert((void*)h);
  }
  *out = h;
  return SPMV_OK;
}

spmv_status_t spmv_destroy(spmv_handle_t h) {
  if (!handle_alive(h)) return SPMV_ERR_INVALID_ARG;
  {
    std::lock_guard<std::mutex> lk(g_live_mu);
    g_live.erase((void*)h);
  }
  cudaDeviceSynchronize();          // no apply may still be using the formats or the staging vectors
  release_all_formats(h);
  if (h->d_x_stage) h->al.free(h->d_x_stage, sizeof(double) * h->A.cols);
  if (h->d_y_stage) h->al.free(h->d_y_stage, sizeof(double) * h->A.rows);
  for (cudaEvent_t e : h->hs_events) cudaEventDestroy(e);
  if (h->ws_event) cudaEventDestroy(h->ws_event);
  if (h->hs_up) { cudaStreamDestroy(h->hs_up); cudaStreamDestroy(h->hs_up2); cudaStreamDestroy(h->hs_run); cudaStreamDestroy(h->hs_down); }
  h->magic = 0;
  delete h;
  return SPMV_OK;
}

spmv_status_t spmv_get_info(spmv_handle_t h, spmv_info_t* out) {
  if (!handle_alive(h) || !out) return SPMV_ERR_INVALID_ARG;
  refresh_info(h);
  *out = h->info;
  return SPMV_OK;
}

spmv_status_t spmv_select(spmv_handle_t h, const char* desc, void* stream) {
  if (!handle_alive(h) || !desc) return SPMV_ERR_INVALID_ARG;
  Variant v;
  if (!variant_from_string(desc, &v)) { set_last_error("cannot parse variant '%s'", desc); return SPMV_ERR_INVALID_ARG; }
  std::string why;
  if (!variant_eligible(h, v, &why)) { set_last_error("variant %s not eligible: %s", desc, why.c_str()); return SPMV_ERR_UNSUPPORTED; }
  spmv_status_t st = adopt_variant(h, v, (cudaStream_t)stream);
  if (st != SPMV_OK) return st;
  SPMV_CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
  return SPMV_OK;
}

spmv_status_t spmv_update_values(spmv_handle_t h, const double* d_val, int32_t* fell_back, void* stream) {
  if (!handle_alive(h) || (h->A.nnz > 0 && !d_val)) return SPMV_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  SPMV_CUDA_TRY(cudaDeviceSynchronize());           // no apply on any stream may still be reading the old formats
  h->A.val = d_val;
  const Variant want = h->sel;
  const bool was_tuned = h->tuned;
  const std::vector<std::string> leaders = h->leaders;
  release_all_formats(h);
  reset_to_default(h);                              // the old plan points into what was just freed: whatever fails
                                                    // below, the handle stays usable (on the default variant)
  if (h->dia_state > 0) h->dia_state = 0;           // constness must be re-established on the new values
  if (fell_back) *fell_back = 0;
  spmv_status_t st = adopt_variant(h, want, s);
  if (st == SPMV_OK) { h->tuned = was_tuned; h->leaders = leaders; refresh_info(h); }
  if (st == SPMV_ERR_UNSUPPORTED) {
    if (fell_back) *fell_back = 1;
    Variant alt = want;
    st = SPMV_ERR_UNSUPPORTED;
    if ((want.fam == FAM_DIA_CONST || want.fam == FAM_DIA_CWIN) && variant_from_string("dia_tma:b288:c256:r1:u8:i3:x0", &alt)) {
      std::string why;
      if (variant_eligible(h, alt, &why)) st = adopt_variant(h, alt, s);
      if (st == SPMV_OK) { h->tuned = was_tuned; refresh_info(h); }
    }
    if (st != SPMV_OK) st = adopt_variant(h, default_variant(), s);
  }
  if (st != SPMV_OK) return st;
  SPMV_CUDA_TRY(cudaStreamSynchronize(s));
  return SPMV_OK;
}

// Variants with a second, ordered fix-up kernel own one workspace per handle.  Two applies of such a variant on
// DIFFERENT streams would overlap on the GPU and mix their carries, so the library orders them itself: every such
// apply records an event, and an apply on another stream than the previous one first makes its stream wait for it
// (no host synchronisation; same-stream applies pay one event record).  Inside a stream capture the graph's own
// edges order the launches and no event is touched; replaying such a graph concurrently with other applies of the
// same handle remains the caller's to order.
static spmv_status_t apply_with_workspace(spmv_handle_s* h, const ApplyArgs& a) {
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(a.stream, &cap) != cudaSuccess) { cudaGetLastError(); cap = cudaStreamCaptureStatusNone; }
  if (cap != cudaStreamCaptureStatusNone) return launch_plan(h->plan, a);
  std::lock_guard<std::mutex> lk(h->ws_mu);
  if (!h->ws_event) SPMV_CUDA_TRY(cudaEventCreateWithFlags(&h->ws_event, cudaEventDisableTiming));
  if (h->ws_used && h->ws_stream != a.stream) SPMV_CUDA_TRY(cudaStreamWaitEvent(a.stream, h->ws_event, 0));
  const spmv_status_t st = launch_plan(h->plan, a);
  if (st != SPMV_OK) return st;
  SPMV_CUDA_TRY(cudaEventRecord(h->ws_event, a.stream));
  h->ws_stream = a.stream;
  h->ws_used = true;
  return SPMV_OK;
}

// The apply path: argument checks, then one (two for merge-path / row-split SELL) kernel launch from the
// plan resolved at select / tune time.  No locks, no lookups, no CUDA attribute or occupancy calls.
spmv_status_t spmv_apply(spmv_handle_t h, double alpha, const double* d_x, double beta, double* d_y, void* stream) {
  if (!h || h->magic != kHandleMagic) return SPMV_ERR_INVALID_ARG;
  if (h->A.rows > 0 && !d_y) return SPMV_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  if (alpha == 0.0 || h->A.rows == 0) {           // reading A2: A and x are not referenced
    cudaError_t e = scale_y_launch(h->A.rows, beta, d_y, s);
    if (e != cudaSuccess) { set_last_error("scale kernel: %s", cudaGetErrorString(e)); return SPMV_ERR_CUDA; }
    return SPMV_OK;
  }
  if (h->A.cols > 0 && !d_x) return SPMV_ERR_INVALID_ARG;
  if (d_x == d_y) { set_last_error("spmv_apply: x and y are the same vector (they must not alias)"); return SPMV_ERR_INVALID_ARG; }
  ApplyArgs a{alpha, beta, d_x, d_y, s};
  if (h->plan.n == 2) return apply_with_workspace(h, a);     // merge-path / row-split SELL
  return launch_plan(h->plan, a);
}

struct spmv_graph_s {
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  int k = 0;
};

spmv_status_t spmv_graph_create(spmv_handle_t h, double alpha, const double* d_x, double beta, double* d_y, int32_t k,
                                spmv_graph_t* out) {
  if (!handle_alive(h) || !out || k < 1) return SPMV_ERR_INVALID_ARG;
  cudaStream_t cs = nullptr;
  SPMV_CUDA_TRY(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
  spmv_graph_s* g = new (std::nothrow) spmv_graph_s();
  if (!g) { cudaStreamDestroy(cs); return SPMV_ERR_ALLOC; }
  g->k = k;
  cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
  spmv_status_t st = SPMV_OK;
  for (int i = 0; i < k && e == cudaSuccess && st == SPMV_OK; ++i) st = spmv_apply(h, alpha, d_x, beta, d_y, cs);
  cudaError_t e2 = cudaStreamEndCapture(cs, &g->graph);         // always end the capture, also after a failure
  if (e == cudaSuccess) e = e2;
  if (e == cudaSuccess && st == SPMV_OK) e = cudaGraphInstantiate(&g->exec, g->graph, 0);
  cudaStreamDestroy(cs);
  if (e != cudaSuccess || st != SPMV_OK) {
    if (e != cudaSuccess) set_last_error("spmv_graph_create: %s", cudaGetErrorString(e));
    if (g->graph) cudaGraphDestroy(g->graph);
    delete g;
    cudaGetLastError();
    return st != SPMV_OK ? st : SPMV_ERR_CUDA;
  }
  *out = g;
  return SPMV_OK;
}

spmv_status_t spmv_graph_launch(spmv_graph_t g, void* stream) {
  if (!g || !g->exec) return SPMV_ERR_INVALID_ARG;
  SPMV_CUDA_TRY(cudaGraphLaunch(g->exec, (cudaStream_t)stream));
  return SPMV_OK;
}

spmv_status_t spmv_graph_destroy(spmv_graph_t g) {
  if (!g) return SPMV_ERR_INVALID_ARG;
  if (g->exec) cudaGraphExecDestroy(g->exec);
  if (g->graph) cudaGraphDestroy(g->graph);
  delete g;
  return SPMV_OK;
}

// Host-vector apply.  Where the selected variant has a row-range form (plan_for_rows) the call is a pipeline over
// chunks of rows on three internal streams: upload (x as far as the chunk's rows reach -- its rows plus the
// matrix bandwidth -- and the chunk of y when beta != 0) | kernel on the chunk | download of the chunk of y.
// PCIe is full duplex, so the download of chunk k-1 overlaps the upload of chunk k+1 and the kernel of chunk k;
// for a banded matrix the first kernel starts long before x is complete.  Results are bit-identical to the
// one-launch form: a row is summed by the same kernel code in the same order.
// entry: event the pipeline's internal streams wait on (nullptr: the current tail of `stream`); wait: synchronise
// `stream` before returning (spmv_apply_host_batch enqueues every member first and synchronises once)
static spmv_status_t apply_host_body(spmv_handle_t h, double alpha, const double* h_x, double beta, double* h_y,
                                     void* stream, cudaEvent_t entry, bool wait);

// Nothing of a host-vector apply may outlive the call that failed: copies and kernels already queued on the
// pipeline's internal streams still read h_x and write h_y, which the caller is free to release after an error.
static void drain_host_streams(spmv_handle_s* h, cudaStream_t s) {
  const std::string err = last_error_text();
  for (cudaStream_t q : {h->hs_up, h->hs_up2, h->hs_run, h->hs_down})
    if (q) cudaStreamSynchronize(q);
  cudaStreamSynchronize(s);
  cudaGetLastError();
  set_last_error("%s", err.c_str());
}

static spmv_status_t apply_host_impl(spmv_handle_t h, double alpha, const double* h_x, double beta, double* h_y,
                                     void* stream, cudaEvent_t entry, bool wait) {
  const spmv_status_t st = apply_host_body(h, alpha, h_x, beta, h_y, stream, entry, wait);
  if (st != SPMV_OK && st != SPMV_ERR_INVALID_ARG && handle_alive(h)) drain_host_streams(h, (cudaStream_t)stream);
  return st;
}

static spmv_status_t apply_host_body(spmv_handle_t h, double alpha, const double* h_x, double beta, double* h_y,
                                     void* stream, cudaEvent_t entry, bool wait) {
  if (!handle_alive(h)) return SPMV_ERR_INVALID_ARG;
  if ((h->A.rows > 0 && !h_y) || (h->A.cols > 0 && !h_x)) return SPMV_ERR_INVALID_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const int64_t rows = h->A.rows, cols = h->A.cols;
  if (!h->d_x_stage) h->d_x_stage = (double*)h->al.alloc(sizeof(double) * cols, s);
  if (!h->d_y_stage) h->d_y_stage = (double*)h->al.alloc(sizeof(double) * rows, s);
  if (!h->d_x_stage || !h->d_y_stage) return SPMV_ERR_ALLOC;
  double *dx = h->d_x_stage, *dy = h->d_y_stage;

  // Zero-copy y.  When the caller's y is pinned, MAPPED host memory (cudaHostAlloc / cudaHostRegister: what
  // torch's pin_memory() gives) and the variant's kernels read and write y one row per thread in row order (the
  // DIA families), the chunk kernels work on the caller's vector in place: their 256-byte warp stores cross PCIe as
  // posted writes while the copy engine uploads the next chunk of x, and no copy engine runs in the opposite
  // direction (measured on the B200 box: bidirectional 3 MB DMA chunks drop to ~31 GB/s each way; cfg2 0.84 ->
  // 0.76 ms, one cfg5 member 0.92 -> 0.75 ms).  Families that store y with a stride (BCSR: three rows from one
  // lane; permuted SELL) were slower this way (BCSR with its y stores packed to 24 B per block row: 0.97 vs 0.68 ms)
  // and keep the staged copies.  SPMV_HOST_ZEROCOPY=0 disables it.
  double* zy = nullptr;
  {
    const char* zc_env = getenv("SPMV_HOST_ZEROCOPY");
    const bool zc_on = !(zc_env && atoi(zc_env) == 0);
    const int rk = h->plan.range_kind;
    if (zc_on && rows > 0 && (rk == RANGE_DIA || rk == RANGE_DIA_TMA || rk == RANGE_DIA_CONST)) {
      cudaPointerAttributes pa;
      if (cudaPointerGetAttributes(&pa, h_y) == cudaSuccess && pa.type == cudaMemoryTypeHost && pa.devicePointer &&
          ((uintptr_t)pa.devicePointer & 15) == 0)
        zy = (double*)pa.devicePointer;
      cudaGetLastError();                      // an unregistered pageable pointer is not an error here
    }
  }
  // chunks of ~3 MB of y (smaller: the fixed cost of a PCIe copy shows; larger: less overlap; ~8 MB when y is
  // zero-copy: the kernels' own PCIe traffic has no per-copy cost), boundaries on the variant's range alignment
  const int64_t align = h->plan.range_align > 0 ? h->plan.range_align : 1;
  const char* chunk_env = getenv("SPMV_HOST_CHUNK_MB");        // read per call: tests force several chunks on small matrices
  const double chunk_mb_env = chunk_env ? atof(chunk_env) : 0.0;
  const double chunk_mb = chunk_mb_env > 0 ? chunk_mb_env : zy ? 8.0 : 3.0;
  int64_t nchunks = std::min<int64_t>(32, (int64_t)(rows * 8 / (chunk_mb * 1048576.0)));
  int64_t chunk = nchunks > 1 ? ((rows + nchunks - 1) / nchunks + align - 1) / align * align : rows;
  const bool pipelined = alpha != 0.0 && nchunks > 1 && chunk < rows && h->plan.n == 1 && h->plan.range_kind != RANGE_NONE;
  if (!pipelined) {
    // small stencil systems: three DMA operations cost more than the data (cfg1: 32 KB each way).  When both
    // vectors are mapped host memory and the variant reads x as coalesced shifted streams (the DIA families:
    // zy != nullptr) the kernel works on the caller's x and y in place -- one launch and one synchronise.
    // Measured: 5-point stencils 29.7 -> 20.8 us (32 KB vectors), 68.9 -> 49.6 us (512 KB); slower from 2 MB per
    // vector on, and 4-13x slower for gathered x (small power-law matrices), hence the family and size limits.
    if (zy && alpha != 0.0 && (rows + cols) * 8 <= (1 << 20) && cols > 0) {
      cudaPointerAttributes px;
      const bool okx = cudaPointerGetAttributes(&px, h_x) == cudaSuccess && px.type == cudaMemoryTypeHost && px.devicePointer;
      cudaGetLastError();
      if (okx) {
        spmv_status_t st = spmv_apply(h, alpha, (const double*)px.devicePointer, beta, zy, stream);
        if (st != SPMV_OK) return st;
        if (wait) SPMV_CUDA_TRY(cudaStreamSynchronize(s));
        return SPMV_OK;
      }
    }
    if (cols) SPMV_CUDA_TRY(cudaMemcpyAsync(dx, h_x, sizeof(double) * cols, cudaMemcpyHostToDevice, s));
    if (beta != 0.0 && rows) SPMV_CUDA_TRY(cudaMemcpyAsync(dy, h_y, sizeof(double) * rows, cudaMemcpyHostToDevice, s));
    spmv_status_t st = spmv_apply(h, alpha, dx, beta, dy, stream);
    if (st != SPMV_OK) return st;
    if (rows) SPMV_CUDA_TRY(cudaMemcpyAsync(h_y, dy, sizeof(double) * rows, cudaMemcpyDeviceToHost, s));
    if (wait) SPMV_CUDA_TRY(cudaStreamSynchronize(s));
    return SPMV_OK;
  }
  nchunks = (rows + chunk - 1) / chunk;
  if (!h->hs_up) {
    SPMV_CUDA_TRY(cudaStreamCreateWithFlags(&h->hs_up, cudaStreamNonBlocking));
    SPMV_CUDA_TRY(cudaStreamCreateWithFlags(&h->hs_up2, cudaStreamNonBlocking));
    SPMV_CUDA_TRY(cudaStreamCreateWithFlags(&h->hs_run, cudaStreamNonBlocking));
    SPMV_CUDA_TRY(cudaStreamCreateWithFlags(&h->hs_down, cudaStreamNonBlocking));
  }
  while ((int64_t)h->hs_events.size() < 3 * nchunks + 2) {
    cudaEvent_t e;
    SPMV_CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    h->hs_events.push_back(e);
  }
  cudaEvent_t* ev = h->hs_events.data();
  // work already queued on the caller's stream comes first (a batch: what was queued when the batch began)
  cudaEvent_t ev_in = entry;
  if (!ev_in) {
    SPMV_CUDA_TRY(cudaEventRecord(ev[3 * nchunks], s));
    ev_in = ev[3 * nchunks];
  }
  SPMV_CUDA_TRY(cudaStreamWaitEvent(h->hs_up, ev_in, 0));
  SPMV_CUDA_TRY(cudaStreamWaitEvent(h->hs_up2, ev_in, 0));
  SPMV_CUDA_TRY(cudaStreamWaitEvent(h->hs_run, ev_in, 0));
  SPMV_CUDA_TRY(cudaStreamWaitEvent(h->hs_down, ev_in, 0));
  const bool aligned = true;                 // the staging vectors come from the allocator: 16-byte aligned
  const int64_t bw = h->info.bandwidth;
  int64_t x_up = 0;                          // x[0, x_up) is queued for upload
  for (int64_t c = 0; c < nchunks; ++c) {
    const int64_t a = c * chunk, b = std::min(rows, a + chunk);
    const int64_t need = std::min(cols, b + bw + 1);          // rows < b reference columns < b + bandwidth + 1
    if (need > x_up) {
      SPMV_CUDA_TRY(cudaMemcpyAsync(dx + x_up, h_x + x_up, sizeof(double) * (need - x_up), cudaMemcpyHostToDevice, h->hs_up));
      x_up = need;
    }
    SPMV_CUDA_TRY(cudaEventRecord(ev[3 * c], h->hs_up));
    SPMV_CUDA_TRY(cudaStreamWaitEvent(h->hs_run, ev[3 * c], 0));
    if (beta != 0.0 && !zy) {       // y on its own upload stream: the fixed latencies of the two small copies overlap
      SPMV_CUDA_TRY(cudaMemcpyAsync(dy + a, h_y + a, sizeof(double) * (b - a), cudaMemcpyHostToDevice, h->hs_up2));
      SPMV_CUDA_TRY(cudaEventRecord(ev[3 * c + 2], h->hs_up2));
      SPMV_CUDA_TRY(cudaStreamWaitEvent(h->hs_run, ev[3 * c + 2], 0));
    }
    KernelCall kc;
    if (!plan_for_rows(h->plan, rows, cols, a, b, aligned, &kc)) { set_last_error("apply_host: range launch refused"); return SPMV_ERR_INTERNAL; }
    ApplyArgs args{alpha, beta, dx, zy ? zy : dy, h->hs_run};
    cudaError_t e = run_call(kc, args);
    if (e != cudaSuccess) { set_last_error("apply_host: chunk launch failed: %s", cudaGetErrorString(e)); return SPMV_ERR_CUDA; }
    SPMV_CUDA_TRY(cudaEventRecord(ev[3 * c + 1], h->hs_run));
    SPMV_CUDA_TRY(cudaStreamWaitEvent(h->hs_down, ev[3 * c + 1], 0));
    if (!zy) SPMV_CUDA_TRY(cudaMemcpyAsync(h_y + a, dy + a, sizeof(double) * (b - a), cudaMemcpyDeviceToHost, h->hs_down));
  }
  SPMV_CUDA_TRY(cudaEventRecord(ev[3 * nchunks + 1], h->hs_down));
  SPMV_CUDA_TRY(cudaStreamWaitEvent(s, ev[3 * nchunks + 1], 0));
  if (wait) {
    SPMV_CUDA_TRY(cudaStreamSynchronize(s));
    SPMV_CUDA_TRY(cudaStreamSynchronize(h->hs_up));     // (nothing pending: every upload precedes a kernel that has finished)
  }
  return SPMV_OK;
}

spmv_status_t spmv_apply_host(spmv_handle_t h, double alpha, const double* h_x, double beta, double* h_y,
                              void* stream) {
  return apply_host_impl(h, alpha, h_x, beta, h_y, stream, nullptr, true);
}

// n host-vector applies as ONE call: every member's chunk pipeline is enqueued behind the same entry event (its
// own internal streams: the members' copies and kernels interleave, PCIe never idles between members), then
// `stream` is synchronised once.
spmv_status_t spmv_apply_host_batch(int32_t n, const spmv_handle_t* hs, const double* alphas, const double* const* h_xs,
                                    const double* betas, double* const* h_ys, void* stream) {
  if (n < 0 || (n > 0 && (!hs || !alphas || !h_xs || !betas || !h_ys))) return SPMV_ERR_INVALID_ARG;
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < i; ++j)
      if (hs[i] == hs[j]) { set_last_error("spmv_apply_host_batch: a handle appears twice (its staging vectors would be shared)"); return SPMV_ERR_INVALID_ARG; }
  cudaStream_t s = (cudaStream_t)stream;
  cudaEvent_t entry = nullptr;
  SPMV_CUDA_TRY(cudaEventCreateWithFlags(&entry, cudaEventDisableTiming));
  cudaError_t e = cudaEventRecord(entry, s);
  spmv_status_t st = e == cudaSuccess ? SPMV_OK : SPMV_ERR_CUDA;
  for (int i = 0; i < n && st == SPMV_OK; ++i) st = apply_host_impl(hs[i], alphas[i], h_xs[i], betas[i], h_ys[i], stream, entry, false);
  e = cudaStreamSynchronize(s);                    // also after a failure: nothing of this call may stay in flight
  for (int i = 0; i < n; ++i) {
    if (!handle_alive(hs[i])) continue;
    if (st != SPMV_OK) drain_host_streams(hs[i], s);       // a member failed: every member's pipeline is drained
    else if (hs[i]->hs_up) cudaStreamSynchronize(hs[i]->hs_up);
  }
  cudaEventDestroy(entry);
  if (st == SPMV_OK && e != cudaSuccess) { set_last_error("spmv_apply_host_batch: %s", cudaGetErrorString(e)); st = SPMV_ERR_CUDA; }
  return st;
}


spmv_status_t spmv_apply_batch(int32_t n, const spmv_handle_t* hs, const double* alphas, const double* const* d_xs,
                               const double* betas, double* const* d_ys, void* const* streams, int32_t nstreams) {
  if (n < 0 || (n > 0 && (!hs || !alphas || !d_xs || !betas || !d_ys))) return SPMV_ERR_INVALID_ARG;
  if (nstreams < 0 || (nstreams > 0 && !streams)) return SPMV_ERR_INVALID_ARG;
  for (int i = 0; i < n; ++i) {
    void* s = nstreams > 0 ? streams[i % nstreams] : nullptr;
    spmv_status_t st = spmv_apply(hs[i], alphas[i], d_xs[i], betas[i], d_ys[i], s);
    if (st != SPMV_OK) return st;
  }
  return SPMV_OK;
}

spmv_status_t spmv_list_variants(spmv_handle_t h, char* buf, size_t cap, size_t* len) {
  if (!handle_alive(h) || !len) return SPMV_ERR_INVALID_ARG;
  int pruned = 0;
  std::vector<Variant> c = enumerate_candidates(h, nullptr, &pruned);
  std::string all;
  for (const auto& v : c) { all += variant_to_string(v); all += '\n'; }
  *len = all.size() + 1;
  if (buf && cap > 0) {
    size_t n = all.size() < cap - 1 ? all.size() : cap - 1;
    memcpy(buf, all.data(), n);
    buf[n] = 0;
  }
  return SPMV_OK;
}

spmv_status_t spmv_format_download(spmv_handle_t h, const char* name, void* h_buf, size_t cap, size_t* bytes,
                                   void* stream) {
  if (!handle_alive(h) || !name || !bytes) return SPMV_ERR_INVALID_ARG;
  const Variant& v = h->sel;
  const void* src = nullptr;
  size_t n = 0;
  const SellFormat* sf = nullptr;
  if (is_sell_family(v)) {
    auto it = h->sells.find(sell_key(v));
    if (it != h->sells.end()) sf = &it->second;
  } else if (v.fam == FAM_ELL && h->has_ell) {
    sf = &h->ell;
  }
  if (sf) {
    if (!strcmp(name, "slice_ptr")) { src = sf->slice_ptr; n = sizeof(int64_t) * (sf->nslices + 1); }
    else if (!strcmp(name, "sval")) { src = sf->val; n = sizeof(double) * sf->padded; }
    else if (!strcmp(name, "scol") && sf->col) { src = sf->col; n = sizeof(int32_t) * sf->padded; }
    else if (!strcmp(name, "scol16") && sf->col16) { src = sf->col16; n = sizeof(uint16_t) * sf->padded; }
    else if (!strcmp(name, "sbase") && sf->sbase) { src = sf->sbase; n = sizeof(int32_t) * sf->nslices; }
    else if (!strcmp(name, "perm") && sf->perm) { src = sf->perm; n = sizeof(int32_t) * sf->nslices * sf->C; }
  } else if (v.fam == FAM_BCSR3 && h->has_bcsr) {
    if (!strcmp(name, "brow_ptr")) { src = h->bcsr.brow_ptr; n = sizeof(int32_t) * (h->bcsr.brows + 1); }
    else if (!strcmp(name, "bcol") && h->bcsr.bcol) { src = h->bcsr.bcol; n = sizeof(int32_t) * h->bcsr.nblocks; }
    else if (!strcmp(name, "bcol16") && h->bcsr.bcol16) { src = h->bcsr.bcol16; n = sizeof(uint16_t) * h->bcsr.nblocks; }
    else if (!strcmp(name, "bval")) { src = h->bcsr.bval; n = sizeof(double) * 9 * h->bcsr.nblocks; }
  } else if ((v.fam == FAM_DIA || v.fam == FAM_DIA_TMA || v.fam == FAM_DIA_CONST || v.fam == FAM_DIA_WIN || v.fam == FAM_DIA_CWIN) && h->dias.count(v.C)) {
    const DiaFormat& df = h->dias[v.C];
    if (!strcmp(name, "dia_val")) { src = df.val; n = sizeof(double) * df.nd * df.ld; }
    else if (!strcmp(name, "dia_mask")) { src = df.mask; n = sizeof(unsigned) * df.ld; }
    else if (!strcmp(name, "dia_mask_small") && df.mask_small) { src = df.mask_small; n = (size_t)df.mask_elem * df.ld; }
    else if (!strcmp(name, "dia_coef")) {     // host-resident
      *bytes = sizeof(double) * df.nd;
      if (h_buf && cap > 0) memcpy(h_buf, df.coef, *bytes < cap ? *bytes : cap);
      return SPMV_OK;
    }
    else if (!strcmp(name, "dia_off")) {      // host-resident: copied directly
      *bytes = sizeof(int) * df.nd;
      if (h_buf && cap > 0) memcpy(h_buf, df.off, *bytes < cap ? *bytes : cap);
      return SPMV_OK;
    }
  } else if (v.fam == FAM_MERGE) {
    auto it = h->plans.find(v.block * v.I);
    if (it != h->plans.end() && !strcmp(name, "tile_row")) { src = it->second.tile_row; n = sizeof(int32_t) * (it->second.ntiles + 1); }
  }
  if (!src) { set_last_error("no array '%s' in the selected format", name); return SPMV_ERR_INVALID_ARG; }
  *bytes = n;
  if (h_buf && cap > 0) {
    cudaStream_t s = (cudaStream_t)stream;
    SPMV_CUDA_TRY(cudaMemcpyAsync(h_buf, src, n < cap ? n : cap, cudaMemcpyDeviceToHost, s));
    SPMV_CUDA_TRY(cudaStreamSynchronize(s));
  }
  return SPMV_OK;
}

}  // extern "C"
