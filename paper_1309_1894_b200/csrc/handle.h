// The handle behind spmv_handle_t and the helpers api.cu / tuner.cu share.
#pragma once
#include <map>
#include <mutex>
#include <string>
#include <tuple>
#include <utility>

#include "spmv_internal.h"

struct spmv_handle_s {
  uint64_t magic = 0;
  spmv::CsrView A;
  spmv::Allocator al;
  spmv::DeviceProps dev;
  int device = 0;
  spmv_info_t info{};
  spmv::Variant sel;
  spmv::LaunchPlan plan;          // resolved launch of `sel` (rebuilt by select / tune / update_values)
  bool tuned = false;
  std::vector<std::string> leaders;   // best three distinct candidates of the last spmv_tune (spmv_cg tune_loop)

  // owned formats, built on demand
  std::map<std::tuple<int, int, int, int>, spmv::SellFormat> sells;   // key (C, sigma, split, 16-bit indices)
  spmv::SellFormat ell;
  bool has_ell = false;
  spmv::BcsrFormat bcsr;
  bool has_bcsr = false;
  std::map<int, spmv::MergePlan> plans;                    // key tile_items
  std::map<int, spmv::DiaFormat> dias;                     // key C
  int dia_state = 0;                                       // 0 not tried, 1 built once, -1 pattern is not diagonal

  // merge-path and row-split SELL keep ONE workspace per handle (tile carries / segment sums): applies of such a
  // variant are chained through this event, so that an apply enqueued on another stream starts after the previous one
  std::mutex ws_mu;
  cudaEvent_t ws_event = nullptr;
  cudaStream_t ws_stream = nullptr;
  bool ws_used = false;

  // staging for spmv_apply_host, and the three internal streams + events of its chunk pipeline
  double* d_x_stage = nullptr;
  double* d_y_stage = nullptr;
  cudaStream_t hs_up = nullptr, hs_up2 = nullptr, hs_run = nullptr, hs_down = nullptr;
  std::vector<cudaEvent_t> hs_events;
};

namespace spmv {

inline bool is_sell16(const Variant& v) { return v.fam == FAM_SELL16 || v.fam == FAM_SELL16_TMA; }
inline bool is_sell_family(const Variant& v) { return v.fam == FAM_SELL || v.fam == FAM_SELL_TMA || is_sell16(v); }
inline std::tuple<int, int, int, int> sell_key(const Variant& v) { return std::make_tuple(v.C, v.S, v.L, is_sell16(v) ? 1 : 0); }

constexpr uint64_t kHandleMagic = 0x53504D5642323030ull;   // "SPMVB200"
constexpr const char* kVersion = "0.1.0";

bool handle_alive(spmv_handle_t h);

// Structural eligibility of a variant for this matrix (SURVEY.md sec. 8(d) "pruning").
bool variant_eligible(const spmv_handle_s* h, const Variant& v, std::string* why);
// Builds (or finds) the format the variant needs.  UNSUPPORTED if the built format turns
// out too padded to be worth keeping.
spmv_status_t ensure_format(spmv_handle_s* h, const Variant& v, cudaStream_t s);
// Resolves kernel, grid, shared memory, carve-out and the argument block of `v` (format must exist).
spmv_status_t build_plan(spmv_handle_s* h, const Variant& v, LaunchPlan* out);
// q = A x with x.q fused into the kernel (solver loop); UNSUPPORTED when the selected family has no such form.
spmv_status_t build_dot_plan(spmv_handle_s* h, double* part, int* n_part, LaunchPlan* out);
// Launches a resolved plan: patch alpha / x / beta / y, one or two kernel launches, nothing else.
spmv_status_t launch_plan(const LaunchPlan& p, const ApplyArgs& a);
// Makes `v` the selected variant: format, plan, info.  Waits for the device first when formats are freed.
spmv_status_t adopt_variant(spmv_handle_s* h, const Variant& v, cudaStream_t s);
// Error paths that may have released the selected variant's format call this: if the format is gone, the handle
// goes back to the fixed default variant (plan on the caller's CSR arrays), tuned = false.
bool selected_format_alive(const spmv_handle_s* h);
void repair_selection_after_failure(spmv_handle_s* h);
void reset_to_default(spmv_handle_s* h);
// Bytes of matrix data the variant streams per apply (format-actual, not algorithmic).
int64_t variant_format_bytes(const spmv_handle_s* h, const Variant& v);
// Frees every owned format the given variant does not need.
void release_formats_except(spmv_handle_s* h, const Variant& keep);
void release_all_formats(spmv_handle_s* h);
// Candidate list of the tuner's first phase for this matrix.
std::vector<Variant> enumerate_candidates(const spmv_handle_s* h, const char* filter, int* n_pruned_structural);
std::string signature_key(const spmv_handle_s* h, bool beta_nonzero);

}  // namespace spmv
