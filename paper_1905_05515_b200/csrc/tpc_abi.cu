// tpc_abi.cu -- the C ABI of include/tpc.h: context, staging of clusters, host-side tables, kernel sequence, result export.
// Everything the path computes runs in the kernels of k1..k6; the host code here only sizes buffers, computes the per-row
// and per-unit constant tables (double -> float once) and moves bytes.  No CPU fallback exists.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <string>
#include <vector>
#include <algorithm>

#include "../../include/tpc.h"
#include "tpc_internal.cuh"

using namespace tpc;

namespace {

std::string g_create_error = "";

// grow-only device buffer
struct DevBuf {
  void* p = nullptr; size_t cap = 0;
  cudaError_t ensure(size_t bytes) {
    if (bytes <= cap) return cudaSuccess;
    size_t want = std::max(bytes, cap + cap / 2);
    want = (want + 255) & ~(size_t)255;
    if (p) { cudaError_t e = cudaFree(p); p = nullptr; cap = 0; if (e != cudaSuccess) return e; }
    cudaError_t e = cudaMalloc(&p, want);
    if (e != cudaSuccess) { p = nullptr; return e; }
    cap = want; return cudaSuccess;
  }
  // grow keeping the first keep_bytes (device-to-device copy on the stream)
  cudaError_t ensure_keep(size_t bytes, size_t keep_bytes, cudaStream_t s) {
    if (bytes <= cap) return cudaSuccess;
    size_t want = std::max(bytes, cap * 2);
    want = (want + 255) & ~(size_t)255;
    void* np = nullptr;
    cudaError_t e = cudaMalloc(&np, want);
    if (e != cudaSuccess) return e;
    keep_bytes = std::min(keep_bytes, cap);
    if (p && keep_bytes) { e = cudaMemcpyAsync(np, p, keep_bytes, cudaMemcpyDeviceToDevice, s); if (e != cudaSuccess) { cudaFree(np); return e; } }
    if (p) { cudaStreamSynchronize(s); cudaFree(p); }
    p = np; cap = want; return cudaSuccess;
  }
  void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
  template <class T> T* as() const { return (T*)p; }
};

// grow-only pinned host buffer
struct PinBuf {
  void* p = nullptr; size_t cap = 0;
  cudaError_t ensure_keep(size_t bytes, size_t keep_bytes) {
    if (bytes <= cap) return cudaSuccess;
    size_t want = std::max(bytes, cap * 2);
    void* np = nullptr;
    cudaError_t e = cudaMallocHost(&np, want);
    if (e != cudaSuccess) return e;
    keep_bytes = std::min(keep_bytes, cap);
    if (p && keep_bytes) memcpy(np, p, keep_bytes);
    if (p) cudaFreeHost(p);
    p = np; cap = want; return cudaSuccess;
  }
  cudaError_t ensure(size_t bytes) { return ensure_keep(bytes, 0); }
  void release() { if (p) cudaFreeHost(p); p = nullptr; cap = 0; }
  template <class T> T* as() const { return (T*)p; }
};

// grow-only pinned host array (result arrays: the device -> host copy is then a true asynchronous DMA)
template <class T> struct PinVec {
  PinBuf b;
  cudaError_t resize(size_t n) { return b.ensure(std::max<size_t>(n, 1) * sizeof(T)); }
  T* data() const { return (T*)b.p; }
  void release() { b.release(); }
};

struct Tunables {   // DESIGN.md table T
  double wy = 1.5, wz = 1.5, dzdx_max = 1.5, wz0 = 0.75, cut2 = 1.75;
  int min_seed = 3;
  double c0[5] = {1.0, 2.25, 1.0, 1.0, 100.0};
  double s_max = 0.95, n_sigma = 4.0, w_max = 3.0;
  int max_gap = 4;
  double edge_margin = 1.0;
  int min_hits = 10;
  double grid_min = 1.0, grid_max = 64.0, grid_scale = 1.0;
  int debug_keep = 0;
  int chunk = 1024;           // clusters per K2/K3 work item (multiple of 32)
  int k2_threads = 0;         // K2 block size (0 = default 256); tuning knob
  int bridge_rows = 0, bridge_min = 3;       // NEXT-2 seed bridging (reading A39): 0 = off
  int link_skip = 0;                         // NEXT-2 (reading A45): 1 = links may skip one pad row (S2')
  double skip_cut2 = 1.75;                   // cut2 of the pairs that skip a row (= cut2 by default; smaller = stricter)
  int bridge_rescue = 0;                     // 1: dropped start hits are fitted in a second wave when the first left their chain unused (A39c)
  double bridge_wy = 1.0, bridge_wz = 1.5;
  double merge_edge = 3.0, merge_dy = 1.5, merge_dz = 2.0, merge_ds = 0.05, merge_dt = 0.05; int merge_rows = 8;   // NEXT-3 (reading A41)
  double loop_qmin = 5.0, loop_dy = 1.0, loop_ds = 0.1, loop_dt = 0.1, loop_dq = 0.5, loop_pmin = 2.0, loop_frac = 0.35; int loop_nmax = 20;   // NEXT-3, second half (reading A46)
};

struct UnitSrc { long long src = 0; int n = 0; };

constexpr int K1_SMEM_CURSOR_MAX = 50 * 1024;   // ints (200 KB) of shared-memory bin cursors per CTA; larger grids use global scratch

}  // namespace

struct tpc_ctx {
  // geometry / physics
  int NS = 0, R = 0;
  std::vector<float> row_x;
  float dphi = 0, z_max = 0, t_frame = 0, sigma_y = 0, sigma_z = 0, bz = 0, vdrift = 0;
  Tunables T;
  int device = 0, sm_count = 148;
  cudaStream_t stream = nullptr;
  std::string err;
  bool loaded_any = false;       // a load happened since create/clear (freezes tpc_set_param)
  bool have_result = false;

  // input staging: one logical arena; host loads land in h_y/h_t (pinned) and are uploaded at find time
  std::vector<UnitSrc> usrc;     // [U]
  long long arena_pos = 0;
  PinBuf h_y, h_t;
  DevBuf d_in_y, d_in_t;
  std::vector<std::pair<long long, long long>> dirty;   // host ranges [a,b) not yet uploaded

  // tables
  std::vector<UnitDesc> h_units; std::vector<Item> h_items;
  PinBuf p_units, p_items, p_small;
  DevBuf d_rows, d_units, d_items;
  bool rows_valid = false;
  bool tables_ready = false;     // per-unit grid descriptors / work items computed and uploaded for the clusters loaded now
  int t_msm = 0, t_max_n = 0, t_max_perm = 0, t_max_yz = 0; long long t_cursor_total = 0;   // K1 launch plan of those tables
  int pinned_async = 0;          // 1: a pinned host source is read by DMA after the load call returned (caller keeps it untouched until tpc_find_tracks*)
  cudaEvent_t ev_tables = nullptr;   // end of the last table upload (the pinned staging copy may be rewritten after it)
  Params P;

  // S1..S4
  long long N = 0, n_bins = 0; int n_items = 0;
  DevBuf d_yz, d_perm, d_bin_start, d_cursor, d_link_up, d_link_dn, d_raw_up, d_raw_dn, d_mask, d_item_count, d_item_base, d_scan_tmp;
  DevBuf d_start_unit, d_start_pos, d_counters, d_keep, d_keep_pos, d_start_unit2, d_start_pos2, d_flag2, d_used;
  // S5/S6
  int M = 0; long long Mpad = 0;
  long long m_cap_hint = 0;      // capacity guess for the per-tracklet buffers of the next call (1.25 x the last count)
  DevBuf d_k5scratch, d_rowhit, d_tl_n, d_tl_first, d_tl_last, d_tl_chi2, d_tl_par, d_tl_cov, d_owner, d_tl_key, d_scan_in, d_scan_out, d_scan_tmp64;
  // outputs (device)
  long long n_tracks = 0, n_refs = 0;
  DevBuf o_sector, o_x, o_par, o_cov, o_chi2, o_ndf, o_tracklet, o_cl_begin, o_cl_row, o_cl_index;
  // outputs / debug copies (host)
  PinVec<int32_t> ho_sector, ho_ndf, ho_tracklet, ho_cl_row, ho_cl_index; PinVec<float> ho_x, ho_par, ho_cov, ho_chi2;
  PinVec<int64_t> ho_cl_begin;
  // S9 merges (device + host)
  DevBuf l_prev, l_prev_n, l_root, l_turn, l_list, l_sec; PinVec<int32_t> hl_prev, hl_root, hl_turn;   // S10 looper turns (device + host)
  DevBuf g_outer, g_row_in, g_row_out, g_leaver, g_sec_begin, g_list, g_blist, g_bucket, g_cand, g_next, g_prev; PinVec<int32_t> hg_next, hg_prev;
  // S8 cluster marks (device + host)
  DevBuf m_att, m_adj, m_status, m_track, m_path, m_path_end; PinVec<int32_t> hm_status, hm_track;
  // S7 refit (device + host)
  DevBuf r_n, r_ndf, r_x, r_par, r_cov, r_chi2, r_z0, r_t0, r_order, r_classes;
  PinVec<int32_t> hr_n, hr_ndf; PinVec<float> hr_x, hr_par, hr_cov, hr_chi2, hr_z0, hr_t0;
  std::vector<int8_t> dbg_up_k, dbg_dn_k;
  std::vector<float> dbg_yz; std::vector<int32_t> dbg_perm, dbg_bins, dbg_up, dbg_dn, dbg_su, dbg_sp;
  std::vector<int32_t> dbg_tl_sector, dbg_tl_row, dbg_tl_n, dbg_tl_first, dbg_tl_last, dbg_rowhit; std::vector<float> dbg_tl_chi2, dbg_tl_x, dbg_tl_par, dbg_tl_cov;

  cudaEvent_t ev[10] = {};
  bool load_pending = false;     // ev_load recorded, not yet waited for
  cudaEvent_t ev_load = nullptr;   // end of a direct H2D copy from the caller's pinned memory (stage_append)
  tpc_timings timings = {};
};

namespace {

int fail(tpc_ctx* c, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof(buf), fmt, ap); va_end(ap);
  if (c) c->err = buf; else g_create_error = buf;
  return code;
}
#define CUDA_TRY(c, expr)                                                                                         \
  do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return fail((c), e_ == cudaErrorMemoryAllocation ? TPC_E_NOMEM : TPC_E_CUDA, \
                                                                   "%s: %s", #expr, cudaGetErrorString(e_)); } while (0)
#define LAUNCH_TRY(c, expr, counter)                                                                              \
  do { int rc_ = (expr); if (rc_ < 0) return fail((c), TPC_E_CUDA, "%s: %s", #expr, cudaGetErrorString((cudaError_t)(-rc_))); (counter) += rc_; } while (0)

// 0 = unregistered host, 1 = pinned host, 2 = device / managed
int pointer_kind(const void* p) {
  cudaPointerAttributes a;
  cudaError_t e = cudaPointerGetAttributes(&a, p);
  if (e != cudaSuccess) { cudaGetLastError(); return 0; }
  if (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) return 2;
  if (a.type == cudaMemoryTypeHost) return 1;
  return 0;
}

int prepare_tables(tpc_ctx* c);

void add_dirty(tpc_ctx* c, long long a, long long b) {
  if (!c->dirty.empty() && c->dirty.back().second == a) c->dirty.back().second = b;
  else c->dirty.emplace_back(a, b);
}

}  // namespace

// =====================================================================================================================
extern "C" {

int tpc_abi_version(void) { return 1; }

// 1 for the checked build (bounds checks in the kernels, -DTPC_CHECKED), 0 for the product build
int tpc_checked_build(void) {
#ifdef TPC_CHECKED
  return 1;
#else
  return 0;
#endif
}

const char* tpc_last_error(const tpc_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

int tpc_create(const tpc_geometry* g, float bz, float vdrift, tpc_ctx** out) {
  if (out) *out = nullptr;
  if (!g || !out) return fail(nullptr, TPC_E_ARG, "tpc_create: null argument");
  if (g->n_sectors < 1 || g->n_rows < 3 || !g->row_x) return fail(nullptr, TPC_E_ARG, "tpc_create: need n_sectors >= 1, n_rows >= 3 and row_x");
  if (g->n_rows > 255) return fail(nullptr, TPC_E_CAPACITY, "tpc_create: n_rows > 255 does not fit the selector key");
  if ((long long)g->n_sectors * g->n_rows > (1 << 24)) return fail(nullptr, TPC_E_CAPACITY, "tpc_create: too many (sector,row) units");
  for (int r = 0; r < g->n_rows; r++) {
    if (!std::isfinite(g->row_x[r]) || !(g->row_x[r] > 0) || (r && !(g->row_x[r] > g->row_x[r - 1])))
      return fail(nullptr, TPC_E_ARG, "tpc_create: row_x must be finite, positive and strictly increasing (row %d)", r);
  }
  if (!std::isfinite(bz) || !std::isfinite(vdrift) || !(vdrift > 0)) return fail(nullptr, TPC_E_ARG, "tpc_create: Bz must be finite and vdrift finite and > 0");
  if (!(g->sector_dphi > 0) || !(g->sector_dphi < 3.14159f) || !(g->z_max > 0) || !(g->t_frame >= 0) || !(g->sigma_y > 0) || !(g->sigma_z > 0) ||
      !std::isfinite(g->z_max) || !std::isfinite(g->t_frame))
    return fail(nullptr, TPC_E_ARG, "tpc_create: sector_dphi in (0,pi), z_max > 0, t_frame >= 0, sigma_y/z > 0 required");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(nullptr, TPC_E_CUDA, "tpc_create: no CUDA device (%s); this library has no CPU fallback", e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
  }
  tpc_ctx* c = new (std::nothrow) tpc_ctx();
  if (!c) return fail(nullptr, TPC_E_NOMEM, "tpc_create: out of host memory");
  c->NS = g->n_sectors; c->R = g->n_rows; c->row_x.assign(g->row_x, g->row_x + g->n_rows);
  c->dphi = g->sector_dphi; c->z_max = g->z_max; c->t_frame = g->t_frame; c->sigma_y = g->sigma_y; c->sigma_z = g->sigma_z;
  c->bz = bz; c->vdrift = vdrift;
  c->usrc.assign((size_t)c->NS * c->R, UnitSrc());
  cudaDeviceProp prop;
  if (cudaGetDevice(&c->device) != cudaSuccess || cudaGetDeviceProperties(&prop, c->device) != cudaSuccess) {
    int rc = fail(nullptr, TPC_E_CUDA, "tpc_create: cannot query the CUDA device: %s", cudaGetErrorString(cudaGetLastError()));
    delete c; return rc;
  }
  c->sm_count = prop.multiProcessorCount;
  for (auto& ev : c->ev) {
    if (cudaEventCreate(&ev) != cudaSuccess) { int rc = fail(nullptr, TPC_E_CUDA, "tpc_create: cudaEventCreate failed"); delete c; return rc; }
  }
  if (cudaEventCreateWithFlags(&c->ev_load, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&c->ev_tables, cudaEventDisableTiming) != cudaSuccess) {
    int rc = fail(nullptr, TPC_E_CUDA, "tpc_create: cudaEventCreate failed"); tpc_destroy(c); return rc;
  }
  *out = c;
  return TPC_OK;
}

void tpc_destroy(tpc_ctx* c) {
  if (!c) return;
  cudaStreamSynchronize(c->stream);
  DevBuf* bufs[] = {&c->d_in_y, &c->d_in_t, &c->d_rows, &c->d_units, &c->d_items, &c->d_yz, &c->d_perm, &c->d_bin_start, &c->d_cursor,
                    &c->d_link_up, &c->d_link_dn, &c->d_raw_up, &c->d_raw_dn, &c->d_mask, &c->d_item_count, &c->d_item_base, &c->d_scan_tmp,
                    &c->d_start_unit, &c->d_start_pos, &c->d_counters, &c->d_k5scratch, &c->d_rowhit, &c->d_tl_n, &c->d_tl_first, &c->d_tl_last, &c->d_tl_chi2,
                    &c->d_tl_par, &c->d_tl_cov, &c->d_owner, &c->d_tl_key, &c->d_scan_in, &c->d_scan_out, &c->d_scan_tmp64, &c->o_sector,
                    &c->o_x, &c->o_par, &c->o_cov, &c->o_chi2, &c->o_ndf, &c->o_tracklet, &c->o_cl_begin, &c->o_cl_row, &c->o_cl_index,
                    &c->r_n, &c->r_ndf, &c->r_x, &c->r_par, &c->r_cov, &c->r_chi2, &c->r_z0, &c->r_t0, &c->r_order, &c->r_classes,
                    &c->d_keep, &c->d_keep_pos, &c->d_start_unit2, &c->d_start_pos2, &c->d_flag2, &c->d_used, &c->m_att, &c->m_adj, &c->m_status, &c->m_track, &c->m_path, &c->m_path_end,
                    &c->g_outer, &c->g_row_in, &c->g_row_out, &c->g_leaver, &c->g_sec_begin, &c->g_list, &c->g_blist, &c->g_bucket, &c->g_cand, &c->g_next, &c->g_prev,
                    &c->l_prev, &c->l_prev_n, &c->l_root, &c->l_turn, &c->l_list, &c->l_sec};
  for (DevBuf* b : bufs) b->release();
  c->h_y.release(); c->h_t.release(); c->p_units.release(); c->p_items.release(); c->p_small.release();
  c->ho_sector.release(); c->ho_ndf.release(); c->ho_tracklet.release(); c->ho_cl_row.release(); c->ho_cl_index.release();
  c->ho_x.release(); c->ho_par.release(); c->ho_cov.release(); c->ho_chi2.release(); c->ho_cl_begin.release();
  c->hr_n.release(); c->hr_ndf.release(); c->hr_x.release(); c->hr_par.release(); c->hr_cov.release(); c->hr_chi2.release();
  c->hr_z0.release(); c->hr_t0.release(); c->hm_status.release(); c->hm_track.release(); c->hg_next.release(); c->hg_prev.release(); c->hl_prev.release(); c->hl_root.release(); c->hl_turn.release();
  for (auto& ev : c->ev) if (ev) cudaEventDestroy(ev);
  if (c->ev_load) cudaEventDestroy(c->ev_load);
  if (c->ev_tables) cudaEventDestroy(c->ev_tables);
  delete c;
}

int tpc_set_stream(tpc_ctx* c, void* s) {
  if (!c) return TPC_E_ARG;
  c->stream = (cudaStream_t)s;
  return TPC_OK;
}

int tpc_set_param(tpc_ctx* c, const char* name, double v) {
  if (!c || !name) return fail(c, TPC_E_ARG, "tpc_set_param: null argument");
  if (c->loaded_any) return fail(c, TPC_E_STATE, "tpc_set_param(%s): only before the first load after tpc_create / tpc_clear", name);
  if (!std::isfinite(v)) return fail(c, TPC_E_ARG, "tpc_set_param(%s): value must be finite", name);
  Tunables& T = c->T; std::string s(name);
  auto pos = [&](double& f) { if (!(v > 0)) return fail(c, TPC_E_ARG, "tpc_set_param(%s): must be > 0", name); f = v; return (int)TPC_OK; };
  auto nonneg = [&](double& f) { if (!(v >= 0)) return fail(c, TPC_E_ARG, "tpc_set_param(%s): must be >= 0", name); f = v; return (int)TPC_OK; };
  int rc = TPC_OK;
  if (s == "wy") rc = pos(T.wy); else if (s == "wz") rc = pos(T.wz); else if (s == "dzdx_max") rc = nonneg(T.dzdx_max);
  else if (s == "wz0") rc = nonneg(T.wz0); else if (s == "cut2") rc = pos(T.cut2);
  else if (s == "min_seed") { if (v < 1 || v > 255) return fail(c, TPC_E_ARG, "min_seed must be in 1..255"); T.min_seed = (int)v; }
  else if (s == "c0_y") rc = pos(T.c0[0]); else if (s == "c0_z") rc = pos(T.c0[1]); else if (s == "c0_sinphi") rc = pos(T.c0[2]);
  else if (s == "c0_dzds") rc = pos(T.c0[3]); else if (s == "c0_qpt") rc = pos(T.c0[4]);
  else if (s == "s_max") { if (!(v > 0 && v < 1)) return fail(c, TPC_E_ARG, "s_max must be in (0,1)"); T.s_max = v; }
  else if (s == "n_sigma") rc = pos(T.n_sigma); else if (s == "w_max") rc = pos(T.w_max);
  else if (s == "max_gap") { if (v < 0 || v > 255) return fail(c, TPC_E_ARG, "max_gap must be in 0..255"); T.max_gap = (int)v; }
  else if (s == "edge_margin") rc = nonneg(T.edge_margin);
  else if (s == "min_hits") { if (v < 3 || v > 255) return fail(c, TPC_E_ARG, "min_hits must be in 3..255 (ndf = 2n-5 > 0)"); T.min_hits = (int)v; }
  else if (s == "grid_scale") rc = pos(T.grid_scale);
  else if (s == "debug_keep") T.debug_keep = v != 0;
  else if (s == "pinned_async") c->pinned_async = v != 0;
  else if (s == "k2_threads") { int k = (int)v; if (k < 32 || k > 256 || (k & 31)) return fail(c, TPC_E_ARG, "k2_threads must be a multiple of 32 in 32..256"); T.k2_threads = k; }
  else if (s == "chunk") { int k = (int)v; if (k < 32 || k > 4096 || (k & 31)) return fail(c, TPC_E_ARG, "chunk must be a multiple of 32 in 32..4096"); T.chunk = k; }
  else if (s == "bridge_rows") { if (v < 0 || v > 16) return fail(c, TPC_E_ARG, "bridge_rows must be in 0..16"); T.bridge_rows = (int)v; }
  else if (s == "bridge_min") { if (v < 3 || v > 255) return fail(c, TPC_E_ARG, "bridge_min must be in 3..255"); T.bridge_min = (int)v; }
  else if (s == "bridge_wy") rc = pos(T.bridge_wy); else if (s == "bridge_wz") rc = pos(T.bridge_wz);
  else if (s == "bridge_rescue") T.bridge_rescue = v != 0;
  else if (s == "link_skip") { if (v != 0 && v != 1) return fail(c, TPC_E_ARG, "link_skip must be 0 or 1"); T.link_skip = (int)v; }
  else if (s == "skip_cut2") { if (!(v > 0)) return fail(c, TPC_E_ARG, "skip_cut2 must be > 0"); T.skip_cut2 = v; }
  else if (s == "merge_edge") rc = nonneg(T.merge_edge); else if (s == "merge_dy") rc = pos(T.merge_dy); else if (s == "merge_dz") rc = pos(T.merge_dz);
  else if (s == "merge_ds") rc = pos(T.merge_ds); else if (s == "merge_dt") rc = pos(T.merge_dt);
  else if (s == "loop_qmin") rc = nonneg(T.loop_qmin); else if (s == "loop_dy") rc = pos(T.loop_dy); else if (s == "loop_ds") rc = pos(T.loop_ds);
  else if (s == "loop_dt") rc = pos(T.loop_dt); else if (s == "loop_dq") rc = pos(T.loop_dq); else if (s == "loop_pmin") rc = pos(T.loop_pmin);
  else if (s == "loop_frac") { if (!(v > 0 && v < 0.5)) return fail(c, TPC_E_ARG, "loop_frac must be in (0, 0.5)"); T.loop_frac = v; }
  else if (s == "loop_nmax") { if (v < 1 || v > 255) return fail(c, TPC_E_ARG, "loop_nmax must be in 1..255"); T.loop_nmax = (int)v; }
  else if (s == "merge_rows") { if (v < 0 || v > 255) return fail(c, TPC_E_ARG, "merge_rows must be in 0..255"); T.merge_rows = (int)v; }
  else return fail(c, TPC_E_ARG, "tpc_set_param: unknown parameter '%s'", name);
  if (rc == TPC_OK) { c->rows_valid = false; c->tables_ready = false; }
  return rc;
}

int tpc_clear(tpc_ctx* c) {
  if (!c) return TPC_E_ARG;
  cudaStreamSynchronize(c->stream);   // staged device copies may still read caller memory; outputs are about to be invalidated
  std::fill(c->usrc.begin(), c->usrc.end(), UnitSrc());
  c->arena_pos = 0; c->dirty.clear(); c->loaded_any = false; c->have_result = false; c->tables_ready = false;
  c->N = 0; c->M = 0; c->n_tracks = 0; c->n_refs = 0;
  return TPC_OK;
}

// append n floats per array at the arena position (rounded up to a multiple of 4 elements for 16-byte vector loads)
static int stage_append(tpc_ctx* c, const float* y, const float* t, long long n, long long* pos_out) {
  long long pos = (c->arena_pos + 3) & ~3LL;
  *pos_out = pos;
  if (n == 0) return TPC_OK;
  const int ky = pointer_kind(y), kt = pointer_kind(t);
  if ((ky == 2) != (kt == 2)) return fail(c, TPC_E_ARG, "tpc_load_clusters: pad_y and time must both be host or both be device pointers");
  const size_t bytes = (size_t)n * sizeof(float), end_bytes = (size_t)(pos + n) * sizeof(float);
  const bool direct = ky == 2 || (ky == 1 && kt == 1 && n >= (1 << 16));
  if (direct) {   // device source (D2D) or large pinned source (DMA straight from the caller's buffer), async on the stream
    const cudaMemcpyKind kind = ky == 2 ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    CUDA_TRY(c, c->d_in_y.ensure_keep(end_bytes + 64, (size_t)c->arena_pos * 4, c->stream));
    CUDA_TRY(c, c->d_in_t.ensure_keep(end_bytes + 64, (size_t)c->arena_pos * 4, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_in_y.as<float>() + pos, y, bytes, kind, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_in_t.as<float>() + pos, t, bytes, kind, c->stream));
    if (ky != 2 && !c->pinned_async) {   // the DMA reads the caller's pinned host memory: it must have finished when the load call
      // returns (tpc.h: host inputs may be freed or overwritten on return) unless the caller opted into pinned_async; the caller of
      // stage_append waits on this event after its own host work.  A device source follows stream order instead.
      CUDA_TRY(c, cudaEventRecord(c->ev_load, c->stream));
      c->load_pending = true;
    }
  } else {        // pageable (or small) host source: copy into the pinned arena now, upload at tpc_find_tracks
    CUDA_TRY(c, c->h_y.ensure_keep(end_bytes + 64, (size_t)c->arena_pos * 4));
    CUDA_TRY(c, c->h_t.ensure_keep(end_bytes + 64, (size_t)c->arena_pos * 4));
    memcpy(c->h_y.as<float>() + pos, y, bytes);
    memcpy(c->h_t.as<float>() + pos, t, bytes);
    add_dirty(c, pos, pos + n);
  }
  c->arena_pos = pos + n;
  return TPC_OK;
}

int tpc_load_clusters(tpc_ctx* c, int sector, int row, const float* pad_y, const float* time, const float* charge, int n) {
  (void)charge;   // carried by the interface, never read on this path (S0)
  if (!c) return TPC_E_ARG;
  if (sector < 0 || sector >= c->NS || row < 0 || row >= c->R) return fail(c, TPC_E_ARG, "tpc_load_clusters: sector %d / row %d out of range", sector, row);
  if (n < 0 || (n > 0 && (!pad_y || !time))) return fail(c, TPC_E_ARG, "tpc_load_clusters: n < 0 or null array with n > 0");
  long long pos = 0;
  int rc = stage_append(c, pad_y, time, n, &pos);
  if (rc != TPC_OK) return rc;
  if (c->load_pending) { c->load_pending = false; CUDA_TRY(c, cudaEventSynchronize(c->ev_load)); }
  UnitSrc& u = c->usrc[(size_t)sector * c->R + row];
  u.src = pos; u.n = n;
  c->loaded_any = true; c->have_result = false; c->tables_ready = false;
  return TPC_OK;
}

int tpc_load_clusters_batch(tpc_ctx* c, const int64_t* unit_off, const float* pad_y, const float* time, const float* charge) {
  (void)charge;
  if (!c) return TPC_E_ARG;
  if (!unit_off) return fail(c, TPC_E_ARG, "tpc_load_clusters_batch: null unit_off");
  const int U = c->NS * c->R;
  if (unit_off[0] < 0) return fail(c, TPC_E_ARG, "tpc_load_clusters_batch: negative offset");
  for (int u = 0; u < U; u++) {
    if (unit_off[u + 1] < unit_off[u]) return fail(c, TPC_E_ARG, "tpc_load_clusters_batch: unit_off must be ascending (unit %d)", u);
    if (unit_off[u + 1] - unit_off[u] > 0x7fffffffLL) return fail(c, TPC_E_CAPACITY, "tpc_load_clusters_batch: more than 2^31-1 clusters in unit %d", u);
  }
  const long long n = unit_off[U] - unit_off[0];
  if (n > 0 && (!pad_y || !time)) return fail(c, TPC_E_ARG, "tpc_load_clusters_batch: null array");
  std::fill(c->usrc.begin(), c->usrc.end(), UnitSrc());   // replaces everything loaded before
  c->arena_pos = 0; c->dirty.clear();
  long long pos = 0;
  int rc = stage_append(c, pad_y ? pad_y + unit_off[0] : nullptr, time ? time + unit_off[0] : nullptr, n, &pos);
  if (rc != TPC_OK) return rc;
  for (int u = 0; u < U; u++) { c->usrc[u].src = pos + (unit_off[u] - unit_off[0]); c->usrc[u].n = (int)(unit_off[u + 1] - unit_off[u]); }
  c->loaded_any = true; c->have_result = false; c->tables_ready = false;
  rc = prepare_tables(c);      // host tables + their upload while the cluster DMA (if any) is running
  if (c->load_pending) { c->load_pending = false; CUDA_TRY(c, cudaEventSynchronize(c->ev_load)); }
  return rc;
}

}  // extern "C"

// =====================================================================================================================
// Host-side tables: formulas evaluated in double, rounded to float once.
namespace {

void make_params_and_rows(tpc_ctx* c, std::vector<RowConst>& rows) {
  const Tunables& T = c->T; const int R = c->R;
  rows.assign(R, RowConst());
  const double dphi = (double)c->dphi;
  for (int r = 0; r < R; r++) {
    const double x = c->row_x[r], xu = r + 1 < R ? (double)c->row_x[r + 1] : x, xd = r > 0 ? (double)c->row_x[r - 1] : x;
    const double a = xu - x, b = x - xd;
    RowConst& k = rows[r];
    k.x = (float)x; k.tu = (float)(xu / x); k.td = (float)(xd / x); k.a = (float)a; k.b = (float)b;
    k.thr = (float)(T.cut2 * 0.5 * (a * a + b * b));
    k.wzu = (float)(T.dzdx_max * a + T.wz0); k.wzd = (float)(T.dzdx_max * b + T.wz0);
    k.yedge = (float)(x * tan(0.5 * dphi));
    const double xu2 = r + 2 < R ? (double)c->row_x[r + 2] : x, xd2 = r > 1 ? (double)c->row_x[r - 2] : x;
    const double a2 = xu2 - x, b2 = x - xd2;
    k.tu2 = (float)(xu2 / x); k.td2 = (float)(xd2 / x); k.a2 = (float)a2; k.b2 = (float)b2;
    k.wzu2 = (float)(T.dzdx_max * a2 + T.wz0); k.wzd2 = (float)(T.dzdx_max * b2 + T.wz0);
    k.thr21 = (float)(T.skip_cut2 * 0.5 * (a2 * a2 + b * b)); k.thr12 = (float)(T.skip_cut2 * 0.5 * (a * a + b2 * b2));
    k.thr22 = (float)(T.skip_cut2 * 0.5 * (a2 * a2 + b2 * b2));
    for (float& f : k.pad) f = 0.f;
  }
  Params& P = c->P;
  P.NS = c->NS; P.R = R; P.continuous = c->t_frame > 0 ? 1 : 0;
  P.zmax = c->z_max; P.vdrift = c->vdrift;
  P.wy = (float)T.wy; P.wz = (float)T.wz; P.min_seed = T.min_seed;
  P.cB = (float)(-0.00299792458 * (double)c->bz);
  for (int i = 0; i < 5; i++) P.c0[i] = (float)T.c0[i];
  P.ry = c->sigma_y * c->sigma_y; P.rz = c->sigma_z * c->sigma_z;
  P.smax = (float)T.s_max; P.nsigma = (float)T.n_sigma; P.wmax = (float)T.w_max; P.edge_margin = (float)T.edge_margin;
  P.max_gap = T.max_gap; P.min_hits = T.min_hits;
  P.bridge_rows = T.link_skip ? 0 : T.bridge_rows; P.bridge_min = T.bridge_min; P.bridge_wy = (float)T.bridge_wy; P.bridge_wz = (float)T.bridge_wz;
  P.link_skip = T.link_skip;
  P.check = nullptr;
}

// S1 grid descriptor of every unit + CSR offsets + K2/K3 work items.  Returns a tpc_status.
int make_units(tpc_ctx* c, int* max_smem_cursor, long long* cursor_total, int* max_n, int* max_perm, int* max_yz) {
  const Tunables& T = c->T; const int R = c->R, U = c->NS * R;
  c->h_units.resize(U); c->h_items.clear();
  const double dphi = (double)c->dphi, vd = (double)c->vdrift, tf = (double)c->t_frame, zmax = (double)c->z_max;
  long long off = 0, boff = 0, coff = 0; int msm = 0, mn = 0; long long mperm = 0, myz = 0;
  for (int u = 0; u < U; u++) {
    const int r = u % R; const int n = c->usrc[u].n;
    const double ye = (double)c->row_x[r] * tan(0.5 * dphi);
    const double y_lo = -ye - 1.0, y_hi = ye + 1.0, z_lo = -vd * tf - 1.0, z_hi = zmax + 1.0;
    double s = sqrt((y_hi - y_lo) * (z_hi - z_lo) / (double)std::max(n, 1)) * T.grid_scale;
    s = std::min(std::max(s, T.grid_min), T.grid_max);
    const double fy = ceil((y_hi - y_lo) / s), fz = ceil((z_hi - z_lo) / s);
    if (fy * fz > 2.0e9) return fail(c, TPC_E_CAPACITY, "grid of unit %d has more than 2e9 bins", u);
    UnitDesc& d = c->h_units[u];
    d.ny = std::max(1, (int)fy); d.nz = std::max(1, (int)fz);
    d.ylo = (float)y_lo; d.zlo = (float)z_lo; d.invs = (float)(1.0 / s);
    d.n = n; d.off = off; d.src = c->usrc[u].src; d.bin_off = boff; d.pad[0] = d.pad[1] = 0;
    const long long nb = (long long)d.ny * d.nz;
    if (nb + 1 <= K1_SMEM_CURSOR_MAX) {
      d.cur_off = -1;
      if (n > 0) {   // K1 shared-memory plan: cursors, then sorted indices, then (y, z) pairs (k1_grid.cu)
        msm = std::max(msm, (int)nb + 1);
        const long long pa = (nb + 1) & ~1LL, ya = (pa + n + 1) & ~1LL;
        mperm = std::max(mperm, pa + n); myz = std::max(myz, ya + 2LL * n);
      }
    }
    else { d.cur_off = coff; coff += nb + 1; }
    for (int s0 = 0; s0 < n; s0 += T.chunk) c->h_items.push_back(Item{u, s0});
    off += n; boff += nb + 1; mn = std::max(mn, n);
  }
  c->N = off; c->n_bins = boff; c->n_items = (int)c->h_items.size();
  *max_smem_cursor = msm; *cursor_total = coff; *max_n = mn;
  *max_perm = (int)std::min(mperm, 1LL << 30); *max_yz = (int)std::min(myz, 1LL << 30);
  return TPC_OK;
}

// Per-row constants, per-unit grid descriptors and K2/K3 work items for the clusters loaded now, computed on the host and uploaded
// (asynchronously, on the context's stream).  Runs once per loaded frame: at the end of tpc_load_clusters_batch, or at the first
// tpc_find_tracks* after per-unit loads.
int prepare_tables(tpc_ctx* c) {
  cudaStream_t st = c->stream;
  const int U = c->NS * c->R;
  std::vector<RowConst> rows;
  make_params_and_rows(c, rows);
  int rc = make_units(c, &c->t_msm, &c->t_cursor_total, &c->t_max_n, &c->t_max_perm, &c->t_max_yz);
  if (rc != TPC_OK) return rc;
  const int n_items = c->n_items;
  CUDA_TRY(c, cudaEventSynchronize(c->ev_tables));   // an earlier upload may still be reading the pinned staging copy
  CUDA_TRY(c, c->d_rows.ensure(rows.size() * sizeof(RowConst)));
  CUDA_TRY(c, c->d_units.ensure((size_t)U * sizeof(UnitDesc)));
  CUDA_TRY(c, c->d_items.ensure((size_t)std::max(n_items, 1) * sizeof(Item)));
  CUDA_TRY(c, c->p_units.ensure((size_t)U * sizeof(UnitDesc) + rows.size() * sizeof(RowConst)));
  CUDA_TRY(c, c->p_items.ensure((size_t)std::max(n_items, 1) * sizeof(Item)));
  memcpy(c->p_units.p, c->h_units.data(), (size_t)U * sizeof(UnitDesc));
  memcpy((char*)c->p_units.p + (size_t)U * sizeof(UnitDesc), rows.data(), rows.size() * sizeof(RowConst));
  if (n_items) memcpy(c->p_items.p, c->h_items.data(), (size_t)n_items * sizeof(Item));
  CUDA_TRY(c, cudaMemcpyAsync(c->d_units.p, c->p_units.p, (size_t)U * sizeof(UnitDesc), cudaMemcpyHostToDevice, st));
  CUDA_TRY(c, cudaMemcpyAsync(c->d_rows.p, (char*)c->p_units.p + (size_t)U * sizeof(UnitDesc), rows.size() * sizeof(RowConst), cudaMemcpyHostToDevice, st));
  if (n_items) CUDA_TRY(c, cudaMemcpyAsync(c->d_items.p, c->p_items.p, (size_t)n_items * sizeof(Item), cudaMemcpyHostToDevice, st));
  CUDA_TRY(c, cudaEventRecord(c->ev_tables, st));
  c->tables_ready = true;
  return TPC_OK;
}

int find_tracks_impl(tpc_ctx* c, tpc_tracks* out, bool to_host) {
  if (!c || !out) return fail(c, TPC_E_ARG, "tpc_find_tracks: null argument");
  memset(out, 0, sizeof(*out));
  const int R = c->R, U = c->NS * R;
  cudaStream_t st = c->stream;
  Launch L{st, c->sm_count, c->T.k2_threads};
  long long launches = 0;
  c->have_result = false;
  tpc_timings& tm = c->timings; memset(&tm, 0, sizeof(tm));

  CUDA_TRY(c, cudaEventRecord(c->ev[0], st));
  // ---- host tables (already computed and uploaded by tpc_load_clusters_batch; per-unit loads: here) + staged host clusters
  int rc = c->tables_ready ? (int)TPC_OK : prepare_tables(c);
  if (rc != TPC_OK) return rc;
  const int msm = c->t_msm, max_n = c->t_max_n, max_perm = c->t_max_perm, max_yz = c->t_max_yz; const long long cursor_total = c->t_cursor_total;
  const long long N = c->N; const int n_items = c->n_items; const int chunk = c->T.chunk;
  const Params& P = c->P;
  CUDA_TRY(c, c->d_in_y.ensure_keep((size_t)(c->arena_pos + 16) * 4, (size_t)c->arena_pos * 4, st));
  CUDA_TRY(c, c->d_in_t.ensure_keep((size_t)(c->arena_pos + 16) * 4, (size_t)c->arena_pos * 4, st));
  for (auto& rg : c->dirty) {
    const size_t b = (size_t)(rg.second - rg.first) * 4;
    CUDA_TRY(c, cudaMemcpyAsync(c->d_in_y.as<float>() + rg.first, c->h_y.as<float>() + rg.first, b, cudaMemcpyHostToDevice, st));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_in_t.as<float>() + rg.first, c->h_t.as<float>() + rg.first, b, cudaMemcpyHostToDevice, st));
  }
  c->dirty.clear();
  CUDA_TRY(c, c->p_small.ensure(256));
  CUDA_TRY(c, cudaEventRecord(c->ev[1], st));

  // ---- buffers of S1..S4
  CUDA_TRY(c, c->d_yz.ensure((size_t)(N + 4) * sizeof(float2)));
  CUDA_TRY(c, c->d_perm.ensure((size_t)(N + 4) * 4));
  CUDA_TRY(c, c->d_bin_start.ensure((size_t)(c->n_bins + 8) * 4));
  CUDA_TRY(c, c->d_cursor.ensure((size_t)(cursor_total + 4) * 4));
  CUDA_TRY(c, c->d_link_up.ensure((size_t)(N + 4) * 4));
  CUDA_TRY(c, c->d_link_dn.ensure((size_t)(N + 4) * 4));
  CUDA_TRY(c, c->d_mask.ensure((size_t)std::max(n_items, 1) * (chunk / 32) * 4));
  CUDA_TRY(c, c->d_item_count.ensure((size_t)std::max(n_items, 1) * 4));
  CUDA_TRY(c, c->d_item_base.ensure((size_t)std::max(n_items, 1) * 4));
  CUDA_TRY(c, c->d_scan_tmp.ensure((size_t)(n_items / SCAN_TILE + 4) * 4));
  const long long start_cap = N / std::max(1, c->T.min_seed) + 4;
  CUDA_TRY(c, c->d_start_unit.ensure((size_t)start_cap * 4));
  CUDA_TRY(c, c->d_start_pos.ensure((size_t)start_cap * 4));
  CUDA_TRY(c, c->d_counters.ensure(256));
#ifdef TPC_CHECKED
  c->P.check = reinterpret_cast<int*>(c->d_counters.as<char>() + 200);
  CUDA_TRY(c, cudaMemsetAsync(c->P.check, 0, sizeof(int), st));
#endif

  // ---- K1: S0 + S1
  LAUNCH_TRY(c, launch_k1_grid(L, U, c->d_units.as<UnitDesc>(), c->d_in_y.as<float>(), c->d_in_t.as<float>(), c->d_yz.as<float2>(),
                               c->d_perm.as<int>(), c->d_bin_start.as<int>(), c->d_cursor.as<int>(), P, std::max(msm, 1), max_n, max_perm, max_yz), launches);
  CUDA_TRY(c, cudaEventRecord(c->ev[2], st));
  // ---- K2: S2
  LAUNCH_TRY(c, launch_k2_neighbours(L, n_items, c->d_items.as<Item>(), chunk, c->d_units.as<UnitDesc>(), c->d_rows.as<RowConst>(),
                                     c->d_yz.as<float2>(), c->d_perm.as<int>(), c->d_bin_start.as<int>(), c->d_link_up.as<int>(),
                                     c->d_link_dn.as<int>(), P), launches);
  if (c->T.link_skip)   // S2': links that may skip a row, for the hits S2 left unlinked (its time counts as neighbour finding)
    LAUNCH_TRY(c, launch_k2_skip_links(L, n_items, c->d_items.as<Item>(), chunk, c->d_units.as<UnitDesc>(), c->d_rows.as<RowConst>(),
                                       c->d_yz.as<float2>(), c->d_perm.as<int>(), c->d_bin_start.as<int>(), c->d_link_up.as<int>(),
                                       c->d_link_dn.as<int>(), P), launches);
  CUDA_TRY(c, cudaEventRecord(c->ev[3], st));
  if (c->T.debug_keep && N > 0) {
    CUDA_TRY(c, c->d_raw_up.ensure((size_t)N * 4)); CUDA_TRY(c, c->d_raw_dn.ensure((size_t)N * 4));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_raw_up.p, c->d_link_up.p, (size_t)N * 4, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_raw_dn.p, c->d_link_dn.p, (size_t)N * 4, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(c, cudaEventRecord(c->ev[3], st));
  }
  // ---- K3: S3 + S4
  int* d_nstart = c->d_counters.as<int>();
  unsigned long long* d_total64 = (unsigned long long*)(c->d_counters.as<char>() + 64);
  LAUNCH_TRY(c, launch_k3_clean_start(L, n_items, c->d_items.as<Item>(), chunk, c->d_units.as<UnitDesc>(), c->d_link_up.as<int>(),
                                      c->d_link_dn.as<int>(), c->d_mask.as<unsigned>(), c->d_item_count.as<int>(), c->d_item_base.as<int>(),
                                      c->d_scan_tmp.as<int>(), c->d_start_unit.as<int>(), c->d_start_pos.as<int>(), d_nstart, P), launches);
  CUDA_TRY(c, cudaEventRecord(c->ev[4], st));
  typedef unsigned long long u64;
  unsigned long long* d_k5cnt = (unsigned long long*)(c->d_counters.as<char>() + 128);
  const bool variant = c->T.bridge_rows > 0 && !c->T.link_skip;   // (seed bridging is not combined with S2')
  // Default path: NO device -> host read between K3 and the end of the call.  The number of start hits M stays in device memory
  // (d_nstart); the per-tracklet buffers are sized for a capacity M_cap guessed from the frame size and from the previous call, the
  // kernels read M themselves, and the guess is checked when the counters are read at the end (a frame that exceeds it is
  // processed again from K5 with larger buffers: the S1-S4 tables stay valid).  The seed-bridging variants (off by default) size
  // their run lists on the host and keep the read-backs.
  long long M_cap = std::min<long long>(start_cap, std::max<long long>(c->m_cap_hint, N / 12 + 1024));
  int M = -1;                    // known on the host only in the variants, or at the end
  long long nt = 0, nr = 0, n_fitted = 0;
  for (int attempt = 0;; attempt++) {
    bool rescue = false;
    if (variant) {
      CUDA_TRY(c, cudaMemcpyAsync(c->p_small.p, d_nstart, sizeof(int), cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaStreamSynchronize(st));
      M = *c->p_small.as<int>();
      if (M < 0 || M > start_cap) return fail(c, TPC_E_CUDA, "start-hit count %d out of range", M);
      rescue = c->T.bridge_rescue && M > 0;
      if (!rescue && M > 0) {   // S4' (NEXT-2 variant): drop the start hits that continue a lower chain, order kept
        const size_t Mb = (size_t)M * 4;
        CUDA_TRY(c, c->d_keep.ensure(Mb)); CUDA_TRY(c, c->d_keep_pos.ensure(Mb)); CUDA_TRY(c, c->d_start_unit2.ensure(Mb));
        CUDA_TRY(c, c->d_start_pos2.ensure(Mb)); CUDA_TRY(c, c->d_scan_tmp.ensure((size_t)(std::max(M, n_items) / SCAN_TILE + 4) * 4));
        LAUNCH_TRY(c, launch_k3_bridge(L, M, c->d_start_unit.as<int>(), c->d_start_pos.as<int>(), c->d_units.as<UnitDesc>(), c->d_rows.as<RowConst>(),
                                       c->d_yz.as<float2>(), c->d_bin_start.as<int>(), c->d_link_up.as<int>(), c->d_link_dn.as<int>(),
                                       c->d_keep.as<int>(), c->d_keep_pos.as<int>(), c->d_scan_tmp.as<int>(), c->d_start_unit2.as<int>(),
                                       c->d_start_pos2.as<int>(), d_nstart, P), launches);
        CUDA_TRY(c, cudaMemcpyAsync(c->p_small.p, d_nstart, sizeof(int), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(c, cudaStreamSynchronize(st));
        const int M2 = *c->p_small.as<int>();
        if (M2 < 0 || M2 > M) return fail(c, TPC_E_CUDA, "bridged start-hit count %d out of range", M2);
        if (M2 > 0) {
          CUDA_TRY(c, cudaMemcpyAsync(c->d_start_unit.p, c->d_start_unit2.p, (size_t)M2 * 4, cudaMemcpyDeviceToDevice, st));
          CUDA_TRY(c, cudaMemcpyAsync(c->d_start_pos.p, c->d_start_pos2.p, (size_t)M2 * 4, cudaMemcpyDeviceToDevice, st));
        }
        CUDA_TRY(c, cudaEventRecord(c->ev[4], st));   // the S4' pass counts as part of K3's time
        M = M2;
      }
      M_cap = M;
    }
    if (M_cap > (1 << 24)) M_cap = 1 << 24;      // capacity of the selector key; a larger M is reported below
    const int Mc = (int)M_cap;
    const int* d_M = variant ? nullptr : d_nstart;   // where the kernels read the tracklet count

    // ---- K5: S5
    const size_t Mz = (size_t)std::max(Mc, 1);
    CUDA_TRY(c, c->d_rowhit.ensure((size_t)(Mz + 32) * R * sizeof(rowhit_t)));
    CUDA_TRY(c, c->d_k5scratch.ensure(k5_scratch_bytes(Mc)));
    CUDA_TRY(c, c->d_tl_n.ensure(Mz * 4)); CUDA_TRY(c, c->d_tl_first.ensure(Mz * 4)); CUDA_TRY(c, c->d_tl_last.ensure(Mz * 4));
    CUDA_TRY(c, c->d_tl_chi2.ensure(Mz * 4)); CUDA_TRY(c, c->d_tl_par.ensure(Mz * 20)); CUDA_TRY(c, c->d_tl_cov.ensure(Mz * 60));
    CUDA_TRY(c, c->d_owner.ensure((size_t)(N + 4) * 8)); CUDA_TRY(c, c->d_tl_key.ensure(Mz * 8));
    CUDA_TRY(c, c->d_scan_in.ensure(Mz * 8)); CUDA_TRY(c, c->d_scan_out.ensure(Mz * 8));
    CUDA_TRY(c, c->d_scan_tmp64.ensure((size_t)(Mc / SCAN_TILE + 4) * 8));
    CUDA_TRY(c, cudaMemsetAsync(d_k5cnt, 0, 32, st));
    auto run_k5 = [&](int n_run, const int* d_n, const int* list) -> int {
      LAUNCH_TRY(c, launch_k5_tracklets(L, n_run, d_n, Mc, list, c->d_start_unit.as<int>(), c->d_start_pos.as<int>(), c->d_units.as<UnitDesc>(),
                                        c->d_rows.as<RowConst>(), c->d_yz.as<float2>(), c->d_perm.as<int>(), c->d_bin_start.as<int>(),
                                        c->d_link_up.as<int>(), c->d_rowhit.as<rowhit_t>(), c->d_tl_n.as<int>(), c->d_tl_first.as<int>(),
                                        c->d_tl_last.as<int>(), c->d_tl_chi2.as<float>(), c->d_tl_par.as<float>(), c->d_tl_cov.as<float>(), d_k5cnt,
                                        c->d_k5scratch.p, P), launches);
      return TPC_OK;
    };
    n_fitted = -1;                 // = M unless the rescue variant skipped duplicates
    if (!rescue) {
      rc = run_k5(Mc, d_M, nullptr);
      if (rc != TPC_OK) return rc;
    } else {
      // S4' with rescue (reading A39c): first wave = the start hits that are not bridged; second wave = the bridged ones whose chain
      // the first wave did not use completely.  Tracklet index = position in the full S4 list in both waves; the others keep n = 0.
      const size_t Mb = (size_t)M * 4;
      CUDA_TRY(c, c->d_keep.ensure(Mb)); CUDA_TRY(c, c->d_keep_pos.ensure(Mb)); CUDA_TRY(c, c->d_start_unit2.ensure(Mb));
      CUDA_TRY(c, c->d_start_pos2.ensure(Mb)); CUDA_TRY(c, c->d_flag2.ensure(Mb));
      CUDA_TRY(c, c->d_scan_tmp.ensure((size_t)(std::max(M, n_items) / SCAN_TILE + 4) * 4));
      CUDA_TRY(c, cudaMemsetAsync(c->d_tl_n.p, 0, Mb, st));
      CUDA_TRY(c, cudaMemsetAsync(c->d_tl_first.p, 0xff, Mb, st)); CUDA_TRY(c, cudaMemsetAsync(c->d_tl_last.p, 0xff, Mb, st));
      int* list1 = c->d_start_unit2.as<int>(); int* list2 = c->d_start_pos2.as<int>();
      LAUNCH_TRY(c, launch_k3_bridge_lists(L, M, c->d_start_unit.as<int>(), c->d_start_pos.as<int>(), c->d_units.as<UnitDesc>(), c->d_rows.as<RowConst>(),
                                           c->d_yz.as<float2>(), c->d_bin_start.as<int>(), c->d_link_up.as<int>(), c->d_link_dn.as<int>(),
                                           c->d_keep.as<int>(), c->d_keep_pos.as<int>(), c->d_scan_tmp.as<int>(), list1, d_nstart, P), launches);
      CUDA_TRY(c, cudaMemcpyAsync(c->p_small.p, d_nstart, sizeof(int), cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaStreamSynchronize(st));
      const int M1 = *c->p_small.as<int>();
      if (M1 < 0 || M1 > M) return fail(c, TPC_E_CUDA, "first-wave start-hit count %d out of range", M1);
      rc = run_k5(M1, nullptr, list1);
      if (rc != TPC_OK) return rc;
      // first half of the selector over the first wave: its owner keys are the "used" marks of the rescue test
      CUDA_TRY(c, cudaMemsetAsync(c->d_owner.p, 0, (size_t)std::max(N, 1LL) * 8, st));
      CUDA_TRY(c, cudaMemsetAsync(c->d_tl_key.p, 0, Mz * 8, st));
      LAUNCH_TRY(c, launch_k6_owner(L, M1, list1, c->d_start_unit.as<int>(), c->d_units.as<UnitDesc>(), c->d_rowhit.as<rowhit_t>(), c->d_tl_n.as<int>(),
                                    c->d_tl_first.as<int>(), c->d_tl_last.as<int>(), c->d_tl_chi2.as<float>(), (unsigned long long*)c->d_owner.p,
                                    (unsigned long long*)c->d_tl_key.p, P), launches);
      LAUNCH_TRY(c, launch_k3_rescue_list(L, M, c->d_keep.as<int>(), c->d_start_unit.as<int>(), c->d_start_pos.as<int>(),
                                          c->d_units.as<UnitDesc>(), c->d_link_up.as<int>(), (const unsigned long long*)c->d_owner.p,
                                          c->d_flag2.as<int>(), c->d_keep_pos.as<int>(), c->d_scan_tmp.as<int>(), list2, d_nstart), launches);
      CUDA_TRY(c, cudaMemcpyAsync(c->p_small.p, d_nstart, sizeof(int), cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaStreamSynchronize(st));
      const int M2 = *c->p_small.as<int>();
      if (M2 < 0 || M2 > M - M1) return fail(c, TPC_E_CUDA, "rescue-wave start-hit count %d out of range", M2);
      if (M2 > 0) {
        rc = run_k5(M2, nullptr, list2);
        if (rc != TPC_OK) return rc;
        LAUNCH_TRY(c, launch_k6_owner(L, M2, list2, c->d_start_unit.as<int>(), c->d_units.as<UnitDesc>(), c->d_rowhit.as<rowhit_t>(), c->d_tl_n.as<int>(),
                                      c->d_tl_first.as<int>(), c->d_tl_last.as<int>(), c->d_tl_chi2.as<float>(), (unsigned long long*)c->d_owner.p,
                                      (unsigned long long*)c->d_tl_key.p, P), launches);
      }
      n_fitted = (long long)M1 + M2;
    }
    CUDA_TRY(c, cudaEventRecord(c->ev[5], st));

    // ---- K6: S6.  Output capacity: every tracklet a track, every cluster referenced once (a cluster has one owner).
    const long long cap_tracks = std::max<long long>(Mc, 1), cap_refs = std::max<long long>(N, 1);
    CUDA_TRY(c, c->o_sector.ensure(cap_tracks * 4)); CUDA_TRY(c, c->o_x.ensure(cap_tracks * 4)); CUDA_TRY(c, c->o_par.ensure(cap_tracks * 20));
    CUDA_TRY(c, c->o_cov.ensure(cap_tracks * 60)); CUDA_TRY(c, c->o_chi2.ensure(cap_tracks * 4)); CUDA_TRY(c, c->o_ndf.ensure(cap_tracks * 4));
    CUDA_TRY(c, c->o_tracklet.ensure(cap_tracks * 4)); CUDA_TRY(c, c->o_cl_begin.ensure((cap_tracks + 1) * 8));
    CUDA_TRY(c, c->o_cl_row.ensure(cap_refs * 4)); CUDA_TRY(c, c->o_cl_index.ensure(cap_refs * 4));
    LAUNCH_TRY(c, launch_k6_select(L, Mc, d_M, N, c->d_start_unit.as<int>(), c->d_units.as<UnitDesc>(),
                                   c->d_rowhit.as<rowhit_t>(), c->d_tl_n.as<int>(), c->d_tl_first.as<int>(), c->d_tl_last.as<int>(),
                                   c->d_tl_chi2.as<float>(), c->d_owner.as<u64>(), c->d_tl_key.as<u64>(), c->d_scan_in.as<u64>(),
                                   c->d_scan_out.as<u64>(), c->d_scan_tmp64.as<u64>(), d_total64, P, rescue), launches);
    LAUNCH_TRY(c, launch_k6_emit(L, Mc, d_M, c->d_start_unit.as<int>(), c->d_units.as<UnitDesc>(), c->d_rows.as<RowConst>(), c->d_perm.as<int>(),
                                 c->d_rowhit.as<rowhit_t>(), c->d_tl_n.as<int>(), c->d_tl_first.as<int>(), c->d_tl_last.as<int>(), c->d_tl_chi2.as<float>(),
                                 c->d_tl_par.as<float>(), c->d_tl_cov.as<float>(), c->d_owner.as<u64>(), c->d_tl_key.as<u64>(), c->d_scan_in.as<u64>(),
                                 c->d_scan_out.as<u64>(), c->o_sector.as<int>(), c->o_x.as<float>(), c->o_par.as<float>(), c->o_cov.as<float>(),
                                 c->o_chi2.as<float>(), c->o_ndf.as<int>(), c->o_tracklet.as<int>(), c->o_cl_begin.as<long long>(),
                                 c->o_cl_row.as<int>(), c->o_cl_index.as<int>(), d_total64, cap_tracks, cap_refs, P), launches);
    CUDA_TRY(c, cudaEventRecord(c->ev[6], st));

    // ---- the one read-back of the call: start-hit count, (tracks, references), S5 work counters
    if (!variant) CUDA_TRY(c, cudaMemcpyAsync(c->p_small.p, d_nstart, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(c, cudaMemcpyAsync(c->p_small.as<char>() + 64, d_total64, 8, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(c, cudaMemcpyAsync(c->p_small.as<char>() + 128, d_k5cnt, 24, cudaMemcpyDeviceToHost, st));
#ifdef TPC_CHECKED
    CUDA_TRY(c, cudaMemcpyAsync(c->p_small.as<char>() + 200, c->P.check, sizeof(int), cudaMemcpyDeviceToHost, st));
#endif
    CUDA_TRY(c, cudaStreamSynchronize(st));
#ifdef TPC_CHECKED
    if (*(int*)(c->p_small.as<char>() + 200) != 0) return fail(c, TPC_E_CUDA, "bounds check %d failed in a kernel (checked build)", *(int*)(c->p_small.as<char>() + 200));
#endif
    if (!variant) {
      M = *c->p_small.as<int>();
      if (M < 0 || M > start_cap) return fail(c, TPC_E_CUDA, "start-hit count %d out of range", M);
      if (M > (1 << 24)) return fail(c, TPC_E_CAPACITY, "%d tracklets exceed the 2^24 capacity of the selector key", M);
      if (M > M_cap) {             // the capacity guess was too small: repeat S5 / S6 with room for all M start hits
        if (attempt >= 2) return fail(c, TPC_E_CUDA, "tracklet capacity did not converge (%d start hits)", M);
        M_cap = std::min<long long>(start_cap, (long long)M + M / 8 + 1024);
        continue;
      }
    } else if (M > (1 << 24)) return fail(c, TPC_E_CAPACITY, "%d tracklets exceed the 2^24 capacity of the selector key", M);
    const u64 total = *(u64*)(c->p_small.as<char>() + 64);
    nt = (long long)(total >> 40); nr = (long long)(total & ((1ull << 40) - 1ull));
    if (nt > cap_tracks || nr > cap_refs) return fail(c, TPC_E_CUDA, "selector totals out of range (%lld tracks, %lld references)", nt, nr);
    if (n_fitted < 0) n_fitted = M;
    break;
  }
  c->m_cap_hint = (long long)M + M / 4 + 1024;   // next frame: 25 % headroom over this one
  c->M = M; c->Mpad = ((long long)M + 31) & ~31LL;
  c->n_tracks = nt; c->n_refs = nr;
  const size_t ntz = (size_t)std::max(nt, 1LL), nrz = (size_t)std::max(nr, 1LL);

  // ---- result
  out->n_tracks = nt; out->n_cluster_refs = nr;
  if (to_host) {
    CUDA_TRY(c, c->ho_sector.resize(ntz)); CUDA_TRY(c, c->ho_x.resize(ntz)); CUDA_TRY(c, c->ho_par.resize(ntz * 5));
    CUDA_TRY(c, c->ho_cov.resize(ntz * 15)); CUDA_TRY(c, c->ho_chi2.resize(ntz)); CUDA_TRY(c, c->ho_ndf.resize(ntz));
    CUDA_TRY(c, c->ho_tracklet.resize(ntz)); CUDA_TRY(c, c->ho_cl_begin.resize(ntz + 1)); CUDA_TRY(c, c->ho_cl_row.resize(nrz));
    CUDA_TRY(c, c->ho_cl_index.resize(nrz));
    if (nt > 0) {
      CUDA_TRY(c, cudaMemcpyAsync(c->ho_sector.data(), c->o_sector.p, nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->ho_x.data(), c->o_x.p, nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->ho_par.data(), c->o_par.p, nt * 20, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->ho_cov.data(), c->o_cov.p, nt * 60, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->ho_chi2.data(), c->o_chi2.p, nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->ho_ndf.data(), c->o_ndf.p, nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->ho_tracklet.data(), c->o_tracklet.p, nt * 4, cudaMemcpyDeviceToHost, st));
    }
    CUDA_TRY(c, cudaMemcpyAsync(c->ho_cl_begin.data(), c->o_cl_begin.p, (nt + 1) * 8, cudaMemcpyDeviceToHost, st));
    if (nr > 0) {
      CUDA_TRY(c, cudaMemcpyAsync(c->ho_cl_row.data(), c->o_cl_row.p, nr * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->ho_cl_index.data(), c->o_cl_index.p, nr * 4, cudaMemcpyDeviceToHost, st));
    }
    out->sector = c->ho_sector.data(); out->x = c->ho_x.data(); out->par = c->ho_par.data(); out->cov = c->ho_cov.data();
    out->chi2 = c->ho_chi2.data(); out->ndf = c->ho_ndf.data(); out->tracklet = c->ho_tracklet.data();
    out->cl_begin = c->ho_cl_begin.data(); out->cl_row = c->ho_cl_row.data(); out->cl_index = c->ho_cl_index.data();
  } else {
    out->sector = c->o_sector.as<int32_t>(); out->x = c->o_x.as<float>(); out->par = c->o_par.as<float>(); out->cov = c->o_cov.as<float>();
    out->chi2 = c->o_chi2.as<float>(); out->ndf = c->o_ndf.as<int32_t>(); out->tracklet = c->o_tracklet.as<int32_t>();
    out->cl_begin = c->o_cl_begin.as<int64_t>(); out->cl_row = c->o_cl_row.as<int32_t>(); out->cl_index = c->o_cl_index.as<int32_t>();
  }
  CUDA_TRY(c, cudaEventRecord(c->ev[7], st));
  CUDA_TRY(c, cudaStreamSynchronize(st));
  float* ms[7] = {&tm.ms_upload, &tm.ms_grid, &tm.ms_neighbours, &tm.ms_clean_start, &tm.ms_tracklets, &tm.ms_selector, &tm.ms_download};
  for (int i = 0; i < 7; i++) CUDA_TRY(c, cudaEventElapsedTime(ms[i], c->ev[i], c->ev[i + 1]));
  CUDA_TRY(c, cudaEventElapsedTime(&tm.ms_total, c->ev[0], c->ev[7]));
  tm.n_clusters = N; tm.n_bins = c->n_bins; tm.n_start_hits = M; tm.n_tracks = nt; tm.n_cluster_refs = nr; tm.launches = launches;
  tm.n_tracklets_kept = n_fitted;   // tracklets actually fitted (= start hits unless the rescue variant skipped duplicates)
  { const unsigned long long* k5 = (const unsigned long long*)(c->p_small.as<char>() + 128);
    tm.n_propagations = (int64_t)k5[0]; tm.n_updates = (int64_t)k5[1]; tm.n_pickups = (int64_t)k5[2]; }
  c->have_result = true;
  return TPC_OK;
}

}  // namespace

extern "C" {
int tpc_find_tracks(tpc_ctx* c, tpc_tracks* out) { return find_tracks_impl(c, out, true); }
int tpc_find_tracks_device(tpc_ctx* c, tpc_tracks* out) { return find_tracks_impl(c, out, false); }
// S7 (NEXT-1): K7 over the tracks of the last call; the S5/S6 buffers it reads (rowhit, sorted clusters, track lists) are still live.
int tpc_refit_tracks(tpc_ctx* c, int device_result, tpc_refit* out) {
  if (!c || !out) return fail(c, TPC_E_ARG, "tpc_refit_tracks: null argument");
  memset(out, 0, sizeof(*out));
  if (!c->have_result) return fail(c, TPC_E_STATE, "tpc_refit_tracks: call tpc_find_tracks first");
  cudaStream_t st = c->stream;
  Launch L{st, c->sm_count, c->T.k2_threads};
  const long long nt = c->n_tracks; const size_t ntz = (size_t)std::max(nt, 1LL);
  CUDA_TRY(c, c->r_n.ensure(ntz * 4)); CUDA_TRY(c, c->r_ndf.ensure(ntz * 4)); CUDA_TRY(c, c->r_x.ensure(ntz * 4));
  CUDA_TRY(c, c->r_par.ensure(ntz * 20)); CUDA_TRY(c, c->r_cov.ensure(ntz * 60)); CUDA_TRY(c, c->r_chi2.ensure(ntz * 4));
  CUDA_TRY(c, c->r_z0.ensure(ntz * 4)); CUDA_TRY(c, c->r_t0.ensure(ntz * 4));
  CUDA_TRY(c, c->r_order.ensure(ntz * 4)); CUDA_TRY(c, c->r_classes.ensure(768 * 4));
  long long launches = 0;
  CUDA_TRY(c, cudaEventRecord(c->ev[8], st));
  LAUNCH_TRY(c, launch_k7_refit(L, nt, c->o_sector.as<int>(), c->o_tracklet.as<int>(), c->o_cl_begin.as<long long>(), c->o_cl_row.as<int>(),
                                c->d_units.as<UnitDesc>(), c->d_rows.as<RowConst>(), c->d_yz.as<float2>(), c->d_rowhit.as<rowhit_t>(),
                                c->r_n.as<int>(), c->r_ndf.as<int>(), c->r_x.as<float>(), c->r_par.as<float>(), c->r_cov.as<float>(),
                                c->r_chi2.as<float>(), c->r_z0.as<float>(), c->r_t0.as<float>(), c->r_order.as<int>(), c->r_classes.as<int>(), c->P), launches);
  CUDA_TRY(c, cudaEventRecord(c->ev[9], st));
  out->n_tracks = nt;
  if (!device_result) {
    CUDA_TRY(c, c->hr_n.resize(ntz)); CUDA_TRY(c, c->hr_ndf.resize(ntz)); CUDA_TRY(c, c->hr_x.resize(ntz)); CUDA_TRY(c, c->hr_par.resize(ntz * 5));
    CUDA_TRY(c, c->hr_cov.resize(ntz * 15)); CUDA_TRY(c, c->hr_chi2.resize(ntz)); CUDA_TRY(c, c->hr_z0.resize(ntz)); CUDA_TRY(c, c->hr_t0.resize(ntz));
    if (nt > 0) {
      CUDA_TRY(c, cudaMemcpyAsync(c->hr_n.data(), c->r_n.p, nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hr_ndf.data(), c->r_ndf.p, nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hr_x.data(), c->r_x.p, nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hr_par.data(), c->r_par.p, nt * 20, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hr_cov.data(), c->r_cov.p, nt * 60, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hr_chi2.data(), c->r_chi2.p, nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hr_z0.data(), c->r_z0.p, nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hr_t0.data(), c->r_t0.p, nt * 4, cudaMemcpyDeviceToHost, st));
    }
    out->n = c->hr_n.data(); out->ndf = c->hr_ndf.data(); out->x = c->hr_x.data(); out->par = c->hr_par.data(); out->cov = c->hr_cov.data();
    out->chi2 = c->hr_chi2.data(); out->z0 = c->hr_z0.data(); out->t0 = c->hr_t0.data();
  } else {
    out->n = c->r_n.as<int32_t>(); out->ndf = c->r_ndf.as<int32_t>(); out->x = c->r_x.as<float>(); out->par = c->r_par.as<float>();
    out->cov = c->r_cov.as<float>(); out->chi2 = c->r_chi2.as<float>(); out->z0 = c->r_z0.as<float>(); out->t0 = c->r_t0.as<float>();
  }
  CUDA_TRY(c, cudaStreamSynchronize(st));
  CUDA_TRY(c, cudaEventElapsedTime(&out->ms_refit, c->ev[8], c->ev[9]));
  return TPC_OK;
}
// S8 (NEXT-4): K8 over the tracks and the grid of the last call.
int tpc_mark_clusters(tpc_ctx* c, float tube_cm, int device_result, tpc_cluster_marks* out) {
  if (!c || !out) return fail(c, TPC_E_ARG, "tpc_mark_clusters: null argument");
  memset(out, 0, sizeof(*out));
  if (!(tube_cm > 0) || !std::isfinite(tube_cm)) return fail(c, TPC_E_ARG, "tpc_mark_clusters: tube_cm must be finite and > 0");
  if (!c->have_result) return fail(c, TPC_E_STATE, "tpc_mark_clusters: call tpc_find_tracks first");
  cudaStream_t st = c->stream;
  Launch L{st, c->sm_count, c->T.k2_threads};
  const long long N = c->N; const size_t Nz = (size_t)std::max(N, 1LL);
  CUDA_TRY(c, c->m_att.ensure(Nz * 4)); CUDA_TRY(c, c->m_adj.ensure(Nz * 8)); CUDA_TRY(c, c->m_status.ensure(Nz * 4));
  CUDA_TRY(c, c->m_track.ensure(Nz * 4));
  { const size_t ntz = (size_t)std::max(c->n_tracks, 1LL); CUDA_TRY(c, c->m_path.ensure(ntz * c->R * 8)); CUDA_TRY(c, c->m_path_end.ensure(ntz * 4)); }
  long long launches = 0;
  CUDA_TRY(c, cudaEventRecord(c->ev[8], st));
  LAUNCH_TRY(c, launch_k8_status(L, c->n_tracks, N, c->NS * c->R, c->o_sector.as<int>(), c->o_tracklet.as<int>(), c->o_par.as<float>(),
                                 c->o_cl_begin.as<long long>(), c->o_cl_row.as<int>(), c->d_tl_first.as<int>(), c->d_units.as<UnitDesc>(),
                                 c->d_rows.as<RowConst>(), c->d_yz.as<float2>(), c->d_perm.as<int>(), c->d_bin_start.as<int>(),
                                 c->d_rowhit.as<rowhit_t>(), c->m_att.as<int>(), (unsigned long long*)c->m_adj.p, c->m_path.as<float2>(), c->m_path_end.as<int>(), c->m_status.as<int>(),
                                 c->m_track.as<int>(), tube_cm, c->P), launches);
  CUDA_TRY(c, cudaEventRecord(c->ev[9], st));
  out->n_clusters = N;
  if (!device_result) {
    CUDA_TRY(c, c->hm_status.resize(Nz)); CUDA_TRY(c, c->hm_track.resize(Nz));
    if (N > 0) {
      CUDA_TRY(c, cudaMemcpyAsync(c->hm_status.data(), c->m_status.p, (size_t)N * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hm_track.data(), c->m_track.p, (size_t)N * 4, cudaMemcpyDeviceToHost, st));
    }
    out->status = c->hm_status.data(); out->track = c->hm_track.data();
  } else {
    out->status = c->m_status.as<int32_t>(); out->track = c->m_track.as<int32_t>();
  }
  CUDA_TRY(c, cudaStreamSynchronize(st));
  CUDA_TRY(c, cudaEventElapsedTime(&out->ms_mark, c->ev[8], c->ev[9]));
  return TPC_OK;
}
// S9 (NEXT-3): K9 over the tracks of the last call.
int tpc_merge_tracks(tpc_ctx* c, int device_result, tpc_merges* out) {
  if (!c || !out) return fail(c, TPC_E_ARG, "tpc_merge_tracks: null argument");
  memset(out, 0, sizeof(*out));
  if (!c->have_result) return fail(c, TPC_E_STATE, "tpc_merge_tracks: call tpc_find_tracks first");
  cudaStream_t st = c->stream;
  Launch L{st, c->sm_count, c->T.k2_threads};
  const long long nt = c->n_tracks; const size_t ntz = (size_t)std::max(nt, 1LL);
  CUDA_TRY(c, c->g_outer.ensure(ntz * 16)); CUDA_TRY(c, c->g_row_in.ensure(ntz * 4)); CUDA_TRY(c, c->g_row_out.ensure(ntz * 4));
  CUDA_TRY(c, c->g_leaver.ensure(ntz * 4)); CUDA_TRY(c, c->g_list.ensure(ntz * 4)); CUDA_TRY(c, c->g_blist.ensure(ntz * 4));
  { const size_t NB = (size_t)c->NS * c->R + 1; CUDA_TRY(c, c->g_bucket.ensure((3 * NB + NB / SCAN_TILE + 4) * 4)); }
  CUDA_TRY(c, c->g_sec_begin.ensure((size_t)(c->NS + 2) * 4)); CUDA_TRY(c, c->g_cand.ensure(ntz * 8));
  CUDA_TRY(c, c->g_next.ensure(ntz * 4)); CUDA_TRY(c, c->g_prev.ensure(ntz * 4));
  const Tunables& T = c->T;
  // sectors per ring: 2 pi / dphi when that is an integer (to 1e-3 rad over the ring) and n_sectors is a whole number of rings
  // (one per side); otherwise the geometry has no neighbouring sectors and nothing is merged
  const double ring = 2.0 * M_PI / (double)c->dphi;
  int per_side = (int)lround(ring);
  if (per_side < 2 || fabs((double)per_side * (double)c->dphi - 2.0 * M_PI) > 1e-3 || c->NS % per_side != 0) per_side = 0;
  K9Params M{(float)T.merge_edge, (float)T.merge_dy, (float)T.merge_dz, (float)T.merge_ds, (float)T.merge_dt,
             (float)cos((double)c->dphi), (float)sin((double)c->dphi), T.merge_rows, per_side};
  long long launches = 0;
  CUDA_TRY(c, cudaEventRecord(c->ev[8], st));
  LAUNCH_TRY(c, launch_k9_merge(L, nt, c->NS, c->o_sector.as<int>(), c->o_tracklet.as<int>(), c->o_par.as<float>(), c->o_cl_begin.as<long long>(),
                                c->o_cl_row.as<int>(), c->d_tl_first.as<int>(), c->d_rows.as<RowConst>(), c->g_outer.as<float>(),
                                c->g_row_in.as<int>(), c->g_row_out.as<int>(), c->g_leaver.as<int>(), c->g_sec_begin.as<int>(), c->g_list.as<int>(), c->g_blist.as<int>(), c->g_bucket.as<int>(),
                                (unsigned long long*)c->g_cand.p, c->g_next.as<int>(), c->g_prev.as<int>(), M, c->P), launches);
  CUDA_TRY(c, cudaEventRecord(c->ev[9], st));
  out->n_tracks = nt;
  if (!device_result) {
    CUDA_TRY(c, c->hg_next.resize(ntz)); CUDA_TRY(c, c->hg_prev.resize(ntz));
    if (nt > 0) {
      CUDA_TRY(c, cudaMemcpyAsync(c->hg_next.data(), c->g_next.p, (size_t)nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hg_prev.data(), c->g_prev.p, (size_t)nt * 4, cudaMemcpyDeviceToHost, st));
    }
    out->next = c->hg_next.data(); out->prev = c->hg_prev.data();
  } else {
    out->next = c->g_next.as<int32_t>(); out->prev = c->g_prev.as<int32_t>();
  }
  CUDA_TRY(c, cudaStreamSynchronize(st));
  CUDA_TRY(c, cudaEventElapsedTime(&out->ms_merge, c->ev[8], c->ev[9]));
  return TPC_OK;
}
// S10 (NEXT-3, second half): K10 over the tracks of the last call.
int tpc_find_loopers(tpc_ctx* c, int device_result, tpc_loopers* out) {
  if (!c || !out) return fail(c, TPC_E_ARG, "tpc_find_loopers: null argument");
  memset(out, 0, sizeof(*out));
  if (!c->have_result) return fail(c, TPC_E_STATE, "tpc_find_loopers: call tpc_find_tracks first");
  cudaStream_t st = c->stream;
  Launch L{st, c->sm_count, c->T.k2_threads};
  const long long nt = c->n_tracks; const size_t ntz = (size_t)std::max(nt, 1LL);
  CUDA_TRY(c, c->l_prev.ensure(ntz * 4)); CUDA_TRY(c, c->l_prev_n.ensure(ntz * 4)); CUDA_TRY(c, c->l_root.ensure(ntz * 4));
  CUDA_TRY(c, c->l_turn.ensure(ntz * 4)); CUDA_TRY(c, c->l_list.ensure(ntz * 4)); CUDA_TRY(c, c->l_sec.ensure((size_t)(c->NS + 1) * 2 * 4));
  const Tunables& T = c->T;
  K10Params K{(float)T.loop_qmin, (float)T.loop_dy, (float)T.loop_ds, (float)T.loop_dt, (float)T.loop_dq, (float)T.loop_pmin,
              (float)T.loop_frac, (float)6.283185307179586, T.loop_nmax};
  long long launches = 0;
  CUDA_TRY(c, cudaEventRecord(c->ev[8], st));
  LAUNCH_TRY(c, launch_k10_loopers(L, nt, c->NS, c->o_sector.as<int>(), c->o_x.as<float>(), c->o_par.as<float>(), c->l_sec.as<int>(), c->l_list.as<int>(),
                                   c->l_prev.as<int>(), c->l_prev_n.as<int>(), c->l_root.as<int>(), c->l_turn.as<int>(), K, c->P), launches);
  CUDA_TRY(c, cudaEventRecord(c->ev[9], st));
  out->n_tracks = nt;
  if (!device_result) {
    CUDA_TRY(c, c->hl_prev.resize(ntz)); CUDA_TRY(c, c->hl_root.resize(ntz)); CUDA_TRY(c, c->hl_turn.resize(ntz));
    if (nt > 0) {
      CUDA_TRY(c, cudaMemcpyAsync(c->hl_prev.data(), c->l_prev.p, (size_t)nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hl_root.data(), c->l_root.p, (size_t)nt * 4, cudaMemcpyDeviceToHost, st));
      CUDA_TRY(c, cudaMemcpyAsync(c->hl_turn.data(), c->l_turn.p, (size_t)nt * 4, cudaMemcpyDeviceToHost, st));
    }
    out->prev = c->hl_prev.data(); out->root = c->hl_root.data(); out->turn = c->hl_turn.data();
  } else {
    out->prev = c->l_prev.as<int32_t>(); out->root = c->l_root.as<int32_t>(); out->turn = c->l_turn.as<int32_t>();
  }
  CUDA_TRY(c, cudaStreamSynchronize(st));
  CUDA_TRY(c, cudaEventElapsedTime(&out->ms_loopers, c->ev[8], c->ev[9]));
  return TPC_OK;
}
// S10 without any allocation (include/tpc.h): caller-owned device inputs / outputs, scratch in a static __device__ array of
// k10_loopers.cu, work queued on the context's stream, no synchronisation.  Needs no tpc_find_tracks* call: the constants it uses
// (cB, s_max, the loop_* tunables) are formed here from the context's field and tunables by the formulas of make_params_and_rows.
static_assert(TPC_NOALLOC_MAX_TRACKS == K10_STATIC_MAX_TRACKS, "tpc.h and tpc_internal.cuh state the same limit");
int tpc_find_loopers_noalloc(tpc_ctx* c, int64_t n_tracks, const int32_t* d_sector, const float* d_x, const float* d_par,
                             int32_t* d_prev, int32_t* d_root, int32_t* d_turn) {
  if (!c) return fail(c, TPC_E_ARG, "tpc_find_loopers_noalloc: null context");
  if (n_tracks < 0) return fail(c, TPC_E_ARG, "tpc_find_loopers_noalloc: n_tracks = %lld is negative", (long long)n_tracks);
  if (n_tracks > TPC_NOALLOC_MAX_TRACKS)
    return fail(c, TPC_E_CAPACITY, "tpc_find_loopers_noalloc: n_tracks = %lld exceeds TPC_NOALLOC_MAX_TRACKS = %d (the static scratch "
                "array holds one word per track); use tpc_find_loopers", (long long)n_tracks, (int)TPC_NOALLOC_MAX_TRACKS);
  if (c->NS > K10_STATIC_MAX_SECTORS)
    return fail(c, TPC_E_CAPACITY, "tpc_find_loopers_noalloc: %d sectors exceed the %d the static scratch array holds", c->NS, K10_STATIC_MAX_SECTORS);
  if (n_tracks == 0) return TPC_OK;
  if (!d_sector || !d_x || !d_par || !d_prev || !d_root || !d_turn) return fail(c, TPC_E_ARG, "tpc_find_loopers_noalloc: null array");
  if (pointer_kind(d_sector) != 2 || pointer_kind(d_x) != 2 || pointer_kind(d_par) != 2 || pointer_kind(d_prev) != 2 ||
      pointer_kind(d_root) != 2 || pointer_kind(d_turn) != 2)
    return fail(c, TPC_E_ARG, "tpc_find_loopers_noalloc: all six arrays must be device memory");
  int dev = -1;
  CUDA_TRY(c, cudaGetDevice(&dev));
  if (dev != c->device) return fail(c, TPC_E_STATE, "tpc_find_loopers_noalloc: current device %d is not the context's device %d", dev, c->device);
  const Tunables& T = c->T;
  const K10Params K{(float)T.loop_qmin, (float)T.loop_dy, (float)T.loop_ds, (float)T.loop_dt, (float)T.loop_dq, (float)T.loop_pmin,
                    (float)T.loop_frac, (float)6.283185307179586, T.loop_nmax};
  Params P = c->P;
  P.NS = c->NS; P.R = c->R;
  P.cB = (float)(-0.00299792458 * (double)c->bz);
  P.smax = (float)T.s_max;
  P.check = nullptr;
  const Launch L{c->stream, c->sm_count, c->T.k2_threads};
  const int rc = launch_k10_loopers_static(L, (long long)n_tracks, c->NS, d_sector, d_x, d_par, d_prev, d_root, d_turn, K, P);
  if (rc < 0) return fail(c, TPC_E_CUDA, "tpc_find_loopers_noalloc: %s", cudaGetErrorString((cudaError_t)(-rc)));
  return TPC_OK;
}
// Measurement utility: fp32 fused-multiply-add throughput of the device at the clocks of the moment (TFLOP/s, 2 flops per FMA).
int tpc_measure_fp32_peak(tpc_ctx* c, float* tflops) {
  if (!c || !tflops) return fail(c, TPC_E_ARG, "tpc_measure_fp32_peak: null argument");
  cudaStream_t st = c->stream;
  Launch L{st, c->sm_count, 0};
  CUDA_TRY(c, c->d_counters.ensure(256));
  float best = 0.f;
  for (int rep = 0; rep < 4; rep++) {           // first launch warms up; best of the next three
    CUDA_TRY(c, cudaEventRecord(c->ev[8], st));
    const long long fmas = launch_fma_peak(L, c->d_counters.as<float>() + 60, 1 << 14);
    if (fmas < 0) return fail(c, TPC_E_CUDA, "fma_peak_kernel: %s", cudaGetErrorString((cudaError_t)(-fmas)));
    CUDA_TRY(c, cudaEventRecord(c->ev[9], st));
    CUDA_TRY(c, cudaStreamSynchronize(st));
    float ms = 0.f;
    CUDA_TRY(c, cudaEventElapsedTime(&ms, c->ev[8], c->ev[9]));
    if (rep > 0 && ms > 0.f) best = std::max(best, (float)(2.0 * (double)fmas / (ms * 1e-3) / 1e12));
  }
  *tflops = best;
  return TPC_OK;
}
int tpc_get_timings(tpc_ctx* c, tpc_timings* out) {
  if (!c || !out) return fail(c, TPC_E_ARG, "tpc_get_timings: null argument");
  if (!c->have_result) return fail(c, TPC_E_STATE, "tpc_get_timings: no tpc_find_tracks call has completed");
  *out = c->timings; return TPC_OK;
}
}

// =====================================================================================================================
// Parity / debug exports: synchronous device -> host copies of intermediate tables of the last call.
extern "C" {

int tpc_debug_get_grid(tpc_ctx* c, int sector, int row, tpc_grid_view* out) {
  if (!c || !out) return fail(c, TPC_E_ARG, "tpc_debug_get_grid: null argument");
  if (!c->have_result) return fail(c, TPC_E_STATE, "tpc_debug_get_grid: call tpc_find_tracks first");
  if (sector < 0 || sector >= c->NS || row < 0 || row >= c->R) return fail(c, TPC_E_ARG, "tpc_debug_get_grid: sector/row out of range");
  const UnitDesc& d = c->h_units[(size_t)sector * c->R + row];
  const int nb = d.ny * d.nz;
  c->dbg_yz.resize((size_t)std::max(d.n, 1) * 2); c->dbg_perm.resize(std::max(d.n, 1)); c->dbg_bins.resize(nb + 1);
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (d.n) {
    CUDA_TRY(c, cudaMemcpy(c->dbg_yz.data(), c->d_yz.as<float2>() + d.off, (size_t)d.n * 8, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(c->dbg_perm.data(), c->d_perm.as<int>() + d.off, (size_t)d.n * 4, cudaMemcpyDeviceToHost));
  }
  CUDA_TRY(c, cudaMemcpy(c->dbg_bins.data(), c->d_bin_start.as<int>() + d.bin_off, (size_t)(nb + 1) * 4, cudaMemcpyDeviceToHost));
  out->n = d.n; out->ny = d.ny; out->nz = d.nz; out->y_lo = d.ylo; out->z_lo = d.zlo; out->inv_s = d.invs;
  out->yz = c->dbg_yz.data(); out->perm = c->dbg_perm.data(); out->bin_start = c->dbg_bins.data();
  return TPC_OK;
}

int tpc_debug_get_links(tpc_ctx* c, int sector, int row, int cleaned, const int32_t** up, const int32_t** dn, int32_t* n) {
  if (!c || !up || !dn || !n) return fail(c, TPC_E_ARG, "tpc_debug_get_links: null argument");
  if (!c->have_result) return fail(c, TPC_E_STATE, "tpc_debug_get_links: call tpc_find_tracks first");
  if (sector < 0 || sector >= c->NS || row < 0 || row >= c->R) return fail(c, TPC_E_ARG, "tpc_debug_get_links: sector/row out of range");
  if (!cleaned && !c->T.debug_keep) return fail(c, TPC_E_STATE, "tpc_debug_get_links: pre-cleaning tables need tpc_set_param(debug_keep, 1)");
  const UnitDesc& d = c->h_units[(size_t)sector * c->R + row];
  c->dbg_up.resize(std::max(d.n, 1)); c->dbg_dn.resize(std::max(d.n, 1));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (d.n) {
    const int* su = cleaned ? c->d_link_up.as<int>() : c->d_raw_up.as<int>();
    const int* sd = cleaned ? c->d_link_dn.as<int>() : c->d_raw_dn.as<int>();
    CUDA_TRY(c, cudaMemcpy(c->dbg_up.data(), su + d.off, (size_t)d.n * 4, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(c->dbg_dn.data(), sd + d.off, (size_t)d.n * 4, cudaMemcpyDeviceToHost));
  }
  // row distance of every link: 1, or what the S2' entries (position << 1 | k - 1) carry; 0 = no link
  c->dbg_up_k.assign(std::max(d.n, 1), 0); c->dbg_dn_k.assign(std::max(d.n, 1), 0);
  for (int i = 0; i < d.n; i++) {
    int32_t& a = c->dbg_up[i]; int32_t& b = c->dbg_dn[i];
    if (c->T.link_skip) {
      if (a >= 0) { c->dbg_up_k[i] = (int8_t)((a & 1) + 1); a >>= 1; }
      if (b >= 0) { c->dbg_dn_k[i] = (int8_t)((b & 1) + 1); b >>= 1; }
    } else { c->dbg_up_k[i] = a >= 0; c->dbg_dn_k[i] = b >= 0; }
  }
  *up = c->dbg_up.data(); *dn = c->dbg_dn.data(); *n = d.n;
  return TPC_OK;
}

int tpc_debug_get_link_rows(tpc_ctx* c, const int8_t** up_k, const int8_t** dn_k, int32_t* n) {
  if (!c || !up_k || !dn_k || !n) return fail(c, TPC_E_ARG, "tpc_debug_get_link_rows: null argument");
  if (c->dbg_up_k.empty()) return fail(c, TPC_E_STATE, "tpc_debug_get_link_rows: call tpc_debug_get_links first");
  *up_k = c->dbg_up_k.data(); *dn_k = c->dbg_dn_k.data(); *n = (int32_t)c->dbg_up.size();
  return TPC_OK;
}

int tpc_debug_get_start_hits(tpc_ctx* c, const int32_t** unit, const int32_t** pos, int64_t* n) {
  if (!c || !unit || !pos || !n) return fail(c, TPC_E_ARG, "tpc_debug_get_start_hits: null argument");
  if (!c->have_result) return fail(c, TPC_E_STATE, "tpc_debug_get_start_hits: call tpc_find_tracks first");
  c->dbg_su.resize(std::max(c->M, 1)); c->dbg_sp.resize(std::max(c->M, 1));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (c->M) {
    CUDA_TRY(c, cudaMemcpy(c->dbg_su.data(), c->d_start_unit.p, (size_t)c->M * 4, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(c->dbg_sp.data(), c->d_start_pos.p, (size_t)c->M * 4, cudaMemcpyDeviceToHost));
  }
  *unit = c->dbg_su.data(); *pos = c->dbg_sp.data(); *n = c->M;
  return TPC_OK;
}

int tpc_debug_get_tracklets(tpc_ctx* c, tpc_tracklet_view* out) {
  if (!c || !out) return fail(c, TPC_E_ARG, "tpc_debug_get_tracklets: null argument");
  if (!c->have_result) return fail(c, TPC_E_STATE, "tpc_debug_get_tracklets: call tpc_find_tracks first");
  const int M = c->M, R = c->R; const size_t Mz = std::max(M, 1);
  c->dbg_tl_sector.resize(Mz); c->dbg_tl_row.resize(Mz); c->dbg_tl_n.resize(Mz); c->dbg_tl_first.resize(Mz); c->dbg_tl_last.resize(Mz);
  c->dbg_tl_chi2.resize(Mz); c->dbg_tl_x.resize(Mz); c->dbg_tl_par.resize(Mz * 5); c->dbg_tl_cov.resize(Mz * 15); c->dbg_rowhit.assign(Mz * R, -1);
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (M) {
    std::vector<int32_t> su(M); std::vector<rowhit_t> raw((size_t)c->Mpad * R);
    CUDA_TRY(c, cudaMemcpy(su.data(), c->d_start_unit.p, (size_t)M * 4, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(c->dbg_tl_n.data(), c->d_tl_n.p, (size_t)M * 4, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(c->dbg_tl_first.data(), c->d_tl_first.p, (size_t)M * 4, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(c->dbg_tl_last.data(), c->d_tl_last.p, (size_t)M * 4, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(c->dbg_tl_chi2.data(), c->d_tl_chi2.p, (size_t)M * 4, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(c->dbg_tl_par.data(), c->d_tl_par.p, (size_t)M * 20, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(c->dbg_tl_cov.data(), c->d_tl_cov.p, (size_t)M * 60, cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(raw.data(), c->d_rowhit.p, raw.size() * sizeof(rowhit_t), cudaMemcpyDeviceToHost));
    for (int i = 0; i < M; i++) {
      c->dbg_tl_sector[i] = su[i] / R; c->dbg_tl_row[i] = su[i] % R; const int f = c->dbg_tl_first[i];
      c->dbg_tl_x[i] = f >= 0 && f < R ? c->row_x[f] : 0.0f;   // tracklets the rescue variant did not fit carry first = last = -1
      for (int r = std::max(f, 0); f >= 0 && r <= c->dbg_tl_last[i] && r < R; r++) c->dbg_rowhit[(size_t)r * M + i] = raw[(size_t)i * R + r];
    }
  }
  out->n_tracklets = M; out->sector = c->dbg_tl_sector.data(); out->start_row = c->dbg_tl_row.data(); out->n_hits = c->dbg_tl_n.data();
  out->first_row = c->dbg_tl_first.data(); out->last_row = c->dbg_tl_last.data(); out->chi2 = c->dbg_tl_chi2.data(); out->x = c->dbg_tl_x.data();
  out->par = c->dbg_tl_par.data(); out->cov = c->dbg_tl_cov.data(); out->rowhit = c->dbg_rowhit.data();
  return TPC_OK;
}

}  // extern "C"
