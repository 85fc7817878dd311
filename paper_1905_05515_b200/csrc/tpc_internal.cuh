// tpc_internal.cuh -- shared declarations of the CUDA path (context layout, per-row / per-unit tables, device helpers).
// Product code: shares nothing with oracle/.  Definitions follow DESIGN.md section 4 (S0..S6).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tpc {

// entry of the rowhit table [tracklet][row]: sorted position of the tracklet's cluster on that row, -1 = none
#ifdef TPC_ROWHIT16
typedef short rowhit_t;
#else
typedef int rowhit_t;
#endif

// Per-row constants, computed on the host in double and rounded once to float ("per-row constants").
struct RowConst {
  float x;       // local x of the row
  float tu, td;  // x_{r+1}/x_r, x_{r-1}/x_r : from-origin projection factors
  float a, b;    // x_{r+1}-x_r, x_r-x_{r-1}
  float thr;     // cut2 * 0.5 * (a^2+b^2)
  float wzu, wzd;// continuous-mode z half-widths up / down
  float yedge;   // x_r * tan(dphi/2)
  // S2' (link_skip, reading A45): the same constants for a row distance of 2, and the acceptance limits of the pairs
  // (k_u, k_d) = (2,1), (1,2), (2,2): cut2 * 0.5 * (a_ku^2 + b_kd^2)
  float tu2, td2, a2, b2, wzu2, wzd2, thr21, thr12, thr22;
  float pad[6];
};
static_assert(sizeof(RowConst) == 96, "RowConst layout");

// One (sector,row) unit: where its clusters come from, where its sorted copy lives, and its S1 grid.
struct UnitDesc {
  long long off;      // offset of the unit in the sorted arrays (CSR over units)
  long long src;      // offset of the unit's clusters in the input arena
  long long bin_off;  // offset of the unit's bin_start table (ny*nz+1 entries)
  long long cur_off;  // K1: offset into the global cursor scratch, or -1 when the cursors fit shared memory
  int n, ny, nz;
  float ylo, zlo, invs;
  int pad[2];
};

// Scalar parameters passed by value to every kernel (table T of DESIGN.md, rounded to float exactly once on the host).
struct Params {
  int NS, R, continuous;
  float zmax, vdrift;             // S0
  float wy, wz;                   // S2
  int min_seed;                   // S4
  float cB;                       // curvature constant -0.00299792458*Bz
  float c0[5];                    // S5 initial covariance diagonal
  float ry, rz;                   // sigma_y^2, sigma_z^2
  float smax, nsigma, wmax, edge_margin;
  int max_gap, min_hits;
  int bridge_rows, bridge_min;    // NEXT-2 seed bridging (reading A39); bridge_rows = 0: off
  float bridge_wy, bridge_wz;
  int* check;                     // TPC_CHECKED builds: device word that receives the code of a failed bounds check (else unused)
  int link_skip;                  // NEXT-2 as SURVEY 8(f).2 wrote it (reading A45): 1 = links may skip one row; link tables then hold (position << 1 | k - 1)
};

// S9 (NEXT-3) matching parameters (reading A41), rounded to float once on the host
struct K9Params { float edge, dy, dz, ds, dt, cd, sd; int rows;
                  int per_side; };   // sectors per closed ring in phi (18 for 20 degree sectors); 0 = the sectors do not close a ring: nothing to merge

// S10 (NEXT-3, second half) parameters (reading A46), rounded to float once on the host
struct K10Params { float qmin, dy, ds, dt, dq, pmin, frac, twopi; int nmax; };
constexpr int K10_STATIC_MAX_TRACKS = 262144;   // limits of the allocation-free S10 entry point (= TPC_NOALLOC_MAX_TRACKS of tpc.h)
constexpr int K10_STATIC_MAX_SECTORS = 1022;

// Work item of K2/K3: a chunk of consecutive sorted hits of one unit.
struct Item { int unit; int start; };

// Bounds checks of the checked build (libtpc_b200_checked.so, -DTPC_CHECKED; compute-sanitizer is closed on the GPU pool, so the
// library carries its own): every gather / scatter index that is computed from data is tested against the size of its array; a
// failed test leaves its code in *P.check, which tpc_find_tracks* turns into TPC_E_CUDA.  Compiled out of the product build.
#ifdef TPC_CHECKED
#define TPC_CHECK(P, cond, code) do { if (!(cond)) atomicMax((P).check, (code)); } while (0)
#else
#define TPC_CHECK(P, cond, code) ((void)0)
#endif

// ---- device helpers ------------------------------------------------------------------------------------------------
// S1 bin of a coordinate: fp32 subtract, fp32 multiply (no FMA), negative / NaN -> 0, clamp to nb-1, truncate.
// (fmaxf(NaN, 0) = 0; clamping before the truncation gives the same integer as truncating first: nb-1 < 2^24 is exact in fp32.)
__device__ __forceinline__ int bin_of(float v, float lo, float inv, int nb) {
  const float f = __fmul_rn(__fsub_rn(v, lo), inv);
  return __float2int_rz(fminf(fmaxf(f, 0.0f), (float)(nb - 1)));
}

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { int t = __shfl_up_sync(0xffffffffu, v, d); if (lane >= d) v += t; }
  return v;
}

// Exclusive scan of one value per thread over the block (blockDim.x multiple of 32, <= 1024).  s_warp: 33 ints of shared memory.
// Returns the exclusive prefix; *total receives the block total.  Contains three __syncthreads.
__device__ __forceinline__ int block_excl_scan(int v, int* s_warp, int* total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  int inc = warp_incl_scan(v, lane);
  if (lane == 31) s_warp[w] = inc;
  __syncthreads();
  if (w == 0) {
    int t = lane < nw ? s_warp[lane] : 0;
    int ti = warp_incl_scan(t, lane);
    s_warp[lane] = ti - t;
    if (lane == 31) s_warp[32] = ti;
  }
  __syncthreads();
  int res = inc - v + s_warp[w];
  *total = s_warp[32];
  __syncthreads();   // s_warp may be reused right away by the caller's next round
  return res;
}

// ---- kernel launchers (one per step; each returns the number of kernels it launched, or a negative cudaError) --------
struct Launch {
  cudaStream_t stream;
  int sm_count;
  int k2_threads;   // 0 = default
};

int launch_k1_grid(const Launch& L, int U, const UnitDesc* d_units, const float* d_in_y, const float* d_in_t, float2* d_yz,
                   int* d_perm, int* d_bin_start, int* d_cursor, const Params& P, int max_cursor_ints_smem, int max_n,
                   int max_perm_ints, int max_yz_ints);

int launch_k2_neighbours(const Launch& L, int n_items, const Item* d_items, int chunk, const UnitDesc* d_units,
                         const RowConst* d_rows, const float2* d_yz, const int* d_perm, const int* d_bin_start, int* d_link_up,
                         int* d_link_dn, const Params& P);

// S2' (link_skip = 1): re-encodes the S2 links as (position << 1 | 0) and gives the hits S2 left unlinked a link that may skip a row
int launch_k2_skip_links(const Launch& L, int n_items, const Item* d_items, int chunk, const UnitDesc* d_units, const RowConst* d_rows,
                         const float2* d_yz, const int* d_perm, const int* d_bin_start, int* d_link_up, int* d_link_dn, const Params& P);

int launch_k3_bridge(const Launch& L, int M, const int* d_start_unit, const int* d_start_pos, const UnitDesc* d_units,
                     const RowConst* d_rows, const float2* d_yz, const int* d_bin_start, const int* d_link_up, const int* d_link_dn,
                     int* d_keep, int* d_keep_pos, int* d_scan_tmp, int* d_out_unit, int* d_out_pos, int* d_total, const Params& P);

int launch_k3_bridge_lists(const Launch& L, int M, const int* d_start_unit, const int* d_start_pos, const UnitDesc* d_units,
                           const RowConst* d_rows, const float2* d_yz, const int* d_bin_start, const int* d_link_up, const int* d_link_dn,
                           int* d_keep, int* d_pos, int* d_scan_tmp, int* d_list1, int* d_total, const Params& P);
int launch_k3_rescue_list(const Launch& L, int M, const int* d_keep, const int* d_start_unit, const int* d_start_pos,
                          const UnitDesc* d_units, const int* d_link_up, const unsigned long long* d_owner,
                          int* d_flag2, int* d_pos, int* d_scan_tmp, int* d_list2, int* d_total);

int launch_k3_clean_start(const Launch& L, int n_items, const Item* d_items, int chunk, const UnitDesc* d_units, int* d_link_up,
                          int* d_link_dn, unsigned* d_mask, int* d_item_count, int* d_item_base, int* d_scan_tmp,
                          int* d_start_unit, int* d_start_pos, int* d_total, const Params& P);

size_t k5_scratch_bytes(long long M);   // handoff records + task lists + control block of the K5 phase kernels
int launch_k5_tracklets(const Launch& L, int n_run, const int* d_n_run, int M, const int* d_run_list, const int* d_start_unit, const int* d_start_pos,
                        const UnitDesc* d_units, const RowConst* d_rows, const float2* d_yz, const int* d_perm, const int* d_bin_start,
                        const int* d_link_up, rowhit_t* d_rowhit, int* d_tl_n, int* d_tl_first, int* d_tl_last, float* d_tl_chi2,
                        float* d_tl_par, float* d_tl_cov, unsigned long long* d_counters, void* d_scratch, const Params& P);

int launch_k6_select(const Launch& L, int M_cap, const int* d_M, long long N, const int* d_start_unit, const UnitDesc* d_units,
                     const rowhit_t* d_rowhit, const int* d_tl_n, const int* d_tl_first,
                     const int* d_tl_last, const float* d_tl_chi2, unsigned long long* d_owner, unsigned long long* d_tl_key,
                     unsigned long long* d_scan_in, unsigned long long* d_scan_out, unsigned long long* d_scan_tmp,
                     unsigned long long* d_total, const Params& P, bool owner_done);
int launch_k6_owner(const Launch& L, int n_run, const int* d_run_list, const int* d_start_unit, const UnitDesc* d_units, const rowhit_t* d_rowhit,
                    const int* d_tl_n, const int* d_tl_first, const int* d_tl_last, const float* d_tl_chi2, unsigned long long* d_owner,
                    unsigned long long* d_tl_key, const Params& P);

int launch_k6_emit(const Launch& L, int M_cap, const int* d_M, const int* d_start_unit, const UnitDesc* d_units, const RowConst* d_rows,
                   const int* d_perm, const rowhit_t* d_rowhit, const int* d_tl_n, const int* d_tl_first, const int* d_tl_last,
                   const float* d_tl_chi2, const float* d_tl_par, const float* d_tl_cov, const unsigned long long* d_owner,
                   const unsigned long long* d_tl_key, const unsigned long long* d_scan_in, const unsigned long long* d_scan_out,
                   int* o_sector, float* o_x, float* o_par, float* o_cov, float* o_chi2, int* o_ndf, int* o_tracklet,
                   long long* o_cl_begin, int* o_cl_row, int* o_cl_index, const unsigned long long* d_total, long long cap_tracks,
                   long long cap_refs, const Params& P);

int launch_k7_refit(const Launch& L, long long n_tracks, const int* o_sector, const int* o_tracklet, const long long* o_cl_begin,
                    const int* o_cl_row, const UnitDesc* d_units, const RowConst* d_rows, const float2* d_yz, const rowhit_t* d_rowhit,
                    int* rf_n, int* rf_ndf, float* rf_x, float* rf_par, float* rf_cov, float* rf_chi2, float* rf_z0, float* rf_t0,
                    int* d_order, int* d_classes /* 768 ints */, const Params& P);

int launch_k8_status(const Launch& L, long long n_tracks, long long N, int U, const int* o_sector, const int* o_tracklet,
                     const float* o_par, const long long* o_cl_begin, const int* o_cl_row, const int* d_tl_first,
                     const UnitDesc* d_units, const RowConst* d_rows, const float2* d_yz, const int* d_perm, const int* d_bin_start,
                     const rowhit_t* d_rowhit, int* d_att, unsigned long long* d_adj, float2* d_path, int* d_path_end, int* cl_status, int* cl_track, float tube,
                     const Params& P);

int launch_k9_merge(const Launch& L, long long n_tracks, int NS, const int* o_sector, const int* o_tracklet, const float* o_par,
                    const long long* o_cl_begin, const int* o_cl_row, const int* d_tl_first, const RowConst* d_rows, float* d_outer,
                    int* d_row_in, int* d_row_out, int* d_leaver, int* d_sec_begin, int* d_list, int* d_blist, int* d_bucket,
                    unsigned long long* d_cand, int* d_next, int* d_prev, const K9Params& M, const Params& P);

int launch_k10_loopers(const Launch& L, long long n_tracks, int NS, const int* o_sector, const float* o_x, const float* o_par,
                       int* d_sec, int* d_list, int* d_prev, int* d_prev_n, int* d_root, int* d_turn, const K10Params& K, const Params& P);
// allocation-free variant: scratch in a file-scope __device__ array of k10_loopers.cu, limits below (tpc_find_loopers_noalloc)
int launch_k10_loopers_static(const Launch& L, long long n_tracks, int NS, const int* o_sector, const float* o_x, const float* o_par,
                              int* d_prev, int* d_root, int* d_turn, const K10Params& K, const Params& P);

// device-wide exclusive scans (own kernels; three launches each)
int launch_scan_i32(const Launch& L, const int* d_in, int* d_out, int n, int* d_tmp, int* d_total);
int launch_scan_u64(const Launch& L, const unsigned long long* d_in, unsigned long long* d_out, int n, unsigned long long* d_tmp,
                    unsigned long long* d_total);
long long launch_fma_peak(const Launch& L, float* d_out, int iters);   // measurement utility (scan.cu)
constexpr int SCAN_TILE = 4096;   // elements per CTA in the scans; tmp needs ceil(n/SCAN_TILE)+1 entries

}  // namespace tpc
