// k6_selector.cu -- K6: S6 tracklet selector, resolves shared clusters (BASELINE north_star; definition in DESIGN.md section 4).
//
// Every cluster referenced by a kept tracklet (n >= min_hits, finite chi2) goes to the tracklet with the maximum key
// (n, -chi2/ndf, -tracklet index).  The key is packed into 64 bits so that one atomicMax per reference resolves the owner:
//   bits 63..56  n (<= 255 rows)
//   bits 55..24  bitwise NOT of the order-preserving image of the fp32 quality chi2/ndf (lower quality wins)
//   bits 23..0   0xFFFFFF - tracklet index (lower index wins)                       -> at most 2^24 tracklets per call
// One warp per tracklet in all three kernels (grid-stride over the tracklets: the tracklet count may live in device memory, so
// that the host does not have to read it back between K3 and K6).
// k6_owner : atomicMax of the key on owner[cluster]          k6_count : owned clusters per tracklet, track flag
// scan     : exclusive prefix sum of (flag << 40 | owned)     k6_emit  : compacted tracks + CSR cluster lists, in tracklet order
#include "tpc_internal.cuh"

namespace tpc {
namespace {

struct CheckOnly { int* check; };   // the K6 kernels take no Params: TPC_CHECK needs only the flag word

constexpr int K6_THREADS = 128;
constexpr int K6_PER_BLOCK = 32;   // consecutive tracklets per CTA: the CTAs are scheduled in launch order, so the tracklets in flight at any
                                   // time are neighbours in (sector, row) order and their owner keys share a small, L2-resident region
constexpr unsigned long long REF_MASK = (1ull << 40) - 1ull;

__device__ __forceinline__ unsigned long long make_key(int n, float chi2, int idx) {
  const float q = chi2 / (float)(2 * n - 5);
  unsigned b = __float_as_uint(q);
  b = (b & 0x80000000u) ? ~b : (b | 0x80000000u);   // monotone map float -> unsigned
  return ((unsigned long long)(unsigned)n << 56) | ((unsigned long long)(~b) << 24) | (unsigned long long)(0xFFFFFFu - (unsigned)idx);
}

// All three kernels map ONE WARP to one tracklet: the lanes read 32 consecutive rows of its rowhit line (coalesced) and issue
// their owner-key atomics / owner reads in parallel.
__global__ void __launch_bounds__(K6_THREADS) k6_owner(const int M_cap, const int* __restrict__ M_dev, const int* __restrict__ run_list, const int R, const int min_hits,
                                                       const int* __restrict__ start_unit, const UnitDesc* __restrict__ units,
                                                       const rowhit_t* __restrict__ rowhit, const int* __restrict__ tl_n,
                                                       const int* __restrict__ tl_first, const int* __restrict__ tl_last,
                                                       const float* __restrict__ tl_chi2, unsigned long long* __restrict__ owner,
                                                       unsigned long long* __restrict__ tl_key, const CheckOnly C) {
  const int lane = threadIdx.x & 31, n_warps = K6_THREADS >> 5;
  const int M = M_dev ? min(*M_dev, M_cap) : M_cap;
  const long long q1 = min((long long)M, ((long long)blockIdx.x + 1) * K6_PER_BLOCK);
  for (long long qq = (long long)blockIdx.x * K6_PER_BLOCK + (threadIdx.x >> 5); qq < q1; qq += n_warps) {
  const int q = (int)qq;
  const int i = run_list ? run_list[q] : q;   // M entries of a run list (rescue variant), or all tracklets
  const int n = tl_n[i];
  const float chi2 = tl_chi2[i];
  const int u0 = start_unit[i], r_lo = tl_first[i], r1 = tl_last[i];   // read with n and chi2, not after the decision they feed
  const bool kept = n >= min_hits && isfinite(chi2);
  const unsigned long long key = kept ? make_key(n, chi2, i) : 0ull;
  if (lane == 0) tl_key[i] = key;
  if (!kept) continue;
  const UnitDesc* __restrict__ su = units + (long long)(u0 / R) * R;
  const rowhit_t* __restrict__ rh = rowhit + (long long)i * R;
  for (int r = r_lo + lane; r <= r1; r += 32) {
    const int p = rh[r];
    TPC_CHECK(C, p < su[r].n && r < R, 61);
    if (p >= 0) atomicMax(&owner[su[r].off + p], key);
  }
  }
}

__global__ void __launch_bounds__(K6_THREADS) k6_count(const int M_cap, const int* __restrict__ M_dev, const int R, const int min_hits,
                                                       const int* __restrict__ start_unit, const UnitDesc* __restrict__ units,
                                                       const rowhit_t* __restrict__ rowhit, const int* __restrict__ tl_first,
                                                       const int* __restrict__ tl_last, const unsigned long long* __restrict__ owner,
                                                       const unsigned long long* __restrict__ tl_key,
                                                       unsigned long long* __restrict__ scan_in, const CheckOnly C) {
  const int lane = threadIdx.x & 31, n_warps = K6_THREADS >> 5;
  const int M = M_dev ? min(*M_dev, M_cap) : M_cap;
  const long long i1 = min((long long)M_cap, ((long long)blockIdx.x + 1) * K6_PER_BLOCK);
  for (long long ii = (long long)blockIdx.x * K6_PER_BLOCK + (threadIdx.x >> 5); ii < i1; ii += n_warps) {
  const int i = (int)ii;
  if (i >= M) { if (lane == 0) scan_in[i] = 0ull; continue; }   // the scan runs over the capacity: entries beyond the count are 0
  const unsigned long long key = tl_key[i];
  const int u0 = start_unit[i], r_lo = tl_first[i], r1 = tl_last[i];     // read with the key, not after the decision it feeds
  int owned = 0;
  if (key) {
    const UnitDesc* __restrict__ su = units + (long long)(u0 / R) * R;
    const rowhit_t* __restrict__ rh = rowhit + (long long)i * R;
    for (int r = r_lo + lane; r <= r1; r += 32) {
      const int p = rh[r];
      TPC_CHECK(C, p < su[r].n && r < R, 62);
      if (p >= 0 && owner[su[r].off + p] == key) owned++;
    }
  }
  owned = __reduce_add_sync(0xffffffffu, owned);
  if (lane == 0) scan_in[i] = owned >= min_hits && key ? ((1ull << 40) | (unsigned long long)owned) : 0ull;
  }
}

__global__ void __launch_bounds__(K6_THREADS) k6_emit(const int M_cap, const int* __restrict__ M_dev, const int R, const int* __restrict__ start_unit,
                                                      const UnitDesc* __restrict__ units, const RowConst* __restrict__ rows,
                                                      const int* __restrict__ perm, const rowhit_t* __restrict__ rowhit,
                                                      const int* __restrict__ tl_n, const int* __restrict__ tl_first,
                                                      const int* __restrict__ tl_last, const float* __restrict__ tl_chi2,
                                                      const float* __restrict__ tl_par, const float* __restrict__ tl_cov,
                                                      const unsigned long long* __restrict__ owner,
                                                      const unsigned long long* __restrict__ tl_key,
                                                      const unsigned long long* __restrict__ scan_in,
                                                      const unsigned long long* __restrict__ scan_out, int* __restrict__ o_sector,
                                                      float* __restrict__ o_x, float* __restrict__ o_par, float* __restrict__ o_cov,
                                                      float* __restrict__ o_chi2, int* __restrict__ o_ndf, int* __restrict__ o_tracklet,
                                                      long long* __restrict__ o_cl_begin, int* __restrict__ o_cl_row,
                                                      int* __restrict__ o_cl_index, const unsigned long long* __restrict__ total,
                                                      const long long cap_tracks, const long long cap_refs, const CheckOnly C) {
  const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31, n_warps = K6_THREADS >> 5;
  const unsigned long long tot = *total;                       // (tracks << 40 | cluster references) of the scan
  const long long n_tracks = (long long)(tot >> 40), n_refs = (long long)(tot & REF_MASK);
  if (n_tracks > cap_tracks || n_refs > cap_refs) return;      // the caller sees the totals and repeats the call with larger buffers
  if (gt == 0) o_cl_begin[n_tracks] = n_refs;
  const int M = M_dev ? min(*M_dev, M_cap) : M_cap;
  const long long i1 = min((long long)M, ((long long)blockIdx.x + 1) * K6_PER_BLOCK);
  for (long long ii = (long long)blockIdx.x * K6_PER_BLOCK + (threadIdx.x >> 5); ii < i1; ii += n_warps) {
  const int i = (int)ii;
  if (scan_in[i] == 0ull) continue;
  const unsigned long long so = scan_out[i];
  const long long t = (long long)(so >> 40);
  long long k = (long long)(so & REF_MASK);
  const int sec = start_unit[i] / R;
  const UnitDesc* __restrict__ su = units + (long long)sec * R;
  const rowhit_t* __restrict__ rh = rowhit + (long long)i * R;
  const unsigned long long key = tl_key[i];
  const int r0 = tl_first[i], r1 = tl_last[i];
  if (lane == 0) {
    o_sector[t] = sec; o_x[t] = rows[r0].x; o_chi2[t] = tl_chi2[i]; o_ndf[t] = 2 * tl_n[i] - 5; o_tracklet[t] = i; o_cl_begin[t] = k;
  }
  if (lane < 5) o_par[t * 5 + lane] = tl_par[(long long)i * 5 + lane];
  if (lane < 15) o_cov[t * 15 + lane] = tl_cov[(long long)i * 15 + lane];
  for (int rb = r0; rb <= r1; rb += 32) {       // ascending rows: ballot + prefix popcount keeps the list ordered
    const int r = rb + lane;
    long long g = 0;
    bool own = false;
    if (r <= r1) { const int p = rh[r]; if (p >= 0) { g = su[r].off + p; own = owner[g] == key; } }
    const unsigned m = __ballot_sync(0xffffffffu, own);
    if (own) { const long long o = k + __popc(m & ((1u << lane) - 1u)); TPC_CHECK(C, o >= 0 && o < n_refs && t < n_tracks, 63); o_cl_row[o] = r; o_cl_index[o] = perm[g]; }
    k += __popc(m);
  }
  }
}

}  // namespace

// grid of the warp-per-tracklet kernels: one CTA per K6_PER_BLOCK consecutive tracklets of the capacity (CTAs beyond the count exit)
static int k6_blocks(const Launch& L, long long M) {
  (void)L;
  const long long want = (M + K6_PER_BLOCK - 1) / K6_PER_BLOCK;
  return (int)(want < 1 ? 1 : want);
}

// d_M: tracklet count in device memory (or nullptr: M_cap is the count); M_cap: capacity of the per-tracklet arrays
int launch_k6_select(const Launch& L, int M_cap, const int* d_M, long long N, const int* d_start_unit, const UnitDesc* d_units,
                     const rowhit_t* d_rowhit, const int* d_tl_n, const int* d_tl_first,
                     const int* d_tl_last, const float* d_tl_chi2, unsigned long long* d_owner, unsigned long long* d_tl_key,
                     unsigned long long* d_scan_in, unsigned long long* d_scan_out, unsigned long long* d_scan_tmp,
                     unsigned long long* d_total, const Params& P, bool owner_done) {
  if (M_cap <= 0) {
    cudaError_t e = cudaMemsetAsync(d_total, 0, sizeof(unsigned long long), L.stream);
    return e == cudaSuccess ? 0 : -(int)e;
  }
  cudaError_t e = cudaSuccess;
  const int blocks = k6_blocks(L, M_cap);
  if (!owner_done) {   // (the rescue variant raised the owner keys wave by wave: launch_k6_owner)
    e = cudaMemsetAsync(d_owner, 0, (size_t)N * sizeof(unsigned long long), L.stream);
    if (e != cudaSuccess) return -(int)e;
    k6_owner<<<blocks, K6_THREADS, 0, L.stream>>>(M_cap, d_M, nullptr, P.R, P.min_hits, d_start_unit, d_units, d_rowhit, d_tl_n, d_tl_first,
                                                   d_tl_last, d_tl_chi2, d_owner, d_tl_key, CheckOnly{P.check});
  }
  k6_count<<<blocks, K6_THREADS, 0, L.stream>>>(M_cap, d_M, P.R, P.min_hits, d_start_unit, d_units, d_rowhit, d_tl_first, d_tl_last, d_owner,
                                                 d_tl_key, d_scan_in, CheckOnly{P.check});
  int rc = launch_scan_u64(L, d_scan_in, d_scan_out, M_cap, d_scan_tmp, d_total);
  if (rc < 0) return rc;
  e = cudaGetLastError();
  return e == cudaSuccess ? (owner_done ? 1 : 2) + rc : -(int)e;
}

// owner keys of the n_run tracklets of a run list (rescue variant: one call per K5 wave; the caller zeroes d_owner and d_tl_key first)
int launch_k6_owner(const Launch& L, int n_run, const int* d_run_list, const int* d_start_unit, const UnitDesc* d_units, const rowhit_t* d_rowhit,
                    const int* d_tl_n, const int* d_tl_first, const int* d_tl_last, const float* d_tl_chi2, unsigned long long* d_owner,
                    unsigned long long* d_tl_key, const Params& P) {
  if (n_run <= 0) return 0;
  k6_owner<<<k6_blocks(L, n_run), K6_THREADS, 0, L.stream>>>(n_run, nullptr, d_run_list, P.R, P.min_hits, d_start_unit, d_units, d_rowhit, d_tl_n,
                                                              d_tl_first, d_tl_last, d_tl_chi2, d_owner, d_tl_key, CheckOnly{P.check});
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 1 : -(int)e;
}

// d_total: (tracks << 40 | references) written by the scan; the output arrays hold cap_tracks tracks / cap_refs references
int launch_k6_emit(const Launch& L, int M_cap, const int* d_M, const int* d_start_unit, const UnitDesc* d_units, const RowConst* d_rows,
                   const int* d_perm, const rowhit_t* d_rowhit, const int* d_tl_n, const int* d_tl_first, const int* d_tl_last,
                   const float* d_tl_chi2, const float* d_tl_par, const float* d_tl_cov, const unsigned long long* d_owner,
                   const unsigned long long* d_tl_key, const unsigned long long* d_scan_in, const unsigned long long* d_scan_out,
                   int* o_sector, float* o_x, float* o_par, float* o_cov, float* o_chi2, int* o_ndf, int* o_tracklet,
                   long long* o_cl_begin, int* o_cl_row, int* o_cl_index, const unsigned long long* d_total, long long cap_tracks,
                   long long cap_refs, const Params& P) {
  k6_emit<<<k6_blocks(L, M_cap), K6_THREADS, 0, L.stream>>>(M_cap, d_M, P.R, d_start_unit, d_units, d_rows, d_perm, d_rowhit, d_tl_n, d_tl_first,
                                                             d_tl_last, d_tl_chi2, d_tl_par, d_tl_cov, d_owner, d_tl_key, d_scan_in, d_scan_out,
                                                             o_sector, o_x, o_par, o_cov, o_chi2, o_ndf, o_tracklet, o_cl_begin, o_cl_row,
                                                             o_cl_index, d_total, cap_tracks, cap_refs, CheckOnly{P.check});
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 1 : -(int)e;
}

}  // namespace tpc
