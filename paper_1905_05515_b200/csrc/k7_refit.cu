// k7_refit.cu -- K7: S7 refit after the selection and collision-time estimate (NEXT-1 of SURVEY.md section 8(f);
// PAPER.md:30 "first preliminary fit ... improve the z-estimation"; readings A37 / A38 of DESIGN.md).
//
// Per output track of S6, over the clusters the track OWNS (ascending row): pass 1 outward from the innermost owned cluster
// (direction from the origin; covariance C0), one exact-helix transport per owned cluster; pass 2 inward from the
// outermost cluster reached with a fresh C0 -> state, covariance, chi2, n, ndf = 2n - 5 at the innermost cluster used.  The
// collision time follows from the extrapolation of that state to the beam line: z0 = z - (dz/ds) * arc, t0 = -z0 / vdrift.
//
// One lane per track, the tracks taken in the order of their length (longest first); the fp32 state lives in registers (same transport / update code as K5, kalman.cuh).  The cluster
// coordinates are fetched through the tracklet's rowhit line and the sorted (y, z) array: the next cluster's row and position
// are read one step ahead of the transport that needs them.
#include "kalman.cuh"

namespace tpc {
namespace {

constexpr int K7_THREADS = 128;
constexpr int K7_CLASSES = 256;   // length classes of the ordering: clusters of a track (at most one per row, n_rows <= 255)

// Tracks ordered by their number of clusters, longest first (counting sort: k7_count, k7_starts, k7_fill): k7_refit runs one
// track per lane from start to end, so a warp takes as long as its longest track; with equally long tracks side by side the lanes
// of a warp finish together.  The order inside a length class is arbitrary and enters no result.
__global__ void __launch_bounds__(256) k7_count(const long long n_tracks, const long long* __restrict__ cl_begin, int* __restrict__ count) {
  __shared__ int s_cnt[K7_CLASSES];   // histogram of the CTA first: most tracks fall into a few classes, global atomics on them would serialise
  s_cnt[threadIdx.x] = 0;
  __syncthreads();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_tracks) atomicAdd(&s_cnt[min((int)(cl_begin[i + 1] - cl_begin[i]), K7_CLASSES - 1)], 1);
  __syncthreads();
  if (s_cnt[threadIdx.x]) atomicAdd(&count[threadIdx.x], s_cnt[threadIdx.x]);
}
__global__ void k7_starts(const int* __restrict__ count, int* __restrict__ start) {   // one thread: K7_CLASSES entries, longest class first
  int acc = 0;
  for (int m = K7_CLASSES - 1; m >= 0; m--) { start[m] = acc; acc += count[m]; }
}
__global__ void __launch_bounds__(256) k7_fill(const long long n_tracks, const long long* __restrict__ cl_begin, const int* __restrict__ start,
                                               int* __restrict__ fill, int* __restrict__ order) {
  __shared__ int s_cnt[K7_CLASSES], s_base[K7_CLASSES];
  s_cnt[threadIdx.x] = 0;
  __syncthreads();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int m = 0, rank = 0;
  if (i < n_tracks) { m = min((int)(cl_begin[i + 1] - cl_begin[i]), K7_CLASSES - 1); rank = atomicAdd(&s_cnt[m], 1); }
  __syncthreads();
  if (s_cnt[threadIdx.x]) s_base[threadIdx.x] = start[threadIdx.x] + atomicAdd(&fill[threadIdx.x], s_cnt[threadIdx.x]);   // one range per class and CTA
  __syncthreads();
  if (i < n_tracks) order[s_base[m] + rank] = (int)i;
}

__global__ void __launch_bounds__(K7_THREADS) k7_refit(const long long n_tracks, const int* __restrict__ order, const int* __restrict__ o_sector,
                                                       const int* __restrict__ o_tracklet, const long long* __restrict__ cl_begin,
                                                       const int* __restrict__ cl_row, const UnitDesc* __restrict__ units,
                                                       const RowConst* __restrict__ rows, const float2* __restrict__ yz,
                                                       const rowhit_t* __restrict__ rowhit, int* __restrict__ rf_n, int* __restrict__ rf_ndf,
                                                       float* __restrict__ rf_x, float* __restrict__ rf_par, float* __restrict__ rf_cov,
                                                       float* __restrict__ rf_chi2, float* __restrict__ rf_z0, float* __restrict__ rf_t0,
                                                       const Params P) {
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_tracks) return;
  const long long i = order[j];
  const int R = P.R;
  const long long a = cl_begin[i];
  const int m = (int)(cl_begin[i + 1] - a);
  const UnitDesc* __restrict__ su = units + (long long)o_sector[i] * R;
  const rowhit_t* __restrict__ rh = rowhit + (long long)o_tracklet[i] * R;
  const int* __restrict__ cr = cl_row + a;
  auto cluster = [&](const int row) { return yz[su[row].off + rh[row]]; };

  // pass 1: outward
  int row = cr[0];
  float2 c = cluster(row);
  const float zref = c.y;
  State st;
  {
    const float x = rows[row].x, y = c.x;
    const float rr = sqrtf(x * x + y * y);
    st.y = y; st.z = 0.0f; st.s = y / rr; st.t = P.continuous ? 0.0f : zref / rr; st.q = 0.0f;
    reset_cov(st, P);
  }
  update(st, c.x, 0.0f, P);
  int last = 0;
  {
    int row_n = m > 1 ? cr[1] : row;
    float2 c_n = cluster(row_n);
    for (int k = 1; k < m; k++) {
      const int row_k = row_n;
      const float2 c_k = c_n;
      if (k + 1 < m) { row_n = cr[k + 1]; c_n = cluster(row_n); }   // next cluster, loaded ahead of this step's arithmetic
      if (!propagate(st, rows[row_k].x - rows[row].x, P)) break;
      update(st, c_k.x, c_k.y - zref, P);
      row = row_k; c = c_k; last = k;
    }
  }
  // pass 2: inward from the outermost cluster reached (row, c)
  reset_cov(st, P);
  float chi2 = update(st, c.x, c.y - zref, P);
  int n = 1;
  State snap = st;
  int row_in = row;
  {
    int row_n = last > 0 ? cr[last - 1] : row;
    float2 c_n = cluster(row_n);
    for (int k = last - 1; k >= 0; k--) {
      const int row_k = row_n;
      const float2 c_k = c_n;
      if (k > 0) { row_n = cr[k - 1]; c_n = cluster(row_n); }
      if (!propagate(st, rows[row_k].x - rows[row].x, P)) break;
      chi2 = chi2 + update(st, c_k.x, c_k.y - zref, P);
      n++; snap = st; row = row_k; row_in = row_k;
    }
  }
  const float x_in = rows[row_in].x;
  const float zabs = snap.z + zref;
  rf_n[i] = n; rf_ndf[i] = 2 * n - 5; rf_chi2[i] = chi2; rf_x[i] = x_in;
  float* __restrict__ op = rf_par + i * 5;
  op[0] = snap.y; op[1] = zabs; op[2] = snap.s; op[3] = snap.t; op[4] = snap.q;
  float* __restrict__ oc = rf_cov + i * 15;
  oc[0] = snap.c00; oc[1] = snap.c10; oc[2] = snap.c11; oc[3] = snap.c20; oc[4] = snap.c21; oc[5] = snap.c22; oc[6] = snap.c30;
  oc[7] = snap.c31; oc[8] = snap.c32; oc[9] = snap.c33; oc[10] = snap.c40; oc[11] = snap.c41; oc[12] = snap.c42; oc[13] = snap.c43;
  oc[14] = snap.c44;
  // collision time (reading A38)
  const float L = sqrtf(x_in * x_in + snap.y * snap.y);
  const float S = arc_of_chord(L, P.cB * snap.q);
  const float z0 = zabs - snap.t * S;
  rf_z0[i] = z0;
  rf_t0[i] = -z0 / P.vdrift;
}

}  // namespace

int launch_k7_refit(const Launch& L, long long n_tracks, const int* o_sector, const int* o_tracklet, const long long* o_cl_begin,
                    const int* o_cl_row, const UnitDesc* d_units, const RowConst* d_rows, const float2* d_yz, const rowhit_t* d_rowhit,
                    int* rf_n, int* rf_ndf, float* rf_x, float* rf_par, float* rf_cov, float* rf_chi2, float* rf_z0, float* rf_t0,
                    int* d_order /* n_tracks ints */, int* d_classes /* 3 * K7_CLASSES ints */, const Params& P) {
  if (n_tracks <= 0) return 0;
  int* d_count = d_classes; int* d_fill = d_classes + K7_CLASSES; int* d_start = d_classes + 2 * K7_CLASSES;
  cudaError_t e0 = cudaMemsetAsync(d_count, 0, (size_t)2 * K7_CLASSES * sizeof(int), L.stream);
  if (e0 != cudaSuccess) return -(int)e0;
  const int b256 = (int)((n_tracks + 255) / 256);
  k7_count<<<b256, 256, 0, L.stream>>>(n_tracks, o_cl_begin, d_count);
  k7_starts<<<1, 1, 0, L.stream>>>(d_count, d_start);
  k7_fill<<<b256, 256, 0, L.stream>>>(n_tracks, o_cl_begin, d_start, d_fill, d_order);
  const int blocks = (int)((n_tracks + K7_THREADS - 1) / K7_THREADS);
  k7_refit<<<blocks, K7_THREADS, 0, L.stream>>>(n_tracks, d_order, o_sector, o_tracklet, o_cl_begin, o_cl_row, d_units, d_rows, d_yz, d_rowhit,
                                                rf_n, rf_ndf, rf_x, rf_par, rf_cov, rf_chi2, rf_z0, rf_t0, P);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 4 : -(int)e;
}

}  // namespace tpc
