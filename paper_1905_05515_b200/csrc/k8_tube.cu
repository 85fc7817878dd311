// k8_tube.cu -- K8: S8 cluster attachment status (NEXT-4 of SURVEY.md section 8(f); "The tracker forms tubes of
// 1.5 cm around each track, and marks unattached clusters as adjacent to the tube of the track with the highest transverse
// momentum it lies in"; reading A40 of DESIGN.md).
//
//   k8_attach : one warp per track marks the clusters of its list (sorted positions through the tracklet's rowhit line)
//   k8_path   : one lane per track transports the S6 state row by row (helix, parameters only -- the covariance part of
//               propagate() is dead code here) from the row of the state to the row of the track's last cluster and stores the
//               position (y, z - z_state) of every row it reaches: the only serial part
//   k8_tube   : one warp per track, one lane per row: scans the grid bins under the tube around the stored position; an unattached
//               cluster inside gets atomicMin of (|q/pT| bits, track index): the track with the highest pT, then the lowest index, wins
//   k8_status : one thread per cluster writes (status, track) in the caller's order through perm
// z is carried relative to the state's z (as in K5), distances are formed term by term in fp32 (library built with -fmad=false).
#include "kalman.cuh"

namespace tpc {
namespace {

constexpr int K8_THREADS = 128;
constexpr unsigned long long K8_NONE = ~0ull;

__global__ void __launch_bounds__(K8_THREADS) k8_attach(const long long n_tracks, const int R, const int* __restrict__ o_sector,
                                                        const int* __restrict__ o_tracklet, const long long* __restrict__ cl_begin,
                                                        const int* __restrict__ cl_row, const UnitDesc* __restrict__ units,
                                                        const rowhit_t* __restrict__ rowhit, int* __restrict__ att) {
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (i >= n_tracks) return;
  const UnitDesc* __restrict__ su = units + (long long)o_sector[i] * R;
  const rowhit_t* __restrict__ rh = rowhit + (long long)o_tracklet[i] * R;
  const long long b = cl_begin[i + 1];
  for (long long k = cl_begin[i] + lane; k < b; k += 32) {
    const int r = cl_row[k];
    att[su[r].off + rh[r]] = (int)i;
  }
}

__global__ void __launch_bounds__(K8_THREADS) k8_path(const long long n_tracks, const int* __restrict__ o_tracklet, const float* __restrict__ o_par,
                                                      const long long* __restrict__ cl_begin, const int* __restrict__ cl_row,
                                                      const int* __restrict__ tl_first, const RowConst* __restrict__ rows,
                                                      float2* __restrict__ path, int* __restrict__ path_end, const Params P) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_tracks) return;
  const float* __restrict__ ip = o_par + i * 5;
  State st = {};
  st.y = ip[0]; st.z = 0.0f; st.s = ip[2]; st.t = ip[3]; st.q = ip[4];
  const int r_first = tl_first[o_tracklet[i]], r_last = cl_row[cl_begin[i + 1] - 1];
  int r_end = r_first - 1;                       // last row with a stored position
  if (isfinite(st.q)) {
    float2* __restrict__ pp = path + i * P.R;
    for (int r = r_first; r <= r_last; r++) {
      if (r > r_first && !propagate(st, rows[r].x - rows[r - 1].x, P)) break;
      pp[r] = make_float2(st.y, st.z);
      r_end = r;
    }
  }
  path_end[i] = r_end;
}

__global__ void __launch_bounds__(K8_THREADS) k8_tube(const long long n_tracks, const int* __restrict__ o_sector,
                                                      const int* __restrict__ o_tracklet, const float* __restrict__ o_par,
                                                      const int* __restrict__ tl_first, const UnitDesc* __restrict__ units,
                                                      const float2* __restrict__ yz, const int* __restrict__ bin_start,
                                                      const int* __restrict__ att, const float2* __restrict__ path,
                                                      const int* __restrict__ path_end, unsigned long long* __restrict__ adj,
                                                      const float tube, const Params P) {
  const long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (i >= n_tracks) return;
  const int r_first = tl_first[o_tracklet[i]], r_end = path_end[i];
  if (r_end < r_first) return;
  const float zref = o_par[i * 5 + 1];
  const unsigned long long key = ((unsigned long long)__float_as_uint(fabsf(o_par[i * 5 + 4])) << 32) | (unsigned long long)(unsigned)i;
  const UnitDesc* __restrict__ su = units + (long long)o_sector[i] * P.R;
  const float2* __restrict__ pp = path + i * P.R;
  const float tube2 = tube * tube, margin = 0.05f;
  for (int r = r_first + lane; r <= r_end; r += 32) {
    const UnitDesc d = su[r];
    if (d.n == 0) continue;
    const float2 pos = pp[r];
    const float y = pos.x, zr = pos.y;
    const float ylo = y - tube, yhi = y + tube, zlo = zr - tube, zhi = zr + tube;
    const int by0 = bin_of(ylo, d.ylo, d.invs, d.ny), by1 = bin_of(yhi, d.ylo, d.invs, d.ny);
    const int bz0 = bin_of((zlo + zref) - margin, d.zlo, d.invs, d.nz), bz1 = bin_of((zhi + zref) + margin, d.zlo, d.invs, d.nz);
    const int* __restrict__ bs = bin_start + d.bin_off;
    for (int bz = bz0; bz <= bz1; bz++) {
      const int pe = bs[bz * d.ny + by1 + 1];
      for (int p = bs[bz * d.ny + by0]; p < pe; p++) {
        const float2 c = yz[d.off + p];
        const float dy = c.x - y, dz = (c.y - zref) - zr;
        const float d2 = dy * dy + dz * dz;
        if (d2 <= tube2 && att[d.off + p] < 0) atomicMin(&adj[d.off + p], key);
      }
    }
  }
}

__global__ void __launch_bounds__(256) k8_status(const int U, const UnitDesc* __restrict__ units, const int* __restrict__ perm,
                                                 const int* __restrict__ att, const unsigned long long* __restrict__ adj,
                                                 int* __restrict__ cl_status, int* __restrict__ cl_track) {
  // one CTA per unit: sorted position p of the unit -> caller's index perm[p] inside the unit
  const UnitDesc d = units[blockIdx.x];
  for (int p = threadIdx.x; p < d.n; p += blockDim.x) {
    const long long g = d.off + p, c = d.off + perm[g];
    const int a = att[g];
    const unsigned long long k = adj[g];
    int s = 0, t = -1;
    if (a >= 0) { s = 1; t = a; }
    else if (k != K8_NONE) { s = 2; t = (int)(unsigned)(k & 0xffffffffull); }
    cl_status[c] = s; cl_track[c] = t;
  }
  (void)U;
}

}  // namespace

int launch_k8_status(const Launch& L, long long n_tracks, long long N, int U, const int* o_sector, const int* o_tracklet,
                     const float* o_par, const long long* o_cl_begin, const int* o_cl_row, const int* d_tl_first,
                     const UnitDesc* d_units, const RowConst* d_rows, const float2* d_yz, const int* d_perm, const int* d_bin_start,
                     const rowhit_t* d_rowhit, int* d_att, unsigned long long* d_adj, float2* d_path /* n_tracks * R */,
                     int* d_path_end /* n_tracks */, int* cl_status, int* cl_track, float tube, const Params& P) {
  if (N <= 0 || U <= 0) return 0;
  cudaError_t e = cudaMemsetAsync(d_att, 0xff, (size_t)N * sizeof(int), L.stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_adj, 0xff, (size_t)N * sizeof(unsigned long long), L.stream);
  if (e != cudaSuccess) return -(int)e;
  int launches = 0;
  if (n_tracks > 0) {
    k8_attach<<<(int)((n_tracks * 32 + K8_THREADS - 1) / K8_THREADS), K8_THREADS, 0, L.stream>>>(n_tracks, P.R, o_sector, o_tracklet,
                                                                                                o_cl_begin, o_cl_row, d_units, d_rowhit,
                                                                                                d_att);
    k8_path<<<(int)((n_tracks + K8_THREADS - 1) / K8_THREADS), K8_THREADS, 0, L.stream>>>(n_tracks, o_tracklet, o_par, o_cl_begin, o_cl_row,
                                                                                         d_tl_first, d_rows, d_path, d_path_end, P);
    k8_tube<<<(int)((n_tracks * 32 + K8_THREADS - 1) / K8_THREADS), K8_THREADS, 0, L.stream>>>(n_tracks, o_sector, o_tracklet, o_par, d_tl_first,
                                                                                              d_units, d_yz, d_bin_start, d_att, d_path,
                                                                                              d_path_end, d_adj, tube, P);
    launches += 3;
  }
  k8_status<<<U, 256, 0, L.stream>>>(U, d_units, d_perm, d_att, d_adj, cl_status, cl_track);
  e = cudaGetLastError();
  return e == cudaSuccess ? launches + 1 : -(int)e;
}

}  // namespace tpc
