// k9_merge.cu -- K9: S9 cross-sector segment matching (NEXT-3 of SURVEY.md section 8(f); PAPER.md:49 says only "Locally, e. g. at the
// TPC sector boundaries, there are still some improvements to be done"; matching segments across the boundary is this build's
// reading A41 of DESIGN.md).  Looper-leg identification is not part of it.
//
//   k9_ranges  : first track of every sector (the S6 tracks are in ascending sector order) by binary search
//   k9_outer   : one lane per track: S6 state transported (parameters only) to the row of the track's last cluster; a track
//                whose outer end lies within merge_edge of the side edge of its sector is a leaver towards the next / previous
//                sector in phi
//   scan, k9_fill : index of the tracks by (sector, first row): k9_outer counts, an exclusive scan gives the bucket starts, k9_fill
//                writes the track indices (arbitrary order inside a bucket; the tie on the index in k9_propose is explicit)
//   k9_propose : one warp per leaver A (the leavers are gathered into a list by k9_outer), one lane per candidate: outer state rotated into the neighbour's frame, transported to the first row of every
//                track B of that sector that starts within merge_rows rows of A's end (one contiguous range of the index),
//                compared inside the four windows; the
//                best B (score, then index) receives atomicMin of (score bits, A)
//   k9_accept  : one thread per track B: its best proposer A -> next[A] = B, prev[B] = A
// fp32, every operation spelled in the order of the definition (reading A41; library built with -fmad=false).
#include "kalman.cuh"

namespace tpc {
namespace {

constexpr int K9_THREADS = 128;
constexpr unsigned long long K9_NONE = ~0ull;

__global__ void k9_ranges(const long long n_tracks, const int NS, const int* __restrict__ o_sector, int* __restrict__ sec_begin) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s > NS) return;
  long long lo = 0, hi = n_tracks;   // first track with sector >= s
  while (lo < hi) { const long long mid = (lo + hi) >> 1; if (o_sector[mid] < s) lo = mid + 1; else hi = mid; }
  sec_begin[s] = (int)lo;
  if (s == 0) sec_begin[NS + 1] = 0;   // number of leavers gathered by k9_outer
}

__global__ void __launch_bounds__(K9_THREADS) k9_outer(const long long n_tracks, const int* __restrict__ o_sector, const int* __restrict__ o_tracklet,
                                                       const float* __restrict__ o_par, const long long* __restrict__ cl_begin,
                                                       const int* __restrict__ cl_row, const int* __restrict__ tl_first,
                                                       const RowConst* __restrict__ rows, float* __restrict__ outer,
                                                       int* __restrict__ row_in, int* __restrict__ row_out, int* __restrict__ leaver,
                                                       int* __restrict__ n_leavers, int* __restrict__ list, int* __restrict__ bucket_count,
                                                       const K9Params M, const Params P) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_tracks) return;
  const float* __restrict__ ip = o_par + i * 5;
  State st = {};
  st.y = ip[0]; st.z = ip[1]; st.s = ip[2]; st.t = ip[3]; st.q = ip[4];
  const int r0 = tl_first[o_tracklet[i]], r1 = cl_row[cl_begin[i + 1] - 1];
  bool ok = isfinite(st.q);
  for (int r = r0 + 1; ok && r <= r1; r++) ok = propagate(st, rows[r].x - rows[r - 1].x, P);
  row_in[i] = r0; row_out[i] = r1;
  atomicAdd(&bucket_count[o_sector[i] * P.R + r0], 1);
  float* __restrict__ o = outer + i * 4;
  int lv = 0;
  if (ok) {
    o[0] = rows[r1].x; o[1] = st.y; o[2] = st.z; o[3] = st.s;
    if (M.per_side > 0 && fabsf(st.y) >= rows[r1].yedge - M.edge) lv = st.y > 0.0f ? 1 : -1;
  } else {
    o[0] = o[1] = o[2] = o[3] = 0.0f;
  }
  leaver[i] = lv;
  if (lv) {   // leavers gathered in arbitrary order (no result depends on it): full warps in k9_propose; one atomic per warp
    const unsigned peers = __activemask();
    const int leader = __ffs(peers) - 1, lane = threadIdx.x & 31;
    int base = 0;
    if (lane == leader) base = atomicAdd(n_leavers, __popc(peers));
    base = __shfl_sync(peers, base, leader);
    list[base + __popc(peers & ((1u << lane) - 1u))] = (int)i;
  }
}

__global__ void __launch_bounds__(256) k9_fill(const long long n_tracks, const int R, const int* __restrict__ o_sector, const int* __restrict__ row_in,
                                               const int* __restrict__ bucket_start, int* __restrict__ bucket_fill, int* __restrict__ blist) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_tracks) return;
  const int u = o_sector[i] * R + row_in[i];
  blist[bucket_start[u] + atomicAdd(&bucket_fill[u], 1)] = (int)i;
}

// One WARP per leaver; the lanes take the candidates of the bucket range in turn and the warp reduces the minimum of
// (score bits : 32 | index : 32) = "smallest score, then lowest index" (score >= 0: its bit pattern orders like its value).
__global__ void __launch_bounds__(K9_THREADS) k9_propose(const long long n_tracks, const int* __restrict__ o_sector,
                                                         const float* __restrict__ o_par, const RowConst* __restrict__ rows,
                                                         const float* __restrict__ outer, const int* __restrict__ row_in,
                                                         const int* __restrict__ row_out, const int* __restrict__ leaver,
                                                         const int* __restrict__ sec_begin, const int* __restrict__ n_leavers,
                                                         const int* __restrict__ list, const int* __restrict__ bucket_start,
                                                         const int* __restrict__ blist, unsigned long long* __restrict__ cand,
                                                         const K9Params M, const Params P) {
  const long long j = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (j >= n_tracks || j >= *n_leavers) return;
  const long long a = list[j];
  const int lv = leaver[a];
  // sectors form closed rings of per_side sectors (one ring per side); the neighbour stays on the ring, hence below NS
  const int sec = o_sector[a], side = sec / M.per_side, k = sec % M.per_side;
  const int nb = side * M.per_side + (k + (lv > 0 ? 1 : M.per_side - 1)) % M.per_side;
  const float sgn = lv > 0 ? 1.0f : -1.0f;
  const float* __restrict__ o = outer + a * 4;
  const float x = o[0], y = o[1], s = o[3], c = sqrtf(1.0f - s * s);
  const float ss = sgn * M.sd;
  State rot = {};
  const float xr = x * M.cd + y * ss;
  rot.y = y * M.cd - x * ss; rot.z = o[2]; rot.s = s * M.cd - c * ss; rot.t = o_par[a * 5 + 3]; rot.q = o_par[a * 5 + 4];
  const int ra = row_out[a];
  unsigned long long best = K9_NONE;
  // the tracks of sector nb that start within merge_rows rows of ra: buckets (nb, ra - rows) .. (nb, ra + rows), one contiguous range
  const int r_lo = max(0, ra - M.rows), r_hi = min(P.R - 1, ra + M.rows);
  const int j1 = bucket_start[nb * P.R + r_hi + 1];
  for (int jb = bucket_start[nb * P.R + r_lo] + lane; jb < j1; jb += 32) {
    const int b = blist[jb];
    const int rb = row_in[b];
    const float* __restrict__ pb = o_par + (long long)b * 5;
    const float dt = pb[3] - rot.t;                 // dz/ds is not changed by the transport: this window is tested before it
    if (!(fabsf(dt) <= M.dt)) continue;
    State st = rot;
    if (!propagate(st, rows[rb].x - xr, P)) continue;
    const float dy = pb[0] - st.y, dz = pb[1] - st.z, ds = pb[2] - st.s;
    if (!(fabsf(dy) <= M.dy && fabsf(dz) <= M.dz && fabsf(ds) <= M.ds)) continue;
    const float ey = dy / M.dy, ez = dz / M.dz, es = ds / M.ds, et = dt / M.dt;
    const float score = ((ey * ey + ez * ez) + es * es) + et * et;
    const unsigned long long key = ((unsigned long long)__float_as_uint(score) << 32) | (unsigned long long)(unsigned)b;
    if (key < best) best = key;
  }
#pragma unroll
  for (int o2 = 16; o2 > 0; o2 >>= 1) { const unsigned long long v = __shfl_xor_sync(0xffffffffu, best, o2); if (v < best) best = v; }
  if (lane == 0 && best != K9_NONE)
    atomicMin(&cand[(unsigned)(best & 0xffffffffull)], (best & 0xffffffff00000000ull) | (unsigned long long)(unsigned)a);
}

__global__ void __launch_bounds__(256) k9_accept(const long long n_tracks, const unsigned long long* __restrict__ cand,
                                                 int* __restrict__ next, int* __restrict__ prev) {
  const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= n_tracks) return;
  const unsigned long long kk = cand[b];
  if (kk == K9_NONE) return;
  const int a = (int)(unsigned)(kk & 0xffffffffull);
  next[a] = (int)b;      // every A proposes to one B only: no two B write the same next[A]
  prev[b] = a;
}

}  // namespace

// d_sec_begin: NS + 2 ints; d_list, d_blist: n_tracks ints each; d_bucket: 3 * (NS * R + 1) + (NS * R + 1) / SCAN_TILE + 4 ints
// (bucket counts, fill counters, starts, scan scratch)
int launch_k9_merge(const Launch& L, long long n_tracks, int NS, const int* o_sector, const int* o_tracklet, const float* o_par,
                    const long long* o_cl_begin, const int* o_cl_row, const int* d_tl_first, const RowConst* d_rows, float* d_outer,
                    int* d_row_in, int* d_row_out, int* d_leaver, int* d_sec_begin, int* d_list, int* d_blist, int* d_bucket,
                    unsigned long long* d_cand, int* d_next, int* d_prev, const K9Params& M, const Params& P) {
  if (n_tracks <= 0) return 0;
  const int NB = NS * P.R + 1;   // one bucket per (sector, row) + the end
  int* d_bcount = d_bucket; int* d_bfill = d_bucket + NB; int* d_bstart = d_bucket + 2 * NB; int* d_btmp = d_bucket + 3 * NB;
  cudaError_t e = cudaMemsetAsync(d_cand, 0xff, (size_t)n_tracks * sizeof(unsigned long long), L.stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_next, 0xff, (size_t)n_tracks * sizeof(int), L.stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_prev, 0xff, (size_t)n_tracks * sizeof(int), L.stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_bcount, 0, (size_t)2 * NB * sizeof(int), L.stream);
  if (e != cudaSuccess) return -(int)e;
  const int blocks = (int)((n_tracks + K9_THREADS - 1) / K9_THREADS);
  k9_ranges<<<(NS + 1 + 63) / 64, 64, 0, L.stream>>>(n_tracks, NS, o_sector, d_sec_begin);
  k9_outer<<<blocks, K9_THREADS, 0, L.stream>>>(n_tracks, o_sector, o_tracklet, o_par, o_cl_begin, o_cl_row, d_tl_first, d_rows, d_outer, d_row_in,
                                               d_row_out, d_leaver, d_sec_begin + NS + 1, d_list, d_bcount, M, P);
  const int rc = launch_scan_i32(L, d_bcount, d_bstart, NB, d_btmp + 1, d_btmp);   // d_bstart[NB - 1] = number of tracks
  if (rc < 0) return rc;
  k9_fill<<<(int)((n_tracks + 255) / 256), 256, 0, L.stream>>>(n_tracks, P.R, o_sector, d_row_in, d_bstart, d_bfill, d_blist);
  const int wblocks = (int)((n_tracks * 32 + K9_THREADS - 1) / K9_THREADS);   // one warp per slot of the leaver list
  k9_propose<<<wblocks, K9_THREADS, 0, L.stream>>>(n_tracks, o_sector, o_par, d_rows, d_outer, d_row_in, d_row_out, d_leaver, d_sec_begin,
                                                 d_sec_begin + NS + 1, d_list, d_bstart, d_blist, d_cand, M, P);
  k9_accept<<<(int)((n_tracks + 255) / 256), 256, 0, L.stream>>>(n_tracks, d_cand, d_next, d_prev);
  e = cudaGetLastError();
  return e == cudaSuccess ? 5 + rc : -(int)e;
}

}  // namespace tpc
