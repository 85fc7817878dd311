// k10_loopers.cu -- K10: S10, turns of one looping particle (NEXT-3, second half, of SURVEY.md section 8(f): "recognise returning
// legs / extra turns"; "looping tracks", "secondary legs of looping tracks below 200 MeV/c"; reading A46 of
// the paper gives no rule).
//
// In a uniform field every turn of a looping particle runs over the same circle in the pad plane, displaced along z by one pitch
// (2 pi / |k|) * dz/ds, so later turns are separate S6 tracks of the same sector with the same (y, sin phi, dz/ds, q/pT) at the same x.
//   k10_ranges  : first track of every sector (the S6 tracks are in ascending sector order) by binary search; zeroes the per-sector
//                 counters of k10_compact
//   k10_compact : the tracks with |q/pT| >= loop_qmin (pT <= 200 MeV/c: about one track in ten) are gathered at the front of their
//                 sector's index range (slot = sec_begin + atomic counter; the order inside a sector is arbitrary and enters no
//                 result); every track gets prev = -1 here
//   k10_match   : one warp per gathered track B, one lane per candidate: B's state is transported (parameters only) to the x of every gathered track A of
//                 its sector and compared inside the four windows; the number of turns tau = dz / pitch must be within loop_frac of
//                 an integer n in 1..loop_nmax; predecessor = smallest n, then smallest score, then lowest index (the tie on the
//                 index is explicit, so the arbitrary gathering order does not matter)
//   k10_roots   : one lane per track: follow the predecessors to the first turn (root), adding up n (turn)
// fp32, every operation spelled in the order of the definition (oracle S10; library built with -fmad=false).
#include "kalman.cuh"

#include <mutex>

// Scratch of the allocation-free entry point tpc_find_loopers_noalloc (end of this file): sec_begin and sec_count
// [K10_STATIC_MAX_SECTORS + 2 each, padded to 1024 words], then list[K10_STATIC_MAX_TRACKS] and prev_n[K10_STATIC_MAX_TRACKS].
// 2 MiB + 8 KiB, held by every GPU that loads the library until exit.
// In HOST code this name is only a stand-in for the symbol, never a device address: the address comes from cudaGetSymbolAddress
// (static_scratch() below), once per device.
static __device__ __align__(256) int k10_static_scratch[2048 + 2 * tpc::K10_STATIC_MAX_TRACKS];

namespace tpc {
namespace {

constexpr int K10_THREADS = 128;

__global__ void k10_ranges(const long long n_tracks, const int NS, const int* __restrict__ o_sector, int* __restrict__ sec_begin,
                           int* __restrict__ sec_count) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s > NS) return;
  long long lo = 0, hi = n_tracks;   // first track with sector >= s
  while (lo < hi) { const long long mid = (lo + hi) >> 1; if (o_sector[mid] < s) lo = mid + 1; else hi = mid; }
  sec_begin[s] = (int)lo;
  sec_count[s] = 0;                  // the counters start every call at zero, whatever the last call left in the scratch
}

__global__ void __launch_bounds__(K10_THREADS) k10_compact(const long long n_tracks, const int* __restrict__ o_sector,
                                                           const float* __restrict__ o_par, const int* __restrict__ sec_begin,
                                                           int* __restrict__ sec_count, int* __restrict__ list, int* __restrict__ prev,
                                                           int* __restrict__ prev_n, const int NS, const K10Params L) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_tracks) return;
  const int sec = o_sector[i];
  // (sector out of range, or a slot beyond the array: only with caller-made arrays that are not in ascending sector order --
  // tpc_find_loopers_noalloc; such a track takes no part, nothing is written out of bounds)
  long long slot = -1;
  const bool take = fabsf(o_par[i * 5 + 4]) >= L.qmin && (unsigned)sec < (unsigned)NS;
  if (take) {   // one atomic per sector and warp (the tracks are in sector order: nearly always one group)
    const unsigned peers = __match_any_sync(__activemask(), sec);
    const int leader = __ffs(peers) - 1, lane = threadIdx.x & 31;
    int base = 0;
    if (lane == leader) base = atomicAdd(&sec_count[sec], __popc(peers));
    base = __shfl_sync(peers, base, leader);
    slot = (long long)sec_begin[sec] + base + __popc(peers & ((1u << lane) - 1u));
  }
  if (slot >= 0 && slot < n_tracks) list[slot] = (int)i;
  prev[i] = -1; prev_n[i] = 0;   // every track starts without a predecessor; k10_match overwrites the gathered ones
}

// One WARP per gathered track B; the lanes take the gathered tracks A of its sector in turn (32 pairs in flight per warp instead of a
// serial loop of several hundred dependent reads per lane) and the warp reduces the minimum of the key
// (n : 8 bits | score bits : 32 | index : 24; loop_nmax <= 255, at most 2^24 tracks as in K6), which is the order "smallest n, then smallest score, then lowest index".
__global__ void __launch_bounds__(K10_THREADS) k10_match(const long long n_tracks, const int* __restrict__ o_sector,
                                                         const float* __restrict__ o_x, const float* __restrict__ o_par,
                                                         const int* __restrict__ sec_begin, const int* __restrict__ sec_count,
                                                         const int* __restrict__ list, int* __restrict__ prev,
                                                         int* __restrict__ prev_n, const K10Params L, const Params P) {
  const long long j = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;   // slot of the gathered list (same sector ranges as the tracks)
  const int lane = threadIdx.x & 31;
  if (j >= n_tracks) return;
  const int sec = o_sector[j];
  if ((unsigned)sec >= (unsigned)P.NS) return;
  const int a0 = sec_begin[sec], a1 = (int)min((long long)a0 + sec_count[sec], n_tracks);
  if (j < a0 || j >= a1) return;                                                 // beyond the gathered tracks of this sector (whole warp)
  const int b = list[j];
  if ((unsigned)b >= (unsigned long long)n_tracks) return;                       // (stale slot: arrays not in ascending sector order)
  const float* __restrict__ pb = o_par + (long long)b * 5;
  const float yb = pb[0], zb = pb[1], sb = pb[2], tb = pb[3], qb = pb[4], xb = o_x[b];
  unsigned long long best = ~0ull;
  for (int ja = a0 + lane; ja < a1; ja += 32) {
    const int a = list[ja];
    if (a == b || (unsigned)a >= (unsigned long long)n_tracks) continue;
    const float* __restrict__ pa = o_par + (long long)a * 5;
    const float qa = pa[4];
    // dz/ds and q/pT are not changed by the transport: their two windows are tested first (same values, same outcome as testing
    // all four after it) and spare most pairs the transport
    const float dt = tb - pa[3], dq = qb - qa;
    if (!(fabsf(dt) <= L.dt && fabsf(dq) <= L.dq * fabsf(qa))) continue;
    State st = {};
    st.y = yb; st.z = zb; st.s = sb; st.t = tb; st.q = qb;
    const float dx = o_x[a] - xb;
    if (dx != 0.0f && !propagate(st, dx, P)) continue;
    const float dy = st.y - pa[0], ds = st.s - pa[2];
    if (!(fabsf(dy) <= L.dy && fabsf(ds) <= L.ds)) continue;
    const float k = P.cB * qa;
    const float tav = 0.5f * (pa[3] + st.t);
    const float pitch = (L.twopi / fabsf(k)) * tav;
    if (!(fabsf(pitch) >= L.pmin)) continue;
    const float tau = (st.z - pa[1]) / pitch;
    const float nr = rintf(tau);
    if (!(nr >= 1.0f && fabsf(tau - nr) <= L.frac && nr <= (float)L.nmax)) continue;
    const float ey = dy / L.dy, es = ds / L.ds, et = dt / L.dt;
    const float score = (ey * ey + es * es) + et * et;          // >= 0: its bit pattern orders like its value
    const unsigned long long key = ((unsigned long long)(unsigned)(int)nr << 56) | ((unsigned long long)__float_as_uint(score) << 24) |
                                   (unsigned long long)(unsigned)a;
    if (key < best) best = key;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { const unsigned long long v = __shfl_xor_sync(0xffffffffu, best, o); if (v < best) best = v; }
  if (lane == 0) {
    prev[b] = best == ~0ull ? -1 : (int)(best & 0xFFFFFFull);
    prev_n[b] = best == ~0ull ? 0 : (int)(best >> 56);
  }
}

__global__ void __launch_bounds__(256) k10_roots(const long long n_tracks, const int* __restrict__ prev, const int* __restrict__ prev_n,
                                                 int* __restrict__ root, int* __restrict__ turn) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_tracks) return;
  int r = (int)i, t = 0;
  for (int it = 0; it < 64 && prev[r] >= 0; it++) { t += prev_n[r]; r = prev[r]; }   // the predecessor lies n >= 1 turns earlier
  root[i] = r; turn[i] = t;
}

}  // namespace

namespace {
// the four launches; scratch: sec_begin[NS + 1], sec_count[NS + 1], list[n_tracks], prev_n[n_tracks]
int k10_launch_all(const Launch& L, long long n_tracks, int NS, const int* o_sector, const float* o_x, const float* o_par, int* d_sec_begin,
                   int* d_sec_count, int* d_list, int* d_prev, int* d_prev_n, int* d_root, int* d_turn, const K10Params& K, const Params& P) {
  k10_ranges<<<(NS + 1 + 63) / 64, 64, 0, L.stream>>>(n_tracks, NS, o_sector, d_sec_begin, d_sec_count);
  const int blocks = (int)((n_tracks + K10_THREADS - 1) / K10_THREADS);
  k10_compact<<<blocks, K10_THREADS, 0, L.stream>>>(n_tracks, o_sector, o_par, d_sec_begin, d_sec_count, d_list, d_prev, d_prev_n, NS, K);
  const int wblocks = (int)((n_tracks * 32 + K10_THREADS - 1) / K10_THREADS);   // one warp per slot of the gathered list
  k10_match<<<wblocks, K10_THREADS, 0, L.stream>>>(n_tracks, o_sector, o_x, o_par, d_sec_begin, d_sec_count, d_list, d_prev, d_prev_n, K, P);
  k10_roots<<<(int)((n_tracks + 255) / 256), 256, 0, L.stream>>>(n_tracks, d_prev, d_prev_n, d_root, d_turn);
  const cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 4 : -(int)e;
}
}  // namespace

// d_sec: 2 * (NS + 1) ints (sec_begin, then the per-sector counters); d_list, d_prev_n: n_tracks ints each
int launch_k10_loopers(const Launch& L, long long n_tracks, int NS, const int* o_sector, const float* o_x, const float* o_par,
                       int* d_sec, int* d_list, int* d_prev, int* d_prev_n, int* d_root, int* d_turn, const K10Params& K, const Params& P) {
  if (n_tracks <= 0) return 0;
  return k10_launch_all(L, n_tracks, NS, o_sector, o_x, o_par, d_sec, d_sec + NS + 1, d_list, d_prev, d_prev_n, d_root, d_turn, K, P);
}

// ---- Allocation-free variant (tpc_find_loopers_noalloc): the same four kernels, their scratch (sec_begin, sec_count, prev_n, list)
// in the file-scope array k10_static_scratch instead of the context's grow-only cudaMalloc buffers.
namespace {

constexpr int K10_MAX_DEVICES = 64;
static_assert(K10_STATIC_MAX_SECTORS + 2 <= 1024, "sec_begin and sec_count have NS + 1 entries each and live in the first 2 x 1024 words of the scratch");
std::mutex g_static_mu;
int* g_static_ptr[K10_MAX_DEVICES] = {};   // device address of k10_static_scratch on each device, resolved once per device

// Device address of the scratch on the CURRENT device (the symbol has one instance per device that loaded the library).
cudaError_t static_scratch(int** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= K10_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, k10_static_scratch);
    if (e != cudaSuccess) return e;
    g_static_ptr[dev] = static_cast<int*>(p);
  }
  *out = g_static_ptr[dev];
  return cudaSuccess;
}

}  // namespace

// Same result as launch_k10_loopers.  No cudaMalloc / cudaFree, no synchronisation.  The array is shared by every call on the device
// and keeps what the last call left in it: the only words that must start at zero, the per-sector counters, are zeroed by
// k10_ranges at the start of every call; sec_begin[0..NS], list[...] and prev_n[0..n_tracks) are written by this call's kernels
// before the kernels that follow read exactly those words.  Two calls that overlap on the GPU (different streams) race on the
// array.  Returns the launches made, or -(cudaError_t).
int launch_k10_loopers_static(const Launch& L, long long n_tracks, int NS, const int* o_sector, const float* o_x, const float* o_par,
                              int* d_prev, int* d_root, int* d_turn, const K10Params& K, const Params& P) {
  if (n_tracks <= 0) return 0;
  if (n_tracks > K10_STATIC_MAX_TRACKS || NS > K10_STATIC_MAX_SECTORS) return -(int)cudaErrorInvalidValue;   // the ABI checks first
  int* scratch = nullptr;
  const cudaError_t e = static_scratch(&scratch);
  if (e != cudaSuccess) return -(int)e;
  return k10_launch_all(L, n_tracks, NS, o_sector, o_x, o_par, scratch, scratch + 1024, scratch + 2048, d_prev,
                        scratch + 2048 + K10_STATIC_MAX_TRACKS, d_root, d_turn, K, P);
}

}  // namespace tpc
