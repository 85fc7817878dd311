// k10_loopers.cu -- K10: S10, turns of one looping particle (NEXT-3, second half, of SURVEY.md section 8(f): "recognise returning
// legs / extra turns"; "looping tracks", "secondary legs of looping tracks below 200 MeV/c"; reading A46 of
// the paper gives no rule).
//
// In a uniform field every turn of a looping particle runs over the same circle in the pad plane, displaced along z by one pitch
// (2 pi / |k|) * dz/ds, so later turns are separate S6 tracks of the same sector with the same (y, sin phi, dz/ds, q/pT) at the same x.
//   k10_ranges : first track of every sector (the S6 tracks are in ascending sector order) by binary search
//   k10_match  : one lane per track B with |q/pT| >= loop_qmin: its state is transported (parameters only) to the x of every
//                track A of its sector with |q/pT| >= loop_qmin and compared inside the four windows; the number of turns
//                tau = dz / pitch must be within loop_frac of an integer n in 1..loop_nmax; predecessor = smallest n, then
//                smallest score, then lowest index
//   k10_roots  : one lane per track: follow the predecessors to the first turn (root), adding up n (turn)
// fp32, every operation spelled in the order of the definition (oracle S10; library built with -fmad=false).
#include "kalman.cuh"

#include <mutex>

// Scratch of the allocation-free entry point tpc_find_loopers_noalloc (end of this file): sec_begin[K10_STATIC_MAX_SECTORS + 2],
// padded to 1024 words, then prev_n[K10_STATIC_MAX_TRACKS].  1 MiB + 4 KiB, held by every GPU that loads the library until exit.
// In HOST code this name is only a stand-in for the symbol, never a device address: the address comes from cudaGetSymbolAddress
// (static_scratch() below), once per device.
static __device__ __align__(256) int k10_static_scratch[1024 + tpc::K10_STATIC_MAX_TRACKS];

namespace tpc {
namespace {

constexpr int K10_THREADS = 128;

__global__ void k10_ranges(const long long n_tracks, const int NS, const int* __restrict__ o_sector, int* __restrict__ sec_begin) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s > NS) return;
  long long lo = 0, hi = n_tracks;   // first track with sector >= s
  while (lo < hi) { const long long mid = (lo + hi) >> 1; if (o_sector[mid] < s) lo = mid + 1; else hi = mid; }
  sec_begin[s] = (int)lo;
}

__global__ void __launch_bounds__(K10_THREADS) k10_match(const long long n_tracks, const int* __restrict__ o_sector,
                                                         const float* __restrict__ o_x, const float* __restrict__ o_par,
                                                         const int* __restrict__ sec_begin, int* __restrict__ prev,
                                                         int* __restrict__ prev_n, const K10Params L, const Params P) {
  const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= n_tracks) return;
  int best = -1, bestn = 0; float bests = 0.0f;
  const float* __restrict__ pb = o_par + b * 5;
  const float qb = pb[4];
  if (fabsf(qb) >= L.qmin) {
    const float xb = o_x[b];
    const int sec = o_sector[b], a1 = sec_begin[sec + 1];
    for (int a = sec_begin[sec]; a < a1; a++) {
      if (a == b) continue;
      const float* __restrict__ pa = o_par + (long long)a * 5;
      const float qa = pa[4];
      if (!(fabsf(qa) >= L.qmin)) continue;
      State st = {};
      st.y = pb[0]; st.z = pb[1]; st.s = pb[2]; st.t = pb[3]; st.q = qb;
      const float dx = o_x[a] - xb;
      if (dx != 0.0f && !propagate(st, dx, P)) continue;
      const float dy = st.y - pa[0], ds = st.s - pa[2], dt = st.t - pa[3], dq = st.q - qa;
      if (!(fabsf(dy) <= L.dy && fabsf(ds) <= L.ds && fabsf(dt) <= L.dt && fabsf(dq) <= L.dq * fabsf(qa))) continue;
      const float k = P.cB * qa;
      const float tav = 0.5f * (pa[3] + st.t);
      const float pitch = (L.twopi / fabsf(k)) * tav;
      if (!(fabsf(pitch) >= L.pmin)) continue;
      const float tau = (st.z - pa[1]) / pitch;
      const float nr = rintf(tau);
      if (!(nr >= 1.0f && fabsf(tau - nr) <= L.frac && nr <= (float)L.nmax)) continue;
      const int n = (int)nr;
      const float ey = dy / L.dy, es = ds / L.ds, et = dt / L.dt;
      const float score = (ey * ey + es * es) + et * et;
      if (best < 0 || n < bestn || (n == bestn && score < bests)) { best = a; bestn = n; bests = score; }
    }
  }
  prev[b] = best; prev_n[b] = bestn;
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

int launch_k10_loopers(const Launch& L, long long n_tracks, int NS, const int* o_sector, const float* o_x, const float* o_par,
                       int* d_sec_begin, int* d_prev, int* d_prev_n, int* d_root, int* d_turn, const K10Params& K, const Params& P) {
  if (n_tracks <= 0) return 0;
  k10_ranges<<<(NS + 1 + 63) / 64, 64, 0, L.stream>>>(n_tracks, NS, o_sector, d_sec_begin);
  const int blocks = (int)((n_tracks + K10_THREADS - 1) / K10_THREADS);
  k10_match<<<blocks, K10_THREADS, 0, L.stream>>>(n_tracks, o_sector, o_x, o_par, d_sec_begin, d_prev, d_prev_n, K, P);
  k10_roots<<<(int)((n_tracks + 255) / 256), 256, 0, L.stream>>>(n_tracks, d_prev, d_prev_n, d_root, d_turn);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 3 : -(int)e;
}

// ---- Allocation-free variant (tpc_find_loopers_noalloc): the same three kernels, their scratch (sec_begin, prev_n) in the
// file-scope array k10_static_scratch instead of the context's grow-only cudaMalloc buffers.
namespace {

constexpr int K10_MAX_DEVICES = 64;
static_assert(K10_STATIC_MAX_SECTORS + 2 <= 1024, "sec_begin has NS + 1 entries and lives in the first 1024 words of the scratch");
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

// Same result as launch_k10_loopers.  No cudaMalloc / cudaFree, no synchronisation.  Nothing in the scratch has to start at zero:
// k10_ranges writes sec_begin[0..NS] and k10_match writes prev_n[0..n_tracks) before the kernels that follow read exactly those words,
// so what an earlier call left behind (the array is shared by every call on the device) is never read.  Two calls that overlap on
// the GPU (different streams) race on the array.  Returns the launches made, or -(cudaError_t).
int launch_k10_loopers_static(const Launch& L, long long n_tracks, int NS, const int* o_sector, const float* o_x, const float* o_par,
                              int* d_prev, int* d_root, int* d_turn, const K10Params& K, const Params& P) {
  if (n_tracks <= 0) return 0;
  if (n_tracks > K10_STATIC_MAX_TRACKS || NS > K10_STATIC_MAX_SECTORS) return -(int)cudaErrorInvalidValue;   // the ABI checks first
  int* scratch = nullptr;
  cudaError_t e = static_scratch(&scratch);
  if (e != cudaSuccess) return -(int)e;
  int* d_sec_begin = scratch;
  int* d_prev_n = scratch + 1024;
  k10_ranges<<<(NS + 1 + 63) / 64, 64, 0, L.stream>>>(n_tracks, NS, o_sector, d_sec_begin);
  const int blocks = (int)((n_tracks + K10_THREADS - 1) / K10_THREADS);
  k10_match<<<blocks, K10_THREADS, 0, L.stream>>>(n_tracks, o_sector, o_x, o_par, d_sec_begin, d_prev, d_prev_n, K, P);
  k10_roots<<<(int)((n_tracks + 255) / 256), 256, 0, L.stream>>>(n_tracks, d_prev, d_prev_n, d_root, d_turn);
  e = cudaGetLastError();
  return e == cudaSuccess ? 3 : -(int)e;
}

}  // namespace tpc
