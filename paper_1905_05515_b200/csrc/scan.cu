// scan.cu -- device-wide exclusive prefix sums used by the S4 start-hit compaction and the S6 track compaction.
// Reduce-then-scan in three launches: per-tile sums, one CTA scanning the tile sums, per-tile rescan with the tile offset.
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int SCAN_THREADS = 1024;
constexpr int SCAN_IPT = SCAN_TILE / SCAN_THREADS;   // 4 consecutive elements per thread

template <class T>
__device__ __forceinline__ T warp_incl(T v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { T t = __shfl_up_sync(0xffffffffu, v, d); if (lane >= d) v += t; }
  return v;
}

// exclusive block scan of one T per thread; s_warp has 33 entries
template <class T>
__device__ __forceinline__ T block_excl(T v, T* s_warp, T* total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  T inc = warp_incl(v, lane);
  if (lane == 31) s_warp[w] = inc;
  __syncthreads();
  if (w == 0) {
    T t = lane < nw ? s_warp[lane] : (T)0;
    T ti = warp_incl(t, lane);
    s_warp[lane] = ti - t;
    if (lane == 31) s_warp[32] = ti;
  }
  __syncthreads();
  T res = inc - v + s_warp[w];
  *total = s_warp[32];
  __syncthreads();   // s_warp may be reused by the caller's next round
  return res;
}

template <class T>
__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_sums(const T* __restrict__ in, int n, T* __restrict__ tile_sum) {
  __shared__ T s_warp[33];
  const long long base = (long long)blockIdx.x * SCAN_TILE + (long long)threadIdx.x * SCAN_IPT;
  T v = 0;
#pragma unroll
  for (int k = 0; k < SCAN_IPT; k++) if (base + k < n) v += in[base + k];
  T total;
  block_excl(v, s_warp, &total);
  if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}

template <class T>
__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_offsets(T* __restrict__ tile_sum, int n_tiles, T* __restrict__ total_out) {
  __shared__ T s_warp[33];
  T carry = 0;
  for (int base = 0; base < n_tiles; base += SCAN_THREADS) {
    int i = base + threadIdx.x;
    T v = i < n_tiles ? tile_sum[i] : (T)0;
    T total;
    T ex = block_excl(v, s_warp, &total);
    if (i < n_tiles) tile_sum[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0) { tile_sum[n_tiles] = carry; *total_out = carry; }
}

template <class T>
__global__ void __launch_bounds__(SCAN_THREADS) scan_tile_apply(const T* __restrict__ in, T* __restrict__ out, int n,
                                                                const T* __restrict__ tile_off) {
  __shared__ T s_warp[33];
  const long long base = (long long)blockIdx.x * SCAN_TILE + (long long)threadIdx.x * SCAN_IPT;
  T x[SCAN_IPT];
  T v = 0;
#pragma unroll
  for (int k = 0; k < SCAN_IPT; k++) { x[k] = base + k < n ? in[base + k] : (T)0; v += x[k]; }
  T total;
  T ex = block_excl(v, s_warp, &total) + tile_off[blockIdx.x];
#pragma unroll
  for (int k = 0; k < SCAN_IPT; k++) { if (base + k < n) out[base + k] = ex; ex += x[k]; }
}

template <class T>
int scan_impl(const Launch& L, const T* d_in, T* d_out, int n, T* d_tmp, T* d_total) {
  int n_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (n_tiles == 0) n_tiles = 1;   // still defines *d_total = 0
  scan_tile_sums<T><<<n_tiles, SCAN_THREADS, 0, L.stream>>>(d_in, n, d_tmp);
  scan_tile_offsets<T><<<1, SCAN_THREADS, 0, L.stream>>>(d_tmp, n_tiles, d_total);
  scan_tile_apply<T><<<n_tiles, SCAN_THREADS, 0, L.stream>>>(d_in, d_out, n, d_tmp);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 3 : -(int)e;
}

}  // namespace

int launch_scan_i32(const Launch& L, const int* d_in, int* d_out, int n, int* d_tmp, int* d_total) {
  return scan_impl<int>(L, d_in, d_out, n, d_tmp, d_total);
}
int launch_scan_u64(const Launch& L, const unsigned long long* d_in, unsigned long long* d_out, int n, unsigned long long* d_tmp,
                    unsigned long long* d_total) {
  return scan_impl<unsigned long long>(L, d_in, d_out, n, d_tmp, d_total);
}

// ---- fp32 FMA-loop peak (measurement utility for bench.py: the roofline denominator of the ALU-bound kernels, measured on the
//      box at the clocks of the run instead of taken from a data sheet).  8 independent chains per thread, explicit __fmaf_rn
//      (the library is compiled with -fmad=false), 2048 resident threads per SM.
namespace {
__global__ void __launch_bounds__(256) fma_peak_kernel(float* __restrict__ out, const int iters, const float a, const float b) {
  float x0 = threadIdx.x * 1e-3f, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
#pragma unroll 4
  for (int i = 0; i < iters; i++) {
    x0 = __fmaf_rn(x0, a, b); x1 = __fmaf_rn(x1, a, b); x2 = __fmaf_rn(x2, a, b); x3 = __fmaf_rn(x3, a, b);
    x4 = __fmaf_rn(x4, a, b); x5 = __fmaf_rn(x5, a, b); x6 = __fmaf_rn(x6, a, b); x7 = __fmaf_rn(x7, a, b);
  }
  const float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 123.456f) out[0] = s;   // keeps the chains alive
}
}  // namespace

// returns fused multiply-adds per launch (each is 2 flops), or a negative cudaError
long long launch_fma_peak(const Launch& L, float* d_out, int iters) {
  const int blocks = L.sm_count * 8;
  fma_peak_kernel<<<blocks, 256, 0, L.stream>>>(d_out, iters, 0.999999f, 1e-7f);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? (long long)blocks * 256 * 8 * (long long)iters : -(long long)e;
}

}  // namespace tpc
