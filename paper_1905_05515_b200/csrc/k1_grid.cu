// k1_grid.cu -- K1: S0 (time -> z) fused with S1 (per-row 2-D grid, stable counting sort).
//
// One CTA per (sector,row) unit.  The bin counters / cursors of the unit live in shared memory (global scratch for units
// whose grid does not fit).  Passes over the unit's clusters:
//   B  count      : float4-vectorised, coalesced loads of pad-y and time; z = z_max - vdrift*t; bin; shared-memory atomicAdd
//   C  scan       : exclusive scan of the counters in place (serial runs per thread + one block scan) -> cursors
//   D  scatter    : pos = atomicAdd(cursor[bin]); perm[pos] = i (from the shared (y,z) copy, or the same loads again: L2 hits);
//                   the advanced cursors are the bin_start table shifted by one bin
//   E  place      : units held in shared memory: one thread per scattered position ranks its index inside its bin and writes
//                   index and (y, z) to the final position -> ascending original index inside a bin, i.e. the counting sort is
//                   stable and independent of the atomic order.  Larger units: E1 one thread per bin insertion-sorts its
//                   (about one) entries, E2 one thread per sorted position gathers float2 (y, z), coalesced
// Algorithmic HBM bytes per cluster: 8 read (y,t) + 8 (yz) + 4 (perm) + ~4 (bin_start) written = 24.
#include "tpc_internal.cuh"

namespace tpc {
namespace {

// Calls f(i, y, t) for every cluster i in [0,n) of a unit whose arrays start at element offset `src` (float4 body when aligned).
template <class F>
__device__ __forceinline__ void for_each_cluster(const float* __restrict__ in_y, const float* __restrict__ in_t, long long src, int n,
                                                 F&& f) {
  const float* py = in_y + src;
  const float* pt = in_t + src;
  int head = (int)((4 - (src & 3)) & 3);
  if (head > n) head = n;
  const int nvec = (n - head) >> 2;
  const int tail0 = head + (nvec << 2);
  if ((int)threadIdx.x < head) f((int)threadIdx.x, py[threadIdx.x], pt[threadIdx.x]);
  const float4* vy = reinterpret_cast<const float4*>(py + head);
  const float4* vt = reinterpret_cast<const float4*>(pt + head);
  for (int v = threadIdx.x; v < nvec; v += blockDim.x) {
    float4 a = __ldg(vy + v), b = __ldg(vt + v);
    int i = head + (v << 2);
    f(i, a.x, b.x); f(i + 1, a.y, b.y); f(i + 2, a.z, b.z); f(i + 3, a.w, b.w);
  }
  int i = tail0 + threadIdx.x;
  if (i < n) f(i, py[i], pt[i]);
}

__global__ void __launch_bounds__(1024, 2) k1_grid_build(const UnitDesc* __restrict__ units, const float* __restrict__ in_y,
                                                       const float* __restrict__ in_t, float2* __restrict__ yz,
                                                       int* __restrict__ perm, int* __restrict__ bin_start, int* __restrict__ cursor_g,
                                                       const float zmax, const float vdrift, const int smem_ints) {
  extern __shared__ __align__(16) int s_cnt[];
  __shared__ int s_warp[33];
  const UnitDesc d = units[blockIdx.x];
  const int n = d.n, ny = d.ny, nz = d.nz, nb = ny * nz;
  int* __restrict__ bs = bin_start + d.bin_off;
  if (n == 0) {
    for (int b = threadIdx.x; b <= nb; b += blockDim.x) bs[b] = 0;
    return;
  }
  // Shared-memory plan of this unit (ints): [0, nb) bin counters / cursors; then, when they fit, the sorted original
  // indices (n) and the unit's (y, z) pairs (2n, 8-byte aligned).  Units too large for that keep them in global memory (L2).
  const bool cnt_s = d.cur_off < 0;
  const int perm_at = (nb + 1) & ~1;
  const bool perm_s = cnt_s && perm_at + n <= smem_ints;
  const int yz_at = (perm_at + n + 1) & ~1;
  const bool yz_s = perm_s && yz_at + 2 * n <= smem_ints;
  int* cnt = cnt_s ? s_cnt : cursor_g + d.cur_off;
  int* __restrict__ pg = perm + d.off;
  int* pm = perm_s ? s_cnt + perm_at : pg;
  float2* syz = reinterpret_cast<float2*>(s_cnt + yz_at);
  for (int b = threadIdx.x; b < nb; b += blockDim.x) cnt[b] = 0;
  __syncthreads();

  // B: count.  S0: product rounded, then subtracted (no FMA).
  for_each_cluster(in_y, in_t, d.src, n, [&](int i, float y, float t) {
    float z = __fsub_rn(zmax, __fmul_rn(vdrift, t));
    int b = bin_of(z, d.zlo, d.invs, nz) * ny + bin_of(y, d.ylo, d.invs, ny);
    if (yz_s) syz[i] = make_float2(y, z);
    atomicAdd(&cnt[b], 1);
  });
  __syncthreads();

  // C: exclusive scan of the counters in place (cnt[b] = start of bin b): every thread scans a run of consecutive bins
  //    serially, one block scan joins the runs.  bin_start is written after pass D from the advanced cursors.
  {
    const int K = (nb + (int)blockDim.x - 1) / (int)blockDim.x;
    const int b0 = min((int)threadIdx.x * K, nb), b1 = min(b0 + K, nb);
    int sum = 0;
#pragma unroll 2
    for (int b = b0; b < b1; b++) sum += cnt[b];
    int total;
    int ex = block_excl_scan(sum, s_warp, &total);
#pragma unroll 2
    for (int b = b0; b < b1; b++) { const int v = cnt[b]; cnt[b] = ex; ex += v; }
  }
  __syncthreads();

  // D: scatter original indices to their bins (order inside a bin arbitrary here).
  if (yz_s) {
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      const float2 c = syz[i];
      int b = bin_of(c.y, d.zlo, d.invs, nz) * ny + bin_of(c.x, d.ylo, d.invs, ny);
      pm[atomicAdd(&cnt[b], 1)] = i;
    }
  } else {
    for_each_cluster(in_y, in_t, d.src, n, [&](int i, float y, float t) {
      float z = __fsub_rn(zmax, __fmul_rn(vdrift, t));
      int b = bin_of(z, d.zlo, d.invs, nz) * ny + bin_of(y, d.ylo, d.invs, ny);
      pm[atomicAdd(&cnt[b], 1)] = i;
    });
  }
  __syncthreads();

  // after D the cursor of bin b stands at the end of bin b = the start of bin b+1: bin_start, coalesced
  for (int b = threadIdx.x; b < nb; b += blockDim.x) bs[b + 1] = cnt[b];
  if (threadIdx.x == 0) bs[0] = 0;
  float2* __restrict__ out = yz + d.off;
  // E (units whose scattered indices are in shared memory): stable placement and payload in one pass, one thread per
  // scattered position.  Position p holds original index i of bin b; its final position is start(b) + #{q in bin b : index at
  // q < i}, so the order inside a bin is ascending original index whatever order the atomics of pass D produced.  Writes
  // stay inside the bin's range.  (y, z) from the shared copy, or re-read from the input (L2) for the larger units.
  if (yz_s) {
    for (int p = threadIdx.x; p < n; p += blockDim.x) {
      const int i = pm[p];
      const float2 c = syz[i];
      const int b = bin_of(c.y, d.zlo, d.invs, nz) * ny + bin_of(c.x, d.ylo, d.invs, ny);
      const int lo = b ? cnt[b - 1] : 0, hi = cnt[b];   // after D, cursor[b] = end of bin b
      int rank = 0;
#pragma unroll 2
      for (int q = lo; q < hi; q++) rank += pm[q] < i;
      pg[lo + rank] = i;
      out[lo + rank] = c;
    }
    return;
  }
  if (perm_s) {
    const float* py = in_y + d.src;
    const float* pt = in_t + d.src;
    for (int p = threadIdx.x; p < n; p += blockDim.x) {
      const int i = pm[p];
      const float2 c = make_float2(py[i], __fsub_rn(zmax, __fmul_rn(vdrift, pt[i])));
      const int b = bin_of(c.y, d.zlo, d.invs, nz) * ny + bin_of(c.x, d.ylo, d.invs, ny);
      const int lo = b ? cnt[b - 1] : 0, hi = cnt[b];
      int rank = 0;
#pragma unroll 2
      for (int q = lo; q < hi; q++) rank += pm[q] < i;
      pg[lo + rank] = i;
      out[lo + rank] = c;
    }
    return;
  }

  // E1: canonical order inside each bin = ascending original index (insertion sort; bins hold about one cluster).
  for (int b = threadIdx.x; b < nb; b += blockDim.x) {
    const int lo = b ? cnt[b - 1] : 0, hi = cnt[b];   // after D, cursor[b] = end of bin b
    for (int i = lo + 1; i < hi; i++) {
      int v = pm[i], j = i - 1;
      while (j >= lo && pm[j] > v) { pm[j + 1] = pm[j]; j--; }
      pm[j + 1] = v;
    }
  }
  __syncthreads();

  // E2: sorted payload, coalesced writes.
  const float* py = in_y + d.src;
  const float* pt = in_t + d.src;
  for (int p = threadIdx.x; p < n; p += blockDim.x) {
    const int i = pm[p];
    out[p] = make_float2(py[i], __fsub_rn(zmax, __fmul_rn(vdrift, pt[i])));
  }
}

}  // namespace

int launch_k1_grid(const Launch& L, int U, const UnitDesc* d_units, const float* d_in_y, const float* d_in_t, float2* d_yz,
                   int* d_perm, int* d_bin_start, int* d_cursor, const Params& P, int max_cursor_ints_smem, int max_n,
                   int max_perm_ints, int max_yz_ints) {
  if (U <= 0) return 0;
  int threads = 128;
  while (threads < 1024 && threads * 16 < max_n) threads <<= 1;   // about 8-16 clusters per thread and pass: small CTAs, more of them per SM
  // Shared memory per CTA: the cursors always; the sorted indices and the (y, z) pairs too while that keeps >= 4 CTAs per SM
  // (56 KB); the sorted indices alone up to 192 KB (one 1024-thread CTA per SM for 20 k-cluster units).
  int ints = max_cursor_ints_smem;
  if (max_yz_ints <= 14 * 1024) ints = ints > max_yz_ints ? ints : max_yz_ints;
  else if (max_perm_ints <= 48 * 1024) ints = ints > max_perm_ints ? ints : max_perm_ints;
  size_t smem = (size_t)ints * sizeof(int);
  if (smem > 48 * 1024) {
    cudaError_t e = cudaFuncSetAttribute(k1_grid_build, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return -(int)e;
  }
  k1_grid_build<<<U, threads, smem, L.stream>>>(d_units, d_in_y, d_in_t, d_yz, d_perm, d_bin_start, d_cursor, P.zmax, P.vdrift, ints);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 1 : -(int)e;
}

}  // namespace tpc
