// k3_clean_start.cu -- K3: S3 mutual-link cleaner + S4 start-hit finder with prefix-sum compaction.
//
// k3_clean_flag : one thread per cluster.  A link survives iff it is mutual (up[h]=u and dn[u]=h).  The tables are cleaned IN
//                 PLACE with no atomics and no second buffer: an entry only ever changes from a non-mutual value to -1, and the
//                 mutuality test gives the same answer whether it reads the raw value or the already cleaned -1, so any thread
//                 order produces the same tables.  The same thread then decides whether h starts a chain (no down link, an up
//                 link, at least min_seed clusters when following cleaned up links -- cleanedness of the links it walks over is
//                 evaluated on the fly by the same mutuality test) and the warp ballots the decision into a bit mask.
// scan          : exclusive prefix sum over the per-item counts (scan.cu).
// k3_compact    : one warp per item turns the bit mask into the ordered start-hit list (ascending sector,row,sorted position).
// Algorithmic HBM bytes per cluster: 8 (own links) + 8 (partner links, gathered) + <=8 (rewritten links) + 1/8 (mask) ~ 24.
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int K3_THREADS = 256;

// cleaned up-link of sorted position p of unit uu (row rr): the raw link if mutual, else -1
__device__ __forceinline__ int clean_up_of(const UnitDesc* __restrict__ units, const int* link_up, const int* link_dn, int uu, int rr,
                                           int R, long long off_uu, int p) {
  const int up = link_up[off_uu + p];
  if (up < 0 || rr + 1 >= R) return -1;
  return link_dn[units[uu + 1].off + up] == p ? up : -1;
}

__global__ void __launch_bounds__(K3_THREADS) k3_clean_flag(const Item* __restrict__ items, const int chunk,
                                                            const UnitDesc* __restrict__ units, int* link_up, int* link_dn,
                                                            unsigned* __restrict__ mask, int* __restrict__ item_count, const int R,
                                                            const int min_seed) {
  __shared__ int s_count;
  const Item it = items[blockIdx.x];
  const int u = it.unit, r = u % R;
  const UnitDesc d = units[u];
  const int cnt = min(chunk, d.n - it.start);
  const int words = chunk >> 5;
  if (threadIdx.x == 0) s_count = 0;
  __syncthreads();
  int my_count = 0;
  for (int base = 0; base < chunk; base += blockDim.x) {   // whole warps stay together for the ballot
    const int k = base + threadIdx.x;
    bool start = false;
    if (k < cnt) {
      const int h = it.start + k;
      const long long g = d.off + h;
      const int up = link_up[g], dn = link_dn[g];
      int cu = -1, cd = -1;
      if (up >= 0 && r + 1 < R && link_dn[units[u + 1].off + up] == h) cu = up;
      if (dn >= 0 && r > 0 && link_up[units[u - 1].off + dn] == h) cd = dn;
      if (cu != up) link_up[g] = -1;
      if (cd != dn) link_dn[g] = -1;
      if (cd < 0 && cu >= 0) {   // S4: chain of at least min_seed clusters starting here
        int len = 2, uu = u + 1, p = cu;
        while (len < min_seed) {
          const int nx = clean_up_of(units, link_up, link_dn, uu, uu % R, R, units[uu].off, p);
          if (nx < 0) break;
          p = nx; uu++; len++;
        }
        start = len >= min_seed;
      }
    }
    const unsigned m = __ballot_sync(0xffffffffu, start);
    if ((threadIdx.x & 31) == 0 && (k >> 5) < words) {
      mask[(long long)blockIdx.x * words + (k >> 5)] = m;
      my_count += __popc(m);
    }
  }
  if ((threadIdx.x & 31) == 0 && my_count) atomicAdd(&s_count, my_count);
  __syncthreads();
  if (threadIdx.x == 0) item_count[blockIdx.x] = s_count;
}

__global__ void __launch_bounds__(K3_THREADS) k3_compact(const Item* __restrict__ items, const int n_items, const int chunk,
                                                         const unsigned* __restrict__ mask, const int* __restrict__ item_base,
                                                         int* __restrict__ start_unit, int* __restrict__ start_pos) {
  const int lane = threadIdx.x & 31;
  const int item = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (item >= n_items) return;
  const Item it = items[item];
  const int words = chunk >> 5;
  int base = item_base[item];
  for (int w0 = 0; w0 < words; w0 += 32) {
    const int w = w0 + lane;
    unsigned m = w < words ? mask[(long long)item * words + w] : 0u;
    const int c = __popc(m);
    const int inc = warp_incl_scan(c, lane);
    int o = base + inc - c;
    while (m) {
      const int b = __ffs(m) - 1;
      m &= m - 1;
      start_unit[o] = it.unit;
      start_pos[o] = it.start + (w << 5) + b;
      o++;
    }
    base += __shfl_sync(0xffffffffu, inc, 31);
  }
}

}  // namespace

int launch_k3_clean_start(const Launch& L, int n_items, const Item* d_items, int chunk, const UnitDesc* d_units, int* d_link_up,
                          int* d_link_dn, unsigned* d_mask, int* d_item_count, int* d_item_base, int* d_scan_tmp,
                          int* d_start_unit, int* d_start_pos, int* d_total, const Params& P) {
  if (n_items <= 0) {
    cudaError_t e = cudaMemsetAsync(d_total, 0, sizeof(int), L.stream);
    return e == cudaSuccess ? 0 : -(int)e;
  }
  k3_clean_flag<<<n_items, K3_THREADS, 0, L.stream>>>(d_items, chunk, d_units, d_link_up, d_link_dn, d_mask, d_item_count, P.R,
                                                       P.min_seed);
  int rc = launch_scan_i32(L, d_item_count, d_item_base, n_items, d_scan_tmp, d_total);
  if (rc < 0) return rc;
  const int warps = K3_THREADS / 32;
  k3_compact<<<(n_items + warps - 1) / warps, K3_THREADS, 0, L.stream>>>(d_items, n_items, chunk, d_mask, d_item_base, d_start_unit,
                                                                        d_start_pos);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 2 + rc : -(int)e;
}

}  // namespace tpc
