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

// cleaned down-link of sorted position p of unit uu (row rr >= 1): the raw link if mutual, else -1
__device__ __forceinline__ int clean_dn_of(const UnitDesc* __restrict__ units, const int* link_up, const int* link_dn, int uu, int rr,
                                           long long off_uu, int p) {
  const int dn = link_dn[off_uu + p];
  if (dn < 0 || rr < 1) return -1;
  return link_up[units[uu - 1].off + dn] == p ? dn : -1;
}

// S4' seed bridging (NEXT-2 of SURVEY.md section 8(f); reading A39 of DESIGN.md; off unless bridge_rows > 0).  The start hit h
// of unit u (row r) continues a lower chain -- and is dropped (k3_bridge_flag / k3_bridge_filter below) -- when the straight line through h and its second chain cluster
// (row r+2), extended down to a row r-g (2 <= g <= bridge_rows), meets the TOP c of a chain of at least bridge_min clusters, and
// the line through c and its second cluster below, extended up to row r, meets h; both within (bridge_wy, bridge_wz).
// Every fp32 operation is spelled in the order of the definition (library built with -fmad=false); links are tested for
// mutuality on the fly, which gives the same answer on raw and on already cleaned tables.
__device__ bool seed_bridged(const UnitDesc* __restrict__ units, const RowConst* __restrict__ rows, const float2* __restrict__ yz,
                             const int* __restrict__ bin_start, const int* link_up, const int* link_dn, const int u, const int r,
                             const int R, const int h, const int u1, const Params& P) {
  if (r + 2 >= R) return false;
  const long long off0 = units[u].off, off1 = units[u + 1].off, off2 = units[u + 2].off;
  const int u2 = clean_up_of(units, link_up, link_dn, u + 1, r + 1, R, off1, u1);
  if (u2 < 0) return false;
  const float2 ch = yz[off0 + h], c2 = yz[off2 + u2];
  const float x_r = rows[r].x;
  const float dxu = rows[r + 2].x - x_r;
  const float sy = (c2.x - ch.x) / dxu, sz = (c2.y - ch.y) / dxu;
  // probed rows in the order 4, 2, 3, 5, 6, ...: one missing cluster leaves exactly four rows between the chains, so most bridged
  // start hits are decided by the first probe ("some row matches" does not depend on the order)
  for (int k = 2; k <= P.bridge_rows; k++) {
    const int g = P.bridge_rows < 4 ? k : (k == 2 ? 4 : (k <= 4 ? k - 1 : k));
    if (r - g < 2) continue;
    const int ud = u - g;
    const UnitDesc d = units[ud];
    if (d.n == 0) continue;
    const float dx = x_r - rows[r - g].x;
    const float yp = ch.x - sy * dx, zp = ch.y - sz * dx;
    const float ylo = yp - P.bridge_wy, yhi = yp + P.bridge_wy, zlo = zp - P.bridge_wz, zhi = zp + P.bridge_wz;
    const int by0 = bin_of(ylo, d.ylo, d.invs, d.ny), by1 = bin_of(yhi, d.ylo, d.invs, d.ny);
    const int bz0 = bin_of(zlo, d.zlo, d.invs, d.nz), bz1 = bin_of(zhi, d.zlo, d.invs, d.nz);
    const int* __restrict__ bs = bin_start + d.bin_off;
    const long long offm1 = units[ud - 1].off, offm2 = units[ud - 2].off;
    for (int bz = bz0; bz <= bz1; bz++) {
      const int pe = bs[bz * d.ny + by1 + 1];
      for (int c = bs[bz * d.ny + by0]; c < pe; c++) {
        const float2 cc = yz[d.off + c];
        if (!(cc.x >= ylo && cc.x <= yhi && cc.y >= zlo && cc.y <= zhi)) continue;
        if (clean_up_of(units, link_up, link_dn, ud, r - g, R, d.off, c) >= 0) continue;      // c must be the top of its chain
        const int d1 = clean_dn_of(units, link_up, link_dn, ud, r - g, d.off, c);
        if (d1 < 0) continue;
        const int d2 = clean_dn_of(units, link_up, link_dn, ud - 1, r - g - 1, offm1, d1);
        if (d2 < 0) continue;
        int len = 3, uu = ud - 2, p = d2;
        while (len < P.bridge_min) {
          const int rr = uu % R;
          if (rr == 0) break;
          const int nx = clean_dn_of(units, link_up, link_dn, uu, rr, units[uu].off, p);
          if (nx < 0) break;
          p = nx; uu--; len++;
        }
        if (len < P.bridge_min) continue;
        const float2 cb = yz[offm2 + d2];
        const float dxd = rows[r - g].x - rows[r - g - 2].x;
        const float ty = (cc.x - cb.x) / dxd, tz = (cc.y - cb.y) / dxd;
        const float yq = cc.x + ty * dx, zq = cc.y + tz * dx;
        if (ch.x >= yq - P.bridge_wy && ch.x <= yq + P.bridge_wy && ch.y >= zq - P.bridge_wz && ch.y <= zq + P.bridge_wz) return true;
      }
    }
  }
  return false;
}

// S2' tables (link_skip = 1): an entry is (position << 1 | k - 1), k = row distance of the link.  Cleaned up-link of sorted position
// p of unit uu (row rr): the raw entry if the partner k rows up points back with the same entry shape, else -1.
__device__ __forceinline__ int clean_up_enc(const UnitDesc* __restrict__ units, const int* link_up, const int* link_dn, int uu, int rr,
                                            int R, long long off_uu, int p) {
  const int e = link_up[off_uu + p];
  if (e < 0) return -1;
  const int k = (e & 1) + 1;
  if (rr + k >= R) return -1;
  return link_dn[units[uu + k].off + (e >> 1)] == ((p << 1) | (k - 1)) ? e : -1;
}

__global__ void __launch_bounds__(K3_THREADS) k3_clean_flag(const Item* __restrict__ items, const int chunk,
                                                            const UnitDesc* __restrict__ units, int* link_up, int* link_dn,
                                                            unsigned* __restrict__ mask, int* __restrict__ item_count,
                                                            const Params P) {
  const int R = P.R, min_seed = P.min_seed;
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
      TPC_CHECK(P, P.link_skip || ((up < 0 || (r + 1 < R && up < units[u + 1].n)) && (dn < 0 || (r > 0 && dn < units[u - 1].n))), 31);
      if (!P.link_skip) {
        if (up >= 0 && r + 1 < R && link_dn[units[u + 1].off + up] == h) cu = up;
        if (dn >= 0 && r > 0 && link_up[units[u - 1].off + dn] == h) cd = dn;
      } else {   // S2' entries carry the row distance: mutual iff the partner k rows away holds (h, k)
        if (up >= 0) { const int k = (up & 1) + 1; if (r + k < R && link_dn[units[u + k].off + (up >> 1)] == ((h << 1) | (k - 1))) cu = up; }
        if (dn >= 0) { const int k = (dn & 1) + 1; if (r - k >= 0 && link_up[units[u - k].off + (dn >> 1)] == ((h << 1) | (k - 1))) cd = dn; }
      }
      if (cu != up) link_up[g] = -1;
      if (cd != dn) link_dn[g] = -1;
      if (cd < 0 && cu >= 0) {   // S4: chain of at least min_seed clusters starting here
        int len = 2, uu = u + 1, p = cu;
        if (P.link_skip) { uu = u + (cu & 1) + 1; p = cu >> 1; }
        while (len < min_seed) {
          const int nx = P.link_skip ? clean_up_enc(units, link_up, link_dn, uu, uu % R, R, units[uu].off, p)
                                     : clean_up_of(units, link_up, link_dn, uu, uu % R, R, units[uu].off, p);
          if (nx < 0) break;
          if (P.link_skip) { uu += (nx & 1) + 1; p = nx >> 1; } else { p = nx; uu++; }
          len++;
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

// S4' pass (only when bridge_rows > 0), on the finished S4 list and the fully cleaned link tables: one thread per start hit.
__global__ void __launch_bounds__(K3_THREADS) k3_bridge_flag(const int M, const int* __restrict__ start_unit,
                                                             const int* __restrict__ start_pos, const UnitDesc* __restrict__ units,
                                                             const RowConst* __restrict__ rows, const float2* __restrict__ yz,
                                                             const int* __restrict__ bin_start, const int* __restrict__ link_up,
                                                             const int* __restrict__ link_dn, int* __restrict__ keep, const Params P) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  const int u = start_unit[i], h = start_pos[i];
  const int cu = link_up[units[u].off + h];   // cleaned: a start hit has an up link
  keep[i] = seed_bridged(units, rows, yz, bin_start, link_up, link_dn, u, u % P.R, P.R, h, cu, P) ? 0 : 1;
}

// order-preserving filter of the start list: entry i moves to position pos[i] (exclusive scan of keep) when kept
__global__ void __launch_bounds__(K3_THREADS) k3_bridge_filter(const int M, const int* __restrict__ start_unit,
                                                               const int* __restrict__ start_pos, const int* __restrict__ keep,
                                                               const int* __restrict__ pos, int* __restrict__ out_unit,
                                                               int* __restrict__ out_pos) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M || !keep[i]) return;
  out_unit[pos[i]] = start_unit[i];
  out_pos[pos[i]] = start_pos[i];
}

// indices of the set flags, in order: list[pos[i]] = i (pos = exclusive scan of flag)
__global__ void __launch_bounds__(K3_THREADS) k3_index_list(const int M, const int* __restrict__ flag, const int* __restrict__ pos,
                                                            int* __restrict__ list) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < M && flag[i]) list[pos[i]] = i;
}

// a dropped start hit is rescued (fitted in the second wave) unless every cluster of its chain lies on a kept first-wave tracklet,
// i.e. carries an owner key (the first half of the selector, k6_owner, has run over the first wave)
__global__ void __launch_bounds__(K3_THREADS) k3_rescue_flag(const int M, const int* __restrict__ keep, const int* __restrict__ start_unit,
                                                             const int* __restrict__ start_pos, const UnitDesc* __restrict__ units,
                                                             const int* __restrict__ link_up, const unsigned long long* __restrict__ owner,
                                                             int* __restrict__ flag2) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  int f = 0;
  if (!keep[i]) {
    int u = start_unit[i], p = start_pos[i];
    for (;;) {
      const long long g = units[u].off + p;
      if (owner[g] == 0ull) { f = 1; break; }
      const int nx = link_up[g];          // cleaned table
      if (nx < 0) break;
      p = nx; u++;
    }
  }
  flag2[i] = f;
}

}  // namespace

// S4' rescue variant, part 1: keep[i] = start hit i is not bridged; list1 = indices of the kept ones (first wave); *d_total = their number
int launch_k3_bridge_lists(const Launch& L, int M, const int* d_start_unit, const int* d_start_pos, const UnitDesc* d_units,
                           const RowConst* d_rows, const float2* d_yz, const int* d_bin_start, const int* d_link_up, const int* d_link_dn,
                           int* d_keep, int* d_pos, int* d_scan_tmp, int* d_list1, int* d_total, const Params& P) {
  if (M <= 0) {
    cudaError_t e = cudaMemsetAsync(d_total, 0, sizeof(int), L.stream);
    return e == cudaSuccess ? 0 : -(int)e;
  }
  const int blocks = (M + K3_THREADS - 1) / K3_THREADS;
  k3_bridge_flag<<<blocks, K3_THREADS, 0, L.stream>>>(M, d_start_unit, d_start_pos, d_units, d_rows, d_yz, d_bin_start, d_link_up,
                                                      d_link_dn, d_keep, P);
  int rc = launch_scan_i32(L, d_keep, d_pos, M, d_scan_tmp, d_total);
  if (rc < 0) return rc;
  k3_index_list<<<blocks, K3_THREADS, 0, L.stream>>>(M, d_keep, d_pos, d_list1);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 2 + rc : -(int)e;
}

// part 2, after the first wave: list2 = dropped start hits whose chain the first wave left (partly) unused; *d_total = their number
int launch_k3_rescue_list(const Launch& L, int M, const int* d_keep, const int* d_start_unit, const int* d_start_pos,
                          const UnitDesc* d_units, const int* d_link_up, const unsigned long long* d_owner,
                          int* d_flag2, int* d_pos, int* d_scan_tmp, int* d_list2, int* d_total) {
  const int blocks = (M + K3_THREADS - 1) / K3_THREADS;
  k3_rescue_flag<<<blocks, K3_THREADS, 0, L.stream>>>(M, d_keep, d_start_unit, d_start_pos, d_units, d_link_up, d_owner, d_flag2);
  int rc = launch_scan_i32(L, d_flag2, d_pos, M, d_scan_tmp, d_total);
  if (rc < 0) return rc;
  k3_index_list<<<blocks, K3_THREADS, 0, L.stream>>>(M, d_flag2, d_pos, d_list2);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 2 + rc : -(int)e;
}

int launch_k3_bridge(const Launch& L, int M, const int* d_start_unit, const int* d_start_pos, const UnitDesc* d_units,
                     const RowConst* d_rows, const float2* d_yz, const int* d_bin_start, const int* d_link_up, const int* d_link_dn,
                     int* d_keep, int* d_keep_pos, int* d_scan_tmp, int* d_out_unit, int* d_out_pos, int* d_total, const Params& P) {
  if (M <= 0) {
    cudaError_t e = cudaMemsetAsync(d_total, 0, sizeof(int), L.stream);
    return e == cudaSuccess ? 0 : -(int)e;
  }
  const int blocks = (M + K3_THREADS - 1) / K3_THREADS;
  k3_bridge_flag<<<blocks, K3_THREADS, 0, L.stream>>>(M, d_start_unit, d_start_pos, d_units, d_rows, d_yz, d_bin_start, d_link_up,
                                                      d_link_dn, d_keep, P);
  int rc = launch_scan_i32(L, d_keep, d_keep_pos, M, d_scan_tmp, d_total);
  if (rc < 0) return rc;
  k3_bridge_filter<<<blocks, K3_THREADS, 0, L.stream>>>(M, d_start_unit, d_start_pos, d_keep, d_keep_pos, d_out_unit, d_out_pos);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 2 + rc : -(int)e;
}

int launch_k3_clean_start(const Launch& L, int n_items, const Item* d_items, int chunk, const UnitDesc* d_units, int* d_link_up,
                          int* d_link_dn, unsigned* d_mask, int* d_item_count, int* d_item_base, int* d_scan_tmp,
                          int* d_start_unit, int* d_start_pos, int* d_total, const Params& P) {
  if (n_items <= 0) {
    cudaError_t e = cudaMemsetAsync(d_total, 0, sizeof(int), L.stream);
    return e == cudaSuccess ? 0 : -(int)e;
  }
  k3_clean_flag<<<n_items, K3_THREADS, 0, L.stream>>>(d_items, chunk, d_units, d_link_up, d_link_dn, d_mask, d_item_count, P);
  int rc = launch_scan_i32(L, d_item_count, d_item_base, n_items, d_scan_tmp, d_total);
  if (rc < 0) return rc;
  const int warps = K3_THREADS / 32;
  k3_compact<<<(n_items + warps - 1) / warps, K3_THREADS, 0, L.stream>>>(d_items, n_items, chunk, d_mask, d_item_base, d_start_unit,
                                                                        d_start_pos);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 2 + rc : -(int)e;
}

}  // namespace tpc
