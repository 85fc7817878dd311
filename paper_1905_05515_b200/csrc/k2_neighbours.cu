// k2_neighbours.cu -- K2: S2 neighbour finder (Cellular-Automaton seeding; definition in DESIGN.md section 4).
//
// For every cluster h of row r (1 <= r <= R-2): the best (up, down) pair on rows r+1 / r-1 by the collinearity residual D, the
// two search windows centred on the projection of h from the origin ("all tracks are primaries coming from the origin").
//
// One CTA per work item = a chunk of consecutive sorted clusters of one (sector,row).  Because the S1 order is z-major, the
// clusters and bins of rows r+1 / r-1 that any window of the chunk can touch are ONE contiguous slab of each row's sorted
// arrays.  Phase 1 finds the slab (block min/max of the window bin rows), thread 0 issues up to four 1-D TMA bulk copies
// (cp.async.bulk, mbarrier complete_tx) that stage the slabs (float2 clusters + bin_start) in shared memory, phase 2 runs
// the window scan and the pair search out of shared memory.  A slab that does not fit falls back to global (L2) reads.
// All decision arithmetic (window bounds, membership, ey, ez, D, D < thr, argmin with index tie-break) is spelled with
// explicit round-to-nearest intrinsics: no FMA contraction, same operation order as the definition -> bit-exact link tables.
// Algorithmic HBM bytes per cluster: 8 (own float2) + 4 (bin table) + 8 (two links written) = 20, rows r+-1 reused from L2/smem.
#include <limits.h>
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int K2_THREADS = 256;
constexpr int K2_STAGE_BYTES = 64 * 1024;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// 1-D TMA bulk copy global -> shared; dst, src 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "K2_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra K2_DONE;\n"
      "bra K2_WAIT;\n"
      "K2_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

struct Stage {          // written by thread 0, read by all
  int staged;
  int pshift_u, pshift_d, bshift_u, bshift_d;
  int hoff_d, boff_u, boff_d;   // byte offsets of the four regions in the staging buffer (hits_u at 0)
};

__global__ void __launch_bounds__(K2_THREADS) k2_neighbours(const Item* __restrict__ items, const int chunk,
                                                            const UnitDesc* __restrict__ units, const RowConst* __restrict__ rows,
                                                            const float2* __restrict__ yz, const int* __restrict__ perm,
                                                            const int* __restrict__ bin_start, int* __restrict__ link_up,
                                                            int* __restrict__ link_dn, const Params P) {
  extern __shared__ __align__(128) unsigned char s_stage[];
  __shared__ __align__(8) uint64_t s_bar;
  __shared__ int s_red[4];
  __shared__ Stage s_st;

  const Item it = items[blockIdx.x];
  const int u = it.unit, r = u % P.R;
  const UnitDesc d = units[u];
  const int cnt = min(chunk, d.n - it.start);
  int* __restrict__ lup = link_up + d.off + it.start;
  int* __restrict__ ldn = link_dn + d.off + it.start;
  const float2* __restrict__ own = yz + d.off + it.start;

  bool searchable = r >= 1 && r <= P.R - 2;
  UnitDesc du, dd;
  if (searchable) { du = units[u + 1]; dd = units[u - 1]; searchable = du.n > 0 && dd.n > 0; }
  if (!searchable) {   // rows 0 and R-1 search nothing; an empty neighbour row leaves no pair
    for (int k = threadIdx.x; k < cnt; k += blockDim.x) { lup[k] = -1; ldn[k] = -1; }
    return;
  }
  const RowConst rc = rows[r];
  const float hw_u = P.continuous ? rc.wzu : P.wz, hw_d = P.continuous ? rc.wzd : P.wz;

  if (threadIdx.x == 0) {
    s_red[0] = INT_MAX; s_red[1] = -1; s_red[2] = INT_MAX; s_red[3] = -1;
    mbar_init(&s_bar, 1);
    mbar_fence_init();
  }
  __syncthreads();

  // ---- phase 1: bin rows of rows r+1 / r-1 touched by any window of this chunk
  {
    int mnu = INT_MAX, mxu = -1, mnd = INT_MAX, mxd = -1;
    for (int k = threadIdx.x; k < cnt; k += blockDim.x) {
      const float z = own[k].y;
      const float zcu = P.continuous ? z : __fmul_rn(z, rc.tu), zcd = P.continuous ? z : __fmul_rn(z, rc.td);
      mnu = min(mnu, bin_of(__fsub_rn(zcu, hw_u), du.zlo, du.invs, du.nz));
      mxu = max(mxu, bin_of(__fadd_rn(zcu, hw_u), du.zlo, du.invs, du.nz));
      mnd = min(mnd, bin_of(__fsub_rn(zcd, hw_d), dd.zlo, dd.invs, dd.nz));
      mxd = max(mxd, bin_of(__fadd_rn(zcd, hw_d), dd.zlo, dd.invs, dd.nz));
    }
    mnu = __reduce_min_sync(0xffffffffu, mnu); mxu = __reduce_max_sync(0xffffffffu, mxu);
    mnd = __reduce_min_sync(0xffffffffu, mnd); mxd = __reduce_max_sync(0xffffffffu, mxd);
    if ((threadIdx.x & 31) == 0) {
      atomicMin(&s_red[0], mnu); atomicMax(&s_red[1], mxu); atomicMin(&s_red[2], mnd); atomicMax(&s_red[3], mxd);
    }
  }
  __syncthreads();

  // ---- staging: thread 0 sizes the two slabs and issues the TMA bulk copies
  if (threadIdx.x == 0) {
    Stage st;
    const int bz0u = s_red[0], bz1u = max(s_red[1], s_red[0]), bz0d = s_red[2], bz1d = max(s_red[3], s_red[2]);
    const long long gbu = du.bin_off + (long long)bz0u * du.ny, gbd = dd.bin_off + (long long)bz0d * dd.ny;
    const int nbu = (bz1u - bz0u + 1) * du.ny + 1, nbd = (bz1d - bz0d + 1) * dd.ny + 1;
    const int p0u = bin_start[gbu], p1u = bin_start[gbu + nbu - 1], p0d = bin_start[gbd], p1d = bin_start[gbd + nbd - 1];
    const long long hau0 = (du.off + p0u) & ~1LL, hau1 = (du.off + p1u + 1) & ~1LL;
    const long long had0 = (dd.off + p0d) & ~1LL, had1 = (dd.off + p1d + 1) & ~1LL;
    const long long bau0 = gbu & ~3LL, bau1 = (gbu + nbu + 3) & ~3LL, bad0 = gbd & ~3LL, bad1 = (gbd + nbd + 3) & ~3LL;
    const long long hbu = (hau1 - hau0) * 8, hbd = (had1 - had0) * 8, bbu = (bau1 - bau0) * 4, bbd = (bad1 - bad0) * 4;
    st.staged = hbu + hbd + bbu + bbd <= (long long)K2_STAGE_BYTES;
    if (st.staged) {
      st.pshift_u = (int)(hau0 - du.off); st.pshift_d = (int)(had0 - dd.off);
      st.bshift_u = (int)(bau0 - du.bin_off); st.bshift_d = (int)(bad0 - dd.bin_off);
      st.hoff_d = (int)hbu; st.boff_u = (int)(hbu + hbd); st.boff_d = (int)(hbu + hbd + bbu);
      mbar_expect_tx(&s_bar, (uint32_t)(hbu + hbd + bbu + bbd));
      if (hbu) tma_load_1d(s_stage, yz + hau0, (uint32_t)hbu, &s_bar);
      if (hbd) tma_load_1d(s_stage + st.hoff_d, yz + had0, (uint32_t)hbd, &s_bar);
      tma_load_1d(s_stage + st.boff_u, bin_start + bau0, (uint32_t)bbu, &s_bar);
      tma_load_1d(s_stage + st.boff_d, bin_start + bad0, (uint32_t)bbd, &s_bar);
    } else {
      st.pshift_u = st.pshift_d = st.bshift_u = st.bshift_d = 0; st.hoff_d = st.boff_u = st.boff_d = 0;
    }
    s_st = st;
  }
  __syncthreads();
  const Stage st = s_st;
  const float2* yzu; const float2* yzd; const int* bsu; const int* bsd;
  if (st.staged) {
    yzu = reinterpret_cast<const float2*>(s_stage); yzd = reinterpret_cast<const float2*>(s_stage + st.hoff_d);
    bsu = reinterpret_cast<const int*>(s_stage + st.boff_u); bsd = reinterpret_cast<const int*>(s_stage + st.boff_d);
    mbar_wait(&s_bar, 0);
  } else {
    yzu = yz + du.off; yzd = yz + dd.off; bsu = bin_start + du.bin_off; bsd = bin_start + dd.bin_off;
  }
  const int psu = st.pshift_u, psd = st.pshift_d, bsu_s = st.bshift_u, bsd_s = st.bshift_d;
  const int* __restrict__ permu = perm + du.off;
  const int* __restrict__ permd = perm + dd.off;

  // ---- phase 2: window scan + best pair, one thread per cluster
  for (int k = threadIdx.x; k < cnt; k += blockDim.x) {
    const float2 h = own[k];
    const float y = h.x, z = h.y;
    // up window (row r+1)
    const float ycu = __fmul_rn(y, rc.tu), zcu = P.continuous ? z : __fmul_rn(z, rc.tu);
    const float ylou = __fsub_rn(ycu, P.wy), yhiu = __fadd_rn(ycu, P.wy), zlou = __fsub_rn(zcu, hw_u), zhiu = __fadd_rn(zcu, hw_u);
    const int by0u = bin_of(ylou, du.ylo, du.invs, du.ny), by1u = bin_of(yhiu, du.ylo, du.invs, du.ny);
    const int bz0u = bin_of(zlou, du.zlo, du.invs, du.nz), bz1u = bin_of(zhiu, du.zlo, du.invs, du.nz);
    // down window (row r-1)
    const float ycd = __fmul_rn(y, rc.td), zcd = P.continuous ? z : __fmul_rn(z, rc.td);
    const float ylod = __fsub_rn(ycd, P.wy), yhid = __fadd_rn(ycd, P.wy), zlod = __fsub_rn(zcd, hw_d), zhid = __fadd_rn(zcd, hw_d);
    const int by0d = bin_of(ylod, dd.ylo, dd.invs, dd.ny), by1d = bin_of(yhid, dd.ylo, dd.invs, dd.ny);
    const int bz0d = bin_of(zlod, dd.zlo, dd.invs, dd.nz), bz1d = bin_of(zhid, dd.zlo, dd.invs, dd.nz);

    bool have = false; float bestD = 0.0f; int bu = -1, bd = -1;
    for (int bz = bz0u; bz <= bz1u; bz++) {
      const int pa = bsu[bz * du.ny + by0u - bsu_s], pb = bsu[bz * du.ny + by1u + 1 - bsu_s];
      for (int p = pa; p < pb; p++) {
        const float2 cu = yzu[p - psu];
        if (!(cu.x >= ylou && cu.x <= yhiu && cu.y >= zlou && cu.y <= zhiu)) continue;
        const float m1 = __fmul_rn(rc.b, __fsub_rn(cu.x, y)), m3 = __fmul_rn(rc.b, __fsub_rn(cu.y, z));
        for (int bzd = bz0d; bzd <= bz1d; bzd++) {
          const int qa = bsd[bzd * dd.ny + by0d - bsd_s], qb = bsd[bzd * dd.ny + by1d + 1 - bsd_s];
          for (int q = qa; q < qb; q++) {
            const float2 cd = yzd[q - psd];
            if (!(cd.x >= ylod && cd.x <= yhid && cd.y >= zlod && cd.y <= zhid)) continue;
            const float ey = __fsub_rn(m1, __fmul_rn(rc.a, __fsub_rn(y, cd.x)));
            const float ez = __fsub_rn(m3, __fmul_rn(rc.a, __fsub_rn(z, cd.y)));
            const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));
            bool better = !have || D < bestD;
            if (have && D == bestD) {   // tie: lower original index of the up cluster, then of the down cluster (rare: global reads)
              const int iu = permu[p], ib = permu[bu];
              better = iu < ib || (iu == ib && permd[q] < permd[bd]);
            }
            if (better) { have = true; bestD = D; bu = p; bd = q; }
          }
        }
      }
    }
    const bool ok = have && bestD < rc.thr;
    lup[k] = ok ? bu : -1;
    ldn[k] = ok ? bd : -1;
  }
}

}  // namespace

int launch_k2_neighbours(const Launch& L, int n_items, const Item* d_items, int chunk, const UnitDesc* d_units,
                         const RowConst* d_rows, const float2* d_yz, const int* d_perm, const int* d_bin_start, int* d_link_up,
                         int* d_link_dn, const Params& P) {
  if (n_items <= 0) return 0;
  {
    cudaError_t e = cudaFuncSetAttribute(k2_neighbours, cudaFuncAttributeMaxDynamicSharedMemorySize, K2_STAGE_BYTES);
    if (e != cudaSuccess) return -(int)e;
  }
  k2_neighbours<<<n_items, K2_THREADS, K2_STAGE_BYTES, L.stream>>>(d_items, chunk, d_units, d_rows, d_yz, d_perm, d_bin_start,
                                                                    d_link_up, d_link_dn, P);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 1 : -(int)e;
}

}  // namespace tpc
