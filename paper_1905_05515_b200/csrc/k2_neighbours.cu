// k2_neighbours.cu -- K2: S2 neighbour finder (Cellular-Automaton seeding; definition in DESIGN.md section 4).
//
// For every cluster h of row r (1 <= r <= R-2): the best (up, down) pair on rows r+1 / r-1 by the collinearity residual D, the
// two search windows centred on the projection of h from the origin ("all tracks are primaries coming from the origin").
//
// One CTA per work item = a chunk of consecutive sorted clusters of one (sector,row).  Because the S1 order is z-major, the
// clusters and bins of rows r+1 / r-1 that any window of the chunk can touch are ONE contiguous slab of each row's sorted
// arrays.  Thread 0 bounds the slab in O(1) from the bin rows of the first and last cluster of the chunk (one bin row of
// safety margin; a superset is all that staging needs), issues up to four 1-D TMA bulk copies (cp.async.bulk, mbarrier
// complete_tx) that stage the slabs (float2 clusters + bin_start) in shared memory, and every thread then runs the window
// scan and the pair search for its clusters out of shared memory.  A slab that does not fit falls back to global (L2) reads.
// The scan is flat: the candidates of the (at most two) bin rows of a window are visited by ONE loop that records the
// in-window ones in a bit mask; the pair search then walks the set bits of the up and down masks (about one each).
// All decision arithmetic (window bounds, membership, ey, ez, D, D < thr, argmin with index tie-break) is spelled with
// explicit round-to-nearest intrinsics: no FMA contraction, same operation order as the definition -> bit-exact link tables.
// Algorithmic HBM bytes per cluster: 8 (own float2) + 4 (bin table) + 8 (two links written) = 20, rows r+-1 reused from L2/smem.
#include <limits.h>
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int K2_THREADS = 256;
constexpr int K2_STAGE_PER_CLUSTER = 40;   // staging bytes per cluster of the chunk: two neighbour slabs of (8 + 4) bytes + margin

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

// One search window on a neighbour row: candidate ranges of its (at most two) bin rows.
struct Win {
  float ylo, yhi, zlo, zhi;
  int a0, n0, a1m, n;  // candidate j < n0 is position a0 + j (bin row 0), else a1m + j (bin row 1; a1m = start - n0); n = total
  bool wide;           // window spans more than two bin rows (tiny bins): generic path
};

__device__ __forceinline__ bool in_win(const float2 c, const Win& w) {
  return c.x >= w.ylo && c.x <= w.yhi && c.y >= w.zlo && c.y <= w.zhi;
}
__device__ __forceinline__ int win_pos(const Win& w, const int j) { return (j < w.n0 ? w.a0 : w.a1m) + j; }

// Window scan + best pair for the `cnt` clusters `own[0..cnt)` of one chunk, one thread per cluster.  yzu / yzd / bsu / bsd are
// indexed by row position / row bin; they point into the staging buffer (shared-memory instance) or into global memory
// (fallback instance) -- the function is inlined at both call sites so that each instance knows its address space.
__device__ __forceinline__ void search_chunk(const float2* __restrict__ yzu, const float2* __restrict__ yzd, const int* __restrict__ bsu,
                                             const int* __restrict__ bsd, const float2* __restrict__ own, const int cnt,
                                             int* __restrict__ lup, int* __restrict__ ldn, const UnitDesc& du, const UnitDesc& dd,
                                             const RowConst& rc, const float hw_u, const float hw_d,
                                             const int* __restrict__ permu, const int* __restrict__ permd, const Params& P) {
  // window on a neighbour row: bounds (one fp32 op each) and the candidate ranges of its bin rows
  auto make_win = [&](const float yc, const float zc, const float hw, const UnitDesc& g, const int* bs) {
    Win w;
    w.ylo = __fsub_rn(yc, P.wy); w.yhi = __fadd_rn(yc, P.wy); w.zlo = __fsub_rn(zc, hw); w.zhi = __fadd_rn(zc, hw);
    const int by0 = bin_of(w.ylo, g.ylo, g.invs, g.ny), by1 = bin_of(w.yhi, g.ylo, g.invs, g.ny);
    const int bz0 = bin_of(w.zlo, g.zlo, g.invs, g.nz), bz1 = bin_of(w.zhi, g.zlo, g.invs, g.nz);
    w.wide = bz1 - bz0 > 1;
    const int ra = bz0 * g.ny;
    w.a0 = bs[ra + by0]; w.n0 = bs[ra + by1 + 1] - w.a0;
    w.a1m = 0; w.n = w.n0;
    if (bz1 > bz0) { const int rb = ra + g.ny; const int a1 = bs[rb + by0]; w.n += bs[rb + by1 + 1] - a1; w.a1m = a1 - w.n0; }
    return w;
  };
  // one flat loop over the candidates of both bin rows of a window: bit j of the result = candidate j lies in the window
  auto scan = [&](const float2* __restrict__ hits, const Win& w) {
    unsigned m = 0u;
#pragma unroll 1
    for (int j = 0; j < w.n; j++) {
      const float2 c = hits[win_pos(w, j)];
      // m |= in_win(c, w) << j, as four chained ordered compares and one predicated OR (NaN compares false, as in in_win)
      asm("{\n.reg .pred p;\n"
          "setp.ge.f32 p, %1, %3;\n"
          "setp.le.and.f32 p, %1, %4, p;\n"
          "setp.ge.and.f32 p, %2, %5, p;\n"
          "setp.le.and.f32 p, %2, %6, p;\n"
          "@p or.b32 %0, %0, %7;\n}"
          : "+r"(m) : "f"(c.x), "f"(c.y), "f"(w.ylo), "f"(w.yhi), "f"(w.zlo), "f"(w.zhi), "r"(1u << j));
    }
    return m;
  };

  for (int k = threadIdx.x; k < cnt; k += blockDim.x) {
    const float2 h = own[k];
    const float y = h.x, z = h.y;
    const Win wu = make_win(__fmul_rn(y, rc.tu), P.continuous ? z : __fmul_rn(z, rc.tu), hw_u, du, bsu);
    const Win wd = make_win(__fmul_rn(y, rc.td), P.continuous ? z : __fmul_rn(z, rc.td), hw_d, dd, bsd);

    bool have = false; float bestD = 0.0f; int bu = -1, bd = -1;
    auto pair = [&](const int p, const float2 cu, const int q, const float2 cd) {
      const float ey = __fsub_rn(__fmul_rn(rc.b, __fsub_rn(cu.x, y)), __fmul_rn(rc.a, __fsub_rn(y, cd.x)));
      const float ez = __fsub_rn(__fmul_rn(rc.b, __fsub_rn(cu.y, z)), __fmul_rn(rc.a, __fsub_rn(z, cd.y)));
      const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));
      TPC_CHECK(P, p >= 0 && p < du.n && q >= 0 && q < dd.n, 21);
      bool better = !have || D < bestD;
      if (have && D == bestD) {   // tie: lower original index of the up cluster, then of the down cluster (rare: global reads)
        const int iu = permu[p], ib = permu[bu];
        better = iu < ib || (iu == ib && permd[q] < permd[bd]);
      }
      if (better) { have = true; bestD = D; bu = p; bd = q; }
    };

    if (!wu.wide && !wd.wide && wu.n <= 32 && wd.n <= 32) {
      // flat scan per side marks the in-window candidates, then the pair search walks the set bits.
      // Down window first: without a down candidate there is no pair and the up scan is skipped.
      const unsigned md = scan(yzd, wd);
      unsigned mu = md ? scan(yzu, wu) : 0u;
      while (mu) {
        const int j = __ffs(mu) - 1; mu &= mu - 1u;
        const int p = win_pos(wu, j);
        const float2 cu = yzu[p];
        unsigned m = md;
        while (m) {
          const int i = __ffs(m) - 1; m &= m - 1u;
          const int q = win_pos(wd, i);
          pair(p, cu, q, yzd[q]);
        }
      }
    } else {
      // generic path (bins smaller than the window, or very dense rows): nested scan over all bin rows of both windows
      const int by0u = bin_of(wu.ylo, du.ylo, du.invs, du.ny), by1u = bin_of(wu.yhi, du.ylo, du.invs, du.ny);
      const int bz0u = bin_of(wu.zlo, du.zlo, du.invs, du.nz), bz1u = bin_of(wu.zhi, du.zlo, du.invs, du.nz);
      const int by0d = bin_of(wd.ylo, dd.ylo, dd.invs, dd.ny), by1d = bin_of(wd.yhi, dd.ylo, dd.invs, dd.ny);
      const int bz0d = bin_of(wd.zlo, dd.zlo, dd.invs, dd.nz), bz1d = bin_of(wd.zhi, dd.zlo, dd.invs, dd.nz);
      for (int bz = bz0u; bz <= bz1u; bz++)
        for (int p = bsu[bz * du.ny + by0u]; p < bsu[bz * du.ny + by1u + 1]; p++) {
          const float2 cu = yzu[p];
          if (!in_win(cu, wu)) continue;
          for (int bzd = bz0d; bzd <= bz1d; bzd++)
            for (int q = bsd[bzd * dd.ny + by0d]; q < bsd[bzd * dd.ny + by1d + 1]; q++) {
              const float2 cd = yzd[q];
              if (in_win(cd, wd)) pair(p, cu, q, cd);
            }
        }
    }
    const bool ok = have && bestD < rc.thr;
    lup[k] = ok ? bu : -1;
    ldn[k] = ok ? bd : -1;
  }
}

__global__ void __launch_bounds__(K2_THREADS) k2_neighbours(const Item* __restrict__ items, const int chunk,
                                                            const UnitDesc* __restrict__ units, const RowConst* __restrict__ rows,
                                                            const float2* __restrict__ yz, const int* __restrict__ perm,
                                                            const int* __restrict__ bin_start, int* __restrict__ link_up,
                                                            int* __restrict__ link_dn, const Params P, const int stage_bytes, const int split) {
  extern __shared__ __align__(128) unsigned char s_stage[];
  __shared__ __align__(8) uint64_t s_bar;
  __shared__ Stage s_st;

  // a K2 CTA covers 1/split of a work item (the items are shared with K3, which wants larger chunks): smaller slabs, more CTAs
  // per SM to overlap the staging latency of one with the search of the others
  Item it = items[blockIdx.x / split];
  it.start += (int)(blockIdx.x % split) * chunk;
  const int u = it.unit, r = u % P.R;
  const UnitDesc d = units[u];
  const int cnt = min(chunk, d.n - it.start);
  if (cnt <= 0) return;
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

  // ---- staging: thread 0 bounds the slabs of rows r+1 / r-1 and issues the TMA bulk copies
  if (threadIdx.x == 0) {
    mbar_init(&s_bar, 1);
    mbar_fence_init();
    // The chunk is sorted by bin (z-major): its clusters lie in the bin rows [bzf, bzl] of this row's grid, hence
    // z in [zA, zB] with one bin row of margin (open-ended at the clamped first / last bin row, which also hold NaN / inf).
    const int bzf = bin_of(own[0].y, d.zlo, d.invs, d.nz), bzl = bin_of(own[cnt - 1].y, d.zlo, d.invs, d.nz);
    const float s = 1.0f / d.invs, inf = __int_as_float(0x7f800000);
    const float zA = bzf <= 0 ? -inf : d.zlo + (float)(bzf - 1) * s;
    const float zB = bzl >= d.nz - 1 ? inf : d.zlo + (float)(bzl + 2) * s;
    const float zAu = P.continuous ? zA : fminf(zA * rc.tu, zA), zBu = P.continuous ? zB : fmaxf(zB * rc.tu, zB);
    const float zAd = P.continuous ? zA : fminf(zA * rc.td, zA), zBd = P.continuous ? zB : fmaxf(zB * rc.td, zB);
    Stage st;
    const int bz0u = bin_of(zAu - hw_u, du.zlo, du.invs, du.nz), bz1u = bin_of(zBu + hw_u, du.zlo, du.invs, du.nz);
    const int bz0d = bin_of(zAd - hw_d, dd.zlo, dd.invs, dd.nz), bz1d = bin_of(zBd + hw_d, dd.zlo, dd.invs, dd.nz);
    const long long gbu = du.bin_off + (long long)bz0u * du.ny, gbd = dd.bin_off + (long long)bz0d * dd.ny;
    const int nbu = (bz1u - bz0u + 1) * du.ny + 1, nbd = (bz1d - bz0d + 1) * dd.ny + 1;
    const int p0u = bin_start[gbu], p1u = bin_start[gbu + nbu - 1], p0d = bin_start[gbd], p1d = bin_start[gbd + nbd - 1];
    const long long hau0 = (du.off + p0u) & ~1LL, hau1 = (du.off + p1u + 1) & ~1LL;
    const long long had0 = (dd.off + p0d) & ~1LL, had1 = (dd.off + p1d + 1) & ~1LL;
    const long long bau0 = gbu & ~3LL, bau1 = (gbu + nbu + 3) & ~3LL, bad0 = gbd & ~3LL, bad1 = (gbd + nbd + 3) & ~3LL;
    const long long hbu = (hau1 - hau0) * 8, hbd = (had1 - had0) * 8, bbu = (bau1 - bau0) * 4, bbd = (bad1 - bad0) * 4;
    st.staged = hbu + hbd + bbu + bbd <= (long long)stage_bytes;
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
  const int* __restrict__ permu = perm + du.off;
  const int* __restrict__ permd = perm + dd.off;
  if (st.staged) {
    // shared-memory instance: the four regions are addressed from the staging buffer directly (LDS with 32-bit addresses)
    mbar_wait(&s_bar, 0);
    search_chunk(reinterpret_cast<const float2*>(s_stage) - st.pshift_u, reinterpret_cast<const float2*>(s_stage + st.hoff_d) - st.pshift_d,
                 reinterpret_cast<const int*>(s_stage + st.boff_u) - st.bshift_u, reinterpret_cast<const int*>(s_stage + st.boff_d) - st.bshift_d,
                 own, cnt, lup, ldn, du, dd, rc, hw_u, hw_d, permu, permd, P);
  } else {
    search_chunk(yz + du.off, yz + dd.off, bin_start + du.bin_off, bin_start + dd.bin_off, own, cnt, lup, ldn, du, dd, rc, hw_u, hw_d,
                 permu, permd, P);
  }
}

// ---------------------------------------------------------------------------------------------------------------------------
// S2' (NEXT-2 as SURVEY.md section 8(f).2 wrote it: "links that may skip a row"; reading A45 of DESIGN.md; link_skip = 1 only).
// Runs after k2_neighbours, one thread per cluster.  A cluster that S2 linked keeps its pair (the tables are re-encoded as
// position << 1 | k - 1 with k = 1).  A cluster S2 left unlinked looks one row further: candidates on rows r+-1, r+-2 in the S2
// windows scaled to the row distance k; pairs (k_u, k_d) = (1,2) and (2,1) first, (2,2) only if none of those is accepted; a pair
// is accepted iff D < cut2 * 0.5 * (a^2 + b^2) with the actual row distances a, b; the accepted pair with the minimum key
// (D, k_u, original index up, original index down) wins.  Reads go to global memory (L2): about one cluster in six takes this path.
struct SkipWin { float ylo, yhi, zlo, zhi; int by0, by1, bz0, bz1; bool any; };

__device__ __forceinline__ SkipWin skip_window(const float y, const float z, const float t, const float hwy, const float hwz,
                                               const bool continuous, const UnitDesc& g) {
  SkipWin w;
  const float yc = __fmul_rn(y, t), zc = continuous ? z : __fmul_rn(z, t);
  w.ylo = __fsub_rn(yc, hwy); w.yhi = __fadd_rn(yc, hwy); w.zlo = __fsub_rn(zc, hwz); w.zhi = __fadd_rn(zc, hwz);
  w.any = g.n > 0;
  w.by0 = bin_of(w.ylo, g.ylo, g.invs, g.ny); w.by1 = bin_of(w.yhi, g.ylo, g.invs, g.ny);
  w.bz0 = bin_of(w.zlo, g.zlo, g.invs, g.nz); w.bz1 = bin_of(w.zhi, g.zlo, g.invs, g.nz);
  return w;
}

struct SkipBest { bool have; float D; int ku, kd, pu, pd; };

// all pairs (candidate of window wu on unit gu) x (candidate of window wd on unit gd) at row distances (ku, kd)
__device__ __forceinline__ void skip_level(SkipBest& best, const int ku, const int kd, const SkipWin& wu, const SkipWin& wd,
                                           const UnitDesc& gu, const UnitDesc& gd, const float a, const float b, const float lim,
                                           const float y, const float z, const float2* __restrict__ yz, const int* __restrict__ perm,
                                           const int* __restrict__ bin_start) {
  if (!wu.any || !wd.any) return;
  const int* __restrict__ bsu = bin_start + gu.bin_off;
  const int* __restrict__ bsd = bin_start + gd.bin_off;
  const float2* __restrict__ hu = yz + gu.off;
  const float2* __restrict__ hd = yz + gd.off;
  for (int bz = wu.bz0; bz <= wu.bz1; bz++) {
    const int pe = bsu[bz * gu.ny + wu.by1 + 1];
    for (int p = bsu[bz * gu.ny + wu.by0]; p < pe; p++) {
      const float2 cu = hu[p];
      if (!(cu.x >= wu.ylo && cu.x <= wu.yhi && cu.y >= wu.zlo && cu.y <= wu.zhi)) continue;
      for (int bzd = wd.bz0; bzd <= wd.bz1; bzd++) {
        const int qe = bsd[bzd * gd.ny + wd.by1 + 1];
        for (int q = bsd[bzd * gd.ny + wd.by0]; q < qe; q++) {
          const float2 cd = hd[q];
          if (!(cd.x >= wd.ylo && cd.x <= wd.yhi && cd.y >= wd.zlo && cd.y <= wd.zhi)) continue;
          const float ey = __fsub_rn(__fmul_rn(b, __fsub_rn(cu.x, y)), __fmul_rn(a, __fsub_rn(y, cd.x)));
          const float ez = __fsub_rn(__fmul_rn(b, __fsub_rn(cu.y, z)), __fmul_rn(a, __fsub_rn(z, cd.y)));
          const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));
          if (!(D < lim)) continue;
          bool better = !best.have || D < best.D;
          if (best.have && D == best.D) {   // exact tie: k_u, then the original indices (rare)
            if (ku != best.ku) better = ku < best.ku;
            else {
              const int iu = perm[gu.off + p], ib = perm[gu.off + best.pu];   // same k_u: same up row
              better = iu < ib || (iu == ib && kd == best.kd && perm[gd.off + q] < perm[gd.off + best.pd]);
            }
          }
          if (better) { best.have = true; best.D = D; best.ku = ku; best.kd = kd; best.pu = p; best.pd = q; }
        }
      }
    }
  }
}

// fast path of S2': like k2_neighbours, the candidates of the (at most two) bin rows of a window are scanned once into a bit mask
struct SkipMask { Win w; unsigned m; bool ok; };   // ok = false: more than two bin rows or more than 32 candidates (generic path)

// first half: the candidate range(s) of the window from the bin table (up to four reads; the four windows of a hit are done
// together so that their 16 reads are in flight at once)
__device__ __forceinline__ SkipMask skip_ranges(const SkipWin& sw, const UnitDesc& g, const int* __restrict__ bin_start) {
  SkipMask r; r.m = 0u; r.ok = true;
  r.w.ylo = sw.ylo; r.w.yhi = sw.yhi; r.w.zlo = sw.zlo; r.w.zhi = sw.zhi; r.w.wide = false; r.w.a0 = r.w.n0 = r.w.a1m = r.w.n = 0;
  if (!sw.any) return r;
  if (sw.bz1 - sw.bz0 > 1) { r.ok = false; return r; }
  const int* __restrict__ bs = bin_start + g.bin_off;
  const int ra = sw.bz0 * g.ny;
  r.w.a0 = bs[ra + sw.by0]; r.w.n0 = bs[ra + sw.by1 + 1] - r.w.a0; r.w.n = r.w.n0;
  if (sw.bz1 > sw.bz0) { const int rb = ra + g.ny; const int a1 = bs[rb + sw.by0]; r.w.n += bs[rb + sw.by1 + 1] - a1; r.w.a1m = a1 - r.w.n0; }
  if (r.w.n > 32) r.ok = false;
  return r;
}
// second half: the candidates inside the window as a bit mask
__device__ __forceinline__ void skip_fill(SkipMask& r, const UnitDesc& g, const float2* __restrict__ yz) {
  if (!r.ok) return;
  const float2* __restrict__ hits = yz + g.off;
#pragma unroll 1
  for (int j = 0; j < r.w.n; j++) { if (in_win(hits[win_pos(r.w, j)], r.w)) r.m |= 1u << j; }
}

__device__ __forceinline__ void skip_level_masks(SkipBest& best, const int ku, const int kd, const SkipMask& mu, const SkipMask& md,
                                                 const UnitDesc& gu, const UnitDesc& gd, const float a, const float b, const float lim,
                                                 const float y, const float z, const float2* __restrict__ yz,
                                                 const int* __restrict__ perm) {
  const float2* __restrict__ hu = yz + gu.off;
  const float2* __restrict__ hd = yz + gd.off;
  unsigned m1 = md.m ? mu.m : 0u;
  while (m1) {
    const int j = __ffs(m1) - 1; m1 &= m1 - 1u;
    const int p = win_pos(mu.w, j);
    const float2 cu = hu[p];
    unsigned m2 = md.m;
    while (m2) {
      const int i = __ffs(m2) - 1; m2 &= m2 - 1u;
      const int q = win_pos(md.w, i);
      const float2 cd = hd[q];
      const float ey = __fsub_rn(__fmul_rn(b, __fsub_rn(cu.x, y)), __fmul_rn(a, __fsub_rn(y, cd.x)));
      const float ez = __fsub_rn(__fmul_rn(b, __fsub_rn(cu.y, z)), __fmul_rn(a, __fsub_rn(z, cd.y)));
      const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));
      if (!(D < lim)) continue;
      bool better = !best.have || D < best.D;
      if (best.have && D == best.D) {   // exact tie: k_u, then the original indices (rare)
        if (ku != best.ku) better = ku < best.ku;
        else { const int iu = perm[gu.off + p], ib = perm[gu.off + best.pu]; better = iu < ib || (iu == ib && perm[gd.off + q] < perm[gd.off + best.pd]); }
      }
      if (better) { best.have = true; best.D = D; best.ku = ku; best.kd = kd; best.pu = p; best.pd = q; }
    }
  }
}

#ifndef K2S_CTAS
#define K2S_CTAS 6   // measured on C3 (K2 + K2'): 0.96 ms at 3 CTAs / SM (the compiler's choice at 80 registers), 0.79 at 4, 0.72 at 5, 0.71 at 6, 0.70 at 8: latency-bound, occupancy pays more than the spills cost
#endif
__global__ void __launch_bounds__(256, K2S_CTAS) k2_skip_links(const Item* __restrict__ items, const int chunk, const UnitDesc* __restrict__ units,
                                                     const RowConst* __restrict__ rows, const float2* __restrict__ yz,
                                                     const int* __restrict__ perm, const int* __restrict__ bin_start,
                                                     int* __restrict__ link_up, int* __restrict__ link_dn, const Params P) {
  const Item it = items[blockIdx.x];
  const int u = it.unit, R = P.R, r = u % R;
  const UnitDesc d = units[u];
  const int cnt = min(chunk, d.n - it.start);
  const bool searchable = r >= 1 && r <= R - 2;
  const RowConst rc = rows[r];
  // pass 1: re-encode the pairs S2 found; the clusters it left unlinked are collected in shared memory, so that pass 2 runs with
  // all lanes busy (they are about one cluster in six)
  __shared__ int s_list[4096];   // chunk <= 4096 (tpc_set_param)
  __shared__ int s_n;
  if (threadIdx.x == 0) s_n = 0;
  __syncthreads();
  for (int k = threadIdx.x; k < cnt; k += blockDim.x) {
    const long long g = d.off + it.start + k;
    const int eu = link_up[g];
    if (eu >= 0) { link_up[g] = eu << 1; link_dn[g] = link_dn[g] << 1; }   // S2's pair: row distance 1 on both sides
    else if (searchable) s_list[atomicAdd(&s_n, 1)] = k;
  }
  __syncthreads();
  const int n_open = s_n;
  if (n_open == 0) return;
  const bool cont = P.continuous != 0;
  const bool up2 = r + 2 <= R - 1, dn2 = r - 2 >= 0;
  // the four neighbour descriptors are the same for every thread: shared memory instead of 4 x 16 registers per thread
  __shared__ UnitDesc s_g[4];
  if (threadIdx.x < 4) {
    const int k = threadIdx.x;   // 0: r+1, 1: r-1, 2: r+2 (or r+1), 3: r-2 (or r-1)
    s_g[k] = units[k == 0 ? u + 1 : k == 1 ? u - 1 : k == 2 ? (up2 ? u + 2 : u + 1) : (dn2 ? u - 2 : u - 1)];
  }
  __syncthreads();
  const UnitDesc& gu1 = s_g[0]; const UnitDesc& gd1 = s_g[1]; const UnitDesc& gu2 = s_g[2]; const UnitDesc& gd2 = s_g[3];
  const float wy1 = __fmul_rn(1.0f, P.wy), wy2 = __fmul_rn(2.0f, P.wy), wz1 = __fmul_rn(1.0f, P.wz), wz2 = __fmul_rn(2.0f, P.wz);
  for (int j = threadIdx.x; j < n_open; j += blockDim.x) {
    const int k = s_list[j];
    const long long g = d.off + it.start + k;
    const float2 h = yz[g];
    const float y = h.x, z = h.y;
    const SkipWin wu1 = skip_window(y, z, rc.tu, wy1, cont ? rc.wzu : wz1, cont, gu1);
    const SkipWin wd1 = skip_window(y, z, rc.td, wy1, cont ? rc.wzd : wz1, cont, gd1);
    SkipBest best; best.have = false; best.D = 0.0f; best.ku = best.kd = 0; best.pu = best.pd = -1;
    SkipWin wu2 = wu1, wd2 = wd1; wu2.any = wd2.any = false;
    if (dn2) wd2 = skip_window(y, z, rc.td2, wy2, cont ? rc.wzd2 : wz2, cont, gd2);
    if (up2) wu2 = skip_window(y, z, rc.tu2, wy2, cont ? rc.wzu2 : wz2, cont, gu2);
    SkipMask mu1 = skip_ranges(wu1, gu1, bin_start), md1 = skip_ranges(wd1, gd1, bin_start);
    SkipMask mu2 = skip_ranges(wu2, gu2, bin_start), md2 = skip_ranges(wd2, gd2, bin_start);
    skip_fill(mu1, gu1, yz); skip_fill(md1, gd1, yz); skip_fill(mu2, gu2, yz); skip_fill(md2, gd2, yz);
    if (mu1.ok && md1.ok && mu2.ok && md2.ok) {
      skip_level_masks(best, 1, 2, mu1, md2, gu1, gd2, rc.a, rc.b2, rc.thr12, y, z, yz, perm);
      skip_level_masks(best, 2, 1, mu2, md1, gu2, gd1, rc.a2, rc.b, rc.thr21, y, z, yz, perm);
      if (!best.have) skip_level_masks(best, 2, 2, mu2, md2, gu2, gd2, rc.a2, rc.b2, rc.thr22, y, z, yz, perm);
    } else {   // tiny bins or very dense rows: nested scan over all bin rows of both windows
      if (dn2) skip_level(best, 1, 2, wu1, wd2, gu1, gd2, rc.a, rc.b2, rc.thr12, y, z, yz, perm, bin_start);
      if (up2) skip_level(best, 2, 1, wu2, wd1, gu2, gd1, rc.a2, rc.b, rc.thr21, y, z, yz, perm, bin_start);
      if (!best.have && up2 && dn2) skip_level(best, 2, 2, wu2, wd2, gu2, gd2, rc.a2, rc.b2, rc.thr22, y, z, yz, perm, bin_start);
    }
    if (best.have) { link_up[g] = (best.pu << 1) | (best.ku - 1); link_dn[g] = (best.pd << 1) | (best.kd - 1); }
  }
}

}  // namespace

int launch_k2_neighbours(const Launch& L, int n_items, const Item* d_items, int chunk, const UnitDesc* d_units,
                         const RowConst* d_rows, const float2* d_yz, const int* d_perm, const int* d_bin_start, int* d_link_up,
                         int* d_link_dn, const Params& P) {
  if (n_items <= 0) return 0;
  // default: half items of 512 clusters, 128 threads (8 CTAs / SM); the k2_threads knob keeps whole items
  const int split = L.k2_threads > 0 || chunk < 512 || (chunk & 63) ? 1 : 2;
  chunk /= split;
  const int stage_bytes = ((chunk * K2_STAGE_PER_CLUSTER + 4096) + 127) & ~127;
  const int threads = L.k2_threads > 0 ? L.k2_threads : (split == 2 ? 128 : K2_THREADS);
  cudaError_t e = cudaFuncSetAttribute(k2_neighbours, cudaFuncAttributeMaxDynamicSharedMemorySize, stage_bytes);
  if (e != cudaSuccess) return -(int)e;
  k2_neighbours<<<n_items * split, threads, stage_bytes, L.stream>>>(d_items, chunk, d_units, d_rows, d_yz, d_perm, d_bin_start,
                                                                   d_link_up, d_link_dn, P, stage_bytes, split);
  e = cudaGetLastError();
  return e == cudaSuccess ? 1 : -(int)e;
}

int launch_k2_skip_links(const Launch& L, int n_items, const Item* d_items, int chunk, const UnitDesc* d_units, const RowConst* d_rows,
                         const float2* d_yz, const int* d_perm, const int* d_bin_start, int* d_link_up, int* d_link_dn, const Params& P) {
  if (n_items <= 0) return 0;
  k2_skip_links<<<n_items, 256, 0, L.stream>>>(d_items, chunk, d_units, d_rows, d_yz, d_perm, d_bin_start, d_link_up, d_link_dn, P);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? 1 : -(int)e;
}

}  // namespace tpc
