// k5_tracklets.cu -- K5: S5 Kalman-filter tracklet constructor ("first preliminary fit, used to find the full track";
// PAPER.md:41 single hypothesis per seed, linear in the event size; definition in DESIGN.md section 4).
//
// Four phase kernels, each a set of persistent CTAs with a global work queue, ONE tracklet per lane, the 5-parameter state
// (y, z_rel, sin phi, dz/ds, q/pT) and the 15 covariance entries in registers, fp32:
//   k5a_seed_fit   Phase A   fit along the cleaned up-links of a start hit (transport + update per row, no search)
//   k5b_extend_out Phase B   outward extrapolation row by row with cluster pick-up from the S1 grid
//   k5c_refit_in   Phase C, rows r_out .. r0: inward refit over the clusters A and B assigned (transport + update; a pick-up only
//                  on the few rows B left empty)
//   k5d_extend_in  Phase C, rows below r0: inward extrapolation with pick-up
// A phase kernel runs ONE kind of row step, so the lanes of a warp execute the same instruction stream at (nearly) full width:
// the single state-machine kernel of round 1 ran its pick-up code at 8 of 32 lanes because only the lanes in an extrapolating
// phase needed it (profiles/r1_ncu_k5_final.md).  Between the phases a tracklet is a 128-byte record in HBM (TlRec) whose `next`
// field names the phase it is due for.  Every kernel walks the tracklets in START-LIST order (queue position = index in the run
// list; a tracklet not due for this phase is skipped after one 16-byte read), so that neighbouring lanes work on neighbouring
// tracks and share rowhit / grid lines in L1 / L2; completion-order task lists doubled the DRAM traffic.
// The order does not enter any result.  A lane that finishes waits until at least K5_FLUSH lanes of its warp have finished: the
// write-out + queue fetch + record load code then runs for several lanes at once instead of for one lane in almost every iteration.
// z is carried relative to the start hit (z_rel = z - z_ref, formed in fp32 before use) so that long continuous time frames
// (|z| up to 2.6e4 cm) keep full fp32 resolution.  Arithmetic is written term by term in the documented order and compiled
// without FMA contraction (the fused multiply-adds of the transport / update are explicit, reading A43), so pick-up decisions
// agree with the fp32 definition.
// rowhit layout: [tracklet][row]; only rows a tracklet visits are written; tl_first / tl_last delimit the valid range.
#include "kalman.cuh"

namespace tpc {
namespace {

constexpr int K5_THREADS = 128;
constexpr int K5_MAX_ROWS = 256;   // rows held in the shared-memory copy of the row table (the launcher checks R)
#ifndef K5_FLUSH_N
#define K5_FLUSH_N 4
#endif
#ifndef K5_CTAS
#define K5_CTAS 6
#endif
#ifndef K5_CTAS_B
#define K5_CTAS_B 7   // measured on C3: k5b 1.58 ms at 6 CTAs / SM (78 registers), 1.49 ms at 7 (72, no spill), 1.73 ms at 5
#endif
#ifndef K5_CTAS_C
#define K5_CTAS_C K5_CTAS
#endif
#ifndef K5_CTAS_D
#define K5_CTAS_D 7   // k5d 1.46 -> 1.41 ms; k5c spills at 72 registers and stays at 6
#endif
// Two passes over the start list per phase kernel: the first takes the tracklets with at least K5_LONG_x rows ahead of them in this
// phase (B: rows above the end of the chain; C: rows between the outermost cluster and the start hit; D: rows below the start hit),
// the second the rest (0 = one pass).  When the queue runs dry every lane finishes the tracklet it holds and the warps run on with
// ever fewer lanes (measured in k5b: 34 % of the warp iterations at 11 of 32 lanes); with the long tracklets taken first that tail
// is made of short ones (19 % of the iterations).  C3: K5 4.63 -> 4.50 ms; a third class gained nothing more.  Each pass walks the
// list in start-list order; the class of a tracklet does not change while a kernel runs, so exactly one pass takes it.
#ifndef K5_LONG_B
#define K5_LONG_B 64
#endif
#ifndef K5_LONG_C
#define K5_LONG_C 40
#endif
#ifndef K5_LONG_D
#define K5_LONG_D 30
#endif
constexpr int K5_FLUSH = K5_FLUSH_N;        // finished lanes of a warp that trigger the write-out / refill code
constexpr unsigned FULL = 0xffffffffu;

// Handoff record of a tracklet between the phase kernels (128 bytes, read / written as float4).
//   A -> B : st = full state after the last chain update (row r_out), cl = that cluster
//   B      : overwrites st[0..4], cl, r_out with the state / cluster / row of its outermost update (if it made one)
//   C1     : reads st[0..4], cl, zref, u0, r_out; writes st = full state at row r0, chi2, n for C2
struct __align__(16) TlRec {
  float st[20];
  float yl, zl, zref, chi2;
  int u0, r_out, n, next;   // next: phase the tracklet is due for (NEXT_B / NEXT_C / NEXT_D / NEXT_NONE)
  int pad[4];
};
static_assert(sizeof(TlRec) == 128, "TlRec is one 128-byte line");

// control block of the four kernels (ints, zeroed by the caller before k5a): the queue heads
enum : int { CT_QA = 0, CT_QB, CT_QC, CT_QD, CT_WORDS = 8 };
enum : int { NEXT_NONE = 0, NEXT_B = 1, NEXT_C = 2, NEXT_D = 3 };

enum : int { MD_FETCH = 0, MD_INIT, MD_RUN, MD_DONE, MD_EXIT };

__device__ __forceinline__ void load_state(State& st, const float4* __restrict__ p) {
  const float4 a = p[0], b = p[1], c = p[2], d = p[3], e = p[4];
  st.y = a.x; st.z = a.y; st.s = a.z; st.t = a.w; st.q = b.x; st.c00 = b.y; st.c10 = b.z; st.c11 = b.w;
  st.c20 = c.x; st.c21 = c.y; st.c22 = c.z; st.c30 = c.w; st.c31 = d.x; st.c32 = d.y; st.c33 = d.z; st.c40 = d.w;
  st.c41 = e.x; st.c42 = e.y; st.c43 = e.z; st.c44 = e.w;
}
__device__ __forceinline__ void store_state(float4* __restrict__ p, const State& st) {
  p[0] = make_float4(st.y, st.z, st.s, st.t); p[1] = make_float4(st.q, st.c00, st.c10, st.c11);
  p[2] = make_float4(st.c20, st.c21, st.c22, st.c30); p[3] = make_float4(st.c31, st.c32, st.c33, st.c40);
  p[4] = make_float4(st.c41, st.c42, st.c43, st.c44);
}

// state <-> per-lane column of a shared-memory array [20][K5_THREADS] (conflict-free: consecutive lanes, consecutive words)
__device__ __forceinline__ void snap_store(float (*s)[K5_THREADS], const int tx, const State& st) {
  s[0][tx] = st.y; s[1][tx] = st.z; s[2][tx] = st.s; s[3][tx] = st.t; s[4][tx] = st.q;
  s[5][tx] = st.c00; s[6][tx] = st.c10; s[7][tx] = st.c11; s[8][tx] = st.c20; s[9][tx] = st.c21;
  s[10][tx] = st.c22; s[11][tx] = st.c30; s[12][tx] = st.c31; s[13][tx] = st.c32; s[14][tx] = st.c33;
  s[15][tx] = st.c40; s[16][tx] = st.c41; s[17][tx] = st.c42; s[18][tx] = st.c43; s[19][tx] = st.c44;
}

// final result of a tracklet: n, first (row of the innermost update), last (row of the outermost), chi2, state of the innermost update
__device__ __forceinline__ void write_tracklet(const int i, const int n, const int r_snap, const int r_out, const float chi2, const float zref,
                                               const float* v /* 20 values */, int* __restrict__ tl_n, int* __restrict__ tl_first,
                                               int* __restrict__ tl_last, float* __restrict__ tl_chi2, float* __restrict__ tl_par,
                                               float* __restrict__ tl_cov) {
  tl_n[i] = n; tl_first[i] = r_snap; tl_last[i] = r_out; tl_chi2[i] = chi2;
  float* __restrict__ op = tl_par + (long long)i * 5;
  op[0] = v[0]; op[1] = v[1] + zref; op[2] = v[2]; op[3] = v[3]; op[4] = v[4];
  float* __restrict__ oc = tl_cov + (long long)i * 15;
#pragma unroll
  for (int k = 0; k < 15; k++) oc[k] = v[5 + k];
}

// warp-aggregated atomicAdd on a counter for the lanes in `m`; returns this lane's slot (valid for lanes in m)
__device__ __forceinline__ int list_append(const unsigned m, int* __restrict__ count, const int lane) {
  int base = 0;
  const int leader = __ffs(m) - 1;
  if (lane == leader) base = atomicAdd(count, __popc(m));
  base = __shfl_sync(FULL, base, leader);
  return base + __popc(m & ((1u << lane) - 1u));
}

// length class of a tracklet with `len` rows ahead of it in a phase: 0 = long (first pass), 1 = short (second pass)
template <int LONG> __device__ __forceinline__ int len_class(const int len, const int passes) { return passes == 2 && len < LONG ? 1 : 0; }
// two passes only while the tail matters: with many tracklets per lane (C5: 32) the tail is a small part of the kernel and the second
// walk over the list costs more than it saves (C5: K5 27.2 ms with one pass, 28.2 ms with two; C3, 4.8 per lane: 4.63 / 4.50 ms)
#ifndef K5_TWO_PASS_MAX_PER_LANE
#define K5_TWO_PASS_MAX_PER_LANE 12
#endif
template <int LONG> __device__ __forceinline__ int len_passes(const int n_tasks) {
  return LONG > 0 && (long long)n_tasks < (long long)K5_TWO_PASS_MAX_PER_LANE * gridDim.x * K5_THREADS ? 2 : 1;
}

// warp-aggregated fetch of queue positions for the lanes in `m`
__device__ __forceinline__ int queue_fetch(const unsigned m, int* __restrict__ head, const int lane) { return list_append(m, head, lane); }

// Cluster pick-up on one row: nearest cluster (dy^2+dz^2, then original index) inside the window
// min(w_max, n_sigma*sqrt(C + sigma^2)) around the extrapolated position; -1 = none.  Returns the cluster in *hit.
__device__ __forceinline__ int pickup(const UnitDesc& d, const float2* __restrict__ yz, const int* __restrict__ perm,
                                      const int* __restrict__ bin_start, const State& st, const float zref, const Params& P,
                                      float2* hit) {
  if (d.n == 0) return -1;
  float wy = P.nsigma * sqrtf(st.c00 + P.ry); if (!(wy <= P.wmax)) wy = P.wmax;
  float wz = P.nsigma * sqrtf(st.c11 + P.rz); if (!(wz <= P.wmax)) wz = P.wmax;
  const float y = st.y, zr = st.z;
  const float ylo = y - wy, yhi = y + wy, zlo = zr - wz, zhi = zr + wz;
  const float margin = 0.05f;   // the bin range only has to cover the z_rel window
  const int by0 = bin_of(ylo, d.ylo, d.invs, d.ny), by1 = bin_of(yhi, d.ylo, d.invs, d.ny);
  const int bz0 = bin_of((zlo + zref) - margin, d.zlo, d.invs, d.nz), bz1 = bin_of((zhi + zref) + margin, d.zlo, d.invs, d.nz);
  // the row's cluster base pointer is materialised once (the empty asm keeps the compiler from re-deriving it from the 64-bit
  // offset at every access): each candidate load below is then one IMAD.WIDE + LDG
  unsigned long long hits_a = (unsigned long long)(yz + d.off);
  asm volatile("" : "+l"(hits_a));
  const int* __restrict__ bs = bin_start + d.bin_off;
  const float2* __restrict__ hits = reinterpret_cast<const float2*>(hits_a);
  int best = -1; float bestd = 0.0f;
  // Two bin rows per round (the window is at most 2*w_max + margin wide, so one round is the rule): the four bin_start
  // reads are issued together, then ONE flat loop runs over the candidates of both rows, so that lanes with different
  // candidate counts share the loop instead of diverging in a nest.  Any visiting order gives the same argmin (total order).
  for (int bz = bz0; bz <= bz1; bz += 2) {
    const int ra = bz * d.ny, rb = ra + d.ny;
    const bool two = bz + 1 <= bz1;
    const int pa0 = bs[ra + by0], pb0 = bs[ra + by1 + 1];
    const int pa1 = two ? bs[rb + by0] : 0, pb1 = two ? bs[rb + by1 + 1] : 0;
    const int n0 = pb0 - pa0, total = n0 + (pb1 - pa1);
#pragma unroll 1
    for (int k0 = 0; k0 < total; k0 += 2) {   // two candidates per round: their loads are independent and issued together
      float2 cc[2];
#pragma unroll
      for (int j = 0; j < 2; j++) {
        const int k = k0 + j;
        cc[j] = k < total ? __ldg(hits + (k < n0 ? pa0 + k : pa1 + (k - n0))) : make_float2(0.f, 0.f);
      }
#pragma unroll
      for (int j = 0; j < 2; j++) {
        const int k = k0 + j;
        const float2 c = cc[j];
        const float yc = c.x, zc = c.y - zref;
        if (k < total && yc >= ylo && yc <= yhi && zc >= zlo && zc <= zhi) {
          const int p = k < n0 ? pa0 + k : pa1 + (k - n0);
          const float dy = yc - y, dz = zc - zr;
          const float dd = dy * dy + dz * dz;
          bool better = best < 0 || dd < bestd;
          if (best >= 0 && dd == bestd) better = perm[d.off + p] < perm[d.off + best];
          if (better) { best = p; bestd = dd; *hit = c; }
        }
      }
    }
  }
  return best;
}

// work counters of a tracklet phase, packed: transports bits 0-10, updates 11-21, pick-ups 22-31 (each < 2 R < 2^9)
__device__ __forceinline__ void work_flush(unsigned& work, unsigned* s_work) {
  if (work) { atomicAdd(&s_work[0], work & 0x7ffu); atomicAdd(&s_work[1], (work >> 11) & 0x7ffu); atomicAdd(&s_work[2], work >> 22); work = 0; }
}

#define K5_PROLOGUE()                                                                                                  \
  const int R = P.R, lane = threadIdx.x & 31, tx = threadIdx.x;                                                        \
  __shared__ float s_rx[K5_MAX_ROWS], s_re[K5_MAX_ROWS];                                                               \
  __shared__ unsigned s_work[3];                                                                                       \
  for (int k = threadIdx.x; k < R && k < K5_MAX_ROWS; k += blockDim.x) { s_rx[k] = rows[k].x; s_re[k] = rows[k].yedge; } \
  if (threadIdx.x < 3) s_work[threadIdx.x] = 0;                                                                        \
  __syncthreads();                                                                                                     \
  int mode = MD_FETCH; bool drained = false; unsigned work = 0

#define K5_EPILOGUE()                                                                                                  \
  __syncthreads();                                                                                                     \
  if (threadIdx.x < 3 && s_work[threadIdx.x]) atomicAdd(&counters[threadIdx.x], (unsigned long long)s_work[threadIdx.x])

// true when the finished lanes of the warp should be written out now: enough of them, or nothing left to wait for
__device__ __forceinline__ bool flush_now(const int mode, const bool drained) {
  const unsigned done = __ballot_sync(FULL, mode == MD_DONE);
  if (!done) return false;
  return __popc(done) >= K5_FLUSH || drained || !__ballot_sync(FULL, mode == MD_RUN || mode == MD_INIT);
}

// ---------------------------------------------------------------------------------------------------------------------------
// Phase A: seed fit along the chain of cleaned up-links (no gate).  Task = start hit (or an entry of run_list).
__global__ void __launch_bounds__(K5_THREADS, 8) k5a_seed_fit(const int M_host, const int* __restrict__ M_dev, const int* __restrict__ run_list,
                                                              const int* __restrict__ start_unit, const int* __restrict__ start_pos,
                                                              const UnitDesc* __restrict__ units, const RowConst* __restrict__ rows,
                                                              const float2* __restrict__ yz, const int* __restrict__ link_up,
                                                              rowhit_t* __restrict__ rowhit, TlRec* __restrict__ rec, int* __restrict__ ctl,
                                                              unsigned long long* __restrict__ counters, const Params P) {
  K5_PROLOGUE();
  const int M = M_dev ? min(*M_dev, M_host) : M_host;   // task count: in device memory (default path: no read-back after K3) or given
  int i = -1, u0 = 0, r = 0, nxt = -1, hit0 = -1;
  bool ok = true;
  float zref = 0.0f;
  float2 cl = make_float2(0.f, 0.f);
  State st = {};
  const UnitDesc* __restrict__ su = units;
  rowhit_t* __restrict__ rh = rowhit;

  for (;;) {
    if (flush_now(mode, drained)) {
      const bool fin = mode == MD_DONE;
      const bool to_b = fin && ok && r + 1 < R;
      if (fin) {
        float4* __restrict__ p = reinterpret_cast<float4*>(rec + i);
        store_state(p, st);
        p[5] = make_float4(cl.x, cl.y, zref, 0.0f);
        reinterpret_cast<int4*>(p)[6] = make_int4(u0, r, r, to_b ? NEXT_B : NEXT_C);   // .z: row Phase B starts from (B moves .y, never .z)
        work_flush(work, s_work);
      }
      if (fin) mode = drained ? MD_EXIT : MD_FETCH;
    }
    const unsigned need = __ballot_sync(FULL, mode == MD_FETCH);
    if (need) {
      const int q = queue_fetch(need, ctl + CT_QA, lane);
      if (mode == MD_FETCH) {
        if (q < M) {
          i = run_list ? run_list[q] : q;
          u0 = start_unit[i];
          hit0 = start_pos[i];
          const int sec = u0 / R;
          r = u0 - sec * R;
          su = units + (long long)sec * R;
          rh = rowhit + (long long)i * R;
          const long long o0 = su[r].off + hit0;
          cl = yz[o0];
          nxt = link_up[o0];
          zref = cl.y; ok = true;
          mode = MD_INIT;
        } else mode = MD_EXIT;
      }
      drained = __any_sync(FULL, mode == MD_EXIT);
    }
    if (__all_sync(FULL, mode == MD_EXIT)) break;

    // ---- one row step: transport along the link (RUN lanes), Kalman update (RUN and INIT lanes)
    const bool run = mode == MD_RUN, init = mode == MD_INIT;
    float2 c = cl;
    int nxt_up = -1;
    // link entry: the position in the next row; with S2' (link_skip) position << 1 | k - 1, k = row distance of the link
    const int kk = P.link_skip ? (nxt & 1) + 1 : 1, pos = P.link_skip ? nxt >> 1 : nxt;
    if (run) {   // linked cluster + its own up-link
      TPC_CHECK(P, r + kk < R && pos >= 0 && pos < su[r + kk < R ? r + kk : r].n, 51);
      const long long o = su[r + kk].off + pos; c = yz[o]; nxt_up = link_up[o];
    }
    bool prop_ok = true;
    __syncwarp();
    if (run) { work += 1u; prop_ok = propagate(st, s_rx[r + kk] - s_rx[r], P); }   // one transport over the whole link
    if (init) {   // direction from the origin, first update with the start hit
      const float x = s_rx[r], y = c.x;
      const float rr = sqrtf(x * x + y * y);
      st.y = y; st.z = 0.0f; st.s = y / rr; st.t = P.continuous ? 0.0f : zref / rr; st.q = 0.0f;
      reset_cov(st, P);
    }
    const bool have = init || (run && prop_ok);
    __syncwarp();
    if (have) { work += 1u << 11; update(st, c.x, c.y - zref, P); }
    __syncwarp();
    if (init) { rh[r] = hit0; mode = nxt >= 0 ? MD_RUN : MD_DONE; }
    else if (run) {
      if (!prop_ok) { ok = false; mode = MD_DONE; }      // a failed transport ends Phase A and skips Phase B
      else {
        if (kk == 2) rh[r + 1] = -1;                       // the skipped row holds no cluster of this tracklet (yet)
        r += kk; rh[r] = pos; cl = c; nxt = nxt_up; if (nxt < 0) mode = MD_DONE;
      }
    }
  }
  K5_EPILOGUE();
}

// ---------------------------------------------------------------------------------------------------------------------------
// Phase B: outward extrapolation with pick-up.  Task = tracklet whose Phase A ended with a good state below the last row.
__global__ void __launch_bounds__(K5_THREADS, K5_CTAS_B) k5b_extend_out(const int M_host, const int* __restrict__ M_dev, const int* __restrict__ run_list,
                                                                const UnitDesc* __restrict__ units,
                                                                const RowConst* __restrict__ rows, const float2* __restrict__ yz,
                                                                const int* __restrict__ perm, const int* __restrict__ bin_start,
                                                                rowhit_t* __restrict__ rowhit, TlRec* __restrict__ rec, int* __restrict__ ctl,
                                                                unsigned long long* __restrict__ counters, const Params P) {
  K5_PROLOGUE();
  __shared__ float s_sv[7][K5_THREADS];   // state after the outermost update (5 parameters) + that cluster (y, z)
  const int n_tasks = M_dev ? min(*M_dev, M_host) : M_host;
  const int passes = len_passes<K5_LONG_B>(n_tasks);
  int i = -1, r = 0, r_out = 0, gap = 0;
  bool extended = false;
  float zref = 0.0f;
  State st = {};
  const UnitDesc* __restrict__ su = units;
  rowhit_t* __restrict__ rh = rowhit;

  for (;;) {
    if (flush_now(mode, drained)) {
      const bool fin = mode == MD_DONE;
      if (fin) {
        if (extended) {
          float4* __restrict__ p = reinterpret_cast<float4*>(rec + i);
          p[0] = make_float4(s_sv[0][tx], s_sv[1][tx], s_sv[2][tx], s_sv[3][tx]);
          rec[i].st[4] = s_sv[4][tx]; rec[i].yl = s_sv[5][tx]; rec[i].zl = s_sv[6][tx]; rec[i].r_out = r_out;
        }
        work_flush(work, s_work);
      }
      if (fin) mode = drained ? MD_EXIT : MD_FETCH;
    }
    const unsigned need = __ballot_sync(FULL, mode == MD_FETCH);
    if (need) {
      const int q = queue_fetch(need, ctl + CT_QB, lane);
      if (mode == MD_FETCH) {
        if (q < passes * n_tasks) {
          const int pass = passes == 1 ? 0 : q / n_tasks, qq = q - pass * n_tasks;
          i = run_list ? run_list[qq] : qq;
          const float4* __restrict__ p = reinterpret_cast<const float4*>(rec + i);
          const int4 k = reinterpret_cast<const int4*>(p)[6];
          // (not NEXT_B: Phase A ended on the last row or with a failed transport; not this pass's class: another pass takes it; the
          // lane fetches again.)  k.z, not k.y: B moves r_out while it runs, the class must not change under a concurrent pass.
          const bool mine = k.w == NEXT_B && len_class<K5_LONG_B>(R - 1 - k.z, passes) == pass;
          if (mine) {
          load_state(st, p);
          zref = p[5].z;
          const int sec = k.x / R;
          r = r_out = k.y; gap = 0; extended = false;
          su = units + (long long)sec * R;
          rh = rowhit + (long long)i * R;
          mode = MD_RUN;
          }
        } else mode = MD_EXIT;
      }
      drained = __any_sync(FULL, mode == MD_EXIT);
    }
    if (__all_sync(FULL, mode == MD_EXIT)) break;

    const bool run = mode == MD_RUN;
    const int rn = r + 1;
    bool do_pick = false;
    __syncwarp();
    if (run) {
      work += 1u;
      const bool prop_ok = propagate(st, s_rx[rn] - s_rx[r], P);
      if (!prop_ok || fabsf(st.y) > s_re[rn] + P.edge_margin) mode = MD_DONE;
      else do_pick = true;
    }
    float2 c = make_float2(0.f, 0.f);
    int hit = -1;
    __syncwarp();
    if (do_pick) { TPC_CHECK(P, rn < R, 52); work += 1u << 22; hit = pickup(su[rn], yz, perm, bin_start, st, zref, P, &c); TPC_CHECK(P, hit < su[rn].n, 53); }
    __syncwarp();
    const bool have = do_pick && hit >= 0;
    if (do_pick) {
      rh[rn] = hit;
      if (!have) { gap++; if (gap > P.max_gap) mode = MD_DONE; }
    }
    __syncwarp();
    if (have) { work += 1u << 11; update(st, c.x, c.y - zref, P); }
    __syncwarp();
    if (have) {
      gap = 0; r_out = rn; extended = true;
      s_sv[0][tx] = st.y; s_sv[1][tx] = st.z; s_sv[2][tx] = st.s; s_sv[3][tx] = st.t; s_sv[4][tx] = st.q; s_sv[5][tx] = c.x; s_sv[6][tx] = c.y;
    }
    if (do_pick) { r = rn; if (rn + 1 >= R) mode = MD_DONE; }
  }
  K5_EPILOGUE();
}

// ---------------------------------------------------------------------------------------------------------------------------
// Phase C, part 1: inward refit from the outermost updated row r_out down to the start row r0 (rows that A / B visited).
// Rows with an assigned cluster are updated without a search; rows B left empty are searched again (rare); no gap counting
// here (first_assigned = r0).  A tracklet with r0 = 0, or whose transport fails, is final; the others continue in k5d.
__global__ void __launch_bounds__(K5_THREADS, K5_CTAS_C) k5c_refit_in(const int M_host, const int* __restrict__ M_dev, const int* __restrict__ run_list,
                                                              const UnitDesc* __restrict__ units,
                                                              const RowConst* __restrict__ rows, const float2* __restrict__ yz,
                                                              const int* __restrict__ perm, const int* __restrict__ bin_start,
                                                              rowhit_t* __restrict__ rowhit, TlRec* __restrict__ rec, int* __restrict__ ctl,
                                                              int* __restrict__ tl_n, int* __restrict__ tl_first,
                                                              int* __restrict__ tl_last, float* __restrict__ tl_chi2,
                                                              float* __restrict__ tl_par, float* __restrict__ tl_cov,
                                                              unsigned long long* __restrict__ counters, const Params P) {
  K5_PROLOGUE();
  __shared__ float s_snap[20][K5_THREADS];   // state after the last update, saved only before a step that may not update
  const int n_tasks = M_dev ? min(*M_dev, M_host) : M_host;
  const int passes = len_passes<K5_LONG_C>(n_tasks);
  int i = -1, u0 = 0, r0 = 0, r = 0, r_out = 0, r_snap = 0, n = 0, a_next = -1, a_next2 = -1;
  bool snap_cur = true, final_ = false;
  float zref = 0.0f, chi2 = 0.0f;
  float2 cl = make_float2(0.f, 0.f);
  State st = {};
  const UnitDesc* __restrict__ su = units;
  rowhit_t* __restrict__ rh = rowhit;

  for (;;) {
    if (flush_now(mode, drained)) {
      const bool fin = mode == MD_DONE;
      const bool to_d = fin && !final_;
      if (fin) {
        if (final_) {
          float v[20];
          if (snap_cur) { v[0] = st.y; v[1] = st.z; v[2] = st.s; v[3] = st.t; v[4] = st.q; v[5] = st.c00; v[6] = st.c10; v[7] = st.c11;
            v[8] = st.c20; v[9] = st.c21; v[10] = st.c22; v[11] = st.c30; v[12] = st.c31; v[13] = st.c32; v[14] = st.c33; v[15] = st.c40;
            v[16] = st.c41; v[17] = st.c42; v[18] = st.c43; v[19] = st.c44; }
          else {
#pragma unroll
            for (int k = 0; k < 20; k++) v[k] = s_snap[k][tx];
          }
          write_tracklet(i, n, r_snap, r_out, chi2, zref, v, tl_n, tl_first, tl_last, tl_chi2, tl_par, tl_cov);
          rec[i].next = NEXT_NONE;
        } else {   // the last step was the update with the start hit on row r0: the state is the snapshot
          float4* __restrict__ p = reinterpret_cast<float4*>(rec + i);
          store_state(p, st);
          p[5] = make_float4(cl.x, cl.y, zref, chi2);
          reinterpret_cast<int4*>(p)[6] = make_int4(u0, r_out, n, NEXT_D);
        }
        work_flush(work, s_work);
      }
      if (fin) mode = drained ? MD_EXIT : MD_FETCH;
    }
    const unsigned need = __ballot_sync(FULL, mode == MD_FETCH);
    if (need) {
      const int q = queue_fetch(need, ctl + CT_QC, lane);
      if (mode == MD_FETCH) {
        if (q < passes * n_tasks) {
          const int pass = passes == 1 ? 0 : q / n_tasks, qq = q - pass * n_tasks;
          i = run_list ? run_list[qq] : qq;   // every tracklet passes through this phase
          const float4* __restrict__ p = reinterpret_cast<const float4*>(rec + i);
          const int4 k = reinterpret_cast<const int4*>(p)[6];
          if (len_class<K5_LONG_C>(k.y - k.x % R, passes) == pass) {   // (else: another pass takes it; the lane fetches again)
          const float4 a = p[0], f = p[5];
          st.y = a.x; st.z = a.y; st.s = a.z; st.t = a.w; st.q = rec[i].st[4];
          cl = make_float2(f.x, f.y); zref = f.z;
          u0 = k.x; r_out = k.y;
          const int sec = u0 / R;
          r0 = u0 - sec * R;
          su = units + (long long)sec * R;
          rh = rowhit + (long long)i * R;
          r = r_out; chi2 = 0.0f; n = 0; final_ = false;
          a_next = r_out - 1 >= r0 ? rh[r_out - 1] : -1;
          a_next2 = r_out - 2 >= r0 ? rh[r_out - 2] : -1;
          mode = MD_INIT;
          }
        } else mode = MD_EXIT;
      }
      drained = __any_sync(FULL, mode == MD_EXIT);
    }
    if (__all_sync(FULL, mode == MD_EXIT)) break;

    const bool run = mode == MD_RUN, init = mode == MD_INIT;
    const int rn = r - 1;
    const int a = a_next;                      // rowhit of row rn, read one step ahead
    float2 c = cl;
    TPC_CHECK(P, !run || (rn >= 0 && rn >= r0 && a < su[rn].n), 54);
    if (run && a >= 0) c = yz[su[rn].off + a]; // assigned cluster: its load hides behind the transport
    if (run && a < 0 && snap_cur) { snap_store(s_snap, tx, st); snap_cur = false; }   // this step may leave the state without an update
    bool have = init, do_pick = false;
    if (init) reset_cov(st, P);                // fresh covariance, refit inward from the outermost cluster
    __syncwarp();
    if (run) {
      work += 1u;
      const bool prop_ok = propagate(st, s_rx[rn] - s_rx[r], P);
      if (!prop_ok) { final_ = true; mode = MD_DONE; }
      else if (a >= 0) have = true;
      else if (!(fabsf(st.y) > s_re[rn] + P.edge_margin)) do_pick = true;   // outside the sector: the row is skipped (rn >= r0)
    }
    int hit = a;
    if (__any_sync(FULL, do_pick)) {           // rare here: rows between r0 and r_out that B left empty
      if (do_pick) { work += 1u << 22; hit = pickup(su[rn], yz, perm, bin_start, st, zref, P, &c); }
      __syncwarp();
      if (do_pick && hit >= 0) { have = true; rh[rn] = hit; }
    }
    float dchi = 0.0f;
    __syncwarp();
    if (have) { work += 1u << 11; dchi = update(st, c.x, c.y - zref, P); }
    __syncwarp();
    if (have) { chi2 = chi2 + dchi; n++; r_snap = init ? r_out : rn; snap_cur = true; }
    if (init) mode = MD_RUN;
    else if (run && mode == MD_RUN) { r = rn; a_next = a_next2; a_next2 = rn - 2 >= r0 ? rh[rn - 2] : -1; }
    if (mode == MD_RUN && r == r0) { final_ = r0 == 0; mode = MD_DONE; }   // rows r_out .. r0 done: finished, or on to k5d
  }
  K5_EPILOGUE();
}

// ---------------------------------------------------------------------------------------------------------------------------
// Phase C, part 2: inward extrapolation below the start row with pick-up (every row is below first_assigned: gaps count).
__global__ void __launch_bounds__(K5_THREADS, K5_CTAS_D) k5d_extend_in(const int M_host, const int* __restrict__ M_dev, const int* __restrict__ run_list,
                                                               const UnitDesc* __restrict__ units,
                                                               const RowConst* __restrict__ rows, const float2* __restrict__ yz,
                                                               const int* __restrict__ perm, const int* __restrict__ bin_start,
                                                               rowhit_t* __restrict__ rowhit, const TlRec* __restrict__ rec,
                                                               int* __restrict__ ctl, int* __restrict__ tl_n,
                                                               int* __restrict__ tl_first, int* __restrict__ tl_last,
                                                               float* __restrict__ tl_chi2, float* __restrict__ tl_par,
                                                               float* __restrict__ tl_cov, unsigned long long* __restrict__ counters,
                                                               const Params P) {
  K5_PROLOGUE();
  __shared__ float s_snap[20][K5_THREADS];   // state after the last update
  const int n_tasks = M_dev ? min(*M_dev, M_host) : M_host;
  const int passes = len_passes<K5_LONG_D>(n_tasks);
  int* const qd = ctl + CT_QD;
  int i = -1, r = 0, r_out = 0, r_snap = 0, n = 0, gap = 0;
  float zref = 0.0f, chi2 = 0.0f;
  State st = {};
  const UnitDesc* __restrict__ su = units;
  rowhit_t* __restrict__ rh = rowhit;

  for (;;) {
    if (flush_now(mode, drained)) {
      if (mode == MD_DONE) {
        float v[20];
#pragma unroll
        for (int k = 0; k < 20; k++) v[k] = s_snap[k][tx];
        write_tracklet(i, n, r_snap, r_out, chi2, zref, v, tl_n, tl_first, tl_last, tl_chi2, tl_par, tl_cov);
        work_flush(work, s_work);
        mode = drained ? MD_EXIT : MD_FETCH;
      }
    }
    const unsigned need = __ballot_sync(FULL, mode == MD_FETCH);
    if (need) {
      const int q = queue_fetch(need, qd, lane);
      if (mode == MD_FETCH) {
        if (q < passes * n_tasks) {
          const int pass = passes == 1 ? 0 : q / n_tasks, qq = q - pass * n_tasks;
          i = run_list ? run_list[qq] : qq;
          const float4* __restrict__ p = reinterpret_cast<const float4*>(rec + i);
          const int4 k = reinterpret_cast<const int4*>(p)[6];
          // (not NEXT_D: the tracklet ended in k5c; not this pass's class: another pass takes it; the lane fetches again)
          const bool mine = k.w == NEXT_D && len_class<K5_LONG_D>(k.x % R, passes) == pass;
          if (mine) {
          load_state(st, p);
          const float4 f = p[5];
          zref = f.z; chi2 = f.w;
          const int sec = k.x / R;
          r = r_snap = k.x - sec * R; r_out = k.y; n = k.z; gap = 0;
          su = units + (long long)sec * R;
          rh = rowhit + (long long)i * R;
          snap_store(s_snap, tx, st);
          mode = MD_RUN;
          }
        } else mode = MD_EXIT;
      }
      drained = __any_sync(FULL, mode == MD_EXIT);
    }
    if (__all_sync(FULL, mode == MD_EXIT)) break;

    const bool run = mode == MD_RUN;
    const int rn = r - 1;
    bool do_pick = false;
    __syncwarp();
    if (run) {
      work += 1u;
      const bool prop_ok = propagate(st, s_rx[rn] - s_rx[r], P);
      if (!prop_ok || fabsf(st.y) > s_re[rn] + P.edge_margin) mode = MD_DONE;   // below first_assigned both end the tracklet
      else do_pick = true;
    }
    float2 c = make_float2(0.f, 0.f);
    int hit = -1;
    __syncwarp();
    if (do_pick) { TPC_CHECK(P, rn >= 0, 55); work += 1u << 22; hit = pickup(su[rn], yz, perm, bin_start, st, zref, P, &c); TPC_CHECK(P, hit < su[rn].n, 56); }
    __syncwarp();
    const bool have = do_pick && hit >= 0;
    if (do_pick) {
      rh[rn] = hit;
      if (!have) { gap++; if (gap > P.max_gap) mode = MD_DONE; }
    }
    float dchi = 0.0f;
    __syncwarp();
    if (have) { work += 1u << 11; dchi = update(st, c.x, c.y - zref, P); }
    __syncwarp();
    if (have) { chi2 = chi2 + dchi; n++; r_snap = rn; gap = 0; snap_store(s_snap, tx, st); }
    if (do_pick) { r = rn; if (rn == 0) mode = MD_DONE; }
  }
  K5_EPILOGUE();
}

template <class K> int persistent_blocks(K kernel, int sm_count) {
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, K5_THREADS, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
  return sm_count * per_sm;
}

}  // namespace

size_t k5_scratch_bytes(long long M) {   // TlRec array + control block
  const size_t m = (size_t)(M > 0 ? M : 1);
  return m * sizeof(TlRec) + 128;
}

// d_scratch: k5_scratch_bytes(M) bytes, 128-byte aligned.  d_counters: three 64-bit work counters (accumulated).
// n_run tasks (entries of d_run_list, or the first n_run start hits); with d_n_run the count is read from device memory and n_run is
// its upper bound.  M: capacity of the per-tracklet arrays / scratch.
int launch_k5_tracklets(const Launch& L, int n_run, const int* d_n_run, int M, const int* d_run_list, const int* d_start_unit, const int* d_start_pos,
                        const UnitDesc* d_units, const RowConst* d_rows, const float2* d_yz, const int* d_perm, const int* d_bin_start,
                        const int* d_link_up, rowhit_t* d_rowhit, int* d_tl_n, int* d_tl_first, int* d_tl_last, float* d_tl_chi2,
                        float* d_tl_par, float* d_tl_cov, unsigned long long* d_counters, void* d_scratch, const Params& P) {
  if (n_run <= 0) return 0;
  if (P.R > K5_MAX_ROWS) return -(int)cudaErrorInvalidValue;   // tpc_create limits n_rows to 255 (selector key)
  char* base = (char*)d_scratch;
  TlRec* rec = (TlRec*)base;
  int* ctl = (int*)(base + (size_t)M * sizeof(TlRec));
  cudaError_t e = cudaMemsetAsync(ctl, 0, CT_WORDS * sizeof(int), L.stream);
  if (e != cudaSuccess) return -(int)e;
  static int nb_a = 0, nb_b = 0, nb_c = 0, nb_d = 0;
  if (!nb_a) {
    nb_a = persistent_blocks(k5a_seed_fit, L.sm_count); nb_b = persistent_blocks(k5b_extend_out, L.sm_count);
    nb_c = persistent_blocks(k5c_refit_in, L.sm_count); nb_d = persistent_blocks(k5d_extend_in, L.sm_count);
  }
  const int need = (n_run + K5_THREADS - 1) / K5_THREADS;
  k5a_seed_fit<<<nb_a < need ? nb_a : need, K5_THREADS, 0, L.stream>>>(n_run, d_n_run, d_run_list, d_start_unit, d_start_pos, d_units, d_rows, d_yz,
                                                                      d_link_up, d_rowhit, rec, ctl, d_counters, P);
  k5b_extend_out<<<nb_b < need ? nb_b : need, K5_THREADS, 0, L.stream>>>(n_run, d_n_run, d_run_list, d_units, d_rows, d_yz, d_perm, d_bin_start,
                                                                        d_rowhit, rec, ctl, d_counters, P);
  k5c_refit_in<<<nb_c < need ? nb_c : need, K5_THREADS, 0, L.stream>>>(n_run, d_n_run, d_run_list, d_units, d_rows, d_yz, d_perm, d_bin_start,
                                                                      d_rowhit, rec, ctl, d_tl_n, d_tl_first, d_tl_last, d_tl_chi2, d_tl_par,
                                                                      d_tl_cov, d_counters, P);
  k5d_extend_in<<<nb_d < need ? nb_d : need, K5_THREADS, 0, L.stream>>>(n_run, d_n_run, d_run_list, d_units, d_rows, d_yz, d_perm, d_bin_start,
                                                                       d_rowhit, rec, ctl, d_tl_n, d_tl_first, d_tl_last, d_tl_chi2, d_tl_par,
                                                                       d_tl_cov, d_counters, P);
  e = cudaGetLastError();
  return e == cudaSuccess ? 4 : -(int)e;
}

}  // namespace tpc
