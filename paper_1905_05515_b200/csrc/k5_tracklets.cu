// k5_tracklets.cu -- K5: S5 Kalman-filter tracklet constructor ("first preliminary fit, used to find the full track";
// PAPER.md:41 single hypothesis per seed, linear in the event size; definition in DESIGN.md section 4).
//
// One lane per tracklet (= start hit) at a time, persistent CTAs with a global work queue.  The 5-parameter state (y, z_rel, sin phi, dz/ds, q/pT) and the 15 covariance
// entries live in registers, fp32.  Phases: A seed fit along the cleaned up-links, B outward extrapolation row by row in the
// uniform Bz helix with cluster pick-up from the S1 grid, C inward refit + inward extrapolation.  z is carried relative to the
// start hit (z_rel = z - z_ref, formed in fp32 before use) so that long continuous time frames (|z| up to 2.6e4 cm) keep
// full fp32 resolution.  Arithmetic is written term by term in the documented order and compiled without FMA contraction (the fused multiply-adds of
// the transport / update are explicit, reading A43),
// so pick-up decisions agree with the fp32 definition.
// rowhit layout: [tracklet][row]: a lane writes and re-reads consecutive rows of its own tracklet (L2-resident while the tracklet
// is alive).  Only rows between the first and the last row a tracklet visits are written; tl_first / tl_last delimit the valid
// range (no memset of the table).
#include "kalman.cuh"

namespace tpc {
namespace {

constexpr int K5_THREADS = 128;
constexpr int K5_MAX_ROWS = 256;   // rows held in the shared-memory copy of the row table (the launcher checks R)

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
  // the row's cluster base pointer is materialised once (the empty asm keeps the compiler from re-deriving them from the 64-bit
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


// Per-lane modes of the row-step state machine.  Every loop iteration of a warp is ONE row step for every lane: (maybe) transport,
// select the measurement for the row, (maybe) Kalman update, bookkeeping.  Lanes in different phases of different tracklets
// therefore execute the same transport / update instruction streams together; a lane that finishes a tracklet pulls the next
// one from a global work queue (persistent CTAs), so short and long tracklets balance out.
enum : int { MD_FETCH = 0, MD_INIT, MD_A, MD_B, MD_TRANS, MD_C, MD_EXIT };

__global__ void __launch_bounds__(K5_THREADS, 6) k5_tracklets(const int M, const int* __restrict__ run_list,
                                                              const int* __restrict__ start_unit,
                                                              const int* __restrict__ start_pos, const UnitDesc* __restrict__ units,
                                                              const RowConst* __restrict__ rows, const float2* __restrict__ yz,
                                                              const int* __restrict__ perm, const int* __restrict__ bin_start,
                                                              const int* __restrict__ link_up, int* __restrict__ rowhit,
                                                              int* __restrict__ tl_n, int* __restrict__ tl_first,
                                                              int* __restrict__ tl_last, float* __restrict__ tl_chi2,
                                                              float* __restrict__ tl_par, float* __restrict__ tl_cov,
                                                              unsigned long long* __restrict__ counters, int* __restrict__ queue,
                                                              const Params P) {
  const unsigned FULL = 0xffffffffu;
  const int R = P.R, lane = threadIdx.x & 31;
  int mode = MD_FETCH;
  int i = -1, r0 = 0, r = 0, nxt = -1, a_next = -1, a_next2 = -1, r_out = 0;
  // four small per-tracklet integers (each below 256: tpc_create limits n_rows to 255) in ONE register, so that the row step stays inside
  // 80 registers: byte 0 = n (updates of phase C), 1 = gap (consecutive rows without a cluster), 2 = first_assigned, 3 = r_snap
  unsigned pk = 0;
  float zref = 0.0f, chi2 = 0.0f;
  State st = {};
  // per-row x and sector half-width in shared memory (2 x 1 KB): read by every lane at every step
  __shared__ float s_rx[K5_MAX_ROWS], s_re[K5_MAX_ROWS];
  for (int k = threadIdx.x; k < R && k < K5_MAX_ROWS; k += blockDim.x) { s_rx[k] = rows[k].x; s_re[k] = rows[k].yedge; }
  __syncthreads();
  __shared__ float s_snap[20][K5_THREADS];   // state after the last Phase-C update, per lane (written often, read once)
  const int tx = threadIdx.x;
  __shared__ float s_sv[7][K5_THREADS];       // state after the outermost update (5 parameters) + that cluster (y, z)
  const UnitDesc* __restrict__ su = units;
  int* __restrict__ rh = rowhit;
  // work counters of the current tracklet packed into one register (transports: bits 0-10, updates: 11-21, pick-ups: 22-31; a tracklet
  // has at most 2 R < 2^9 of each), added to the CTA's shared counters when the tracklet finishes
  unsigned work = 0;
  __shared__ unsigned s_work[3];
  if (threadIdx.x < 3) s_work[threadIdx.x] = 0;
  __syncthreads();

  for (;;) {
    // ---- work queue: lanes without a tracklet take the next start hits (one atomic per warp)
    const unsigned need = __ballot_sync(FULL, mode == MD_FETCH);
    if (need) {
      const int leader = __ffs(need) - 1;
      int base = 0;
      if (lane == leader) base = atomicAdd(queue, __popc(need));
      base = __shfl_sync(FULL, base, leader);
      if (mode == MD_FETCH) {
        i = base + __popc(need & ((1u << lane) - 1u));   // queue position; M = entries to run
        if (i < M) {
          if (run_list) i = run_list[i];                 // a sub-list of the start hits (rescue variant): tracklet index = list entry
          const int u0 = start_unit[i];
          const int h0 = start_pos[i];
          const int sec = u0 / R;
          r0 = u0 - sec * R;
          su = units + (long long)sec * R;
          rh = rowhit + (long long)i * R;
          const long long o0 = su[r0].off + h0;
          const float2 c0 = yz[o0];   // the start hit: read once, here; INIT takes it from (st.y, zref), its position from nxt
          st.y = c0.x; zref = c0.y; nxt = h0;
          a_next = link_up[o0];       // and its up-link (a_next is free until phase C)
          mode = MD_INIT;
        } else {
          mode = MD_EXIT;
        }
      }
    }
    if (__all_sync(FULL, mode == MD_EXIT)) break;

    // ---- 1. transport to the next row (phases A, B outward; C inward).  __syncwarp() before each shared stage makes the
    //         lanes of all phases reconverge, so the transport / pick-up / update code runs once per warp and step.
    const bool moving = mode == MD_A || mode == MD_B || mode == MD_C;
    const int rn = mode == MD_C ? r - 1 : r + 1;
    bool prop_ok = true;
    // measurement prefetch: a linked (phase A) or already assigned (phase C) cluster of the target row is known before the
    // transport, so its load is issued here and its latency hides behind the transport arithmetic
    const int hit_pref = mode == MD_A ? nxt : (mode == MD_C ? a_next : -1);
    float2 c_pref = make_float2(0.f, 0.f);
    int nxt_up = -1;   // phase A: the up-link of the linked cluster is read here as well, a whole transport + update ahead of its use
    if (hit_pref >= 0) { const long long o = su[rn].off + hit_pref; c_pref = yz[o]; if (mode == MD_A) nxt_up = link_up[o]; }
    __syncwarp();
    if (moving) { work += 1u; prop_ok = propagate(st, s_rx[rn] - s_rx[r], P); }

    // ---- 2a. per-phase decision: which measurement this step uses (a linked / assigned hit, a pick-up, or none)
    bool have = false, finish = false, do_pick = false;
    float2 c = make_float2(0.f, 0.f);
    int hit = -1;
    if (mode == MD_INIT) {
      hit = nxt;
      c = make_float2(st.y, zref);  // Phase A start: direction from the origin, first update with the start hit
      const float x = s_rx[r0], y = c.x;
      const float rr = sqrtf(x * x + y * y);
      st.y = y; st.z = 0.0f; st.s = y / rr; st.t = P.continuous ? 0.0f : zref / rr; st.q = 0.0f;
      reset_cov(st, P);
      have = true;
    } else if (mode == MD_A) {      // follow the cleaned up-link, no gate
      if (!prop_ok) mode = MD_TRANS;
      else { hit = nxt; c = c_pref; have = true; }
    } else if (mode == MD_B) {      // outward extrapolation with pick-up
      if (!prop_ok || fabsf(st.y) > s_re[rn] + P.edge_margin) mode = MD_TRANS;
      else { do_pick = true; r = rn; }
    } else if (mode == MD_TRANS) {  // Phase C start: state after the outermost update, fresh covariance, refit inward
      st.y = s_sv[0][tx]; st.z = s_sv[1][tx]; st.s = s_sv[2][tx]; st.t = s_sv[3][tx]; st.q = s_sv[4][tx];
      reset_cov(st, P);
      chi2 = 0.0f; pk = (pk & 0xff000000u) | ((unsigned)r0 << 16);   // n = 0, gap = 0, first_assigned = r0
      c = make_float2(s_sv[5][tx], s_sv[6][tx]); have = true; r = r_out;
    } else if (mode == MD_C) {
      if (!prop_ok) finish = true;
      else {
        const int a = a_next;                   // rowhit of this row, read one step ahead (-1 below r0: never visited before)
        r = rn;
        if (a >= 0) { hit = a; c = c_pref; have = true; }
        else if (fabsf(st.y) > s_re[rn] + P.edge_margin) {
          if (rn < (int)((pk >> 16) & 0xffu)) finish = true;
          else if (rn < r0) rh[rn] = -1;       // skipped row inside the tracklet's range: reads as "no cluster"
        } else do_pick = true;
      }
    }
    // ---- 2b. cluster pick-up from the grid (phase B and phase C lanes together)
    __syncwarp();
    if (do_pick) { work += 1u << 22; hit = pickup(su[rn], yz, perm, bin_start, st, zref, P, &c); }
    __syncwarp();
    if (do_pick) {
      have = hit >= 0;
      if (mode == MD_B) {
        rh[rn] = hit;
        if (!have) { pk += 0x100u; if ((int)((pk >> 8) & 0xffu) > P.max_gap) mode = MD_TRANS; }
      } else {
        if (rn < r0 || have) rh[rn] = hit;
        const int fa = (int)((pk >> 16) & 0xffu);
        if (have) { if (rn < fa) pk = (pk & 0xff0000ffu) | ((unsigned)rn << 16); }   // first_assigned = rn, gap = 0
        else if (rn < fa) { pk += 0x100u; if ((int)((pk >> 8) & 0xffu) > P.max_gap) finish = true; }
      }
    }

    // ---- 3. Kalman update (all lanes that have a measurement, whatever their phase)
    float dchi = 0.0f;
    __syncwarp();
    if (have) { work += 1u << 11; dchi = update(st, c.x, c.y - zref, P); }
    __syncwarp();

    // ---- 4. bookkeeping and phase transitions
    bool save_snap = false;
    if (mode == MD_INIT) {
      rh[r0] = hit; r = r0;
      s_sv[0][tx] = st.y; s_sv[1][tx] = st.z; s_sv[2][tx] = st.s; s_sv[3][tx] = st.t; s_sv[4][tx] = st.q; r_out = r0; s_sv[5][tx] = c.x; s_sv[6][tx] = c.y;
      nxt = a_next;
      pk &= 0xffff00ffu;   // gap = 0
      mode = nxt >= 0 ? MD_A : (r0 + 1 < R ? MD_B : MD_TRANS);
    } else if (mode == MD_A) {      // (a failed transport already switched the lane to MD_TRANS)
      r = rn; rh[rn] = hit;
      s_sv[0][tx] = st.y; s_sv[1][tx] = st.z; s_sv[2][tx] = st.s; s_sv[3][tx] = st.t; s_sv[4][tx] = st.q; r_out = rn; s_sv[5][tx] = c.x; s_sv[6][tx] = c.y;
      nxt = nxt_up;
      if (nxt < 0) { pk &= 0xffff00ffu; mode = rn + 1 < R ? MD_B : MD_TRANS; }
    } else if (mode == MD_B) {
      if (have) { pk &= 0xffff00ffu; s_sv[0][tx] = st.y; s_sv[1][tx] = st.z; s_sv[2][tx] = st.s; s_sv[3][tx] = st.t; s_sv[4][tx] = st.q; r_out = rn; s_sv[5][tx] = c.x; s_sv[6][tx] = c.y; }
      if (rn + 1 >= R) mode = MD_TRANS;
    } else if (mode == MD_TRANS) {
      if (have) {                   // (have is false only for lanes that switched to MD_TRANS in step 2 of this iteration)
        chi2 = chi2 + dchi; pk = (pk & 0x00ffff00u) | 1u | ((unsigned)r_out << 24); save_snap = true;   // n = 1, r_snap = r_out
        if (r_out - 1 >= 0) { mode = MD_C; a_next = r_out - 1 >= r0 ? rh[r_out - 1] : -1; a_next2 = r_out - 2 >= r0 ? rh[r_out - 2] : -1; }
        else finish = true;
      }
    } else if (mode == MD_C) {
      if (have) { chi2 = chi2 + dchi; pk = ((pk + 1u) & 0x00ffffffu) | ((unsigned)rn << 24); save_snap = true; }   // n++, r_snap = rn
      if (!finish && rn == 0) finish = true;
      if (!finish) { a_next = a_next2; a_next2 = rn - 2 >= r0 ? rh[rn - 2] : -1; }   // rowhit is read two rows ahead
    }

    if (save_snap) { s_snap[0][tx] = st.y; s_snap[1][tx] = st.z; s_snap[2][tx] = st.s; s_snap[3][tx] = st.t; s_snap[4][tx] = st.q;
          s_snap[5][tx] = st.c00; s_snap[6][tx] = st.c10; s_snap[7][tx] = st.c11; s_snap[8][tx] = st.c20; s_snap[9][tx] = st.c21;
          s_snap[10][tx] = st.c22; s_snap[11][tx] = st.c30; s_snap[12][tx] = st.c31; s_snap[13][tx] = st.c32; s_snap[14][tx] = st.c33;
          s_snap[15][tx] = st.c40; s_snap[16][tx] = st.c41; s_snap[17][tx] = st.c42; s_snap[18][tx] = st.c43; s_snap[19][tx] = st.c44; }

    if (finish) {   // tracklet complete: hits exist exactly on the rows [r_snap, r_out] that carry a non-negative rowhit
      tl_n[i] = (int)(pk & 0xffu); tl_first[i] = (int)(pk >> 24); tl_last[i] = r_out; tl_chi2[i] = chi2;
      float* __restrict__ op = tl_par + (long long)i * 5;
      op[0] = s_snap[0][tx]; op[1] = s_snap[1][tx] + zref; op[2] = s_snap[2][tx]; op[3] = s_snap[3][tx]; op[4] = s_snap[4][tx];
      float* __restrict__ oc = tl_cov + (long long)i * 15;
#pragma unroll
      for (int k = 0; k < 15; k++) oc[k] = s_snap[5 + k][tx];
      atomicAdd(&s_work[0], work & 0x7ffu); atomicAdd(&s_work[1], (work >> 11) & 0x7ffu); atomicAdd(&s_work[2], work >> 22);
      work = 0;
      mode = MD_FETCH;
    }
  }
  // work counters: one atomic per CTA and counter (every tracklet has flushed its counts when its lane left the loop)
  __syncthreads();
  if (threadIdx.x < 3) atomicAdd(&counters[threadIdx.x], (unsigned long long)s_work[threadIdx.x]);
}

}  // namespace

int launch_k5_tracklets(const Launch& L, int M, long long Mpad, const int* d_run_list, const int* d_start_unit, const int* d_start_pos,
                        const UnitDesc* d_units,
                        const RowConst* d_rows, const float2* d_yz, const int* d_perm, const int* d_bin_start, const int* d_link_up,
                        int* d_rowhit, int* d_tl_n, int* d_tl_first, int* d_tl_last, float* d_tl_chi2, float* d_tl_par,
                        float* d_tl_cov, unsigned long long* d_counters, const Params& P) {
  (void)Mpad;
  if (M <= 0) return 0;
  if (P.R > K5_MAX_ROWS) return -(int)cudaErrorInvalidValue;   // tpc_create limits n_rows to 255 (selector key)
  int* d_queue = reinterpret_cast<int*>(d_counters + 3);   // work-queue head, zeroed with the counters by the caller
  int per_sm = 0;
  cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k5_tracklets, K5_THREADS, 0);
  if (e != cudaSuccess) return -(int)e;
  if (per_sm < 1) per_sm = 1;
  int blocks = L.sm_count * per_sm;                         // persistent CTAs: one resident wave
  const int need = (M + K5_THREADS - 1) / K5_THREADS;
  if (blocks > need) blocks = need;
  k5_tracklets<<<blocks, K5_THREADS, 0, L.stream>>>(M, d_run_list, d_start_unit, d_start_pos, d_units, d_rows, d_yz, d_perm, d_bin_start, d_link_up,
                                                    d_rowhit, d_tl_n, d_tl_first, d_tl_last, d_tl_chi2, d_tl_par, d_tl_cov, d_counters,
                                                    d_queue, P);
  e = cudaGetLastError();
  return e == cudaSuccess ? 1 : -(int)e;
}

}  // namespace tpc
