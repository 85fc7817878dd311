// k5_tracklets.cu -- K5: S5 Kalman-filter tracklet constructor ("first preliminary fit, used to find the full track";
// PAPER.md:41 single hypothesis per seed, linear in the event size; definition in DESIGN.md section 4).
//
// One lane per tracklet (= start hit) at a time, persistent CTAs with a global work queue.  The 5-parameter state (y, z_rel, sin phi, dz/ds, q/pT) and the 15 covariance
// entries live in registers, fp32.  Phases: A seed fit along the cleaned up-links, B outward extrapolation row by row in the
// uniform Bz helix with cluster pick-up from the S1 grid, C inward refit + inward extrapolation.  z is carried relative to the
// start hit (z_rel = z - z_ref, formed in fp32 before use) so that long continuous time frames (|z| up to 2.6e4 cm) keep
// full fp32 resolution.  Arithmetic is written term by term in the documented order and compiled without FMA contraction,
// so pick-up decisions agree with the fp32 definition.
// rowhit layout: [tracklet][row]: a lane writes and re-reads consecutive rows of its own tracklet (L2-resident while the tracklet
// is alive).  Only rows between the first and the last row a tracklet visits are written; tl_first / tl_last delimit the valid
// range (no memset of the table).
#include "tpc_internal.cuh"

namespace tpc {
namespace {

constexpr int K5_THREADS = 128;

// lower-triangle indices of the symmetric 5x5 covariance, row-major: (0,0)(1,0)(1,1)(2,0)(2,1)(2,2)(3,0)...(4,4)
struct State {
  float y, z, s, t, q;
  float c00, c10, c11, c20, c21, c22, c30, c31, c32, c33, c40, c41, c42, c43, c44;
};

__device__ __forceinline__ void reset_cov(State& st, const Params& P) {
  st.c00 = P.c0[0]; st.c11 = P.c0[1]; st.c22 = P.c0[2]; st.c33 = P.c0[3]; st.c44 = P.c0[4];
  st.c10 = st.c20 = st.c21 = st.c30 = st.c31 = st.c32 = st.c40 = st.c41 = st.c42 = st.c43 = 0.0f;
}

// Helix transport x -> x+dx in uniform Bz, covariance C' = F C F^T (F written out: only F02 F04 F12 F13 F14 F24 are non-trivial).
// false: |sin phi| would leave [-s_max, s_max].
__device__ __forceinline__ bool propagate(State& st, const float dx, const Params& P) {
  const float cB = P.cB;
  const float s = st.s, t = st.t;
  const float k = cB * st.q;
  const float kdx = k * dx;
  const float s1 = s + kdx;
  if (!(fabsf(s) <= P.smax) || !(fabsf(s1) <= P.smax)) return false;
  const float c = sqrtf(1.0f - s * s), c1 = sqrtf(1.0f - s1 * s1);
  const float cc = c + c1, ss = s + s1, tq = ss / cc;
  const float g = 1.0f + tq * tq;
  const float L = dx * sqrtf(g);
  const float h = (0.5f * k) * L, h2 = h * h;
  float S;
  if (fabsf(h) < 0.25f) {   // asin(h)/h = 1 + h^2/6 + 3h^4/40 + 15h^6/336 + 105h^8/3456
    float poly = (float)(105.0 / 3456.0);
    poly = (float)(15.0 / 336.0) + h2 * poly;
    poly = (float)(3.0 / 40.0) + h2 * poly;
    poly = (float)(1.0 / 6.0) + h2 * poly;
    poly = 1.0f + h2 * poly;
    S = L * poly;
  } else {
    S = (2.0f / k) * asinf(h);
  }
  float dSdk;
  if (fabsf(kdx) >= 1e-2f) {
    dSdk = (dx / c1 - S) / k;
  } else {
    const float sm = (s + 2.0f * s1) / 3.0f;
    const float cm2 = 1.0f - sm * sm;
    const float cm = sqrtf(cm2);
    dSdk = ((dx * dx) * sm) / (2.0f * (cm2 * cm));
  }
  const float cc1 = c * c1;
  const float f02 = ((dx * g) * cc) / (2.0f * cc1);
  const float f04 = (((dx * dx) * cB) * g) / (2.0f * c1);
  const float f12 = ((t * dx) * tq) / cc1;
  const float f13 = S;
  const float f14 = (t * cB) * dSdk;
  const float f24 = cB * dx;
  st.y = st.y + dx * tq;
  st.z = st.z + t * S;
  st.s = s1;
  // T = F C   (row i of T = sum_m F[i][m] C[m][:], accumulated in the order m = 0..4; zero terms add exactly nothing)
  const float t00 = (st.c00 + f02 * st.c20) + f04 * st.c40;
  const float t01 = (st.c10 + f02 * st.c21) + f04 * st.c41;
  const float t02 = (st.c20 + f02 * st.c22) + f04 * st.c42;
  const float t03 = (st.c30 + f02 * st.c32) + f04 * st.c43;
  const float t04 = (st.c40 + f02 * st.c42) + f04 * st.c44;
  const float t10 = ((st.c10 + f12 * st.c20) + f13 * st.c30) + f14 * st.c40;
  const float t11 = ((st.c11 + f12 * st.c21) + f13 * st.c31) + f14 * st.c41;
  const float t12 = ((st.c21 + f12 * st.c22) + f13 * st.c32) + f14 * st.c42;
  const float t13 = ((st.c31 + f12 * st.c32) + f13 * st.c33) + f14 * st.c43;
  const float t14 = ((st.c41 + f12 * st.c42) + f13 * st.c43) + f14 * st.c44;
  const float t20 = st.c20 + f24 * st.c40;
  const float t21 = st.c21 + f24 * st.c41;
  const float t22 = st.c22 + f24 * st.c42;
  const float t23 = st.c32 + f24 * st.c43;
  const float t24 = st.c42 + f24 * st.c44;
  const float t30 = st.c30, t31 = st.c31, t32 = st.c32, t33 = st.c33, t34 = st.c43;
  const float t40 = st.c40, t41 = st.c41, t42 = st.c42, t43 = st.c43, t44 = st.c44;
  // C' = T F^T, lower triangle: C'[i][j] = sum_m T[i][m] F[j][m]
  st.c00 = (t00 + t02 * f02) + t04 * f04;
  st.c10 = (t10 + t12 * f02) + t14 * f04;
  st.c11 = ((t11 + t12 * f12) + t13 * f13) + t14 * f14;
  st.c20 = (t20 + t22 * f02) + t24 * f04;
  st.c21 = ((t21 + t22 * f12) + t23 * f13) + t24 * f14;
  st.c22 = t22 + t24 * f24;
  st.c30 = (t30 + t32 * f02) + t34 * f04;
  st.c31 = ((t31 + t32 * f12) + t33 * f13) + t34 * f14;
  st.c32 = t32 + t34 * f24;
  st.c33 = t33;
  st.c40 = (t40 + t42 * f02) + t44 * f04;
  st.c41 = ((t41 + t42 * f12) + t43 * f13) + t44 * f14;
  st.c42 = t42 + t44 * f24;
  st.c43 = t43;
  st.c44 = t44;
  (void)t01; (void)t03;
  return true;
}

// Kalman update with the joint 2-D measurement (ym, zm), R = diag(sigma_y^2, sigma_z^2); returns the chi2 increment.
__device__ __forceinline__ float update(State& st, const float ym, const float zm, const Params& P) {
  const float s00 = st.c00 + P.ry, s10 = st.c10, s11 = st.c11 + P.rz;
  const float det = s00 * s11 - s10 * s10;
  const float i00 = s11 / det, i11 = s00 / det, i10 = -s10 / det;
  const float r0 = ym - st.y, r1 = zm - st.z;
  // K = C[:,0:2] S^-1
  const float k00 = st.c00 * i00 + st.c10 * i10, k01 = st.c00 * i10 + st.c10 * i11;
  const float k10 = st.c10 * i00 + st.c11 * i10, k11 = st.c10 * i10 + st.c11 * i11;
  const float k20 = st.c20 * i00 + st.c21 * i10, k21 = st.c20 * i10 + st.c21 * i11;
  const float k30 = st.c30 * i00 + st.c31 * i10, k31 = st.c30 * i10 + st.c31 * i11;
  const float k40 = st.c40 * i00 + st.c41 * i10, k41 = st.c40 * i10 + st.c41 * i11;
  // C' = C - K C[0:2,:], lower triangle; C[0][j] = c_j0, C[1][j] = c_j1 (symmetric storage)
  const float o00 = st.c00, o10 = st.c10, o11 = st.c11, o20 = st.c20, o21 = st.c21, o30 = st.c30, o31 = st.c31, o40 = st.c40, o41 = st.c41;
  st.c00 = o00 - (k00 * o00 + k01 * o10);
  st.c10 = o10 - (k10 * o00 + k11 * o10);
  st.c11 = o11 - (k10 * o10 + k11 * o11);
  st.c20 = o20 - (k20 * o00 + k21 * o10);
  st.c21 = o21 - (k20 * o10 + k21 * o11);
  st.c22 = st.c22 - (k20 * o20 + k21 * o21);
  st.c30 = o30 - (k30 * o00 + k31 * o10);
  st.c31 = o31 - (k30 * o10 + k31 * o11);
  st.c32 = st.c32 - (k30 * o20 + k31 * o21);
  st.c33 = st.c33 - (k30 * o30 + k31 * o31);
  st.c40 = o40 - (k40 * o00 + k41 * o10);
  st.c41 = o41 - (k40 * o10 + k41 * o11);
  st.c42 = st.c42 - (k40 * o20 + k41 * o21);
  st.c43 = st.c43 - (k40 * o30 + k41 * o31);
  st.c44 = st.c44 - (k40 * o40 + k41 * o41);
  st.y = st.y + (k00 * r0 + k01 * r1);
  st.z = st.z + (k10 * r0 + k11 * r1);
  st.s = st.s + (k20 * r0 + k21 * r1);
  st.t = st.t + (k30 * r0 + k31 * r1);
  st.q = st.q + (k40 * r0 + k41 * r1);
  return r0 * (i00 * r0 + i10 * r1) + r1 * (i10 * r0 + i11 * r1);
}

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
  const int* __restrict__ bs = bin_start + d.bin_off;
  const float2* __restrict__ hits = yz + d.off;
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
        cc[j] = k < total ? hits[k < n0 ? pa0 + k : pa1 + (k - n0)] : make_float2(0.f, 0.f);
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

__global__ void __launch_bounds__(K5_THREADS, 6) k5_tracklets(const int M, const int* __restrict__ start_unit,
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
  int i = -1, r0 = 0, r = 0, nxt = -1, a_next = -1, a_next2 = -1, r_out = 0, gap = 0, n = 0, r_snap = 0, first_assigned = 0;
  float zref = 0.0f, chi2 = 0.0f;
  State st = {};
  __shared__ float s_snap[20][K5_THREADS];   // state after the last Phase-C update, per lane (written often, read once)
  const int tx = threadIdx.x;
  __shared__ float s_sv[7][K5_THREADS];       // state after the outermost update (5 parameters) + that cluster (y, z)
  const UnitDesc* __restrict__ su = units;
  int* __restrict__ rh = rowhit;
  unsigned n_prop = 0, n_upd = 0, n_pick = 0;

  for (;;) {
    // ---- work queue: lanes without a tracklet take the next start hits (one atomic per warp)
    const unsigned need = __ballot_sync(FULL, mode == MD_FETCH);
    if (need) {
      const int leader = __ffs(need) - 1;
      int base = 0;
      if (lane == leader) base = atomicAdd(queue, __popc(need));
      base = __shfl_sync(FULL, base, leader);
      if (mode == MD_FETCH) {
        i = base + __popc(need & ((1u << lane) - 1u));
        if (i < M) {
          const int u0 = start_unit[i];
          const int h0 = start_pos[i];
          const int sec = u0 / R;
          r0 = u0 - sec * R;
          su = units + (long long)sec * R;
          rh = rowhit + (long long)i * R;
          zref = yz[su[r0].off + h0].y;
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
    if (hit_pref >= 0) c_pref = yz[su[rn].off + hit_pref];
    __syncwarp();
    if (moving) { n_prop++; prop_ok = propagate(st, rows[rn].x - rows[r].x, P); }

    // ---- 2a. per-phase decision: which measurement this step uses (a linked / assigned hit, a pick-up, or none)
    bool have = false, finish = false, do_pick = false;
    float2 c = make_float2(0.f, 0.f);
    int hit = -1;
    if (mode == MD_INIT) {
      hit = start_pos[i];
      c = yz[su[r0].off + hit];
      const float2 c0 = c;          // Phase A start: direction from the origin, first update with the start hit
      const float x = rows[r0].x, y = c0.x;
      const float rr = sqrtf(x * x + y * y);
      st.y = y; st.z = 0.0f; st.s = y / rr; st.t = P.continuous ? 0.0f : zref / rr; st.q = 0.0f;
      reset_cov(st, P);
      have = true;
    } else if (mode == MD_A) {      // follow the cleaned up-link, no gate
      if (!prop_ok) mode = MD_TRANS;
      else { hit = nxt; c = c_pref; have = true; }
    } else if (mode == MD_B) {      // outward extrapolation with pick-up
      if (!prop_ok || fabsf(st.y) > rows[rn].yedge + P.edge_margin) mode = MD_TRANS;
      else { do_pick = true; r = rn; }
    } else if (mode == MD_TRANS) {  // Phase C start: state after the outermost update, fresh covariance, refit inward
      st.y = s_sv[0][tx]; st.z = s_sv[1][tx]; st.s = s_sv[2][tx]; st.t = s_sv[3][tx]; st.q = s_sv[4][tx];
      reset_cov(st, P);
      chi2 = 0.0f; n = 0; first_assigned = r0; gap = 0;
      c = make_float2(s_sv[5][tx], s_sv[6][tx]); have = true; r = r_out;
    } else if (mode == MD_C) {
      if (!prop_ok) finish = true;
      else {
        const int a = a_next;                   // rowhit of this row, read one step ahead (-1 below r0: never visited before)
        r = rn;
        if (a >= 0) { hit = a; c = c_pref; have = true; }
        else if (fabsf(st.y) > rows[rn].yedge + P.edge_margin) {
          if (rn < first_assigned) finish = true;
          else if (rn < r0) rh[rn] = -1;       // skipped row inside the tracklet's range: reads as "no cluster"
        } else do_pick = true;
      }
    }
    // ---- 2b. cluster pick-up from the grid (phase B and phase C lanes together)
    __syncwarp();
    if (do_pick) { n_pick++; hit = pickup(su[rn], yz, perm, bin_start, st, zref, P, &c); }
    __syncwarp();
    if (do_pick) {
      have = hit >= 0;
      if (mode == MD_B) {
        rh[rn] = hit;
        if (!have && ++gap > P.max_gap) mode = MD_TRANS;
      } else {
        if (rn < r0 || have) rh[rn] = hit;
        if (have) { if (rn < first_assigned) { first_assigned = rn; gap = 0; } }
        else if (rn < first_assigned && ++gap > P.max_gap) finish = true;
      }
    }

    // ---- 3. Kalman update (all lanes that have a measurement, whatever their phase)
    float dchi = 0.0f;
    __syncwarp();
    if (have) { n_upd++; dchi = update(st, c.x, c.y - zref, P); }
    __syncwarp();

    // ---- 4. bookkeeping and phase transitions
    bool save_snap = false;
    if (mode == MD_INIT) {
      rh[r0] = hit; r = r0;
      s_sv[0][tx] = st.y; s_sv[1][tx] = st.z; s_sv[2][tx] = st.s; s_sv[3][tx] = st.t; s_sv[4][tx] = st.q; r_out = r0; s_sv[5][tx] = c.x; s_sv[6][tx] = c.y;
      nxt = link_up[su[r0].off + hit];
      gap = 0;
      mode = nxt >= 0 ? MD_A : (r0 + 1 < R ? MD_B : MD_TRANS);
    } else if (mode == MD_A) {      // (a failed transport already switched the lane to MD_TRANS)
      r = rn; rh[rn] = hit;
      s_sv[0][tx] = st.y; s_sv[1][tx] = st.z; s_sv[2][tx] = st.s; s_sv[3][tx] = st.t; s_sv[4][tx] = st.q; r_out = rn; s_sv[5][tx] = c.x; s_sv[6][tx] = c.y;
      nxt = link_up[su[rn].off + hit];
      if (nxt < 0) { gap = 0; mode = rn + 1 < R ? MD_B : MD_TRANS; }
    } else if (mode == MD_B) {
      if (have) { gap = 0; s_sv[0][tx] = st.y; s_sv[1][tx] = st.z; s_sv[2][tx] = st.s; s_sv[3][tx] = st.t; s_sv[4][tx] = st.q; r_out = rn; s_sv[5][tx] = c.x; s_sv[6][tx] = c.y; }
      if (rn + 1 >= R) mode = MD_TRANS;
    } else if (mode == MD_TRANS) {
      if (have) {                   // (have is false only for lanes that switched to MD_TRANS in step 2 of this iteration)
        chi2 = chi2 + dchi; n = 1; r_snap = r_out; save_snap = true;
        if (r_out - 1 >= 0) { mode = MD_C; a_next = r_out - 1 >= r0 ? rh[r_out - 1] : -1; a_next2 = r_out - 2 >= r0 ? rh[r_out - 2] : -1; }
        else finish = true;
      }
    } else if (mode == MD_C) {
      if (have) { chi2 = chi2 + dchi; n++; r_snap = rn; save_snap = true; }
      if (!finish && rn == 0) finish = true;
      if (!finish) { a_next = a_next2; a_next2 = rn - 2 >= r0 ? rh[rn - 2] : -1; }   // rowhit is read two rows ahead
    }

    if (save_snap) { s_snap[0][tx] = st.y; s_snap[1][tx] = st.z; s_snap[2][tx] = st.s; s_snap[3][tx] = st.t; s_snap[4][tx] = st.q;
          s_snap[5][tx] = st.c00; s_snap[6][tx] = st.c10; s_snap[7][tx] = st.c11; s_snap[8][tx] = st.c20; s_snap[9][tx] = st.c21;
          s_snap[10][tx] = st.c22; s_snap[11][tx] = st.c30; s_snap[12][tx] = st.c31; s_snap[13][tx] = st.c32; s_snap[14][tx] = st.c33;
          s_snap[15][tx] = st.c40; s_snap[16][tx] = st.c41; s_snap[17][tx] = st.c42; s_snap[18][tx] = st.c43; s_snap[19][tx] = st.c44; }

    if (finish) {   // tracklet complete: hits exist exactly on the rows [r_snap, r_out] that carry a non-negative rowhit
      tl_n[i] = n; tl_first[i] = r_snap; tl_last[i] = r_out; tl_chi2[i] = chi2;
      float* __restrict__ op = tl_par + (long long)i * 5;
      op[0] = s_snap[0][tx]; op[1] = s_snap[1][tx] + zref; op[2] = s_snap[2][tx]; op[3] = s_snap[3][tx]; op[4] = s_snap[4][tx];
      float* __restrict__ oc = tl_cov + (long long)i * 15;
#pragma unroll
      for (int k = 0; k < 15; k++) oc[k] = s_snap[5 + k][tx];
      mode = MD_FETCH;
    }
  }
  // work counters: one atomic per warp
  for (int d = 16; d > 0; d >>= 1) {
    n_prop += __shfl_down_sync(FULL, n_prop, d); n_upd += __shfl_down_sync(FULL, n_upd, d); n_pick += __shfl_down_sync(FULL, n_pick, d);
  }
  if (lane == 0) {
    atomicAdd(&counters[0], (unsigned long long)n_prop); atomicAdd(&counters[1], (unsigned long long)n_upd);
    atomicAdd(&counters[2], (unsigned long long)n_pick);
  }
}

}  // namespace

int launch_k5_tracklets(const Launch& L, int M, long long Mpad, const int* d_start_unit, const int* d_start_pos, const UnitDesc* d_units,
                        const RowConst* d_rows, const float2* d_yz, const int* d_perm, const int* d_bin_start, const int* d_link_up,
                        int* d_rowhit, int* d_tl_n, int* d_tl_first, int* d_tl_last, float* d_tl_chi2, float* d_tl_par,
                        float* d_tl_cov, unsigned long long* d_counters, const Params& P) {
  (void)Mpad;
  if (M <= 0) return 0;
  int* d_queue = reinterpret_cast<int*>(d_counters + 3);   // work-queue head, zeroed with the counters by the caller
  int per_sm = 0;
  cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k5_tracklets, K5_THREADS, 0);
  if (e != cudaSuccess) return -(int)e;
  if (per_sm < 1) per_sm = 1;
  int blocks = L.sm_count * per_sm;                         // persistent CTAs: one resident wave
  const int need = (M + K5_THREADS - 1) / K5_THREADS;
  if (blocks > need) blocks = need;
  k5_tracklets<<<blocks, K5_THREADS, 0, L.stream>>>(M, d_start_unit, d_start_pos, d_units, d_rows, d_yz, d_perm, d_bin_start, d_link_up,
                                                    d_rowhit, d_tl_n, d_tl_first, d_tl_last, d_tl_chi2, d_tl_par, d_tl_cov, d_counters,
                                                    d_queue, P);
  e = cudaGetLastError();
  return e == cudaSuccess ? 1 : -(int)e;
}

}  // namespace tpc
