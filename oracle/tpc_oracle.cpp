/*
 * tpc_oracle.cpp -- plain, slow, single-threaded CPU ORACLE of the TPC sector track finding.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code with the CUDA library
 * (paper_1905_05515_b200/csrc) and neither includes the other.
 *
 * What it computes: PAPER.md:27-30 (section 2: time scaled to z with the average drift velocity, all
 * tracks assumed primary from the origin, a first preliminary fit used to find the full track) and
 * PAPER.md:37-41 (section 3: Cellular-Automaton seeding, then single-hypothesis Kalman track following).
 * The paper gives no formula for any step (it defers to its refs [6]-[9], not available), so every
 * step below follows the readings listed in DESIGN.md section 4 (S0..S6, A1..A33), in that order and
 * notation; each function names the step it implements.
 *
 * Two instances: Real=float (the parity reference: decisions are taken in fp32, the kernel's
 * precision, with contraction off; the only fused multiply-adds are the std::fma calls of the S5 transport / update, reading A43)
 * and Real=double (closed-form pins).
 * Build: g++ -O2 -ffp-contract=off -shared -fPIC oracle/tpc_oracle.cpp -o oracle/libtpc_oracle.so
 *
 * Pins (tests/test_oracle_*.py): S0 closed form; S1 invariants; S2 brute force O(N^2) + bin-size and
 * permutation invariance + straight lines; S3/S4 invariants; S5 propagate vs closed-form circle,
 * composition, round trip, Jacobian vs finite differences; S5 fit: noise-free helix recovery 1e-5,
 * Bz=0 exact, chi2/ndf = 1 and pulls on smeared tracks; S6 hand-built sharing cases, order invariance.
 * S4' (NEXT-2) seed bridging: hand-made single dropouts (one start hit per track), subset of the S4 list, brute-force probe.
 * S9 (NEXT-3) cross-sector matching: rotated + transported outer state against the closed-form helix in the neighbour's frame,
 *   generator labels of the matched pairs, structural invariants.  Looper-leg identification: not built.
 * S8 (NEXT-4) tube adjacency: independent numpy restatement with the closed-form helix, brute force over the rows, truth labels.
 * S7 (NEXT-1) refit + collision time: noise-free recovery, chi2/ndf = 1, t0 against the generator's collision times.
 * S5 pick-up (window n_sigma*sqrt(C+sigma^2) capped at w_max, plain squared distance, original-index tie-break) and the Phase B / C
 *   control flow (max_gap, sector edge + margin, first_assigned, reading A33, ungated Phase A / assigned rows): hand-built cases in
 *   tests/test_oracle_s5_control.py, each listing the one-line mutations it fails under.  S2 in continuous mode (the benchmarked
 *   mode): numpy restatement with unequal row pitch, tests/test_oracle_ca.py.
 * Second, TEST-ONLY fp32 build -DS5_PLAIN_ORDER (reading A44): the S5 arithmetic in SURVEY 8(c)'s first operation order; the margin
 *   of the parity claim against an independently ordered reference (tests/test_oracle_plain_order.py, tests/test_gpu_parity.py).
 * The file is also built with -fsanitize=address,undefined and run in tests/test_oracle_sanitize.py.
 * Absolute efficiency / resolution versus the paper: parity unpinned (PAPER.md:49 gives no number).
 */
#include <cmath>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>
#include <algorithm>
#include <limits>

namespace {

struct Tunables {            // DESIGN.md table T (all are readings; the paper is silent)
  double wy = 1.5, wz = 1.5, dzdx_max = 1.5, wz0 = 0.75, cut2 = 1.75;
  int min_seed = 3;
  double c0[5] = {1.0, 2.25, 1.0, 1.0, 100.0};
  double s_max = 0.95, n_sigma = 4.0, w_max = 3.0;
  int max_gap = 4;
  double edge_margin = 1.0;
  int min_hits = 10;
  double grid_min = 1.0, grid_max = 64.0, grid_scale = 1.0;   // S1 bin size clamp; scale is a test knob
  int bridge_rows = 0;          // NEXT-2 (reading A39): 0 = off; else the deepest row gap a start hit may bridge to a lower chain
  double bridge_wy = 1.0, bridge_wz = 1.5;
  int bridge_min = 3;           // clusters the lower chain must have
  int bridge_rescue = 0;        // 1: dropped start hits get their tracklet after all when the first wave left their chain unused
  int link_skip = 0;            // NEXT-2 as SURVEY 8(f).2 wrote it (reading A45): 1 = a link may skip one pad row
  double skip_cut2 = 1.75;      // cut2 of the pairs that skip a row (S2'; = cut2 by default, smaller = stricter: DESIGN.md section 11.1)
  double tube = 1.5;            // NEXT-4: radius of the tube around a track, cm
  // NEXT-3 (reading A41): cross-sector segment matching
  double merge_edge = 3.0; int merge_rows = 8; double merge_dy = 1.5, merge_dz = 2.0, merge_ds = 0.05, merge_dt = 0.05;
  // NEXT-3, second half (reading A46): legs / turns of one looping particle
  double loop_qmin = 5.0, loop_dy = 1.0, loop_ds = 0.1, loop_dt = 0.1, loop_dq = 0.5, loop_pmin = 2.0, loop_frac = 0.35; int loop_nmax = 20;
};

struct OracleBase {
  virtual ~OracleBase() {}
  virtual int load(const int64_t* unit_off, const float* y, const float* t) = 0;
  virtual int run(int upto, int brute) = 0;
  virtual int get(const char* name, const void** p, int64_t* n, int* kind) = 0;
  virtual int propagate(double* par, double* cov, double dx) = 0;
  virtual int update(double* par, double* cov, double ym, double zm, double* chi2) = 0;
  virtual int set_tracklets(int64_t n, const int32_t* sector, const int32_t* nh, const double* chi2, const int32_t* rowhit) = 0;
  virtual int pickup_hook(const double* par, const double* cov, int sector, int row, double zref, int brute) = 0;
  virtual int set_links(const int32_t* up, const int32_t* dn) = 0;
  virtual int run_range(int from, int upto, int brute) = 0;
  Tunables T;
  std::string err;
};

template <class Real>
struct Oracle : OracleBase {
  // geometry
  int NS, R; std::vector<float> row_x; double dphi, z_max, t_frame, sigma_y, sigma_z, bz, vdrift;
  bool continuous;
  // per-row constants (double -> Real once)
  std::vector<Real> X, tu, td, ar, br, thr, wzu, wzd, yedge;
  std::vector<Real> tu2, td2, ar2, br2, wzu2, wzd2, thr21, thr12, thr22;   // S2' (link_skip): the same constants for a row distance of 2
  Real cB;
  // clusters
  int64_t N = 0; std::vector<int64_t> off;           // [U+1]
  std::vector<float> in_y, in_t;
  std::vector<Real> z;                                // S0, input order
  // S1
  std::vector<Real> ys, zs; std::vector<int32_t> perm; std::vector<int64_t> bin_off; std::vector<int32_t> bin_start;
  std::vector<int32_t> g_ny, g_nz; std::vector<Real> g_ylo, g_zlo, g_invs;
  std::vector<double> g_ylo_d, g_zlo_d, g_invs_d;
  // S2/S3
  std::vector<int32_t> link_up, link_dn, clean_up, clean_dn;
  std::vector<int32_t> link_up_k, link_dn_k, clean_up_k, clean_dn_k;   // row distance of each link (1, or 2 with link_skip; 0 = no link)
  // S4
  std::vector<int32_t> start_unit, start_pos;
  // S5
  std::vector<int32_t> tl_n, tl_first, tl_last, tl_rowhit, tl_sector; std::vector<double> tl_chi2, tl_x, tl_par, tl_cov, tl_zref;
  // S6
  std::vector<int32_t> trk_sector, trk_ndf, trk_tracklet, trk_cl_row, trk_cl_index; std::vector<int64_t> trk_cl_begin;
  std::vector<double> trk_x, trk_par, trk_cov, trk_chi2;
  // S7 (NEXT-1): refit of the owned clusters + collision-time estimate
  std::vector<int32_t> rf_n, rf_ndf; std::vector<double> rf_x, rf_par, rf_cov, rf_chi2, rf_z0, rf_t0;
  // S8 (NEXT-4): attachment status of every cluster, caller's order (CSR offset of the unit + index inside the unit)
  std::vector<int32_t> cl_status, cl_track;
  std::vector<int32_t> start_wave;   // 1 = first wave, 2 = bridged start hit kept for the rescue wave (bridge_rescue)
  // S9 (NEXT-3): cross-sector segment matching
  std::vector<int32_t> mg_next, mg_prev, mg_leaver; std::vector<double> mg_outer;   // outer: x, y, z, sinphi per track
  // S10 (NEXT-3, second half): turns of one looping particle
  std::vector<int32_t> lp_prev, lp_root, lp_turn;
  std::vector<double> z_d, ys_d, zs_d;   // export copies

  Oracle(int ns, int nr, const float* rx, double dphi_, double zmax, double tframe, double sy, double sz, double bz_, double vd)
      : NS(ns), R(nr), row_x(rx, rx + nr), dphi(dphi_), z_max(zmax), t_frame(tframe), sigma_y(sy), sigma_z(sz), bz(bz_), vdrift(vd) {
    continuous = t_frame > 0;
  }

  // ---- per-row constant table: formulas of DESIGN.md section 4 "per-row constants", double -> Real once ----
  void make_tables() {
    X.assign(R, 0); tu.assign(R, 0); td.assign(R, 0); ar.assign(R, 0); br.assign(R, 0); thr.assign(R, 0);
    wzu.assign(R, 0); wzd.assign(R, 0); yedge.assign(R, 0);
    for (int r = 0; r < R; r++) {
      double x = row_x[r], xu = r + 1 < R ? row_x[r + 1] : x, xd = r > 0 ? row_x[r - 1] : x;
      double a = xu - x, b = x - xd;
      X[r] = (Real)x; tu[r] = (Real)(xu / x); td[r] = (Real)(xd / x); ar[r] = (Real)a; br[r] = (Real)b;
      thr[r] = (Real)(T.cut2 * 0.5 * (a * a + b * b));
      wzu[r] = (Real)(T.dzdx_max * a + T.wz0); wzd[r] = (Real)(T.dzdx_max * b + T.wz0);
      yedge[r] = (Real)(x * std::tan(0.5 * dphi));
    }
    // S2' (reading A45): row distance 2 upwards (index "2" first) / downwards; thr_{ku kd} = skip_cut2 * 0.5 * (a_ku^2 + b_kd^2)
    tu2.assign(R, 1); td2.assign(R, 1); ar2.assign(R, 0); br2.assign(R, 0); wzu2.assign(R, 0); wzd2.assign(R, 0);
    thr21.assign(R, 0); thr12.assign(R, 0); thr22.assign(R, 0);
    for (int r = 0; r < R; r++) {
      double x = row_x[r], xu = r + 1 < R ? row_x[r + 1] : x, xd = r > 0 ? row_x[r - 1] : x;
      double xu2 = r + 2 < R ? row_x[r + 2] : x, xd2 = r > 1 ? row_x[r - 2] : x;
      double a = xu - x, b = x - xd, a2 = xu2 - x, b2 = x - xd2;
      tu2[r] = (Real)(xu2 / x); td2[r] = (Real)(xd2 / x); ar2[r] = (Real)a2; br2[r] = (Real)b2;
      wzu2[r] = (Real)(T.dzdx_max * a2 + T.wz0); wzd2[r] = (Real)(T.dzdx_max * b2 + T.wz0);
      thr21[r] = (Real)(T.skip_cut2 * 0.5 * (a2 * a2 + b * b)); thr12[r] = (Real)(T.skip_cut2 * 0.5 * (a * a + b2 * b2));
      thr22[r] = (Real)(T.skip_cut2 * 0.5 * (a2 * a2 + b2 * b2));
    }
    cB = (Real)(-0.00299792458 * bz);
  }

  int load(const int64_t* unit_off, const float* y, const float* t) override {
    int U = NS * R; off.assign(unit_off, unit_off + U + 1); N = off[U];
    in_y.assign(y, y + N); in_t.assign(t, t + N);
    return 0;
  }

  // ---- S0: z = z_max - vdrift * t ("scales the time to z linearly using the average drift velocity") ----
  void s0_time_to_z() {
    z.resize(N);
    const Real zm = (Real)z_max, vd = (Real)vdrift;
    for (int64_t i = 0; i < N; i++) { Real prod = vd * (Real)in_t[i]; z[i] = zm - prod; }
  }

  // ---- S1: per (sector,row) 2-D grid, stable counting sort ----
  static int bin_of(Real v, Real lo, Real inv, int nb) {
    Real f = (v - lo) * inv;
    if (!(f > (Real)0)) return 0;            // negative or NaN -> bin 0
    if (f >= (Real)nb) return nb - 1;
    int b = (int)f; return b > nb - 1 ? nb - 1 : b;
  }
  void s1_grid() {
    int U = NS * R;
    g_ny.assign(U, 1); g_nz.assign(U, 1); g_ylo.assign(U, 0); g_zlo.assign(U, 0); g_invs.assign(U, 1);
    g_ylo_d.assign(U, 0); g_zlo_d.assign(U, 0); g_invs_d.assign(U, 0);
    bin_off.assign(U + 1, 0);
    for (int u = 0; u < U; u++) {
      int r = u % R; int64_t n = off[u + 1] - off[u];
      double ye = (double)row_x[r] * std::tan(0.5 * dphi);
      double y_lo = -ye - 1.0, y_hi = ye + 1.0, z_lo = -vdrift * t_frame - 1.0, z_hi = z_max + 1.0;
      double s = std::sqrt((y_hi - y_lo) * (z_hi - z_lo) / (double)std::max<int64_t>(n, 1)) * T.grid_scale;
      s = std::min(std::max(s, T.grid_min), T.grid_max);
      int ny = std::max(1, (int)std::ceil((y_hi - y_lo) / s)), nz = std::max(1, (int)std::ceil((z_hi - z_lo) / s));
      g_ny[u] = ny; g_nz[u] = nz;
      g_ylo[u] = (Real)(float)y_lo; g_zlo[u] = (Real)(float)z_lo; g_invs[u] = (Real)(float)(1.0 / s);
      g_ylo_d[u] = (double)g_ylo[u]; g_zlo_d[u] = (double)g_zlo[u]; g_invs_d[u] = (double)g_invs[u];
      bin_off[u + 1] = bin_off[u] + (int64_t)ny * nz + 1;
    }
    bin_start.assign(bin_off[U], 0); ys.resize(N); zs.resize(N); perm.resize(N);
    std::vector<int32_t> b;
    for (int u = 0; u < U; u++) {
      int64_t o = off[u], n = off[u + 1] - o; int ny = g_ny[u], nz = g_nz[u], nb = ny * nz;
      int32_t* bs = &bin_start[bin_off[u]];
      b.resize(n);
      for (int64_t i = 0; i < n; i++) {
        int by = bin_of((Real)in_y[o + i], g_ylo[u], g_invs[u], ny), bz_ = bin_of(z[o + i], g_zlo[u], g_invs[u], nz);
        b[i] = bz_ * ny + by; bs[b[i] + 1]++;
      }
      for (int k = 0; k < nb; k++) bs[k + 1] += bs[k];
      std::vector<int32_t> cur(bs, bs + nb);
      for (int64_t i = 0; i < n; i++) {      // ascending original index inside each bin
        int32_t p = cur[b[i]]++; ys[o + p] = (Real)in_y[o + i]; zs[o + p] = z[o + i]; perm[o + p] = (int32_t)i;
      }
    }
  }

  // hits of unit u (sorted positions) inside [ylo,yhi]x[zlo,zhi] bins; brute: every hit of the unit
  template <class F> void for_bins(int u, Real ylo, Real yhi, Real zlo, Real zhi, bool brute, F&& f) const {
    int64_t n = off[u + 1] - off[u];
    if (n == 0) return;
    if (brute) { for (int32_t p = 0; p < n; p++) f(p); return; }
    int ny = g_ny[u], nz = g_nz[u]; const int32_t* bs = &bin_start[bin_off[u]];
    int by0 = bin_of(ylo, g_ylo[u], g_invs[u], ny), by1 = bin_of(yhi, g_ylo[u], g_invs[u], ny);
    int bz0 = bin_of(zlo, g_zlo[u], g_invs[u], nz), bz1 = bin_of(zhi, g_zlo[u], g_invs[u], nz);
    for (int bz_ = bz0; bz_ <= bz1; bz_++)
      for (int32_t p = bs[bz_ * ny + by0]; p < bs[bz_ * ny + by1 + 1]; p++) f(p);
  }

  // ---- S2: neighbour finder -- best (up,down) pair by collinearity, window centred on the from-origin projection ----
  void s2_neighbours(bool brute) {
    link_up.assign(N, -1); link_dn.assign(N, -1); link_up_k.assign(N, 0); link_dn_k.assign(N, 0);
    const Real wy = (Real)T.wy, wz = (Real)T.wz;
    std::vector<int32_t> cu, cd;
    for (int sec = 0; sec < NS; sec++)
      for (int r = 1; r <= R - 2; r++) {
        int u = sec * R + r, uu = u + 1, ud = u - 1; int64_t o = off[u], ou = off[uu], od = off[ud], n = off[u + 1] - o;
        for (int64_t h = 0; h < n; h++) {
          Real y = ys[o + h], zz = zs[o + h];
          cu.clear(); cd.clear();
          { Real yc = y * tu[r], zc = continuous ? zz : zz * tu[r], hw = continuous ? wzu[r] : wz;
            Real ylo = yc - wy, yhi = yc + wy, zlo = zc - hw, zhi = zc + hw;
            for_bins(uu, ylo, yhi, zlo, zhi, brute, [&](int32_t p) {
              Real yu = ys[ou + p], zu = zs[ou + p];
              if (yu >= ylo && yu <= yhi && zu >= zlo && zu <= zhi) cu.push_back(p); }); }
          if (cu.empty()) continue;
          { Real yc = y * td[r], zc = continuous ? zz : zz * td[r], hw = continuous ? wzd[r] : wz;
            Real ylo = yc - wy, yhi = yc + wy, zlo = zc - hw, zhi = zc + hw;
            for_bins(ud, ylo, yhi, zlo, zhi, brute, [&](int32_t p) {
              Real yd = ys[od + p], zd = zs[od + p];
              if (yd >= ylo && yd <= yhi && zd >= zlo && zd <= zhi) cd.push_back(p); }); }
          if (cd.empty()) continue;
          bool have = false; Real bestD = 0; int32_t bu = -1, bd = -1, bpu = 0, bpd = 0;
          for (int32_t pu : cu)
            for (int32_t pd : cd) {
              Real dyu = ys[ou + pu] - y, dyd = y - ys[od + pd]; Real m1 = br[r] * dyu, m2 = ar[r] * dyd; Real ey = m1 - m2;
              Real dzu = zs[ou + pu] - zz, dzd = zz - zs[od + pd]; Real m3 = br[r] * dzu, m4 = ar[r] * dzd; Real ez = m3 - m4;
              Real e1 = ey * ey, e2 = ez * ez; Real D = e1 + e2;
              int32_t iu = perm[ou + pu], id = perm[od + pd];
              if (!have || D < bestD || (D == bestD && (iu < bpu || (iu == bpu && id < bpd)))) {
                have = true; bestD = D; bu = pu; bd = pd; bpu = iu; bpd = id; }
            }
          if (have && bestD < thr[r]) { link_up[o + h] = bu; link_dn[o + h] = bd; link_up_k[o + h] = 1; link_dn_k[o + h] = 1; }
        }
      }
    if (T.link_skip) s2_skip_links(brute);
  }

  // ---- S2' (NEXT-2 as SURVEY.md section 8(f).2 wrote it: "links that may skip a row"; reading A45; off unless link_skip = 1).
  //      A hit WITHOUT an accepted pair on the adjacent rows (S2 above is unchanged and final for the others) looks one row
  //      further: candidates on rows r+1, r+2 / r-1, r-2 in the windows of S2 scaled to the row distance k (centre y * x_{r+-k}/x_r;
  //      half-width k*wy; z: centre z * x_{r+-k}/x_r with half-width k*wz in triggered mode, centre z with half-width
  //      dzdx_max*|dx| + wz0 in continuous mode).  Pair residual as in S2 with the actual distances a = x_u - x_r, b = x_r - x_d:
  //      ey = b (y_u - y) - a (y - y_d), ez likewise, D = ey^2 + ez^2, accepted iff D < skip_cut2 * 0.5 * (a^2 + b^2)
  //      (skip_cut2 = cut2 unless set: a stricter cut for the longer lever arm keeps the efficiency of the r+-1 path).
  //      Level 3: pairs that skip one row on one side, (k_u, k_d) = (2,1) and (1,2); if none is accepted, level 4: (2,2).
  //      Within a level the accepted pair with the minimum key (D, k_u, original index of up, original index of down) wins.
  void s2_skip_links(bool brute) {
    const Real wy = (Real)T.wy, wz = (Real)T.wz;
    std::vector<int32_t> cu[3], cd[3];   // [k] candidates at row distance k
    for (int sec = 0; sec < NS; sec++)
      for (int r = 1; r <= R - 2; r++) {
        const int u = sec * R + r; const int64_t o = off[u], n = off[u + 1] - o;
        for (int64_t h = 0; h < n; h++) {
          if (link_up[o + h] >= 0) continue;
          const Real y = ys[o + h], zz = zs[o + h];
          for (int k = 1; k <= 2; k++) {
            cu[k].clear(); cd[k].clear();
            const Real kk = (Real)k;
            if (r + k <= R - 1) {
              const Real t_ = k == 1 ? tu[r] : tu2[r];
              const Real yc = y * t_, zc = continuous ? zz : zz * t_, hwy = kk * wy, hw = continuous ? (k == 1 ? wzu[r] : wzu2[r]) : kk * wz;
              const Real ylo = yc - hwy, yhi = yc + hwy, zlo = zc - hw, zhi = zc + hw;
              const int64_t ou = off[u + k];
              for_bins(u + k, ylo, yhi, zlo, zhi, brute, [&](int32_t p) {
                const Real yu = ys[ou + p], zu = zs[ou + p];
                if (yu >= ylo && yu <= yhi && zu >= zlo && zu <= zhi) cu[k].push_back(p); });
            }
            if (r - k >= 0) {
              const Real t_ = k == 1 ? td[r] : td2[r];
              const Real yc = y * t_, zc = continuous ? zz : zz * t_, hwy = kk * wy, hw = continuous ? (k == 1 ? wzd[r] : wzd2[r]) : kk * wz;
              const Real ylo = yc - hwy, yhi = yc + hwy, zlo = zc - hw, zhi = zc + hw;
              const int64_t od = off[u - k];
              for_bins(u - k, ylo, yhi, zlo, zhi, brute, [&](int32_t p) {
                const Real yd = ys[od + p], zd = zs[od + p];
                if (yd >= ylo && yd <= yhi && zd >= zlo && zd <= zhi) cd[k].push_back(p); });
            }
          }
          bool have = false; Real bestD = 0; int bku = 0, bkd = 0; int32_t bu = -1, bd = -1, bpu = 0, bpd = 0;
          auto level = [&](int ku, int kd) {
            const Real a = ku == 1 ? ar[r] : ar2[r], b = kd == 1 ? br[r] : br2[r];
            const Real lim = ku == 1 ? thr12[r] : (kd == 1 ? thr21[r] : thr22[r]);
            const int64_t ou = off[u + ku], od = off[u - kd];
            for (int32_t pu : cu[ku])
              for (int32_t pd : cd[kd]) {
                Real dyu = ys[ou + pu] - y, dyd = y - ys[od + pd]; Real m1 = b * dyu, m2 = a * dyd; Real ey = m1 - m2;
                Real dzu = zs[ou + pu] - zz, dzd = zz - zs[od + pd]; Real m3 = b * dzu, m4 = a * dzd; Real ez = m3 - m4;
                Real e1 = ey * ey, e2 = ez * ez; Real D = e1 + e2;
                if (!(D < lim)) continue;
                const int32_t iu = perm[ou + pu], id = perm[od + pd];
                if (!have || D < bestD || (D == bestD && (ku < bku || (ku == bku && (iu < bpu || (iu == bpu && id < bpd)))))) {
                  have = true; bestD = D; bku = ku; bkd = kd; bu = pu; bd = pd; bpu = iu; bpd = id; }
              }
          };
          level(1, 2); level(2, 1);
          if (!have) level(2, 2);
          if (have) { link_up[o + h] = bu; link_dn[o + h] = bd; link_up_k[o + h] = bku; link_dn_k[o + h] = bkd; }
        }
      }
  }

  // ---- S3: mutual-link cleaner (double-buffered definition) ----
  void s3_clean() {
    clean_up.assign(N, -1); clean_dn.assign(N, -1); clean_up_k.assign(N, 0); clean_dn_k.assign(N, 0);
    for (int sec = 0; sec < NS; sec++)
      for (int r = 0; r < R; r++) {
        int u = sec * R + r; int64_t o = off[u], n = off[u + 1] - o;
        for (int64_t h = 0; h < n; h++) {
          int32_t up = link_up[o + h], dn = link_dn[o + h];
          const int ku = link_up_k[o + h], kd = link_dn_k[o + h];   // row distance of the link (1; 2 only with link_skip)
          if (up >= 0 && r + ku < R && link_dn[off[u + ku] + up] == (int32_t)h && link_dn_k[off[u + ku] + up] == ku) { clean_up[o + h] = up; clean_up_k[o + h] = ku; }
          if (dn >= 0 && r - kd >= 0 && link_up[off[u - kd] + dn] == (int32_t)h && link_up_k[off[u - kd] + dn] == kd) { clean_dn[o + h] = dn; clean_dn_k[o + h] = kd; }
        }
      }
  }

  // ---- S4: start hits = chain beginnings with >= min_seed hits, ascending (sector,row,sorted pos) ----
  void s4_start_hits(bool brute = false) {
    start_unit.clear(); start_pos.clear(); start_wave.clear();
    for (int u = 0; u < NS * R; u++) {
      int64_t o = off[u], n = off[u + 1] - o;
      for (int64_t h = 0; h < n; h++) {
        if (!(clean_dn[o + h] < 0 && clean_up[o + h] >= 0)) continue;
        int len = 1; int uu = u; int32_t p = (int32_t)h;
        while (len < T.min_seed) { int32_t nx = clean_up[off[uu] + p]; if (nx < 0) break; const int k = clean_up_k[off[uu] + p]; p = nx; uu += k; len++; }
        if (len < T.min_seed) continue;
        int wave = 1;
        if (T.bridge_rows > 0 && !T.link_skip && bridged(u, (int32_t)h, brute)) { if (!T.bridge_rescue) continue; wave = 2; }
        start_unit.push_back(u); start_pos.push_back((int32_t)h); start_wave.push_back(wave);
      }
    }
  }

  // ---- S4' (NEXT-2; reading A39): seed bridging.  A missing cluster breaks a chain of mutual links over
  //      three rows, and every piece longer than min_seed seeds its own tracklet of the SAME track (about 6 per track at 5 %
  //      dropout, all but one discarded by S6).  A start hit h (row r) is dropped when it continues a lower chain: the straight
  //      line through h and its second chain cluster w (row r+2), extended down to a row r-g (2 <= g <= bridge_rows), meets the
  //      TOP c of a chain (no up link, a down link, at least min_seed clusters below), and the line through c and its second
  //      cluster below, extended up to row r, meets h -- both within (bridge_wy, bridge_wz).  The lower chain's tracklet then
  //      collects h's clusters in its outward pass (max_gap >= the bridged rows).
  bool bridged(int u, int32_t h, bool brute) const {
    const int sec = u / R, r = u % R;
    if (r + 2 >= R) return false;
    const int32_t u1 = clean_up[off[u] + h]; if (u1 < 0) return false;
    const int32_t u2 = clean_up[off[u + 1] + u1]; if (u2 < 0) return false;
    const Real wy = (Real)T.bridge_wy, wz = (Real)T.bridge_wz;
    const Real yh = ys[off[u] + h], zh = zs[off[u] + h];
    const Real dxu = X[r + 2] - X[r];
    const Real sy = (ys[off[u + 2] + u2] - yh) / dxu, sz = (zs[off[u + 2] + u2] - zh) / dxu;
    for (int g = 2; g <= T.bridge_rows && r - g >= 2; g++) {
      const int ud = sec * R + (r - g);
      const Real dx = X[r] - X[r - g];
      const Real yp = yh - sy * dx, zp = zh - sz * dx;
      const Real ylo = yp - wy, yhi = yp + wy, zlo = zp - wz, zhi = zp + wz;
      bool found = false;
      for_bins(ud, ylo, yhi, zlo, zhi, brute, [&](int32_t c) {
        if (found) return;
        const int64_t gc = off[ud] + c;
        const Real yc = ys[gc], zc = zs[gc];
        if (!(yc >= ylo && yc <= yhi && zc >= zlo && zc <= zhi)) return;
        if (clean_up[gc] >= 0) return;                       // c must be the top of its chain
        int32_t d1 = clean_dn[gc]; if (d1 < 0) return;
        int32_t d2 = clean_dn[off[ud - 1] + d1]; if (d2 < 0) return;
        { int len = 3; int uu = ud - 2; int32_t p = d2;      // at least min_seed clusters: the lower chain has its own start hit
          while (len < T.bridge_min) { if (uu <= sec * R) break; int32_t nx = clean_dn[off[uu] + p]; if (nx < 0) break; p = nx; uu--; len++; }
          if (len < T.bridge_min) return; }
        const Real dxd = X[r - g] - X[r - g - 2];
        const Real ty = (yc - ys[off[ud - 2] + d2]) / dxd, tz = (zc - zs[off[ud - 2] + d2]) / dxd;
        const Real yq = yc + ty * dx, zq = zc + tz * dx;     // lower chain extended up to row r
        if (yh >= yq - wy && yh <= yq + wy && zh >= zq - wz && zh <= zq + wz) found = true;
      });
      if (found) return true;
    }
    return false;
  }

  // ---- S5 building blocks ----
  struct State { Real p[5]; Real C[5][5]; };

#ifdef S5_PLAIN_ORDER
  // ---- TEST-ONLY second fp32 build (-DS5_PLAIN_ORDER, liboracle "plain"): the S5 transport / update in the operation order of
  //      SURVEY.md section 8(c) as first written -- every Jacobian entry and every entry of S^-1 with its own division, every
  //      a + p*q as a rounded product followed by a rounded sum (no std::fma, no shared reciprocal).  Mathematically identical to
  //      the default build below (readings A42 / A43 only regroup roundings); tests/test_gpu_parity.py::test_parity_against_plain_order_oracle
  //      checks that the CUDA path also meets the north_star bars against THIS independently ordered reference.
  bool propagate_state(State& st, Real dx) const {
    const Real smax = (Real)T.s_max;
    Real y = st.p[0], zz = st.p[1], s = st.p[2], t = st.p[3], q = st.p[4];
    Real k = cB * q;
    Real kdx = k * dx;
    Real s1 = s + kdx;
    if (!(std::fabs(s) <= smax) || !(std::fabs(s1) <= smax)) return false;
    Real c = std::sqrt((Real)1 - s * s), c1 = std::sqrt((Real)1 - s1 * s1);
    Real cc = c + c1, ss = s + s1, tq = ss / cc;
    Real g = (Real)1 + tq * tq;
    Real L = dx * std::sqrt(g);
    Real h = ((Real)0.5 * k) * L, h2 = h * h;
    const Real hthr = sizeof(Real) == 4 ? (Real)0.25 : (Real)1e-3;
    Real S;
    if (std::fabs(h) < hthr) {   // asin(h)/h = 1 + h^2/6 + 3h^4/40 + 15h^6/336 + 105h^8/3456 + ...
      Real poly = (Real)(105.0 / 3456.0);
      poly = (Real)(15.0 / 336.0) + h2 * poly;
      poly = (Real)(3.0 / 40.0) + h2 * poly;
      poly = (Real)(1.0 / 6.0) + h2 * poly;
      poly = (Real)1 + h2 * poly;
      S = L * poly;
    } else S = ((Real)2 / k) * std::asin(h);
    Real dSdk;
    const Real kthr = sizeof(Real) == 4 ? (Real)1e-2 : (Real)1e-3;
    if (std::fabs(kdx) >= kthr) dSdk = (dx / c1 - S) / k;
    else { Real sm = (s + (Real)2 * s1) / (Real)3; Real cm2 = (Real)1 - sm * sm; Real cm = std::sqrt(cm2);
      dSdk = ((dx * dx) * sm) / ((Real)2 * (cm2 * cm)); }
    Real cc1 = c * c1;
    Real F[5][5]; for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) F[i][j] = i == j ? (Real)1 : (Real)0;
    F[0][2] = ((dx * g) * cc) / ((Real)2 * cc1);
    F[0][4] = (((dx * dx) * cB) * g) / ((Real)2 * c1);
    F[1][2] = ((t * dx) * tq) / cc1;
    F[1][3] = S;
    F[1][4] = (t * cB) * dSdk;
    F[2][4] = cB * dx;
    st.p[0] = y + dx * tq; st.p[1] = zz + t * S; st.p[2] = s1;
    Real Tm[5][5], Cn[5][5];
    for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) { Real a = 0; for (int m = 0; m < 5; m++) a = a + F[i][m] * st.C[m][j]; Tm[i][j] = a; }
    for (int i = 0; i < 5; i++) for (int j = 0; j <= i; j++) { Real a = 0; for (int m = 0; m < 5; m++) a = a + Tm[i][m] * F[j][m]; Cn[i][j] = a; }
    for (int i = 0; i < 5; i++) for (int j = 0; j <= i; j++) { st.C[i][j] = Cn[i][j]; st.C[j][i] = Cn[i][j]; }
    return true;
  }
  Real update_state(State& st, Real ym, Real zm) const {
    const Real ry = (Real)sigma_y * (Real)sigma_y, rz = (Real)sigma_z * (Real)sigma_z;
    Real s00 = st.C[0][0] + ry, s10 = st.C[1][0], s11 = st.C[1][1] + rz;
    Real det = s00 * s11 - s10 * s10;
    Real i00 = s11 / det, i11 = s00 / det, i10 = -s10 / det;
    Real r0 = ym - st.p[0], r1 = zm - st.p[1];
    Real K0[5], K1[5];
    for (int i = 0; i < 5; i++) { K0[i] = st.C[i][0] * i00 + st.C[i][1] * i10; K1[i] = st.C[i][0] * i10 + st.C[i][1] * i11; }
    Real Cn[5][5];
    for (int i = 0; i < 5; i++) for (int j = 0; j <= i; j++) Cn[i][j] = st.C[i][j] - (K0[i] * st.C[0][j] + K1[i] * st.C[1][j]);
    for (int i = 0; i < 5; i++) st.p[i] = st.p[i] + (K0[i] * r0 + K1[i] * r1);
    for (int i = 0; i < 5; i++) for (int j = 0; j <= i; j++) { st.C[i][j] = Cn[i][j]; st.C[j][i] = Cn[i][j]; }
    return r0 * (i00 * r0 + i10 * r1) + r1 * (i10 * r0 + i11 * r1);
  }
#else
  // propagate the state from its x to x+dx on the helix in uniform Bz; false = |sin(phi)| leaves [-s_max, s_max]
  bool propagate_state(State& st, Real dx) const {
    const Real smax = (Real)T.s_max;
    Real y = st.p[0], zz = st.p[1], s = st.p[2], t = st.p[3], q = st.p[4];
    Real k = cB * q;
    Real kdx = k * dx;
    Real s1 = s + kdx;
    if (!(std::fabs(s) <= smax) || !(std::fabs(s1) <= smax)) return false;
    // reading A43: every a + p*q of the transport and of the update below is ONE fused multiply-add, std::fma(p, q, a)
    Real c = std::sqrt(std::fma(-s, s, (Real)1)), c1 = std::sqrt(std::fma(-s1, s1, (Real)1));
    // reading A42: one reciprocal per distinct denominator (1/(c+c1), 1/(c c1), 1/c1 = c * 1/(c c1)), products rounded one by one
    Real cc = c + c1, ss = s + s1, icc = (Real)1 / cc, tq = ss * icc;
    Real g = std::fma(tq, tq, (Real)1);
    Real L = dx * std::sqrt(g);
    Real h = ((Real)0.5 * k) * L, h2 = h * h;
    const Real hthr = sizeof(Real) == 4 ? (Real)0.25 : (Real)1e-3;
    Real S;
    if (std::fabs(h) < hthr) {   // asin(h)/h = 1 + h^2/6 + 3h^4/40 + 15h^6/336 + 105h^8/3456 + ...
      Real poly = (Real)(105.0 / 3456.0);
      poly = std::fma(h2, poly, (Real)(15.0 / 336.0));
      poly = std::fma(h2, poly, (Real)(3.0 / 40.0));
      poly = std::fma(h2, poly, (Real)(1.0 / 6.0));
      poly = std::fma(h2, poly, (Real)1);
      S = L * poly;
    } else S = ((Real)2 / k) * std::asin(h);
    Real dSdk;
    const Real kthr = sizeof(Real) == 4 ? (Real)1e-2 : (Real)1e-3;
    Real cc1 = c * c1, icc1 = (Real)1 / cc1, ic1 = c * icc1;
    if (std::fabs(kdx) >= kthr) dSdk = std::fma(dx, ic1, -S) / k;
    else { Real sm = (s + (Real)2 * s1) * (Real)(1.0 / 3.0); Real cm2 = std::fma(-sm, sm, (Real)1); Real cm = std::sqrt(cm2);
      dSdk = ((dx * dx) * sm) / ((Real)2 * (cm2 * cm)); }
    Real F[5][5]; for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) F[i][j] = i == j ? (Real)1 : (Real)0;
    F[0][2] = ((dx * g) * cc) * ((Real)0.5 * icc1);
    F[0][4] = (((dx * dx) * cB) * g) * ((Real)0.5 * ic1);
    F[1][2] = ((t * dx) * tq) * icc1;
    F[1][3] = S;
    F[1][4] = (t * cB) * dSdk;
    F[2][4] = cB * dx;
    st.p[0] = std::fma(dx, tq, y); st.p[1] = std::fma(t, S, zz); st.p[2] = s1;
    Real Tm[5][5], Cn[5][5];
    for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) { Real a = 0; for (int m = 0; m < 5; m++) a = std::fma(F[i][m], st.C[m][j], a); Tm[i][j] = a; }
    for (int i = 0; i < 5; i++) for (int j = 0; j <= i; j++) { Real a = 0; for (int m = 0; m < 5; m++) a = std::fma(Tm[i][m], F[j][m], a); Cn[i][j] = a; }
    for (int i = 0; i < 5; i++) for (int j = 0; j <= i; j++) { st.C[i][j] = Cn[i][j]; st.C[j][i] = Cn[i][j]; }   // symmetrise: lower triangle mirrored
    return true;
  }

  // Kalman update with the joint 2-D measurement (ym, zm), R = diag(sigma_y^2, sigma_z^2); returns chi2 increment
  Real update_state(State& st, Real ym, Real zm) const {
    const Real ry = (Real)sigma_y * (Real)sigma_y, rz = (Real)sigma_z * (Real)sigma_z;
    Real s00 = st.C[0][0] + ry, s10 = st.C[1][0], s11 = st.C[1][1] + rz;
    Real det = std::fma(-s10, s10, s00 * s11);   // reading A43: fused multiply-adds, as in the transport
    Real idet = (Real)1 / det;   // reading A42: S^-1 through one reciprocal
    Real i00 = s11 * idet, i11 = s00 * idet, i10 = -s10 * idet;
    Real r0 = ym - st.p[0], r1 = zm - st.p[1];
    Real K0[5], K1[5];
    for (int i = 0; i < 5; i++) { K0[i] = std::fma(st.C[i][1], i10, st.C[i][0] * i00); K1[i] = std::fma(st.C[i][1], i11, st.C[i][0] * i10); }
    Real Cn[5][5];
    for (int i = 0; i < 5; i++) for (int j = 0; j <= i; j++) Cn[i][j] = std::fma(-K1[i], st.C[1][j], std::fma(-K0[i], st.C[0][j], st.C[i][j]));
    for (int i = 0; i < 5; i++) st.p[i] = std::fma(K1[i], r1, std::fma(K0[i], r0, st.p[i]));
    for (int i = 0; i < 5; i++) for (int j = 0; j <= i; j++) { st.C[i][j] = Cn[i][j]; st.C[j][i] = Cn[i][j]; }
    Real u0 = std::fma(i10, r1, i00 * r0), u1 = std::fma(i11, r1, i10 * r0);
    return std::fma(r1, u1, r0 * u0);
  }

#endif   // S5_PLAIN_ORDER

  void reset_cov(State& st) const { for (int i = 0; i < 5; i++) for (int j = 0; j < 5; j++) st.C[i][j] = i == j ? (Real)T.c0[i] : (Real)0; }

  // cluster pick-up on row r of a sector: nearest hit inside min(w_max, n_sigma*sqrt(C+sigma^2)); -1 = none
  int32_t pickup(int sec, int r, const State& st, Real zref, bool brute) const {
    int u = sec * R + r; int64_t o = off[u];
    const Real wmax = (Real)T.w_max, ns = (Real)T.n_sigma;
    Real wy = ns * std::sqrt(st.C[0][0] + (Real)sigma_y * (Real)sigma_y); if (!(wy <= wmax)) wy = wmax;
    Real wz = ns * std::sqrt(st.C[1][1] + (Real)sigma_z * (Real)sigma_z); if (!(wz <= wmax)) wz = wmax;
    Real y = st.p[0], zr = st.p[1];
    Real ylo = y - wy, yhi = y + wy, zlo = zr - wz, zhi = zr + wz;
    const Real margin = (Real)0.05;   // the bin range only has to be a superset of the z_rel window
    int32_t best = -1; Real bestd = 0; int32_t besti = 0;
    for_bins(u, ylo, yhi, (zlo + zref) - margin, (zhi + zref) + margin, brute, [&](int32_t p) {
      Real yc = ys[o + p], zc = zs[o + p] - zref;
      if (!(yc >= ylo && yc <= yhi && zc >= zlo && zc <= zhi)) return;
      Real dy = yc - y, dz = zc - zr; Real d = dy * dy + dz * dz; int32_t ip = perm[o + p];
      if (best < 0 || d < bestd || (d == bestd && ip < besti)) { best = p; bestd = d; besti = ip; } });
    return best;
  }

  // ---- S5: tracklet constructor, one hypothesis per start hit ----
  void s5_tracklets(bool brute) {
    int64_t M = (int64_t)start_unit.size();
    tl_n.assign(M, 0); tl_first.assign(M, -1); tl_last.assign(M, -1); tl_rowhit.assign(M * R, -1); tl_sector.assign(M, 0);
    tl_chi2.assign(M, 0); tl_x.assign(M, 0); tl_par.assign(M * 5, 0); tl_cov.assign(M * 15, 0); tl_zref.assign(M, 0);
    auto fit = [&](int64_t i) {
      int u0 = start_unit[i], sec = u0 / R, r0 = u0 % R; int32_t h0 = start_pos[i];
      int32_t* rowhit = &tl_rowhit[i * R];
      auto Y = [&](int r, int32_t p) { return ys[off[sec * R + r] + p]; };
      auto Z = [&](int r, int32_t p) { return zs[off[sec * R + r] + p]; };
      const Real zref = Z(r0, h0);
      State st;
      { // Phase A init: direction from the origin
        Real x = X[r0], y = Y(r0, h0); Real rr = std::sqrt(x * x + y * y);
        st.p[0] = y; st.p[1] = 0; st.p[2] = y / rr; st.p[3] = continuous ? (Real)0 : zref / rr; st.p[4] = 0; reset_cov(st);
      }
      update_state(st, Y(r0, h0), (Real)0); rowhit[r0] = h0;
      int r = r0; int32_t h = h0; bool ok = true;
      State saved = st; int r_out = r0;
      for (;;) {   // Phase A: follow the cleaned up-links, no gate
        int32_t up = clean_up[off[sec * R + r] + h]; if (up < 0) break;
        const int k = clean_up_k[off[sec * R + r] + h];     // 1; 2 = the link skips a row (S2', link_skip): one transport over both rows
        if (!propagate_state(st, X[r + k] - X[r])) { ok = false; break; }
        r += k; h = up; update_state(st, Y(r, h), Z(r, h) - zref); rowhit[r] = h; saved = st; r_out = r;
      }
      if (ok) {    // Phase B: extrapolate outward with pick-up
        int gap = 0;
        for (int rr = r + 1; rr < R; rr++) {
          if (!propagate_state(st, X[rr] - X[rr - 1])) break;
          if (std::fabs(st.p[0]) > yedge[rr] + (Real)T.edge_margin) break;
          int32_t p = pickup(sec, rr, st, zref, brute);
          if (p >= 0) { update_state(st, Y(rr, p), Z(rr, p) - zref); rowhit[rr] = p; gap = 0; saved = st; r_out = rr; }
          else { gap++; if (gap > T.max_gap) break; }
        }
      }
      // Phase C: inward refit from the outermost assigned hit, then extrapolate inward
      st = saved; reset_cov(st);
      Real chi2 = 0; int n = 0;
      chi2 = chi2 + update_state(st, Y(r_out, rowhit[r_out]), Z(r_out, rowhit[r_out]) - zref); n = 1;
      State snap = st; int r_snap = r_out; int first_assigned = r0; int gap = 0; int stop_row = -1;
      for (int rr = r_out - 1; rr >= 0; rr--) {
        if (!propagate_state(st, X[rr] - X[rr + 1])) { stop_row = rr; break; }
        if (rowhit[rr] >= 0) { chi2 = chi2 + update_state(st, Y(rr, rowhit[rr]), Z(rr, rowhit[rr]) - zref); n++; snap = st; r_snap = rr; continue; }
        if (std::fabs(st.p[0]) > yedge[rr] + (Real)T.edge_margin) { if (rr < first_assigned) break; else continue; }
        int32_t p = pickup(sec, rr, st, zref, brute);
        if (p >= 0) { chi2 = chi2 + update_state(st, Y(rr, p), Z(rr, p) - zref); n++; rowhit[rr] = p; snap = st; r_snap = rr;
          if (rr < first_assigned) { first_assigned = rr; gap = 0; } }
        else if (rr < first_assigned) { gap++; if (gap > T.max_gap) break; }
      }
      for (int rr = 0; rr <= stop_row; rr++) rowhit[rr] = -1;   // hits never reached by the refit are not part of the tracklet
      tl_sector[i] = sec; tl_n[i] = n; tl_chi2[i] = (double)chi2; tl_first[i] = r_snap; tl_last[i] = r_out; tl_x[i] = (double)X[r_snap]; tl_zref[i] = (double)zref;
      for (int k = 0; k < 5; k++) tl_par[i * 5 + k] = (double)snap.p[k];
      tl_par[i * 5 + 1] = (double)(snap.p[1] + zref);
      int c = 0; for (int a = 0; a < 5; a++) for (int b = 0; b <= a; b++) tl_cov[i * 15 + c++] = (double)snap.C[a][b];
    };
    const bool two = T.bridge_rows > 0 && T.bridge_rescue;
    for (int64_t i = 0; i < M; i++) { tl_sector[i] = start_unit[i] / R; if (!two || start_wave[i] == 1) fit(i); }
    // S4' with rescue (reading A39c): the first wave fits the start hits that are not bridged; a bridged start hit is fitted in the
    // second wave unless every cluster of its chain is used by a kept first-wave tracklet (then that tracklet covers its track)
    if (two) {
      std::vector<char> used(N, 0);
      for (int64_t i = 0; i < M; i++) if (start_wave[i] == 1 && tracklet_kept(i)) {
        const int sec = tl_sector[i];
        for (int r = tl_first[i]; r <= tl_last[i]; r++) { int32_t p = tl_rowhit[i * R + r]; if (p >= 0) used[off[sec * R + r] + p] = 1; }
      }
      for (int64_t i = 0; i < M; i++) if (start_wave[i] == 2) {
        int uu = start_unit[i]; int32_t p = start_pos[i]; bool all = true;
        for (;;) { if (!used[off[uu] + p]) { all = false; break; } int32_t nx = clean_up[off[uu] + p]; if (nx < 0) break; p = nx; uu++; }
        if (!all) fit(i);
      }
    }
  }

  bool tracklet_kept(int64_t i) const { return tl_n[i] >= T.min_hits && std::isfinite(tl_chi2[i]); }
  Real quality(int64_t i) const { return (Real)tl_chi2[i] / (Real)(2 * tl_n[i] - 5); }
  // true if tracklet a beats tracklet b for a shared cluster: more hits, then lower chi2/ndf, then lower index
  bool beats(int64_t a, int64_t b) const {
    if (tl_n[a] != tl_n[b]) return tl_n[a] > tl_n[b];
    Real qa = quality(a), qb = quality(b);
    if (qa != qb) return qa < qb;
    return a < b;
  }

  // ---- S6: selector -- winner takes the cluster; a track = a tracklet with >= min_hits owned clusters ----
  void s6_select() {
    int64_t M = (int64_t)tl_n.size();
    std::vector<int64_t> owner(N, -1);
    for (int64_t i = 0; i < M; i++) {
      if (!tracklet_kept(i)) continue;
      int sec = tl_sector[i];
      for (int r = 0; r < R; r++) { int32_t p = tl_rowhit[i * R + r]; if (p < 0) continue;
        int64_t g = off[sec * R + r] + p; if (owner[g] < 0 || beats(i, owner[g])) owner[g] = i; }
    }
    trk_sector.clear(); trk_ndf.clear(); trk_tracklet.clear(); trk_cl_row.clear(); trk_cl_index.clear(); trk_cl_begin.assign(1, 0);
    trk_x.clear(); trk_par.clear(); trk_cov.clear(); trk_chi2.clear();
    for (int64_t i = 0; i < M; i++) {
      if (!tracklet_kept(i)) continue;
      int sec = tl_sector[i]; int owned = 0;
      for (int r = 0; r < R; r++) { int32_t p = tl_rowhit[i * R + r]; if (p >= 0 && owner[off[sec * R + r] + p] == i) owned++; }
      if (owned < T.min_hits) continue;
      for (int r = 0; r < R; r++) { int32_t p = tl_rowhit[i * R + r]; if (p >= 0 && owner[off[sec * R + r] + p] == i) {
        trk_cl_row.push_back(r); trk_cl_index.push_back(perm[off[sec * R + r] + p]); } }
      trk_cl_begin.push_back((int64_t)trk_cl_row.size());
      trk_sector.push_back(sec); trk_ndf.push_back(2 * tl_n[i] - 5); trk_tracklet.push_back((int32_t)i);
      trk_x.push_back(tl_x[i]); trk_chi2.push_back(tl_chi2[i]);
      for (int k = 0; k < 5; k++) trk_par.push_back(tl_par[i * 5 + k]);
      for (int k = 0; k < 15; k++) trk_cov.push_back(tl_cov[i * 15 + k]);
    }
  }

  // ---- S7 (NEXT-1; "improve the z-estimation"): refit of the clusters a track OWNS after the
  //      selection, so that state, covariance and chi2/ndf describe the returned cluster list (reading A17 -> A37), and the
  //      collision time of a continuous-read-out track from its extrapolation to the beam line (reading A38).
  //      Pass 1 outward over the owned clusters (seed direction from the origin, C0), pass 2 inward with a fresh C0.
  void s7_refit() {
    int64_t NT = (int64_t)trk_sector.size();
    rf_n.assign(NT, 0); rf_ndf.assign(NT, 0); rf_x.assign(NT, 0); rf_par.assign(NT * 5, 0); rf_cov.assign(NT * 15, 0);
    rf_chi2.assign(NT, 0); rf_z0.assign(NT, 0); rf_t0.assign(NT, 0);
    for (int64_t i = 0; i < NT; i++) {
      const int sec = trk_sector[i]; const int64_t a = trk_cl_begin[i], m = trk_cl_begin[i + 1] - a;
      const int32_t T_ = trk_tracklet[i];
      auto row = [&](int64_t k) { return (int)trk_cl_row[a + k]; };
      auto pos = [&](int64_t k) { return off[sec * R + row(k)] + tl_rowhit[(int64_t)T_ * R + row(k)]; };
      const Real zref = zs[pos(0)];
      State st;
      { Real x = X[row(0)], y = ys[pos(0)]; Real rr = std::sqrt(x * x + y * y);
        st.p[0] = y; st.p[1] = 0; st.p[2] = y / rr; st.p[3] = continuous ? (Real)0 : zref / rr; st.p[4] = 0; reset_cov(st); }
      update_state(st, ys[pos(0)], (Real)0);
      int64_t last = 0;
      for (int64_t k = 1; k < m; k++) {                       // pass 1: outward
        if (!propagate_state(st, X[row(k)] - X[row(k - 1)])) break;
        update_state(st, ys[pos(k)], zs[pos(k)] - zref); last = k;
      }
      reset_cov(st);                                          // pass 2: inward from the outermost cluster reached
      Real chi2 = 0; int n = 0;
      chi2 = chi2 + update_state(st, ys[pos(last)], zs[pos(last)] - zref); n = 1;
      State snap = st; int64_t kin = last;
      for (int64_t k = last - 1; k >= 0; k--) {
        if (!propagate_state(st, X[row(k)] - X[row(k + 1)])) break;
        chi2 = chi2 + update_state(st, ys[pos(k)], zs[pos(k)] - zref); n++; snap = st; kin = k;
      }
      rf_n[i] = n; rf_ndf[i] = 2 * n - 5; rf_chi2[i] = (double)chi2; rf_x[i] = (double)X[row(kin)];
      for (int k = 0; k < 5; k++) rf_par[i * 5 + k] = (double)snap.p[k];
      const Real zabs = snap.p[1] + zref;
      rf_par[i * 5 + 1] = (double)zabs;
      int c = 0; for (int u = 0; u < 5; u++) for (int v = 0; v <= u; v++) rf_cov[i * 15 + c++] = (double)snap.C[u][v];
      // collision time (A38): a primary passes the beam line (x = y = 0); the chord from there to the state point has length
      // L, the arc over it S = L * asin(h)/h with h = k L / 2 (same series / switch as propagate_state); z at the beam line
      // z0 = z - (dz/ds) * S; a collision at time t0 shifts the scaled z rigidly by -vdrift * t0 (A6), hence t0 = -z0 / vdrift.
      { Real x = X[row(kin)], y = snap.p[0]; Real L = std::sqrt(x * x + y * y); Real k = cB * snap.p[4];
        Real h = ((Real)0.5 * k) * L, h2 = h * h;
        const Real hthr = sizeof(Real) == 4 ? (Real)0.25 : (Real)1e-3;
        Real S;
        if (std::fabs(h) < hthr) {
          Real poly = (Real)(105.0 / 3456.0);
          poly = (Real)(15.0 / 336.0) + h2 * poly;
          poly = (Real)(3.0 / 40.0) + h2 * poly;
          poly = (Real)(1.0 / 6.0) + h2 * poly;
          poly = (Real)1 + h2 * poly;
          S = L * poly;
        } else {
          if (h > (Real)1) h = (Real)1; if (h < (Real)-1) h = (Real)-1;
          S = ((Real)2 / k) * std::asin(h);
        }
        Real z0 = zabs - snap.p[3] * S;
        rf_z0[i] = (double)z0;
        rf_t0[i] = (double)(-z0 / (Real)vdrift); }
    }
  }

  // ---- S8 (NEXT-4; "The tracker forms tubes of 1.5 cm around each track, and marks
  //      unattached clusters as adjacent to the tube of the track with the highest transverse momentum it lies in"; reading A40).
  //      status 1 = attached (in the cluster list of a track), 2 = adjacent, 0 = neither; cl_track = that track, or -1.
  //      The tube follows the S6 state of the track, transported row by row (helix, parameters only) from the row of the state
  //      to the row of the track's last cluster; distance in the (y, z) plane of the pad row.
  void s8_adjacent(bool brute) {
    const int64_t NT = (int64_t)trk_sector.size();
    std::vector<int32_t> att(N, -1), adj_t(N, -1); std::vector<Real> adj_q(N, (Real)0);
    for (int64_t i = 0; i < NT; i++) {
      const int sec = trk_sector[i]; const int32_t T_ = trk_tracklet[i];
      for (int64_t k = trk_cl_begin[i]; k < trk_cl_begin[i + 1]; k++) { int r = trk_cl_row[k]; att[off[sec * R + r] + tl_rowhit[(int64_t)T_ * R + r]] = (int32_t)i; }
    }
    const Real tube = (Real)T.tube, tube2 = tube * tube, margin = (Real)0.05;
    for (int64_t i = 0; i < NT; i++) {
      const int sec = trk_sector[i]; const int32_t T_ = trk_tracklet[i];
      const int r_first = tl_first[T_], r_last = trk_cl_row[trk_cl_begin[i + 1] - 1];
      State st; for (int a = 0; a < 5; a++) for (int b = 0; b < 5; b++) st.C[a][b] = 0;
      const Real zref = (Real)trk_par[i * 5 + 1];
      st.p[0] = (Real)trk_par[i * 5 + 0]; st.p[1] = 0; st.p[2] = (Real)trk_par[i * 5 + 2]; st.p[3] = (Real)trk_par[i * 5 + 3]; st.p[4] = (Real)trk_par[i * 5 + 4];
      if (!std::isfinite(st.p[4])) continue;
      const Real aq = std::fabs(st.p[4]);
      for (int r = r_first; r <= r_last; r++) {
        if (r > r_first && !propagate_state(st, X[r] - X[r - 1])) break;
        const int u = sec * R + r; const int64_t o = off[u];
        const Real y = st.p[0], zr = st.p[1];
        const Real ylo = y - tube, yhi = y + tube, zlo = zr - tube, zhi = zr + tube;
        for_bins(u, ylo, yhi, (zlo + zref) - margin, (zhi + zref) + margin, brute, [&](int32_t p) {
          const Real dy = ys[o + p] - y, dz = (zs[o + p] - zref) - zr;
          const Real d2 = dy * dy + dz * dz;
          if (!(d2 <= tube2) || att[o + p] >= 0) return;
          if (adj_t[o + p] < 0 || aq < adj_q[o + p] || (aq == adj_q[o + p] && (int32_t)i < adj_t[o + p])) { adj_q[o + p] = aq; adj_t[o + p] = (int32_t)i; }
        });
      }
    }
    cl_status.assign(N, 0); cl_track.assign(N, -1);
    for (int u = 0; u < NS * R; u++)
      for (int64_t g = off[u]; g < off[u + 1]; g++) {
        const int64_t c = off[u] + perm[g];
        if (att[g] >= 0) { cl_status[c] = 1; cl_track[c] = att[g]; }
        else if (adj_t[g] >= 0) { cl_status[c] = 2; cl_track[c] = adj_t[g]; }
      }
  }

  // ---- S9 (NEXT-3; PAPER.md:49 says only "Locally, e. g. at the TPC sector boundaries, there are still some improvements to be done"; matching segments across the boundary is this build's reading A41 of that sentence, not a rule the paper prints;
  //      reading A41): a track that leaves its sector through the side edge continues in the neighbouring sector of
  //      the same side as a separate S6 track.  Outer state of A = its S6 state transported (parameters only) to the row of its
  //      last cluster.  A is a leaver iff |y_out| >= yedge - merge_edge; the neighbour is the next sector in phi for y_out > 0,
  //      the previous one for y_out < 0.  The outer state is rotated into the neighbour's frame (x' = x c + y s, y' = -x s + y c,
  //      sinphi' = sinphi c - cosphi s with (c, s) = (cos, sin)(+-dphi)) and transported to the x of every candidate B of that
  //      sector with |row_in(B) - row_out(A)| <= merge_rows; B matches iff |dy| <= merge_dy, |dz| <= merge_dz, |dsinphi| <=
  //      merge_ds, |d(dz/ds)| <= merge_dt.  score = sum of the squared normalised differences; A proposes its best B (score, then
  //      index), B accepts its best proposer: next[A] = B, prev[B] = A (-1 elsewhere).
  void s9_merge() {
    const int64_t NT = (int64_t)trk_sector.size();
    // sectors per closed ring in phi (18 for 20 degree sectors), one ring per side; 0 when the sectors do not close a ring
    int ring = (int)std::lround(2.0 * M_PI / dphi);
    if (ring < 2 || std::fabs(ring * dphi - 2.0 * M_PI) > 1e-3 || NS % ring != 0) ring = 0;
    mg_next.assign(NT, -1); mg_prev.assign(NT, -1); mg_leaver.assign(NT, 0); mg_outer.assign(NT * 4, 0);
    std::vector<int> r_in(NT), r_out(NT); std::vector<State> outer(NT);
    for (int64_t i = 0; i < NT; i++) {
      const int32_t T_ = trk_tracklet[i];
      r_in[i] = tl_first[T_]; r_out[i] = trk_cl_row[trk_cl_begin[i + 1] - 1];
      State st; for (int a = 0; a < 5; a++) for (int b = 0; b < 5; b++) st.C[a][b] = 0;
      for (int k = 0; k < 5; k++) st.p[k] = (Real)trk_par[i * 5 + k];
      bool ok = std::isfinite(st.p[4]);
      for (int r = r_in[i] + 1; ok && r <= r_out[i]; r++) ok = propagate_state(st, X[r] - X[r - 1]);
      outer[i] = st;
      if (!ok) continue;
      mg_outer[i * 4 + 0] = (double)X[r_out[i]]; mg_outer[i * 4 + 1] = (double)st.p[0]; mg_outer[i * 4 + 2] = (double)st.p[1]; mg_outer[i * 4 + 3] = (double)st.p[2];
      if (ring == 0) continue;
      const Real ya = std::fabs(st.p[0]);
      if (ya >= yedge[r_out[i]] - (Real)T.merge_edge) mg_leaver[i] = st.p[0] > 0 ? 1 : -1;
    }
    const Real cd = (Real)std::cos(dphi), sd = (Real)std::sin(dphi);
    const Real my = (Real)T.merge_dy, mz = (Real)T.merge_dz, ms = (Real)T.merge_ds, mt = (Real)T.merge_dt;
    std::vector<int32_t> bestB(NT, -1); std::vector<Real> bestS(NT, (Real)0);
    for (int64_t a = 0; a < NT; a++) {
      if (!mg_leaver[a]) continue;
      const int sec = trk_sector[a], side = sec / ring, k = sec % ring;
      const int nb = side * ring + (k + (mg_leaver[a] > 0 ? 1 : ring - 1)) % ring;
      const Real sgn = mg_leaver[a] > 0 ? (Real)1 : (Real)-1;
      const State& o = outer[a];
      const Real x = X[r_out[a]], y = o.p[0], s = o.p[2], c = std::sqrt((Real)1 - s * s);
      const Real ss = sgn * sd;                          // sin of the signed rotation angle
      State rot = o;
      const Real xr = x * cd + y * ss;
      rot.p[0] = y * cd - x * ss;
      rot.p[2] = s * cd - c * ss;
      for (int64_t b = 0; b < NT; b++) {
        if (trk_sector[b] != nb) continue;
        int dr = r_in[b] - r_out[a]; if (dr < 0) dr = -dr;
        if (dr > T.merge_rows) continue;
        State st = rot;
        if (!propagate_state(st, X[r_in[b]] - xr)) continue;
        const Real dy = (Real)trk_par[b * 5 + 0] - st.p[0], dz = (Real)trk_par[b * 5 + 1] - st.p[1];
        const Real ds = (Real)trk_par[b * 5 + 2] - st.p[2], dt = (Real)trk_par[b * 5 + 3] - st.p[3];
        if (!(std::fabs(dy) <= my && std::fabs(dz) <= mz && std::fabs(ds) <= ms && std::fabs(dt) <= mt)) continue;
        const Real ey = dy / my, ez = dz / mz, es = ds / ms, et = dt / mt;
        const Real score = ((ey * ey + ez * ez) + es * es) + et * et;
        if (bestB[a] < 0 || score < bestS[a]) { bestB[a] = (int32_t)b; bestS[a] = score; }
      }
    }
    std::vector<int32_t> bestA(NT, -1); std::vector<Real> bestAS(NT, (Real)0);
    for (int64_t a = 0; a < NT; a++) { const int32_t b = bestB[a]; if (b < 0) continue;
      if (bestA[b] < 0 || bestS[a] < bestAS[b]) { bestA[b] = (int32_t)a; bestAS[b] = bestS[a]; } }
    for (int64_t b = 0; b < NT; b++) if (bestA[b] >= 0) { mg_next[bestA[b]] = (int32_t)b; mg_prev[b] = bestA[b]; }
  }

  // ---- S10 (NEXT-3, second half, SURVEY.md section 8(f).3 "recognise returning legs / extra turns"; "looping tracks",
  //      PAPER.md:104 "secondary legs of looping tracks below 200 MeV/c"; reading A46).  In a uniform field every turn of a looping
  //      particle runs over the SAME circle in the pad plane and is displaced along z by one pitch = (2 pi / |k|) * dz/ds, so the
  //      later turns appear in the same sector as separate S6 tracks with the same (y, sin phi, dz/ds, q/pT) at the same x.
  //      For tracks A, B of one sector, both with |q/pT| >= loop_qmin (pT <= 200 MeV/c): B's state is transported (parameters only)
  //      to x_A; B follows A iff |dy| <= loop_dy, |d sin phi| <= loop_ds, |d dz/ds| <= loop_dt, |dq| <= loop_dq |q_A|, the pitch
  //      p = (2 pi / |cB q_A|) * (t_A + t_B)/2 has |p| >= loop_pmin, and the number of turns tau = (z_B - z_A) / p is within
  //      loop_frac of an integer n, 1 <= n <= loop_nmax.  B takes as predecessor the A with the smallest n, then the smallest score
  //      (dy/loop_dy)^2 + (ds/loop_ds)^2 + (dt/loop_dt)^2, then the lowest index.  root = first turn of the group, turn = turns
  //      after the root (0 for a track that follows nobody).
  void s10_loopers() {
    const int64_t NT = (int64_t)trk_sector.size();
    lp_prev.assign(NT, -1); lp_root.assign(NT, 0); lp_turn.assign(NT, 0);
    std::vector<int32_t> lp_n(NT, 0);
    const Real qmin = (Real)T.loop_qmin, wy = (Real)T.loop_dy, ws = (Real)T.loop_ds, wt = (Real)T.loop_dt, wq = (Real)T.loop_dq;
    const Real pmin = (Real)T.loop_pmin, frac = (Real)T.loop_frac, twopi = (Real)6.283185307179586;
    for (int64_t b = 0; b < NT; b++) {
      const Real qb = (Real)trk_par[b * 5 + 4];
      if (!(std::fabs(qb) >= qmin)) continue;
      bool have = false; int32_t best = -1, bestn = 0; Real bests = 0;
      for (int64_t a = 0; a < NT; a++) {
        if (a == b || trk_sector[a] != trk_sector[b]) continue;
        const Real qa = (Real)trk_par[a * 5 + 4];
        if (!(std::fabs(qa) >= qmin)) continue;
        State st; for (int u = 0; u < 5; u++) for (int v = 0; v < 5; v++) st.C[u][v] = 0;
        for (int k = 0; k < 5; k++) st.p[k] = (Real)trk_par[b * 5 + k];
        const Real dx = (Real)trk_x[a] - (Real)trk_x[b];
        if (dx != (Real)0 && !propagate_state(st, dx)) continue;
        const Real dy = st.p[0] - (Real)trk_par[a * 5 + 0], ds = st.p[2] - (Real)trk_par[a * 5 + 2];
        const Real dt = st.p[3] - (Real)trk_par[a * 5 + 3], dq = st.p[4] - qa;
        if (!(std::fabs(dy) <= wy && std::fabs(ds) <= ws && std::fabs(dt) <= wt && std::fabs(dq) <= wq * std::fabs(qa))) continue;
        const Real k = cB * qa;
        const Real tav = (Real)0.5 * ((Real)trk_par[a * 5 + 3] + st.p[3]);
        const Real pitch = (twopi / std::fabs(k)) * tav;
        if (!(std::fabs(pitch) >= pmin)) continue;
        const Real tau = (st.p[1] - (Real)trk_par[a * 5 + 1]) / pitch;
        const Real nr = std::nearbyint(tau);
        if (!(nr >= (Real)1 && std::fabs(tau - nr) <= frac && nr <= (Real)T.loop_nmax)) continue;
        const int32_t n = (int32_t)nr;
        const Real ey = dy / wy, es = ds / ws, et = dt / wt;
        const Real score = (ey * ey + es * es) + et * et;
        if (!have || n < bestn || (n == bestn && score < bests)) { have = true; best = (int32_t)a; bestn = n; bests = score; }
      }
      if (have) { lp_prev[b] = best; lp_n[b] = bestn; }
    }
    for (int64_t i = 0; i < NT; i++) {     // the predecessor lies n >= 1 turns earlier: following it ends at the first turn
      int32_t r = (int32_t)i, t = 0;
      for (int it = 0; it < 64 && lp_prev[r] >= 0; it++) { t += lp_n[r]; r = lp_prev[r]; }
      lp_root[i] = r; lp_turn[i] = t;
    }
  }

  int run(int upto, int brute) override { return run_range(0, upto, brute); }
  // stages from..upto (the earlier ones must have run, or been set by hand: set_links); test hook for hand-built cases
  int run_range(int from, int upto, int brute) override {
    make_tables();
    for (int st = from; st <= upto; st++) {
      switch (st) {
        case 0: s0_time_to_z(); break;
        case 1: s1_grid(); break;
        case 2: s2_neighbours(brute & 1); break;
        case 3: s3_clean(); break;
        case 4: s4_start_hits((brute & 1) != 0); break;
        case 5: s5_tracklets((brute & 2) != 0); break;
        case 6: s6_select(); break;
        case 7: s7_refit(); break;
        case 8: s8_adjacent((brute & 2) != 0); break;
        case 9: s9_merge(); break;
        case 10: s10_loopers(); break;
        default: break;
      }
    }
    return 0;
  }

  // test hooks: the S5 pick-up alone on a hand-given state (S1 must have run), and hand-set cleaned link tables (sorted positions)
  int pickup_hook(const double* par, const double* cov, int sector, int row, double zref, int brute) override {
    make_tables(); State st; to_state(st, par, cov); return pickup(sector, row, st, (Real)zref, brute != 0);
  }
  int set_links(const int32_t* up, const int32_t* dn) override {
    clean_up.assign(up, up + N); clean_dn.assign(dn, dn + N); link_up = clean_up; link_dn = clean_dn;
    clean_up_k.assign(N, 0); clean_dn_k.assign(N, 0);
    for (int64_t g = 0; g < N; g++) { clean_up_k[g] = clean_up[g] >= 0; clean_dn_k[g] = clean_dn[g] >= 0; }
    link_up_k = clean_up_k; link_dn_k = clean_dn_k; return 0;
  }

  // hand-built tracklets for S6 pins (requires S1 to have run so that perm/off exist)
  int set_tracklets(int64_t n, const int32_t* sector, const int32_t* nh, const double* chi2, const int32_t* rowhit) override {
    tl_n.assign(nh, nh + n); tl_sector.assign(sector, sector + n); tl_chi2.assign(chi2, chi2 + n);
    tl_rowhit.assign(rowhit, rowhit + n * R); tl_first.assign(n, 0); tl_last.assign(n, 0); tl_x.assign(n, 0);
    tl_par.assign(n * 5, 0); tl_cov.assign(n * 15, 0); tl_zref.assign(n, 0);
    s6_select(); return 0;
  }

  static void to_state(State& st, const double* par, const double* cov) {
    for (int i = 0; i < 5; i++) st.p[i] = (Real)par[i];
    int c = 0; for (int a = 0; a < 5; a++) for (int b = 0; b <= a; b++) { st.C[a][b] = (Real)cov[c]; st.C[b][a] = (Real)cov[c]; c++; }
  }
  static void from_state(const State& st, double* par, double* cov) {
    for (int i = 0; i < 5; i++) par[i] = (double)st.p[i];
    int c = 0; for (int a = 0; a < 5; a++) for (int b = 0; b <= a; b++) cov[c++] = (double)st.C[a][b];
  }
  int propagate(double* par, double* cov, double dx) override {
    make_tables(); State st; to_state(st, par, cov); bool ok = propagate_state(st, (Real)dx); from_state(st, par, cov); return ok ? 0 : 1; }
  int update(double* par, double* cov, double ym, double zm, double* chi2) override {
    make_tables(); State st; to_state(st, par, cov); *chi2 = (double)update_state(st, (Real)ym, (Real)zm); from_state(st, par, cov); return 0; }

  // kind: 0 int32, 1 int64, 2 double, 3 float
  template <class V> static void dcopy(const std::vector<V>& a, std::vector<double>& d) { d.assign(a.begin(), a.end()); }
  int get(const char* name, const void** p, int64_t* n, int* kind) override {
    std::string s(name);
#define RET(vec, k) { *p = (vec).data(); *n = (int64_t)(vec).size(); *kind = (k); return 0; }
    if (s == "z") { dcopy(z, z_d); RET(z_d, 2) }
    if (s == "ys") { dcopy(ys, ys_d); RET(ys_d, 2) }
    if (s == "zs") { dcopy(zs, zs_d); RET(zs_d, 2) }
    if (s == "perm") RET(perm, 0)
    if (s == "bin_off") RET(bin_off, 1)
    if (s == "bin_start") RET(bin_start, 0)
    if (s == "grid_ny") RET(g_ny, 0)
    if (s == "grid_nz") RET(g_nz, 0)
    if (s == "grid_ylo") RET(g_ylo_d, 2)
    if (s == "grid_zlo") RET(g_zlo_d, 2)
    if (s == "grid_invs") RET(g_invs_d, 2)
    if (s == "link_up") RET(link_up, 0)
    if (s == "link_dn") RET(link_dn, 0)
    if (s == "link_up_k") RET(link_up_k, 0)
    if (s == "link_dn_k") RET(link_dn_k, 0)
    if (s == "clean_up_k") RET(clean_up_k, 0)
    if (s == "clean_dn_k") RET(clean_dn_k, 0)
    if (s == "clean_up") RET(clean_up, 0)
    if (s == "clean_dn") RET(clean_dn, 0)
    if (s == "start_unit") RET(start_unit, 0)
    if (s == "start_pos") RET(start_pos, 0)
    if (s == "tl_n") RET(tl_n, 0)
    if (s == "tl_first") RET(tl_first, 0)
    if (s == "tl_last") RET(tl_last, 0)
    if (s == "tl_rowhit") RET(tl_rowhit, 0)
    if (s == "tl_sector") RET(tl_sector, 0)
    if (s == "tl_chi2") RET(tl_chi2, 2)
    if (s == "tl_x") RET(tl_x, 2)
    if (s == "tl_par") RET(tl_par, 2)
    if (s == "tl_cov") RET(tl_cov, 2)
    if (s == "tl_zref") RET(tl_zref, 2)
    if (s == "trk_sector") RET(trk_sector, 0)
    if (s == "trk_ndf") RET(trk_ndf, 0)
    if (s == "trk_tracklet") RET(trk_tracklet, 0)
    if (s == "trk_cl_begin") RET(trk_cl_begin, 1)
    if (s == "trk_cl_row") RET(trk_cl_row, 0)
    if (s == "trk_cl_index") RET(trk_cl_index, 0)
    if (s == "trk_x") RET(trk_x, 2)
    if (s == "trk_par") RET(trk_par, 2)
    if (s == "trk_cov") RET(trk_cov, 2)
    if (s == "trk_chi2") RET(trk_chi2, 2)
    if (s == "start_wave") RET(start_wave, 0)
    if (s == "lp_prev") RET(lp_prev, 0)
    if (s == "lp_root") RET(lp_root, 0)
    if (s == "lp_turn") RET(lp_turn, 0)
    if (s == "mg_next") RET(mg_next, 0)
    if (s == "mg_prev") RET(mg_prev, 0)
    if (s == "mg_leaver") RET(mg_leaver, 0)
    if (s == "mg_outer") RET(mg_outer, 2)
    if (s == "cl_status") RET(cl_status, 0)
    if (s == "cl_track") RET(cl_track, 0)
    if (s == "rf_n") RET(rf_n, 0)
    if (s == "rf_ndf") RET(rf_ndf, 0)
    if (s == "rf_x") RET(rf_x, 2)
    if (s == "rf_par") RET(rf_par, 2)
    if (s == "rf_cov") RET(rf_cov, 2)
    if (s == "rf_chi2") RET(rf_chi2, 2)
    if (s == "rf_z0") RET(rf_z0, 2)
    if (s == "rf_t0") RET(rf_t0, 2)
#undef RET
    return -1;
  }
};

}  // namespace

extern "C" {
void* orc_create(int use_double, int n_sectors, int n_rows, const float* row_x, double dphi, double z_max, double t_frame,
                 double sigma_y, double sigma_z, double bz, double vdrift) {
  if (use_double) return new Oracle<double>(n_sectors, n_rows, row_x, dphi, z_max, t_frame, sigma_y, sigma_z, bz, vdrift);
  return new Oracle<float>(n_sectors, n_rows, row_x, dphi, z_max, t_frame, sigma_y, sigma_z, bz, vdrift);
}
void orc_destroy(void* h) { delete (OracleBase*)h; }
int orc_set_param(void* h, const char* name, double v) {
  Tunables& T = ((OracleBase*)h)->T; std::string s(name);
  if (s == "wy") T.wy = v; else if (s == "wz") T.wz = v; else if (s == "dzdx_max") T.dzdx_max = v; else if (s == "wz0") T.wz0 = v;
  else if (s == "cut2") T.cut2 = v; else if (s == "min_seed") T.min_seed = (int)v; else if (s == "s_max") T.s_max = v;
  else if (s == "n_sigma") T.n_sigma = v; else if (s == "w_max") T.w_max = v; else if (s == "max_gap") T.max_gap = (int)v;
  else if (s == "edge_margin") T.edge_margin = v; else if (s == "min_hits") T.min_hits = (int)v;
  else if (s == "c0_y") T.c0[0] = v; else if (s == "c0_z") T.c0[1] = v; else if (s == "c0_sinphi") T.c0[2] = v;
  else if (s == "c0_dzds") T.c0[3] = v; else if (s == "c0_qpt") T.c0[4] = v;
  else if (s == "grid_scale") T.grid_scale = v;
  else if (s == "bridge_rows") T.bridge_rows = (int)v; else if (s == "bridge_wy") T.bridge_wy = v; else if (s == "bridge_wz") T.bridge_wz = v; else if (s == "bridge_min") T.bridge_min = (int)v; else if (s == "bridge_rescue") T.bridge_rescue = (int)v; else if (s == "tube") T.tube = v; else if (s == "link_skip") T.link_skip = (int)v; else if (s == "skip_cut2") T.skip_cut2 = v;
  else if (s == "merge_edge") T.merge_edge = v; else if (s == "merge_rows") T.merge_rows = (int)v; else if (s == "merge_dy") T.merge_dy = v;
  else if (s == "merge_dz") T.merge_dz = v; else if (s == "merge_ds") T.merge_ds = v; else if (s == "merge_dt") T.merge_dt = v;
  else if (s == "loop_qmin") T.loop_qmin = v; else if (s == "loop_dy") T.loop_dy = v; else if (s == "loop_ds") T.loop_ds = v; else if (s == "loop_dt") T.loop_dt = v;
  else if (s == "loop_dq") T.loop_dq = v; else if (s == "loop_pmin") T.loop_pmin = v; else if (s == "loop_frac") T.loop_frac = v; else if (s == "loop_nmax") T.loop_nmax = (int)v;
  else return -1;
  return 0;
}
int orc_load(void* h, const int64_t* unit_off, const float* y, const float* t) { return ((OracleBase*)h)->load(unit_off, y, t); }
int orc_run(void* h, int upto, int brute) { return ((OracleBase*)h)->run(upto, brute); }
int orc_get(void* h, const char* name, const void** p, int64_t* n, int* kind) { return ((OracleBase*)h)->get(name, p, n, kind); }
int orc_propagate(void* h, double* par, double* cov, double dx) { return ((OracleBase*)h)->propagate(par, cov, dx); }
int orc_update(void* h, double* par, double* cov, double ym, double zm, double* chi2) { return ((OracleBase*)h)->update(par, cov, ym, zm, chi2); }
int orc_pickup(void* h, const double* par, const double* cov, int sector, int row, double zref, int brute) {
  return ((OracleBase*)h)->pickup_hook(par, cov, sector, row, zref, brute); }
int orc_set_links(void* h, const int32_t* up, const int32_t* dn) { return ((OracleBase*)h)->set_links(up, dn); }
int orc_run_range(void* h, int from, int upto, int brute) { return ((OracleBase*)h)->run_range(from, upto, brute); }
int orc_plain_order(void) {
#ifdef S5_PLAIN_ORDER
  return 1;
#else
  return 0;
#endif
}
int orc_set_tracklets(void* h, int64_t n, const int32_t* sector, const int32_t* nh, const double* chi2, const int32_t* rowhit) {
  return ((OracleBase*)h)->set_tracklets(n, sector, nh, chi2, rowhit); }
}
