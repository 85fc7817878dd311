// kalman.cuh -- fp32 track state, helix transport and Kalman update shared by K5 (tracklet constructor) and K7 (refit).
// Definition: DESIGN.md section 4, S5.  Written term by term in the documented order; the library is compiled
// with -fmad=false, so a product is rounded before it is added unless the definition asks for a fused multiply-add (reading A43),
// which is then written as fma1(p, q, a) = __fmaf_rn.
#pragma once
#include "tpc_internal.cuh"

namespace tpc {

// explicit fused multiply-add (round once); the only place the library fuses a product into a sum
__device__ __forceinline__ float fma1(const float p, const float q, const float a) { return __fmaf_rn(p, q, a); }

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
  // reading A43: every a + p*q below is ONE fused multiply-add, written out as fma1(p, q, a) (the library is compiled with
  // -fmad=false, so nothing else is contracted)
  const float c = sqrtf(fma1(-s, s, 1.0f)), c1 = sqrtf(fma1(-s1, s1, 1.0f));
  // reading A42: one reciprocal per distinct denominator
  const float cc = c + c1, ss = s + s1, icc = 1.0f / cc, tq = ss * icc;
  const float g = fma1(tq, tq, 1.0f);
  const float L = dx * sqrtf(g);
  const float h = (0.5f * k) * L, h2 = h * h;
  float S;
  if (fabsf(h) < 0.25f) {   // asin(h)/h = 1 + h^2/6 + 3h^4/40 + 15h^6/336 + 105h^8/3456
    float poly = (float)(105.0 / 3456.0);
    poly = fma1(h2, poly, (float)(15.0 / 336.0));
    poly = fma1(h2, poly, (float)(3.0 / 40.0));
    poly = fma1(h2, poly, (float)(1.0 / 6.0));
    poly = fma1(h2, poly, 1.0f);
    S = L * poly;
  } else {
    S = (2.0f / k) * asinf(h);
  }
  const float cc1 = c * c1, icc1 = 1.0f / cc1, ic1 = c * icc1;
  float dSdk;
  if (fabsf(kdx) >= 1e-2f) {
    dSdk = fma1(dx, ic1, -S) / k;
  } else {
    const float sm = (s + 2.0f * s1) * (float)(1.0 / 3.0);
    const float cm2 = fma1(-sm, sm, 1.0f);
    const float cm = sqrtf(cm2);
    dSdk = ((dx * dx) * sm) / (2.0f * (cm2 * cm));
  }
  const float f02 = ((dx * g) * cc) * (0.5f * icc1);
  const float f04 = (((dx * dx) * cB) * g) * (0.5f * ic1);
  const float f12 = ((t * dx) * tq) * icc1;
  const float f13 = S;
  const float f14 = (t * cB) * dSdk;
  const float f24 = cB * dx;
  st.y = fma1(dx, tq, st.y);
  st.z = fma1(t, S, st.z);
  st.s = s1;
  // T = F C   (row i of T = sum_m F[i][m] C[m][:], accumulated by fma in the order m = 0..4; zero terms add exactly nothing)
  const float t00 = fma1(f04, st.c40, fma1(f02, st.c20, st.c00));
  const float t02 = fma1(f04, st.c42, fma1(f02, st.c22, st.c20));
  const float t04 = fma1(f04, st.c44, fma1(f02, st.c42, st.c40));
  const float t10 = fma1(f14, st.c40, fma1(f13, st.c30, fma1(f12, st.c20, st.c10)));
  const float t11 = fma1(f14, st.c41, fma1(f13, st.c31, fma1(f12, st.c21, st.c11)));
  const float t12 = fma1(f14, st.c42, fma1(f13, st.c32, fma1(f12, st.c22, st.c21)));
  const float t13 = fma1(f14, st.c43, fma1(f13, st.c33, fma1(f12, st.c32, st.c31)));
  const float t14 = fma1(f14, st.c44, fma1(f13, st.c43, fma1(f12, st.c42, st.c41)));
  const float t20 = fma1(f24, st.c40, st.c20);
  const float t21 = fma1(f24, st.c41, st.c21);
  const float t22 = fma1(f24, st.c42, st.c22);
  const float t23 = fma1(f24, st.c43, st.c32);
  const float t24 = fma1(f24, st.c44, st.c42);
  const float t30 = st.c30, t31 = st.c31, t32 = st.c32, t33 = st.c33, t34 = st.c43;
  const float t40 = st.c40, t41 = st.c41, t42 = st.c42, t43 = st.c43, t44 = st.c44;
  // C' = T F^T, lower triangle: C'[i][j] = sum_m T[i][m] F[j][m], accumulated by fma in the order m = 0..4
  st.c00 = fma1(t04, f04, fma1(t02, f02, t00));
  st.c10 = fma1(t14, f04, fma1(t12, f02, t10));
  st.c11 = fma1(t14, f14, fma1(t13, f13, fma1(t12, f12, t11)));
  st.c20 = fma1(t24, f04, fma1(t22, f02, t20));
  st.c21 = fma1(t24, f14, fma1(t23, f13, fma1(t22, f12, t21)));
  st.c22 = fma1(t24, f24, t22);
  st.c30 = fma1(t34, f04, fma1(t32, f02, t30));
  st.c31 = fma1(t34, f14, fma1(t33, f13, fma1(t32, f12, t31)));
  st.c32 = fma1(t34, f24, t32);
  st.c33 = t33;
  st.c40 = fma1(t44, f04, fma1(t42, f02, t40));
  st.c41 = fma1(t44, f14, fma1(t43, f13, fma1(t42, f12, t41)));
  st.c42 = fma1(t44, f24, t42);
  st.c43 = t43;
  st.c44 = t44;
  return true;
}

// Kalman update with the joint 2-D measurement (ym, zm), R = diag(sigma_y^2, sigma_z^2); returns the chi2 increment.
// Reading A43: fused multiply-adds in the order written.
__device__ __forceinline__ float update(State& st, const float ym, const float zm, const Params& P) {
  const float s00 = st.c00 + P.ry, s10 = st.c10, s11 = st.c11 + P.rz;
  const float det = fma1(-s10, s10, s00 * s11);
  const float idet = 1.0f / det;
  const float i00 = s11 * idet, i11 = s00 * idet, i10 = -s10 * idet;
  const float r0 = ym - st.y, r1 = zm - st.z;
  // K = C[:,0:2] S^-1
  const float k00 = fma1(st.c10, i10, st.c00 * i00), k01 = fma1(st.c10, i11, st.c00 * i10);
  const float k10 = fma1(st.c11, i10, st.c10 * i00), k11 = fma1(st.c11, i11, st.c10 * i10);
  const float k20 = fma1(st.c21, i10, st.c20 * i00), k21 = fma1(st.c21, i11, st.c20 * i10);
  const float k30 = fma1(st.c31, i10, st.c30 * i00), k31 = fma1(st.c31, i11, st.c30 * i10);
  const float k40 = fma1(st.c41, i10, st.c40 * i00), k41 = fma1(st.c41, i11, st.c40 * i10);
  // C' = C - K C[0:2,:], lower triangle: C'[i][j] = fma1(-K1[i], C[1][j], fma1(-K0[i], C[0][j], C[i][j])); C[0][j] = c_j0, C[1][j] = c_j1
  const float o00 = st.c00, o10 = st.c10, o11 = st.c11, o20 = st.c20, o21 = st.c21, o30 = st.c30, o31 = st.c31, o40 = st.c40, o41 = st.c41;
  st.c00 = fma1(-k01, o10, fma1(-k00, o00, o00));
  st.c10 = fma1(-k11, o10, fma1(-k10, o00, o10));
  st.c11 = fma1(-k11, o11, fma1(-k10, o10, o11));
  st.c20 = fma1(-k21, o10, fma1(-k20, o00, o20));
  st.c21 = fma1(-k21, o11, fma1(-k20, o10, o21));
  st.c22 = fma1(-k21, o21, fma1(-k20, o20, st.c22));
  st.c30 = fma1(-k31, o10, fma1(-k30, o00, o30));
  st.c31 = fma1(-k31, o11, fma1(-k30, o10, o31));
  st.c32 = fma1(-k31, o21, fma1(-k30, o20, st.c32));
  st.c33 = fma1(-k31, o31, fma1(-k30, o30, st.c33));
  st.c40 = fma1(-k41, o10, fma1(-k40, o00, o40));
  st.c41 = fma1(-k41, o11, fma1(-k40, o10, o41));
  st.c42 = fma1(-k41, o21, fma1(-k40, o20, st.c42));
  st.c43 = fma1(-k41, o31, fma1(-k40, o30, st.c43));
  st.c44 = fma1(-k41, o41, fma1(-k40, o40, st.c44));
  st.y = fma1(k01, r1, fma1(k00, r0, st.y));
  st.z = fma1(k11, r1, fma1(k10, r0, st.z));
  st.s = fma1(k21, r1, fma1(k20, r0, st.s));
  st.t = fma1(k31, r1, fma1(k30, r0, st.t));
  st.q = fma1(k41, r1, fma1(k40, r0, st.q));
  const float u0 = fma1(i10, r1, i00 * r0), u1 = fma1(i11, r1, i10 * r0);
  return fma1(r1, u1, r0 * u0);
}

// arc length over a chord of length L on a circle of curvature k: L * asin(h)/h, h = k L / 2 (series below 0.25, reading A32)
__device__ __forceinline__ float arc_of_chord(const float L, const float k) {
  float h = (0.5f * k) * L;
  const float h2 = h * h;
  if (fabsf(h) < 0.25f) {
    float poly = (float)(105.0 / 3456.0);
    poly = (float)(15.0 / 336.0) + h2 * poly;
    poly = (float)(3.0 / 40.0) + h2 * poly;
    poly = (float)(1.0 / 6.0) + h2 * poly;
    poly = 1.0f + h2 * poly;
    return L * poly;
  }
  if (h > 1.0f) h = 1.0f;
  if (h < -1.0f) h = -1.0f;
  return (2.0f / k) * asinf(h);
}

}  // namespace tpc
