// gray_math.cuh — per-photon arithmetic of the integrator: Kerr geodesic right-hand side, RK4
// step, step rules, theta remap.  Templated on the scalar type (float / double builds).
//
// The equations are the second-order geodesic equations of the Kerr metric in Boyer-Lindquist
// coordinates (paper P:23; the 20 non-zero Christoffel symbols are listed in SURVEY.md
// App. A.3).  They are not evaluated symbol by symbol.  With
//     Sigma = r^2 + a^2 cos^2(th),  Delta = (r - r_+)(r - r_-),  P = r^2 - a^2 cos^2(th),
//     rho = r^2 + a^2,  s = sin(th),  c = cos(th),
//     u = k^t - a s^2 k^phi,        w = a k^t - rho k^phi
// the contractions -Gamma^mu_ab k^a k^b collapse to (DESIGN.md "Kernel arithmetic" derives them):
//   dk^t  /dl = -2/Sigma^2 [ (k^r/Delta) (rho P u - 2 a s^2 r^2 Sigma k^phi) - 2 a^2 r s c k^th u ]
//   dk^phi/dl = -2/Sigma^2 [ (k^r/Delta) (a P u + r Sigma (Sigma - 2r) k^phi)
//                            + (c/s) k^th (Sigma^2 k^phi - 2 a r u) ]
//   dk^r  /dl = (r - 1) (k^r)^2/Delta
//               - 1/Sigma [ Delta (P u^2/Sigma^2 - r (s^2 (k^phi)^2 + (k^th)^2)) + r (k^r)^2
//                           - 2 a^2 s c k^r k^th ]
//   dk^th /dl = 1/Sigma [ s c (2 r w^2/Sigma^2 + Delta (k^phi)^2 + a^2 ((k^th)^2 - (k^r)^2/Delta))
//                         - 2 r k^r k^th ]
// One sincos and three reciprocals (1/Sigma, 1/Delta, 1/s) per evaluation.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#if defined(__CUDACC__)
#define GRAY_DEV __device__ __forceinline__
#else
#define GRAY_DEV inline
#endif

namespace gray {

template <typename T>
struct KerrConst {
  T a, a2;        // spin and its square
  T rp, rm;       // r_+ = 1 + sqrt(1 - a^2) (the horizon r_bh) and r_- = 1 - sqrt(1 - a^2)
  T h;            // step parameter (paper's Delta)
  T r_cap, r_esc; // termination radii
};

// ---- scalar helpers -------------------------------------------------------------------------
GRAY_DEV float rcp(float x) {
#if defined(__CUDA_ARCH__)
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));   // MUFU.RCP, ~1 ulp
  float e = fmaf(-x, y, 1.0f);                             // one Newton step -> < 1 ulp
  return fmaf(y, e, y);
#else
  return 1.0f / x;
#endif
}
GRAY_DEV double rcp(double x) { return 1.0 / x; }

GRAY_DEV void sincos_t(float x, float* s, float* c) { sincosf(x, s, c); }
GRAY_DEV void sincos_t(double x, double* s, double* c) { sincos(x, s, c); }
GRAY_DEV float abs_t(float x) { return fabsf(x); }
GRAY_DEV double abs_t(double x) { return fabs(x); }
GRAY_DEV float min_t(float x, float y) { return fminf(x, y); }
GRAY_DEV double min_t(double x, double y) { return fmin(x, y); }

// ---- right-hand side: accelerations dk^mu/dlambda at (r, th) for momentum (kt, kr, kh, kp) ------
template <typename T>
GRAY_DEV void geodesic_accel(const KerrConst<T>& K, T r, T th, T kt, T kr, T kh, T kp,
                             T& at, T& ar, T& ah, T& ap) {
  T s, c;
  sincos_t(th, &s, &c);
  const T r2 = r * r, c2 = c * c, s2 = s * s, sc = s * c;
  const T a2c2 = K.a2 * c2;
  const T Sg = r2 + a2c2;                       // Sigma
  const T P = r2 - a2c2;
  const T rho = r2 + K.a2;
  const T Dl = (r - K.rp) * (r - K.rm);         // Delta, product form: no cancellation at the horizon
  const T iS = rcp(Sg), iD = rcp(Dl), is = rcp(s);
  const T cot = c * is;
  const T iS2 = iS * iS;
  const T as2 = K.a * s2;
  const T u = kt - as2 * kp;
  const T w = K.a * kt - rho * kp;
  const T krD = kr * iD;                        // k^r / Delta
  const T rSg = r * Sg;
  const T two = T(2);

  const T e1 = rho * P * u - two * as2 * r * rSg * kp;
  at = -two * iS2 * (krD * e1 - two * K.a2 * r * sc * kh * u);

  const T e2 = K.a * P * u + rSg * (Sg - two * r) * kp;
  const T e3 = Sg * Sg * kp - two * K.a * r * u;
  ap = -two * iS2 * (krD * e2 + cot * kh * e3);

  const T kh2 = kh * kh;
  ar = (r - T(1)) * krD * kr -
       iS * (Dl * (P * iS2 * u * u - r * (s2 * kp * kp + kh2)) + r * kr * kr - two * K.a2 * sc * kr * kh);

  ah = iS * (sc * (two * r * iS2 * w * w + Dl * kp * kp + K.a2 * (kh2 - krD * kr)) - two * r * kr * kh);
}

// ---- step size (gray.h gray_step_rule; paper eq. (2)) -----------------------------------------
template <typename T, int RULE>
GRAY_DEV T step_size(const KerrConst<T>& K, const T y[8]) {
  if (RULE == 0) return -K.h * y[1];
  const T akr = abs_t(y[5]);
  const T d1 = K.h / (akr / y[1] + abs_t(y[6]) + abs_t(y[7]));
  const T d2 = (y[1] - K.rp) / (T(2) * akr);
  return -(d1 < d2 ? d1 : d2);
}

// ---- one classical RK4 step of y = (t, r, th, phi, k^t, k^r, k^th, k^phi) -------------------
template <typename T>
GRAY_DEV void rk4_step(const KerrConst<T>& K, T y[8], T dl) {
  T acc[8], w[8], f[4];
  const T hdl = T(0.5) * dl;
  // stage 1
  geodesic_accel(K, y[1], y[2], y[4], y[5], y[6], y[7], f[0], f[1], f[2], f[3]);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    acc[i] = y[4 + i];
    acc[4 + i] = f[i];
    w[i] = y[i] + hdl * y[4 + i];
    w[4 + i] = y[4 + i] + hdl * f[i];
  }
  // stage 2
  geodesic_accel(K, w[1], w[2], w[4], w[5], w[6], w[7], f[0], f[1], f[2], f[3]);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    acc[i] += T(2) * w[4 + i];
    acc[4 + i] += T(2) * f[i];
    const T kx = w[4 + i];
    w[i] = y[i] + hdl * kx;
    w[4 + i] = y[4 + i] + hdl * f[i];
  }
  // stage 3
  geodesic_accel(K, w[1], w[2], w[4], w[5], w[6], w[7], f[0], f[1], f[2], f[3]);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    acc[i] += T(2) * w[4 + i];
    acc[4 + i] += T(2) * f[i];
    const T kx = w[4 + i];
    w[i] = y[i] + dl * kx;
    w[4 + i] = y[4 + i] + dl * f[i];
  }
  // stage 4
  geodesic_accel(K, w[1], w[2], w[4], w[5], w[6], w[7], f[0], f[1], f[2], f[3]);
  const T dl6 = dl * T(1.0 / 6.0);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    y[i] += dl6 * (acc[i] + w[4 + i]);
    y[4 + i] += dl6 * (acc[4 + i] + f[i]);
  }
}

// ---- theta remap, paper eq. (3), P:87 ---------------------------------------------------------------
template <typename T>
GRAY_DEV void remap_theta(T y[8]) {
  const T pi = T(3.14159265358979323846);
  if (y[2] > pi) {
    y[2] = T(2) * pi - y[2];
    y[3] += pi;
    y[6] = -y[6];
  } else if (y[2] < T(0)) {
    y[2] = -y[2];
    y[3] -= pi;
    y[6] = -y[6];
  }
}

// ---- status of a state after a full step: BAD(3) / CAPTURED(1) / ESCAPED(2) / LIVE(0), in that order
template <typename T>
GRAY_DEV int state_status(const KerrConst<T>& K, const T y[8]) {
  T z = T(0);
#pragma unroll
  for (int i = 0; i < 8; ++i) z += T(0) * y[i];     // inf * 0 = NaN, NaN * 0 = NaN, finite * 0 = 0
  if (!(z == T(0))) return 3;
  if (y[1] < K.r_cap) return 1;
  if (y[1] > K.r_esc) return 2;
  return 0;
}

}  // namespace gray
