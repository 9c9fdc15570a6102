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
//
// Conditioning: inside the kernel the radial variable is the
// height above the horizon  d = r - r_+  (so Delta = d (d + r_+ - r_-) keeps full relative
// precision where the equations are singular), and the polar angle is kept in [0, pi/2] by the
// reflection symmetry theta -> pi - theta, k^theta -> -k^theta of the Kerr metric (so the
// absolute rounding of theta shrinks towards either pole, where the equations are singular
// too).  Both are exact changes of variable of the same ODE; they are undone on store.
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
  T rp;           // r_+ = 1 + sqrt(1 - a^2): the horizon r_bh of P:75
  T rpm;          // r_+ - r_- = 2 sqrt(1 - a^2)
  T h;            // step parameter (paper's Delta)
  T r_cap, r_esc; // termination radii
};

// Photon state as the kernel carries it: y = (t, d, th, phi, k^t, k^r, k^th, k^phi) with d = r - r_+ and
// th in [0, pi/2]; `mirrored` says that the true polar angle is pi - th (and the true k^theta is -k^th).
template <typename T>
struct Photon {
  T y[8];
  int mirrored;
};

// ---- scalar helpers -------------------------------------------------------------------------
// Reciprocal.  float: MUFU.RCP (relative error <= 1 ulp, B300_MICROARCH "XU"); its three uses per
// right-hand side sit among ~80 roundings of half an ulp each, so it is not refined.
GRAY_DEV float rcp(float x) {
#if defined(__CUDA_ARCH__)
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
#else
  return 1.0f / x;
#endif
}
GRAY_DEV double rcp(double x) { return 1.0 / x; }

// sin and cos of x for |x| < ~100 (the kernel's theta stays within a step of [0, pi/2]).
// float: quadrant j = rint(x 2/pi) by the add-magic-constant trick, r = x - j pi/2 with pi/2 split in
// two floats (exact enough for small |j|), then near-minimax polynomials on [-pi/4, pi/4] fitted for
// this kernel (max error 0.86 ulp for both, checked against fp64 over 2e6 points); no slow path, no
// int<->float conversions (those run on the quarter-rate XU pipe).
GRAY_DEV void sincos_t(float x, float* s, float* c) {
#if defined(__CUDA_ARCH__)
  const float q = fmaf(x, 0.636619772f, 12582912.0f);      // 1.5 * 2^23: the low mantissa bits of q hold j
  const int j = __float_as_int(q);
  const float jf = q - 12582912.0f;
  float r = fmaf(jf, -1.57079637050628662109375f, x);      // float(pi/2)
  r = fmaf(jf, 4.371139000186241e-08f, r);                 // pi/2 - float(pi/2)
  const float u = r * r;
  const float sp = fmaf(fmaf(-1.957778732e-04f, u, 8.332700469e-03f), u, -1.666666418e-01f);
  const float sn = fmaf(r * u, sp, r);
  const float cp = fmaf(fmaf(fmaf(2.445036807e-05f, u, -1.388748409e-03f), u, 4.166664928e-02f), u, -0.5f);
  const float cs = fmaf(u, cp, 1.0f);
  const bool swap = (j & 1) != 0;
  const float ss = swap ? cs : sn, cc = swap ? sn : cs;
  *s = __int_as_float(__float_as_int(ss) ^ ((j & 2) << 30));          // quadrants 2, 3: sin < 0
  *c = __int_as_float(__float_as_int(cc) ^ (((j + 1) & 2) << 30));    // quadrants 1, 2: cos < 0
#else
  *s = sinf(x); *c = cosf(x);
#endif
}
GRAY_DEV void sincos_t(double x, double* s, double* c) { sincos(x, s, c); }
GRAY_DEV float abs_t(float x) { return fabsf(x); }
GRAY_DEV double abs_t(double x) { return fabs(x); }
GRAY_DEV float min_t(float x, float y) { return fminf(x, y); }
GRAY_DEV double min_t(double x, double y) { return fmin(x, y); }

// ---- right-hand side: accelerations dk^mu/dlambda at (d = r - r_+, th) for momentum (kt, kr, kh, kp) ----
template <typename T>
GRAY_DEV void geodesic_accel(const KerrConst<T>& K, T d, T th, T kt, T kr, T kh, T kp,
                             T& at, T& ar, T& ah, T& ap) {
  T s, c;
  sincos_t(th, &s, &c);
  const T r = d + K.rp;
  const T r2 = r * r, c2 = c * c, s2 = s * s, sc = s * c;
  const T a2c2 = K.a2 * c2;
  const T Sg = r2 + a2c2;                       // Sigma
  const T P = r2 - a2c2;
  const T rho = r2 + K.a2;
  const T Dl = d * (d + K.rpm);                 // Delta = (r - r_+)(r - r_-): no cancellation at the horizon
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
// y[1] = d = r - r_+.  float: the two quotients of eq. (2) are formed with MUFU.RCP (1 ulp): the step
// size is a free parameter of the scheme, an ulp of it is far below the truncation error it controls.
template <typename T, int RULE>
GRAY_DEV T step_size(const KerrConst<T>& K, const T y[8]) {
  const T r = y[1] + K.rp;
  if (RULE == 0) return -K.h * r;
  const T akr = abs_t(y[5]);
  if (sizeof(T) == 4) {
    const T d1 = K.h * r * rcp(akr + r * (abs_t(y[6]) + abs_t(y[7])));
    const T d2 = T(0.5) * y[1] * rcp(akr);
    return -min_t(d1, d2);
  }
  const T d1 = K.h / (akr / r + abs_t(y[6]) + abs_t(y[7]));
  const T d2 = y[1] / (T(2) * akr);
  return -(d1 < d2 ? d1 : d2);
}

// ---- one classical RK4 step of y = (t, d, th, phi, k^t, k^r, k^th, k^phi) -------------------
// `comp` carries, for the float build, the rounding error of each state update into the next one
// (compensated summation): y + comp is the state to roughly twice the working precision.
template <typename T>
GRAY_DEV void rk4_step(const KerrConst<T>& K, T y[8], T comp[8], T dl) {
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
  if (sizeof(T) == 4) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const T inc = dl6 * (acc[i] + (i < 4 ? w[4 + i] : f[i - 4])) + comp[i];
      const T s = y[i] + inc;
      comp[i] = inc - (s - y[i]);          // Fast2Sum: exact whenever |y| >= |inc|
      y[i] = s;
    }
  } else {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      y[i] += dl6 * (acc[i] + w[4 + i]);
      y[4 + i] += dl6 * (acc[4 + i] + f[i]);
    }
  }
}

// pi and 2 pi minus x with pi split in two parts of the working precision
GRAY_DEV float pi_minus(float x) { return (3.14159274101257324219f - x) - 8.742278000372485e-08f; }
GRAY_DEV double pi_minus(double x) { return (3.141592653589793116 - x) + 1.2246467991473532e-16; }
GRAY_DEV float two_pi_minus(float x) { return (6.28318548202514648438f - x) - 1.748455600074497e-07f; }
GRAY_DEV double two_pi_minus(double x) { return (6.283185307179586232 - x) + 2.4492935982947064e-16; }

// ---- theta remap, paper eq. (3), followed by the reflection that keeps th in [0, pi/2] ----------
// Eq. (3) acts on the true polar angle.  For a mirrored photon (true angle pi - th) the true angle
// exceeds pi when th < 0 and is negative when th > pi, so the sign of the phi shift flips with it.
template <typename T>
GRAY_DEV void remap_theta(T y[8], T comp[8], int& mirrored) {
  const T pi = T(3.14159265358979323846);
  const T shift = mirrored ? -pi : pi;
  if (y[2] > pi) {
    y[2] = two_pi_minus(y[2]);
    y[3] += shift;
    y[6] = -y[6];
    comp[2] = -comp[2]; comp[6] = -comp[6];
  } else if (y[2] < T(0)) {
    y[2] = -y[2];
    y[3] -= shift;
    y[6] = -y[6];
    comp[2] = -comp[2]; comp[6] = -comp[6];
  }
  if (y[2] > T(1.57079632679489661923)) {
    y[2] = pi_minus(y[2]);
    y[6] = -y[6];
    comp[2] = -comp[2]; comp[6] = -comp[6];
    mirrored ^= 1;
  }
}

// ---- status of a state after a full step: BAD(3) / CAPTURED(1) / ESCAPED(2) / LIVE(0), in that order
template <typename T>
GRAY_DEV int state_status(const KerrConst<T>& K, const T y[8]) {
  T z = T(0);
#pragma unroll
  for (int i = 0; i < 8; ++i) z += T(0) * y[i];     // inf * 0 = NaN, NaN * 0 = NaN, finite * 0 = 0
  if (!(z == T(0))) return 3;
  const T r = y[1] + K.rp;
  if (r < K.r_cap) return 1;
  if (r > K.r_esc) return 2;
  return 0;
}

}  // namespace gray
