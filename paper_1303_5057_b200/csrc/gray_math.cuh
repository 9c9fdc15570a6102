// gray_math.cuh — per-photon arithmetic of the integrator: Kerr geodesic right-hand side, RK4 step,
// step rules, theta remap, termination tests.  Templated on the vector type V of gray_vec.cuh
// (float, double, or f2 = two fp32 photons per thread in packed FFMA2 / FMUL2 / FADD2 instructions).
//
// The equations are the second-order geodesic equations of the Kerr metric in Boyer-Lindquist
// coordinates (paper P:23; the 20 non-zero Christoffel symbols are listed in SURVEY.md
// App. A.3).  They are not evaluated symbol by symbol.  With
//     Sigma = r^2 + a^2 cos^2(th),  Delta = (r - r_+)(r - r_-),  P = r^2 - a^2 cos^2(th),
//     rho = r^2 + a^2,  s = sin(th),  c = cos(th),
//     q = (k^t - a s^2 k^phi) / Sigma,        v = k^phi - a q   (= (rho k^phi - a k^t) / Sigma)
// the contractions -Gamma^mu_ab k^a k^b collapse to:
//   dk^t  /dl = -2/Sigma [ (k^r/Delta) (rho P q - 2 a s^2 r^2 k^phi) - 2 a^2 r s c k^th q ]
//   dk^phi/dl = -2/Sigma [ (k^r/Delta) (a P q + r (Sigma - 2r) k^phi) + (c/s) k^th (Sigma k^phi - 2 a r q) ]
//   dk^r  /dl = (k^r)^2 [ (r - 1)/Delta - r/Sigma ]
//               + 1/Sigma [ Delta (r (s^2 (k^phi)^2 + (k^th)^2) - P q^2) + 2 a^2 s c k^r k^th ]
//   dk^th /dl = 1/Sigma [ s c (2 r v^2 + Delta (k^phi)^2 + a^2 ((k^th)^2 - (k^r)^2/Delta)) - 2 r k^r k^th ]
// Three reciprocals (1/Sigma, 1/Delta, 1/s) and 63 FP-pipe operations (26 of them fused multiply-adds) per
// evaluation, besides the sine and cosine.
//
// Conditioning: inside the kernel the radial variable is the height above
// the horizon  d = r - r_+  (so Delta = d (d + r_+ - r_-) keeps full relative precision where the
// equations are singular), and the polar angle is kept in [0, pi/2] by the reflection symmetry
// theta -> pi - theta, k^theta -> -k^theta of the Kerr metric (so the absolute rounding of theta shrinks
// towards either pole, where the equations are singular too).  Both are affine changes of variable of the
// same ODE (they commute with RK4); they are undone on store.
#pragma once
#include "gray_vec.cuh"

// Components of y = (t, d, th, phi, k^t, k^r, k^th, k^phi) whose update is a compensated sum in the float builds
// (bit i = component i).  t (bit 0) and phi (bit 3) are left out: the metric depends on neither, so they feed nothing
// back.  Measured on B200: with or without t the final (r, theta, phi) and the drift of E, L_z, Q
// are bit-for-bit the same; without phi the error of the final state against the oracle is unchanged at the 99th
// percentile and at the maximum (phi's own rounding, ~ 1e-7 per step, stays far below the error r and theta carry).
#ifndef GRAY_COMP_MASK
#define GRAY_COMP_MASK 0xf6
#endif

namespace gray {

// Largest |dlt| for which sincos_rotate's series are used (beyond it: sincos_wide)
template <typename S> struct RotateMax;
template <> struct RotateMax<float> { static constexpr float value = 0.045f; };
template <> struct RotateMax<double> { static constexpr double value = 0.04; };

// Constants of a launch, already broadcast to V (for f2 both halves hold the same number, so the packed
// instructions can take them straight from the constant bank / uniform registers).
template <typename V>
struct Consts {
  using S = typename VT<V>::S;
  V a, na, a2, na2, twoa2, n2a2, n2a;     // a, -a, a^2, -a^2, 2a^2, -2a^2, -2a
  V rp, rpm, rpm1;                        // r_+ (the horizon r_bh of P:75), r_+ - r_-, r_+ - 1
  V nh;                                   // -h (step parameter, the paper's Delta)
  V zero, one, mone, two, m2, half, nhalf, sixth, ninth;
  // sin / cos (float builds): quadrant reduction and minimax polynomials, see sincos_v
  V two_over_pi, magic, npio2_hi, npio2_lo, s1, s2, s3, c1, c2, c3, c4;
  V fs1, fs2, fs3, fs4, fc1, fc2, fc3, fc4, fc5;   // sincos_folded (float builds)
  V nsixth, r24;                                   // sincos_rotate (float builds): -1/6, 1/24
  S r_cap, r_esc;                         // termination radii, as heights above the horizon (r - r_+): the kernel's radial variable
  S xi_eps;                               // epsilon of the xi monitor (paper eq. 4); 0 = off
  int stage2_in_range;                    // h / 2 <= RotateMax: under the eq. (2) rule the theta offset of stage 2, dl/2 k^th with
                                          // |dl k^th| <= h, needs no range test before the angle-addition formulas (sincos_stage)
};

template <typename V>
__host__ inline Consts<V> make_consts(double a, double h, double r_cap, double r_esc, double xi_eps) {
  using S = typename VT<V>::S;
  Consts<V> K;
  auto B = [](double v) { V r; S s = (S)v; S* p = (S*)&r; for (int i = 0; i < VT<V>::N; ++i) p[i] = s; return r; };
  const double root = sqrt(1.0 - a * a);
  K.a = B(a); K.na = B(-a); K.a2 = B(a * a); K.na2 = B(-a * a); K.twoa2 = B(2 * a * a); K.n2a2 = B(-2 * a * a);
  K.n2a = B(-2 * a);
  K.rp = B(1.0 + root); K.rpm = B(2.0 * root); K.rpm1 = B(root);
  K.nh = B(-h);
  K.zero = B(0); K.one = B(1); K.two = B(2); K.m2 = B(-2); K.half = B(0.5); K.nhalf = B(-0.5); K.sixth = B(1.0 / 6.0);
  K.mone = B(-1); K.ninth = B(1.0 / 9.0); K.xi_eps = (S)xi_eps;
  K.two_over_pi = B(0.636619772); K.magic = B(12582912.0);
  K.npio2_hi = B(-1.57079637050628662109375); K.npio2_lo = B(4.371139000186241e-08);
  K.s1 = B(-1.666666418e-01); K.s2 = B(8.332700469e-03); K.s3 = B(-1.957778732e-04);
  K.c1 = B(-0.5); K.c2 = B(4.166664928e-02); K.c3 = B(-1.388748409e-03); K.c4 = B(2.445036807e-05);
  K.fs1 = B(-1.6666642594e-01); K.fs2 = B(8.3326730771e-03); K.fs3 = B(-1.9783720104e-04); K.fs4 = B(2.5544161709e-06);
  K.fc1 = B(-4.9999998057e-01); K.fc2 = B(4.1666583344e-02); K.fc3 = B(-1.3887727202e-03); K.fc4 = B(2.4730754562e-05);
  K.fc5 = B(-2.5585777763e-07);
  K.nsixth = B(-1.0 / 6.0); K.r24 = B(1.0 / 24.0);
  K.r_cap = (S)(r_cap - (1.0 + root)); K.r_esc = (S)(r_esc - (1.0 + root));   // differences formed in double
  K.stage2_in_range = 0.5 * h * 1.001 <= (double)RotateMax<S>::value;
  return K;
}

// ---- sin and cos ---------------------------------------------------------------------------------------
// float builds, |x| < ~100 (the kernel's theta stays within a step of [0, pi/2]): quadrant
// j = rint(x 2/pi) by the add-magic-constant trick (1.5 * 2^23: the low mantissa bits of q hold j),
// r = x - j pi/2 with pi/2 split in two floats, then near-minimax polynomials on [-pi/4, pi/4] fitted
// for this kernel (max error 0.86 ulp for both, checked against fp64 over 2e6 points); no slow path and
// no int<->float conversions.  13 FP-pipe operations; the quadrant logic is sign-bit / select work.
GRAY_DEV void quadrant_fix(float q, float sn, float cs, float& s, float& c) {
  const int j = __float_as_int(q);
  const bool swap = (j & 1) != 0;
  const float ss = swap ? cs : sn, cc = swap ? sn : cs;
  s = __int_as_float(__float_as_int(ss) ^ ((j & 2) << 30));          // quadrants 2, 3: sin < 0
  c = __int_as_float(__float_as_int(cc) ^ (((j + 1) & 2) << 30));    // quadrants 1, 2: cos < 0
}
template <typename V>
GRAY_DEV void sincos_v(const Consts<V>& K, V x, V& s, V& c) {
  const V q = vfma(x, K.two_over_pi, K.magic);
  const V jf = vsub(q, K.magic);
  V r = vfma(jf, K.npio2_hi, x);
  r = vfma(jf, K.npio2_lo, r);
  const V u = vmul(r, r);
  const V sp = vfma(vfma(K.s3, u, K.s2), u, K.s1);
  const V sn = vfma(vmul(r, u), sp, r);
  const V cp = vfma(vfma(vfma(K.c4, u, K.c3), u, K.c2), u, K.c1);
  const V cs = vfma(u, cp, K.one);
#pragma unroll
  for (int l = 0; l < VT<V>::N; ++l) {
    float sl, cl;
    quadrant_fix(vget(q, l), vget(sn, l), vget(cs, l), sl, cl);
    vset(s, l, sl);
    vset(c, l, cl);
  }
}
// double build, same scheme: quadrant by the magic constant 1.5 * 2^52, two-term Cody-Waite reduction (exact for the
// |j| <= 2 that occur), Taylor polynomials to r^17 / r^16 on [-pi/4, pi/4] (truncation < 1e-18), Horner in FMAs:
// 22 FP64-pipe operations, no slow path, against ~40 plus a Payne-Hanek branch in the CUDA library's sincos.
template <>
GRAY_DEV void sincos_v<double>(const Consts<double>&, double x, double& s, double& c) {
  const double magic = 6755399441055744.0;
  const double q = __fma_rn(x, 0.63661977236758134308, magic);
  const int j = __double2loint(q);
  const double jf = __dsub_rn(q, magic);
  double r = __fma_rn(jf, -1.57079632679489655800e+00, x);
  r = __fma_rn(jf, -6.12323399573676603587e-17, r);
  const double u = __dmul_rn(r, r);
  double sp = -7.6471637318198164759e-13;                       // -1/15!
  sp = __fma_rn(sp, u, 1.6059043836821614599e-10);              //  1/13!
  sp = __fma_rn(sp, u, -2.5052108385441718775e-08);             // -1/11!
  sp = __fma_rn(sp, u, 2.7557319223985890653e-06);              //  1/9!
  sp = __fma_rn(sp, u, -1.9841269841269841270e-04);             // -1/7!
  sp = __fma_rn(sp, u, 8.3333333333333332177e-03);              //  1/5!
  sp = __fma_rn(sp, u, -1.6666666666666665741e-01);             // -1/3!
  const double sn = __fma_rn(__dmul_rn(r, u), sp, r);
  double cp = 4.7794773323873852974e-14;                        //  1/16!
  cp = __fma_rn(cp, u, -1.1470745597729724714e-11);             // -1/14!
  cp = __fma_rn(cp, u, 2.0876756987868098979e-09);              //  1/12!
  cp = __fma_rn(cp, u, -2.7557319223985888276e-07);             // -1/10!
  cp = __fma_rn(cp, u, 2.4801587301587301566e-05);              //  1/8!
  cp = __fma_rn(cp, u, -1.3888888888888889419e-03);             // -1/6!
  cp = __fma_rn(cp, u, 4.1666666666666664354e-02);              //  1/4!
  cp = __fma_rn(cp, u, -0.5);
  const double cs = __fma_rn(u, cp, 1.0);
  const bool swap = (j & 1) != 0;
  const double ss = swap ? cs : sn, cc = swap ? sn : cs;
  s = (j & 2) ? -ss : ss;                                       // quadrants 2, 3: sin < 0
  c = ((j + 1) & 2) ? -cc : cc;                                 // quadrants 1, 2: cos < 0
}

// ---- sin and cos inside one RK4 step ---------------------------------------------------------------------
// The four right-hand sides of a step are evaluated at th0 (stage 1) and at th0 + dlt with small dlt (stages 2-4:
// dlt = dlambda/2 k^th or dlambda k^th, and eq. (2) keeps |dlambda k^th| <= h).  So only stage 1 needs a sine and
// a cosine of an angle; the others follow by the angle-addition formulas from (s0, c0) and the Taylor series of
// sin, cos of dlt, which needs no range reduction, no quadrant logic and fewer operations.
//
// sincos_folded, float builds: x is the kernel's folded polar angle, in [0, pi/2] at the start of every step
// (remap_theta) - fitted polynomials on [-0.25, pi/2 + 0.25] (sin: odd, relative error 2.8e-8; cos: even, absolute
// error 1.4e-9), 11 FP-pipe operations and no integer / select work at all.  The double build keeps sincos_v.
template <typename V>
GRAY_DEV void sincos_folded(const Consts<V>& K, V x, V& s, V& c) {
  const V u = vmul(x, x);
  const V sp = vfma(vfma(vfma(K.fs4, u, K.fs3), u, K.fs2), u, K.fs1);
  s = vfma(vmul(x, u), sp, x);
  const V cp = vfma(vfma(vfma(vfma(K.fc5, u, K.fc4), u, K.fc3), u, K.fc2), u, K.fc1);
  c = vfma(u, cp, K.one);
}
template <>
GRAY_DEV void sincos_folded<double>(const Consts<double>& K, double x, double& s, double& c) { sincos_v(K, x, s, c); }

// the part of sincos_folded's fitted range that callers who have to ask (rk4_step FOLD = 2) accept
template <typename S> GRAY_DEV S fold_lo() { return S(-0.2); }
template <typename S> GRAY_DEV S fold_hi() { return S(1.7707963); }      // pi/2 + 0.2

// (s, c) = (sin, cos)(th0 + dlt) from (s0, c0) = (sin, cos)(th0):  s = s0 + c0 sd + s0 cm,  c = c0 - s0 sd + c0 cm
// with sd = sin(dlt), cm = cos(dlt) - 1 by their Taylor series.  float: sd = dlt - dlt^3/6, cm = -dlt^2/2 + dlt^4/24
// (9 operations; truncation < 3.4e-8 relative for |dlt| <= RotateMax).  double: through dlt^7 / dlt^8
// (13 operations; truncation dlt^8 / 9! < 2e-17 relative for |dlt| <= RotateMax = 0.04; under eq. (2) with h = 1/32 the
// stage offsets stay below 1/32).
template <typename V>
GRAY_DEV void sincos_rotate(const Consts<V>& K, V s0, V c0, V dlt, V& s, V& c) {
  const V u = vmul(dlt, dlt);
  const V sd = vfma(vmul(dlt, u), K.nsixth, dlt);
  const V cm = vmul(u, vfma(u, K.r24, K.nhalf));
  s = vfma(s0, cm, vfma(c0, sd, s0));
  c = vfma(c0, cm, vfma(s0, vneg(sd), c0));
}
template <>
GRAY_DEV void sincos_rotate<double>(const Consts<double>&, double s0, double c0, double dlt, double& s, double& c) {
  const double u = __dmul_rn(dlt, dlt);
  double sp = -1.9841269841269841270e-04;                       // -1/7!
  sp = __fma_rn(sp, u, 8.3333333333333332177e-03);              //  1/5!
  sp = __fma_rn(sp, u, -1.6666666666666665741e-01);             // -1/3!
  const double sd = __fma_rn(__dmul_rn(dlt, u), sp, dlt);
  double cp = 2.4801587301587301566e-05;                        //  1/8!
  cp = __fma_rn(cp, u, -1.3888888888888889419e-03);             // -1/6!
  cp = __fma_rn(cp, u, 4.1666666666666664354e-02);              //  1/4!
  cp = __fma_rn(cp, u, -0.5);
  const double cm = __dmul_rn(u, cp);
  s = __fma_rn(s0, cm, __fma_rn(c0, sd, s0));
  c = __fma_rn(c0, cm, __fma_rn(-s0, sd, c0));
}
// One photon whose stage offset is outside the series' range (a large k^th next to the axis, or a step rule
// without an angular limit: rare): sine and cosine of th0 + dlt from the CUDA math library.  Kept out of line so that
// its constants and slow path cost the loop nothing.
__device__ __noinline__ float2 sincos_wide(float th0, float dlt) { float2 r; sincosf(__fadd_rn(th0, dlt), &r.x, &r.y); return r; }
__device__ __noinline__ double2 sincos_wide(double th0, double dlt) { double2 r; sincos(__dadd_rn(th0, dlt), &r.x, &r.y); return r; }
// sine and cosine of th0 + dlt for a stage, from (s0, c0) = (sin, cos)(th0).  Each photon by its own |dlt| (its
// result must not depend on the photon it shares a thread with): the rotation within the series' range, else
// sincos_wide.  A NaN dlt goes through the rotation and comes out NaN.
// check = false (uniform over the launch): the caller knows that |dlt| is within the range (no test, rotation only).
template <typename V>
GRAY_DEV void sincos_stage(const Consts<V>& K, V th0, V s0, V c0, V dlt, V& s, V& c, bool check = true) {
  using S = typename VT<V>::S;
  constexpr int N = VT<V>::N;
  sincos_rotate(K, s0, c0, dlt, s, c);
  if (!check) return;
  S a[N];
  vunpack(dlt, a);
  bool wide = false;
#pragma unroll
  for (int l = 0; l < N; ++l) wide |= sabs(a[l]) > RotateMax<S>::value;
  if (wide) {
    S sr[N], cr[N], tb[N];
    vunpack(s, sr); vunpack(c, cr); vunpack(th0, tb);
#pragma unroll
    for (int l = 0; l < N; ++l)
      if (sabs(a[l]) > RotateMax<S>::value) { const auto sc = sincos_wide(tb[l], a[l]); sr[l] = sc.x; cr[l] = sc.y; }
    vpack(s, sr); vpack(c, cr);
  }
}

// ---- right-hand side: accelerations dk^mu/dlambda at d = r - r_+, (s, c) = (sin, cos)(theta) for momentum (kt, kr, kh, kp) ----
// out[i] = dk^i/dlambda (i = t, r, th, phi) if !ACC, else add[i] + dk^i/dlambda with the addition fused into the
// last multiply of each component (stage 4 of RK4 needs only that sum).  No addition or subtraction below
// takes a single-use product as an operand: ptxas contracts such pairs of packed instructions into FFMA2
// even though both carry .rn, which would make the f2 build round differently from the float build.
template <bool ACC, typename V>
GRAY_DEV void geodesic_accel(const Consts<V>& K, V d, V s, V c, V kt, V kr, V kh, V kp, const V* add, V out[4]) {
  const V r = vadd(d, K.rp);
  const V r2 = vmul(r, r);
  const V c2 = vmul(c, c);
  const V Sg = vfma(K.a2, c2, r2);              // Sigma
  const V P = vfma(K.na2, c2, r2);
  const V rho = vadd(r2, K.a2);
  const V Dl = vmul(d, vadd(d, K.rpm));         // Delta = (r - r_+)(r - r_-): no cancellation at the horizon
  const V iS = vrcp(Sg), iD = vrcp(Dl), is = vrcp(s);
  const V niS = vneg(iS);
  const V tniS = vadd(niS, niS);                // -2/Sigma
  const V s2 = vmul(s, s);
  const V sc = vmul(s, c);
  const V as2n = vmul(K.na, s2);                // -a s^2
  const V u = vfma(as2n, kp, kt);
  const V q = vmul(u, iS);                      // u / Sigma
  const V krD = vmul(kr, iD);                   // k^r / Delta
  const V Pq = vmul(P, q);
  const V rk = vmul(r, kp);
  const V rq = vmul(r, q);
  const V Sgk = vmul(Sg, kp);
  // dk^t = -2/Sigma [ (k^r/Delta) (rho P q - 2 a s^2 r^2 k^phi) - 2 a^2 r s c k^th q ]
  const V e1 = vfma(K.two, vmul(vmul(as2n, r), rk), vmul(rho, Pq));
  const V tk = vmul(sc, kh);
  const V Xt = vfma(K.n2a2, vmul(rq, tk), vmul(krD, e1));
  out[0] = ACC ? vfma(tniS, Xt, add[0]) : vmul(tniS, Xt);
  // dk^phi = -2/Sigma [ (k^r/Delta) (a P q + r (Sigma - 2r) k^phi) + (c/s) k^th (Sigma k^phi - 2 a r q) ]
  const V e2 = vfma(K.a, Pq, vmul(vfma(K.m2, r, Sg), rk));
  const V e3 = vfma(K.n2a, rq, Sgk);
  const V ck = vmul(vmul(c, is), kh);
  const V Xp = vfma(ck, e3, vmul(krD, e2));
  out[3] = ACC ? vfma(tniS, Xp, add[3]) : vmul(tniS, Xp);
  // dk^r = (k^r)^2 [(r - 1)/Delta - r/Sigma] + 1/Sigma [ Delta (r (s^2 (k^phi)^2 + (k^th)^2) - P q^2) + 2 a^2 s c k^r k^th ]
  const V krkr = vmul(kr, kr);
  const V G = vfma(vadd(d, K.rpm1), iD, vmul(r, niS));      // (r - 1)/Delta - r/Sigma
  const V kp2 = vmul(kp, kp), kh2 = vmul(kh, kh);
  const V rA1 = vmul(r, vfma(s2, kp2, kh2));
  const V Bp = vfma(vneg(Pq), q, rA1);
  const V J2 = vfma(K.twoa2, vmul(tk, kr), vmul(Dl, Bp));
  out[1] = vfma(krkr, G, ACC ? vfma(iS, J2, add[1]) : vmul(iS, J2));
  // dk^theta = 1/Sigma [ s c (2 r v^2 + Delta (k^phi)^2 + a^2 ((k^th)^2 - (k^r)^2 / Delta)) - 2 r k^r k^th ],  v = w/Sigma = k^phi - a q
  const V v = vfma(K.na, q, kp);
  const V z2 = vfma(K.a2, vfma(vneg(krD), kr, kh2), vmul(Dl, kp2));
  const V z3 = vfma(K.two, vmul(r, vmul(v, v)), z2);
  const V z5 = vfma(K.m2, vmul(vmul(r, kr), kh), vmul(sc, z3));
  out[2] = ACC ? vfma(iS, z5, add[2]) : vmul(iS, z5);
}

// ---- step size (gray.h gray_step_rule; paper eq. (2)) -----------------------------------------
// Returns dlambda < 0.  float builds form the two quotients of eq. (2) with MUFU.RCP (1 ulp): the step
// size is a free parameter of the scheme, an ulp of it is far below the truncation error it controls.
template <typename V, int RULE>
GRAY_DEV V step_size(const Consts<V>& K, V d, V kr, V kh, V kp) {
  const V r = vadd(d, K.rp);
  const V nhr = vmul(K.nh, r);
  if (RULE == 0) return nhr;
  const V akr = vabs(kr);
  const V den = vfma(r, vadd(vabs(kh), vabs(kp)), akr);       // r (|k^r|/r + |k^th| + |k^phi|)
  const V d1 = vmul(nhr, vrcp_step(den));
  const V d2 = vmul(vmul(K.nhalf, d), vrcp_step(akr));
  return vmax(d1, d2);
}

// ---- state update y <- y + scale * rate (scale_x for the four positions, scale_k for the four momenta) ----
// `comp` carries, for the float builds, the rounding error of each update into the next one (compensated
// summation): y + comp is the state to roughly twice the working precision.
template <bool MASKED = false, typename V>
GRAY_DEV void advance_state(const V y[8], const V comp[8], V scale_x, V scale_k, const V rate[8], V yn[8], V cn[8],
                            const bool* adv = nullptr) {
  using S = typename VT<V>::S;
  constexpr int N = VT<V>::N;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const V scale = i < 4 ? scale_x : scale_k;
    if (sizeof(typename VT<V>::S) == 4 && ((GRAY_COMP_MASK >> i) & 1)) {
      const V inc = vfma(scale, rate[i], comp[i]);
      const V s = vadd(y[i], inc);
      cn[i] = vsub(inc, vsub(s, y[i]));        // Fast2Sum: exact whenever |y| >= |inc|
      yn[i] = s;
      if (MASKED) {
        // a slot that does not advance keeps its value and its residual, whatever (finite or not) its rate came out as
        S a[N], b[N], ca[N], cb[N];
        vunpack(yn[i], a); vunpack(y[i], b); vunpack(cn[i], ca); vunpack(comp[i], cb);
#pragma unroll
        for (int l = 0; l < N; ++l) { a[l] = adv[l] ? a[l] : b[l]; ca[l] = adv[l] ? ca[l] : cb[l]; }
        vpack(yn[i], a); vpack(cn[i], ca);
      }
    } else {
      yn[i] = vfma(scale, rate[i], y[i]);
      if (MASKED) {
        S a[N], b[N];
        vunpack(yn[i], a); vunpack(y[i], b);
#pragma unroll
        for (int l = 0; l < N; ++l) a[l] = adv[l] ? a[l] : b[l];
        vpack(yn[i], a);
      }
      cn[i] = comp[i];
    }
  }
}

// ---- the paper's xi (eq. 4): N = g_mu_nu k^mu k^nu and D = g_tt (k^t)^2, xi + 1 = N / D ---------------
//   N = -(k^t)^2 + (2r/Sigma) u^2 + Sigma ((k^r)^2/Delta + (k^th)^2) + rho s^2 (k^phi)^2,  D = (2r/Sigma - 1) (k^t)^2
// (s, c) = (sin, cos)(y[2]), supplied by the caller.
template <typename V>
GRAY_DEV void null_norm(const Consts<V>& K, const V y[8], V s, V c, V& Nn, V& Dn) {
  const V d = y[1], kt = y[4], kr = y[5], kh = y[6], kp = y[7];
  const V r = vadd(d, K.rp);
  const V r2 = vmul(r, r);
  const V Sg = vfma(K.a2, vmul(c, c), r2);
  const V rho = vadd(r2, K.a2);
  const V Dl = vmul(d, vadd(d, K.rpm));
  const V iS = vrcp(Sg), iD = vrcp(Dl);
  const V s2 = vmul(s, s);
  const V u = vfma(vmul(K.na, s2), kp, kt);
  const V riS = vmul(r, iS);
  const V kt2 = vmul(kt, kt);
  const V B = vfma(vmul(kr, iD), kr, vmul(kh, kh));
  const V n1 = vfma(K.two, vmul(riS, vmul(u, u)), vmul(Sg, B));
  const V n2 = vfma(vmul(rho, vmul(s2, kp)), kp, n1);
  Nn = vfma(vneg(kt), kt, n2);
  Dn = vmul(vfma(K.two, riS, K.mone), kt2);
}

// ---- one classical RK4 step of y = (t, d, th, phi, k^t, k^r, k^th, k^phi) -------------------
// XI: the paper's production pole treatment: if the state the RK4 step produced has |xi + 1| > epsilon
// (or a non-finite xi), the step is re-integrated from the old state as one forward Euler step of dlambda / 9,
// which is not tested itself.  rejected[l] reports it per photon.
// FOLD: whether y[2] lies in the range of sincos_folded at the start of the step.  1: always (the kernel's folded theta
// under the eq. (2) rule, whose steps cannot leave [0, pi/2] by more than h); 2: the caller says in `fold_ok` whether
// all photons of the thread are within [fold_lo, fold_hi] (stop_at_equator under eq. (2): a photon being landed on
// the plane sits just beyond pi/2, and a Newton landing step is not bounded by the rule); 0: never (the REL rule, whose
// steps are not bounded in theta).
// MASKED (gray.h `frozen`): only the slots with adv[l] advance; the others keep their state bit for bit while the
// arithmetic of the step is carried out for them all the same (the caller passes them dlambda = 0).
template <bool XI, int FOLD, bool MASKED = false, typename V>
GRAY_DEV void rk4_step(const Consts<V>& K, V y[8], V comp[8], V dl, bool rejected[VT<V>::N], const bool* adv = nullptr,
                       bool fold_ok = false) {
  using S = typename VT<V>::S;
  constexpr int N = VT<V>::N;
  constexpr bool FOLDED = FOLD == 1;
  V acc[8], w[8], f[4], f1[4];
  const V hdl = vmul(K.half, dl);
  const V dl6 = vmul(K.sixth, dl);
  // stage 1
  V s0, c0, ss, cc;
  if (FOLD != 0) {
    sincos_folded(K, y[2], s0, c0);
    if (FOLD == 2 && !fold_ok) {
      // rare: some photon of this thread is outside the polynomial's range; it alone takes the quadrant-reduced values
      // (a photon's arithmetic must not depend on the photon it shares a thread with)
      V sv, cv;
      sincos_v(K, y[2], sv, cv);
      S th[N], a[N], b[N], c[N], d[N];
      vunpack(y[2], th); vunpack(s0, a); vunpack(c0, b); vunpack(sv, c); vunpack(cv, d);
#pragma unroll
      for (int l = 0; l < N; ++l) {
        const bool in = th[l] >= fold_lo<S>() && th[l] <= fold_hi<S>();
        a[l] = in ? a[l] : c[l];
        b[l] = in ? b[l] : d[l];
      }
      vpack(s0, a); vpack(c0, b);
    }
  } else sincos_v(K, y[2], s0, c0);
  geodesic_accel<false>(K, y[1], s0, c0, y[4], y[5], y[6], y[7], (const V*)nullptr, f);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    f1[i] = f[i];
    acc[i] = y[4 + i];
    acc[4 + i] = f[i];
    w[i] = i == 2 ? vmul(hdl, y[6]) : vfma(hdl, y[4 + i], y[i]);      // w[2]: the stage's offset in theta, not theta
    w[4 + i] = vfma(hdl, f[i], y[4 + i]);
  }
  // stages 2 and 3.  Stage 2 under the eq. (2) rule (FOLDED): |dl k^th| <= h by the rule itself, so with h / 2 inside the
  // rotation's range (Consts::stage2_in_range) its offset needs no range test
#pragma unroll
  for (int stage = 2; stage <= 3; ++stage) {
    const V hs = stage == 2 ? hdl : dl;
    sincos_stage(K, y[2], s0, c0, w[2], ss, cc, !(stage == 2 && FOLDED && K.stage2_in_range));
    geodesic_accel<false>(K, w[1], ss, cc, w[4], w[5], w[6], w[7], (const V*)nullptr, f);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const V kx = w[4 + i];
      acc[i] = vfma(K.two, kx, acc[i]);
      acc[4 + i] = vfma(K.two, f[i], acc[4 + i]);
      w[i] = i == 2 ? vmul(hs, kx) : vfma(hs, kx, y[i]);
      w[4 + i] = vfma(hs, f[i], y[4 + i]);
    }
  }
  // stage 4: the sums k1 + 2 k2 + 2 k3 + k4
#pragma unroll
  for (int i = 0; i < 4; ++i) acc[i] = vadd(acc[i], w[4 + i]);
  sincos_stage(K, y[2], s0, c0, w[2], ss, cc);
  geodesic_accel<true>(K, w[1], ss, cc, w[4], w[5], w[6], w[7], acc + 4, acc + 4);
  V yn[8], cn[8];
  advance_state<MASKED>(y, comp, dl6, dl6, acc, yn, cn, adv);
#pragma unroll
  for (int l = 0; l < N; ++l) rejected[l] = false;
  if (XI) {
    // sine and cosine at the new state: (s0, c0) turned by the step's own increment of theta (yn[2] and y[2] differ by
    // it up to the rounding the compensation carries)
    V Nn, Dn, sn, cn2;
    sincos_stage(K, y[2], s0, c0, vsub(yn[2], y[2]), sn, cn2);
    null_norm(K, yn, sn, cn2, Nn, Dn);
    S nn[N], dn[N];
    vunpack(Nn, nn); vunpack(Dn, dn);
    bool any = false;
#pragma unroll
    for (int l = 0; l < N; ++l) {
      rejected[l] = !(sabs(nn[l]) <= vmul(K.xi_eps, sabs(dn[l])));
      any |= rejected[l];
    }
    if (any) {
      V re[8], ye[8], ce[8];
#pragma unroll
      for (int i = 0; i < 4; ++i) { re[i] = y[4 + i]; re[4 + i] = f1[i]; }
      const V dl9 = vmul(K.ninth, dl);
      advance_state(y, comp, dl9, dl9, re, ye, ce);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        S a[N], b[N], ca[N], cb[N];
        vunpack(yn[i], a); vunpack(ye[i], b); vunpack(cn[i], ca); vunpack(ce[i], cb);
#pragma unroll
        for (int l = 0; l < N; ++l) { a[l] = rejected[l] ? b[l] : a[l]; ca[l] = rejected[l] ? cb[l] : ca[l]; }
        vpack(yn[i], a); vpack(cn[i], ca);
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) { y[i] = yn[i]; comp[i] = cn[i]; }
}

// ======================================================================================================
// Reduced system (NEXT-3; R21): the Killing constants E = -k_t, L = k_phi eliminate k^t and k^phi.
//   u = k^t - a s^2 k^phi = (rho E - a L)/Delta,    w = Sigma k^phi - a u = L/s^2 - a E,
//   k^phi = (w + a u)/Sigma,                        k^t = u + a s^2 k^phi
// (the inverse Kerr metric applied to (-E, L), regrouped), and dk^r/dl, dk^theta/dl are the same expressions as
// in geodesic_accel.  49 FP-pipe operations besides the sincos, against 63.
// ======================================================================================================
GRAY_DEV void sincos_s(float x, float& s, float& c) { sincosf(x, &s, &c); }
GRAY_DEV void sincos_s(double x, double& s, double& c) { sincos(x, &s, &c); }

// E, L of a stored state (scalar, once per photon on load)
template <typename S>
GRAY_DEV void killing_constants(S a, S rp, S d, S th, S kt, S kp, S& E, S& L) {
  S s, c;
  sincos_s(th, s, c);
  const S r = vadd(d, rp);
  const S r2 = vmul(r, r), s2 = vmul(s, s);
  const S Sg = vfma(vmul(a, a), vmul(c, c), r2);
  const S rho = vfma(a, a, r2);
  const S f = vmul(vadd(r, r), vrcp_exact(Sg));                  // 2r/Sigma
  const S af = vmul(a, f);
  // E = (1 - 2r/Sigma) k^t + (2 a r s^2/Sigma) k^phi;  L = s^2 [(rho + a s^2 (2 a r/Sigma)) k^phi - (2 a r/Sigma) k^t]
  E = vfma(vmul(af, s2), kp, vfma(vneg(f), kt, kt));
  L = vmul(s2, vfma(vfma(vmul(a, s2), af, rho), kp, vneg(vmul(af, kt))));
}
// k^t, k^phi of a state from its constants (scalar, once per photon on retirement)
template <typename S>
GRAY_DEV void killing_velocities(S a, S rp, S rpm, S d, S th, S E, S L, S& kt, S& kp) {
  S s, c;
  sincos_s(th, s, c);
  const S r = vadd(d, rp);
  const S r2 = vmul(r, r), s2 = vmul(s, s);
  const S Sg = vfma(vmul(a, a), vmul(c, c), r2);
  const S rho = vfma(a, a, r2);
  const S Dl = vmul(d, vadd(d, rpm));
  const S u = vmul(vfma(rho, E, vneg(vmul(a, L))), vrcp_exact(Dl));
  const S w = vfma(L, vrcp_exact(s2), vneg(vmul(a, E)));
  kp = vmul(vfma(a, u, w), vrcp_exact(Sg));
  kt = vfma(vmul(a, s2), kp, u);
}

// accelerations of (k^r, k^theta) -> out[0], out[1] (ACC: added to add[0], add[1]); k^t, k^phi of the point -> kt, kp
template <bool ACC, typename V>
GRAY_DEV void geodesic_accel_reduced(const Consts<V>& K, V d, V s, V c, V kr, V kh, V E, V L, V naE, V naL, const V* add,
                                     V out[2], V& kt, V& kp) {
  const V r = vadd(d, K.rp);
  const V r2 = vmul(r, r);
  const V c2 = vmul(c, c);
  const V Sg = vfma(K.a2, c2, r2);
  const V P = vfma(K.na2, c2, r2);
  const V rho = vadd(r2, K.a2);
  const V Dl = vmul(d, vadd(d, K.rpm));
  const V iS = vrcp(Sg), iD = vrcp(Dl), is = vrcp(s);
  const V niS = vneg(iS);
  const V s2 = vmul(s, s);
  const V sc = vmul(s, c);
  const V u = vmul(vfma(rho, E, naL), iD);
  const V w = vfma(L, vmul(is, is), naE);
  const V q = vmul(u, iS);                      // u / Sigma
  const V v = vmul(w, iS);                      // w / Sigma
  kp = vfma(K.a, q, v);
  kt = vfma(vmul(K.a, s2), kp, u);
  const V krD = vmul(kr, iD);
  const V Pq = vmul(P, q);
  const V tk = vmul(sc, kh);
  // dk^r
  const V krkr = vmul(kr, kr);
  const V G = vfma(vadd(d, K.rpm1), iD, vmul(r, niS));
  const V kp2 = vmul(kp, kp), kh2 = vmul(kh, kh);
  const V rA1 = vmul(r, vfma(s2, kp2, kh2));
  const V Bp = vfma(vneg(Pq), q, rA1);
  const V J2 = vfma(K.twoa2, vmul(tk, kr), vmul(Dl, Bp));
  out[0] = vfma(krkr, G, ACC ? vfma(iS, J2, add[0]) : vmul(iS, J2));
  // dk^theta
  const V z2 = vfma(K.a2, vfma(vneg(krD), kr, kh2), vmul(Dl, kp2));     // Delta (k^phi)^2 + a^2 ((k^th)^2 - (k^r)^2 / Delta)
  const V z3 = vfma(K.two, vmul(r, vmul(v, v)), z2);
  const V z5 = vfma(K.m2, vmul(vmul(r, kr), kh), vmul(sc, z3));
  out[1] = ACC ? vfma(iS, z5, add[1]) : vmul(iS, z5);
}

// One RK4 step of the reduced system.  y[4], y[7] hold the constants E, L of the photon and comp[4], comp[7] hold
// -a E, -a L; neither is touched.  The step size (which needs k^phi) is formed after the first evaluation.
template <int RULE, typename V>
GRAY_DEV void rk4_step_reduced(const Consts<V>& K, V y[8], V comp[8]) {
  const V E = y[4], L = y[7], naE = comp[4], naL = comp[7];
  V f[2], kt, kp, acc[8], w1, w2, w5, w6, s0, c0, ss, cc;
  if (RULE == 1) sincos_folded(K, y[2], s0, c0);
  else sincos_v(K, y[2], s0, c0);
  geodesic_accel_reduced<false>(K, y[1], s0, c0, y[5], y[6], E, L, naE, naL, (const V*)nullptr, f, kt, kp);
  const V dl = step_size<V, RULE>(K, y[1], y[5], y[6], kp);
  const V hdl = vmul(K.half, dl);
  acc[0] = kt; acc[3] = kp; acc[1] = y[5]; acc[2] = y[6]; acc[5] = f[0]; acc[6] = f[1];
  w1 = vfma(hdl, y[5], y[1]); w2 = vmul(hdl, y[6]); w5 = vfma(hdl, f[0], y[5]); w6 = vfma(hdl, f[1], y[6]);   // w2: offset in theta
#pragma unroll
  for (int stage = 2; stage <= 3; ++stage) {
    const V hs = stage == 2 ? hdl : dl;
    sincos_stage(K, y[2], s0, c0, w2, ss, cc);
    geodesic_accel_reduced<false>(K, w1, ss, cc, w5, w6, E, L, naE, naL, (const V*)nullptr, f, kt, kp);
    acc[0] = vfma(K.two, kt, acc[0]); acc[3] = vfma(K.two, kp, acc[3]);
    acc[1] = vfma(K.two, w5, acc[1]); acc[2] = vfma(K.two, w6, acc[2]);
    acc[5] = vfma(K.two, f[0], acc[5]); acc[6] = vfma(K.two, f[1], acc[6]);
    const V k5 = w5, k6 = w6;
    w1 = vfma(hs, k5, y[1]); w2 = vmul(hs, k6); w5 = vfma(hs, f[0], y[5]); w6 = vfma(hs, f[1], y[6]);
  }
  acc[1] = vadd(acc[1], w5); acc[2] = vadd(acc[2], w6);
  sincos_stage(K, y[2], s0, c0, w2, ss, cc);
  geodesic_accel_reduced<true>(K, w1, ss, cc, w5, w6, E, L, naE, naL, acc + 5, acc + 5, kt, kp);
  acc[0] = vadd(acc[0], kt); acc[3] = vadd(acc[3], kp);
  const V dl6 = vmul(K.sixth, dl);
#pragma unroll
  for (int i = 0; i < 7; ++i) {
    if (i == 4) continue;
    if (sizeof(typename VT<V>::S) == 4 && ((GRAY_COMP_MASK >> i) & 1)) {
      const V inc = vfma(dl6, acc[i], comp[i]);
      const V s = vadd(y[i], inc);
      comp[i] = vsub(inc, vsub(s, y[i]));
      y[i] = s;
    } else {
      y[i] = vfma(dl6, acc[i], y[i]);
    }
  }
}

// pi and 2 pi minus x with pi split in two parts of the working precision
GRAY_DEV float pi_minus(float x) { return __fsub_rn(__fsub_rn(3.14159274101257324219f, x), 8.742278000372485e-08f); }
GRAY_DEV double pi_minus(double x) { return (3.141592653589793116 - x) + 1.2246467991473532e-16; }
GRAY_DEV float two_pi_minus(float x) { return __fsub_rn(__fsub_rn(6.28318548202514648438f, x), 1.748455600074497e-07f); }
GRAY_DEV double two_pi_minus(double x) { return (6.283185307179586232 - x) + 2.4492935982947064e-16; }

// ---- theta remap, paper eq. (3), followed by the reflection that keeps th in [0, pi/2] ----------
// One photon (scalar S).  Eq. (3) acts on the true polar angle.  For a mirrored photon (true angle
// pi - th) the true angle exceeds pi when th < 0 and is negative when th > pi, so the sign of the phi
// shift flips with it.  Returns whether the (eq. (3)-remapped) folded angle exceeds pi/2, i.e. whether the step
// crossed the equatorial plane; the fold itself is applied only if `fold` (gray.h stop_at_equator lands the
// photon on the plane instead).
template <typename S>
GRAY_DEV bool remap_theta(S& th, S& ph, S& kh, S& c_th, S& c_kh, int& mirrored, bool fold) {
  const S pi = S(3.14159265358979323846);
  const S shift = mirrored ? -pi : pi;
  if (th > pi) {
    th = two_pi_minus(th);
    ph += shift;
    kh = sneg(kh); c_th = sneg(c_th); c_kh = sneg(c_kh);
  } else if (th < S(0)) {
    th = sneg(th);
    ph -= shift;
    kh = sneg(kh); c_th = sneg(c_th); c_kh = sneg(c_kh);
  }
  const bool over = th > S(1.57079632679489661923);      // the true polar angle has crossed the equatorial plane
  if (over && fold) {
    th = pi_minus(th);
    kh = sneg(kh); c_th = sneg(c_th); c_kh = sneg(c_kh);
    mirrored ^= 1;
  }
  return over;
}

// ---- non-finite detector: z = sum_i 0 * k^i is 0 iff the four momentum components are finite ------------
// The positions need no probe: x_new = x + dlambda/6 (sum of the stage momenta), and a stage momentum is
// non-finite only if an acceleration is, which makes the new momentum non-finite as well; so with finite
// momenta the positions stay finite (short of the overflow of a finite sum beyond 3e38, which r_escape
// excludes).  The oracle's test on all eight components (R10) fires on the same step.
template <typename V>
GRAY_DEV V nonfinite_probe(const Consts<V>& K, const V y[8]) {
  V z = vmul(K.zero, y[4]);
#pragma unroll
  for (int i = 5; i < 8; ++i) z = vfma(K.zero, y[i], z);
  return z;
}

// status of one photon after a full step: BAD(3) / CAPTURED(1) / ESCAPED(2) / LIVE(0), in that order
template <typename S>
GRAY_DEV int state_status(S z, S r, S r_cap, S r_esc) {     // r, r_cap, r_esc: heights above the horizon
  if (!(z == S(0))) return 3;
  if (r < r_cap) return 1;
  if (r > r_esc) return 2;
  return 0;
}

}  // namespace gray
