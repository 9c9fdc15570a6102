// gray_vec.cuh — the arithmetic layer of the integrator: every floating-point operation of the hot loop
// is one of the functions below, written for three "vector" types V:
//     float    one photon per thread, fp32
//     double   one photon per thread, fp64
//     f2       TWO photons per thread, fp32, in the packed sm_100a instructions FFMA2 / FMUL2 / FADD2
//              (PTX fma/mul/add/sub.rn.f32x2): one issue slot carries the operation for both photons, so
//              the FP32 pipe (128 lanes per SM) is fed from half the issue slots and the integer, select
//              and MUFU instructions of the loop issue in its shadow.
// Every operation is a single correctly rounded IEEE operation with the contraction written out
// (vfma) — nothing is left to the compiler's -fmad — so the float and the f2 builds execute the same
// operations in the same order and give the same bits per photon (tested).
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#define GRAY_DEV __device__ __forceinline__

namespace gray {

// Two floats in one 64-bit register pair (x = photon 0 in the low word, y = photon 1 in the high word).  Held as
// a single 64-bit value so that the register allocator keeps the pair together across the loop: the packed
// instructions need an aligned pair, and assembling one from two free-floating scalars costs a MOV per half.
struct f2 { unsigned long long v; };
GRAY_DEV f2 f2_pack(float lo, float hi) {
  f2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
  return r;
}
GRAY_DEV void f2_unpack(f2 a, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); }

template <typename V> struct VT;
template <> struct VT<float>  { using S = float;  static constexpr int N = 1; };
template <> struct VT<double> { using S = double; static constexpr int N = 1; };
template <> struct VT<f2>     { using S = float;  static constexpr int N = 2; };

// ---- broadcast, lane access --------------------------------------------------------------------------
template <typename V> GRAY_DEV V vsplat(typename VT<V>::S s);
template <> GRAY_DEV float vsplat<float>(float s) { return s; }
template <> GRAY_DEV double vsplat<double>(double s) { return s; }
template <> GRAY_DEV f2 vsplat<f2>(float s) { return f2_pack(s, s); }

GRAY_DEV float vget(float v, int) { return v; }
GRAY_DEV double vget(double v, int) { return v; }
GRAY_DEV float vget(f2 v, int l) { float lo, hi; f2_unpack(v, lo, hi); return l ? hi : lo; }
GRAY_DEV void vset(float& v, int, float s) { v = s; }
GRAY_DEV void vset(double& v, int, double s) { v = s; }
GRAY_DEV void vset(f2& v, int l, float s) { float lo, hi; f2_unpack(v, lo, hi); v = l ? f2_pack(lo, s) : f2_pack(s, hi); }
// all lanes at once: v <-> s[0 .. N-1]
GRAY_DEV void vunpack(float v, float s[1]) { s[0] = v; }
GRAY_DEV void vunpack(double v, double s[1]) { s[0] = v; }
GRAY_DEV void vunpack(f2 v, float s[2]) { f2_unpack(v, s[0], s[1]); }
GRAY_DEV void vpack(float& v, const float s[1]) { v = s[0]; }
GRAY_DEV void vpack(double& v, const double s[1]) { v = s[0]; }
GRAY_DEV void vpack(f2& v, const float s[2]) { v = f2_pack(s[0], s[1]); }

// ---- add, sub, mul, fma: one rounding each -----------------------------------------------------------
GRAY_DEV float vadd(float a, float b) { return __fadd_rn(a, b); }
GRAY_DEV float vsub(float a, float b) {      // sub.rn spelled out: the same instruction form as the packed build's
  float d;
  asm("sub.rn.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  return d;
}
GRAY_DEV float vmul(float a, float b) { return __fmul_rn(a, b); }
GRAY_DEV float vfma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
GRAY_DEV double vadd(double a, double b) { return __dadd_rn(a, b); }
GRAY_DEV double vsub(double a, double b) {
  double d;
  asm("sub.rn.f64 %0, %1, %2;" : "=d"(d) : "d"(a), "d"(b));
  return d;
}
GRAY_DEV double vmul(double a, double b) { return __dmul_rn(a, b); }
GRAY_DEV double vfma(double a, double b, double c) { return __fma_rn(a, b, c); }

#define GRAY_F2_BINARY(name, op)                                                     \
  GRAY_DEV f2 name(f2 a, f2 b) {                                                     \
    f2 d;                                                                            \
    asm(op " %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v));                         \
    return d;                                                                        \
  }
GRAY_F2_BINARY(vadd, "add.rn.f32x2")
GRAY_F2_BINARY(vsub, "sub.rn.f32x2")
GRAY_F2_BINARY(vmul, "mul.rn.f32x2")
#undef GRAY_F2_BINARY
GRAY_DEV f2 vfma(f2 a, f2 b, f2 c) {
  f2 d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.v) : "l"(a.v), "l"(b.v), "l"(c.v));
  return d;
}

// ---- negation and absolute value: sign-bit logic on the ALU pipe, not an FP32-pipe operation -----------
GRAY_DEV float sneg(float x) { return __int_as_float(__float_as_int(x) ^ (int)0x80000000); }
GRAY_DEV float sabs(float x) { return __int_as_float(__float_as_int(x) & 0x7fffffff); }
GRAY_DEV double sneg(double x) { return -x; }
GRAY_DEV double sabs(double x) { return fabs(x); }
GRAY_DEV float vneg(float x) { return sneg(x); }
GRAY_DEV double vneg(double x) { return -x; }
GRAY_DEV f2 vneg(f2 v) { float lo, hi; f2_unpack(v, lo, hi); return f2_pack(sneg(lo), sneg(hi)); }
GRAY_DEV float vabs(float x) { return sabs(x); }
GRAY_DEV double vabs(double x) { return fabs(x); }
GRAY_DEV f2 vabs(f2 v) { float lo, hi; f2_unpack(v, lo, hi); return f2_pack(sabs(lo), sabs(hi)); }

// ---- reciprocal -------------------------------------------------------------------------------------
// float: MUFU.RCP (relative error <= 1 ulp); its uses sit among ~80 half-ulp roundings per right-hand
// side, so it is not refined.
GRAY_DEV float srcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
GRAY_DEV float vrcp(float x) { return srcp(x); }
// double: MUFU.RCP64H seed y0 (rcp.approx.ftz.f64, relative error e ~ 2^-20) refined to third order in FMAs,
// y = y0 (1 + e + e^2) with e = 1 - x y0: relative error e^3 ~ 1e-18, i.e. the rounding of the last FMA (not correctly
// rounded, like the float build's); 3 FP64 operations, no special-case branch.
GRAY_DEV double vrcp(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = __fma_rn(-x, y, 1.0);
  const double t = __fma_rn(e, e, e);
  return __fma_rn(y, t, y);
}
// reciprocals that only scale the step size (eq. 2): one Newton iteration, relative error ~ 2^-40 - the step size is a
// free parameter of the scheme, and 1e-12 of it is far below the 1e-9 the results are compared at
GRAY_DEV float vrcp_step(float x) { return srcp(x); }
GRAY_DEV double vrcp_step(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return __fma_rn(y, __fma_rn(-x, y, 1.0), y);
}
GRAY_DEV f2 vrcp(f2 v) { float lo, hi; f2_unpack(v, lo, hi); return f2_pack(srcp(lo), srcp(hi)); }
GRAY_DEV f2 vrcp_step(f2 v) { return vrcp(v); }

// exact (IEEE) reciprocal for the scalar once-per-photon work of the reduced system
GRAY_DEV float vrcp_exact(float x) { return __frcp_rn(x); }
GRAY_DEV double vrcp_exact(double x) { return __drcp_rn(x); }

// ---- min / max (ALU pipe for float) --------------------------------------------------------------------
GRAY_DEV float vmax(float a, float b) { return fmaxf(a, b); }
GRAY_DEV double vmax(double a, double b) { return fmax(a, b); }
GRAY_DEV f2 vmax(f2 a, f2 b) {
  float al, ah, bl, bh;
  f2_unpack(a, al, ah);
  f2_unpack(b, bl, bh);
  return f2_pack(fmaxf(al, bl), fmaxf(ah, bh));
}

}  // namespace gray
