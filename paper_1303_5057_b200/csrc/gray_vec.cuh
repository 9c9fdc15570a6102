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

struct f2 { float x, y; };

template <typename V> struct VT;
template <> struct VT<float>  { using S = float;  static constexpr int N = 1; };
template <> struct VT<double> { using S = double; static constexpr int N = 1; };
template <> struct VT<f2>     { using S = float;  static constexpr int N = 2; };

// ---- broadcast, lane access --------------------------------------------------------------------------
template <typename V> GRAY_DEV V vsplat(typename VT<V>::S s);
template <> GRAY_DEV float vsplat<float>(float s) { return s; }
template <> GRAY_DEV double vsplat<double>(double s) { return s; }
template <> GRAY_DEV f2 vsplat<f2>(float s) { f2 r; r.x = s; r.y = s; return r; }

GRAY_DEV float vget(float v, int) { return v; }
GRAY_DEV double vget(double v, int) { return v; }
GRAY_DEV float vget(f2 v, int l) { return l ? v.y : v.x; }
GRAY_DEV void vset(float& v, int, float s) { v = s; }
GRAY_DEV void vset(double& v, int, double s) { v = s; }
GRAY_DEV void vset(f2& v, int l, float s) { if (l) v.y = s; else v.x = s; }

// ---- add, sub, mul, fma: one rounding each -----------------------------------------------------------
GRAY_DEV float vadd(float a, float b) { return __fadd_rn(a, b); }
GRAY_DEV float vsub(float a, float b) {      // explicit sub.rn: __fsub_rn was seen contracted with a feeding __fmul_rn
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

#define GRAY_F2_BINARY(name, op)                                                                     \
  GRAY_DEV f2 name(f2 a, f2 b) {                                                                     \
    f2 d;                                                                                            \
    asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t" op        \
        " rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"                                                 \
        : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));                            \
    return d;                                                                                        \
  }
GRAY_F2_BINARY(vadd, "add.rn.f32x2")
GRAY_F2_BINARY(vsub, "sub.rn.f32x2")
GRAY_F2_BINARY(vmul, "mul.rn.f32x2")
#undef GRAY_F2_BINARY
GRAY_DEV f2 vfma(f2 a, f2 b, f2 c) {
  f2 d;
  asm("{\n\t.reg .b64 ra, rb, rc, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\tmov.b64 rc, {%6, %7};\n\t"
      "fma.rn.f32x2 rd, ra, rb, rc;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
  return d;
}

// ---- negation and absolute value: sign-bit logic on the ALU pipe, not an FP32-pipe operation -----------
GRAY_DEV float sneg(float x) { return __int_as_float(__float_as_int(x) ^ (int)0x80000000); }
GRAY_DEV float sabs(float x) { return __int_as_float(__float_as_int(x) & 0x7fffffff); }
GRAY_DEV double sneg(double x) { return -x; }
GRAY_DEV double sabs(double x) { return fabs(x); }
GRAY_DEV float vneg(float x) { return sneg(x); }
GRAY_DEV double vneg(double x) { return -x; }
GRAY_DEV f2 vneg(f2 v) { f2 r; r.x = sneg(v.x); r.y = sneg(v.y); return r; }
GRAY_DEV float vabs(float x) { return sabs(x); }
GRAY_DEV double vabs(double x) { return fabs(x); }
GRAY_DEV f2 vabs(f2 v) { f2 r; r.x = sabs(v.x); r.y = sabs(v.y); return r; }

// ---- reciprocal -------------------------------------------------------------------------------------
// float: MUFU.RCP (relative error <= 1 ulp); its uses sit among ~80 half-ulp roundings per right-hand
// side, so it is not refined.  double: IEEE division.
GRAY_DEV float srcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
GRAY_DEV float vrcp(float x) { return srcp(x); }
GRAY_DEV double vrcp(double x) { return __drcp_rn(x); }
GRAY_DEV f2 vrcp(f2 v) { f2 r; r.x = srcp(v.x); r.y = srcp(v.y); return r; }

// ---- min / max (ALU pipe for float) --------------------------------------------------------------------
GRAY_DEV float vmax(float a, float b) { return fmaxf(a, b); }
GRAY_DEV double vmax(double a, double b) { return fmax(a, b); }
GRAY_DEV f2 vmax(f2 a, f2 b) { f2 r; r.x = fmaxf(a.x, b.x); r.y = fmaxf(a.y, b.y); return r; }

}  // namespace gray
