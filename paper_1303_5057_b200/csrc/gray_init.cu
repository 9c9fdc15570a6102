// gray_init.cu — gray_init_rays / gray_init_rays_random (include/gray.h): image plane -> photon states.
//
// One thread per photon, double precision throughout, rounded to the build's precision on store
// (readings R1-R4).  Nothing here is timed on the hot loop: it runs once.
#include "gray_internal.h"

namespace gray {

struct InitArgs {
  void* x;
  void* k;
  uint8_t* status;
  uint32_t* steps;
  unsigned long long n, p0, seed;
  double a, r_obs, sin_i, cos_i, W, R_lo;
  unsigned long long nx, ny;
};

// 64-bit finaliser of the splitmix64 generator (Steele, Lea & Flood 2014), used as a stateless hash
// of (seed, photon index): the counter-based pixel generator of DESIGN.md "Input recipe".
__device__ __forceinline__ unsigned long long mix64(unsigned long long z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

template <typename T, int PIXELS>
__global__ void __launch_bounds__(256) init_kernel(const __grid_constant__ InitArgs A) {
  const unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= A.n) return;
  const unsigned long long p = A.p0 + j;
  double alpha, beta;
  if (PIXELS == GRAY_PIXELS_POLAR) {
    // nx radii (cell centres of (R_lo, W)), ny angles in [0, pi] including both ends; explicit roundings
    const unsigned long long jr = p % A.nx, kt = p / A.nx;
    const double dR = __ddiv_rn(__dadd_rn(A.W, -A.R_lo), (double)A.nx);
    const double R = __dadd_rn(A.R_lo, __dmul_rn(__dadd_rn((double)jr, 0.5), dR));
    const double vt = __dmul_rn((double)kt, __ddiv_rn(3.14159265358979323846, (double)(A.ny - 1)));
    double sv, cv;
    sincos(vt, &sv, &cv);
    alpha = __dmul_rn(R, cv);
    beta = __dmul_rn(R, sv);
  } else if (PIXELS == GRAY_PIXELS_GRID) {
    // pixel centres; explicit roundings so that (alpha, beta) are the same doubles on any machine
    const unsigned long long col = p % A.nx, row = p / A.nx;
    const double da = __ddiv_rn(__dmul_rn(2.0, A.W), (double)A.nx);
    const double db = __ddiv_rn(__dmul_rn(2.0, A.W), (double)A.ny);
    alpha = __dadd_rn(-A.W, __dmul_rn(__dadd_rn((double)col, 0.5), da));
    beta = __dadd_rn(-A.W, __dmul_rn(__dadd_rn((double)row, 0.5), db));
  } else {
    // two 24-bit integers from one 64-bit hash -> cell centres of a 2^24 x 2^24 lattice, defined as
    // the fp32 rounding so that every implementation starts from identical pixels
    const unsigned long long z = mix64(mix64(A.seed) ^ p);
    const long long u = (long long)(z >> 40), v = (long long)((z >> 16) & 0xFFFFFFull);
    const double fa = __dmul_rn(__dmul_rn((double)(2 * u + 1 - (1ll << 24)), A.W), 1.0 / 16777216.0);
    const double fb = __dmul_rn(__dmul_rn((double)(2 * v + 1 - (1ll << 24)), A.W), 1.0 / 16777216.0);
    alpha = (double)__double2float_rn(fa);
    beta = (double)__double2float_rn(fb);
  }
  // Cartesian position of the pixel: r_obs o + alpha yhat + beta bhat
  const double X = A.r_obs * A.sin_i - beta * A.cos_i;
  const double Y = alpha;
  const double Z = A.r_obs * A.cos_i + beta * A.sin_i;
  const double q2 = X * X + Y * Y;            // (r sin th)^2
  const double q = sqrt(q2);
  const double r = sqrt(q2 + Z * Z);
  const double ct = Z / r, st = q / r;
  const double th = atan2(q, Z);              // well conditioned for observers near the spin axis, where acos(Z / r) is not
  const double ph = atan2(Y, X);
  // velocity o = (sin i, 0, cos i) in spherical components: o.rhat = r_obs / r,
  // o.thhat / r, o.phhat / (r sin th)
  double kr = A.r_obs / r;
  double kh = (A.sin_i * ct * (X / q) - A.cos_i * st) / r;
  double kp = -A.sin_i * Y / q2;
  // A pixel exactly on the spin axis (q = 0: a face-on observer's central pixel) has no azimuth; o is then parallel to
  // the axis and its theta and phi components vanish in the limit.  The state is finite; the ray itself cannot be
  // followed in Boyer-Lindquist coordinates (1 / sin(theta) in the first right-hand side) and ends GRAY_BAD (gray.h).
  if (q == 0.0) { kh = 0.0; kp = 0.0; }
  // null condition for k^t (future-directed root), then normalise to E = -k_t = 1
  const double a = A.a, a2 = a * a, r2 = r * r, s2 = st * st;
  const double Sg = r2 + a2 * ct * ct;
  const double Dl = r2 - 2.0 * r + a2;
  const double g_tt = -(1.0 - 2.0 * r / Sg);
  const double g_tp = -2.0 * a * r * s2 / Sg;
  const double g_pp = (r2 + a2 + 2.0 * a2 * r * s2 / Sg) * s2;
  const double C = Sg / Dl * kr * kr + Sg * kh * kh + g_pp * kp * kp;
  const double B = g_tp * kp;
  double kt = (-B - sqrt(B * B - g_tt * C)) / g_tt;
  const double iE = -1.0 / (g_tt * kt + g_tp * kp);
  kt *= iE; kr *= iE; kh *= iE; kp *= iE;
  if (sizeof(T) == 4) {
    ((float4*)A.x)[j] = make_float4(0.0f, (float)r, (float)th, (float)ph);
    ((float4*)A.k)[j] = make_float4((float)kt, (float)kr, (float)kh, (float)kp);
  } else {
    ((double4*)A.x)[j] = make_double4(0.0, r, th, ph);
    ((double4*)A.k)[j] = make_double4(kt, kr, kh, kp);
  }
  A.status[j] = GRAY_LIVE;
  A.steps[j] = 0;
}

static int init_common(gray_state* st, double a, double r_obs, double inc_deg, double W, int pixels,
                       int32_t nx, int32_t ny, uint64_t seed, uint64_t p0, cudaStream_t stream, double R_lo = 0.0) {
  int rc = check_state(st, false);
  if (rc) return rc;
  if (!(a > -1.0 && a < 1.0)) { set_error("spin a = %g outside (-1, 1)", a); return GRAY_ERR_DOMAIN; }
  if (!(r_obs > 0.0) || !(W > 0.0)) { set_error("r_obs and half_width must be positive"); return GRAY_ERR_DOMAIN; }
  if (!(inc_deg >= 0.0 && inc_deg <= 180.0)) { set_error("inclination %g outside [0, 180] degrees", inc_deg); return GRAY_ERR_DOMAIN; }
  if (pixels == GRAY_PIXELS_POLAR && (!(R_lo >= 0.0 && R_lo < W) || ny < 2)) { set_error("polar grid needs 0 <= R_lo < R_hi and n_theta >= 2"); return GRAY_ERR_DOMAIN; }
  if (!(sqrt(r_obs * r_obs + 2.0 * W * W) < 1.01 * r_obs)) { set_error("half_width %g too large for r_obs %g: a pixel would start outside 1.01 r_obs", W, r_obs); return GRAY_ERR_DOMAIN; }
  if (pixels == GRAY_PIXELS_GRID || pixels == GRAY_PIXELS_POLAR) {
    if (nx <= 0 || ny <= 0) { set_error("nx, ny must be positive"); return GRAY_ERR_ARG; }
    if (p0 + st->n > (uint64_t)nx * (uint64_t)ny) { set_error("p0 + n = %llu exceeds nx * ny = %llu", (unsigned long long)(p0 + st->n), (unsigned long long)nx * ny); return GRAY_ERR_ARG; }
  }
  st->pixels = pixels;
  st->a = a; st->r_obs = r_obs; st->inc_deg = inc_deg; st->half_width = W;
  st->nx = pixels != GRAY_PIXELS_RANDOM ? nx : 0;
  st->ny = pixels != GRAY_PIXELS_RANDOM ? ny : 0;
  st->seed = seed; st->p0 = p0; st->r_lo = R_lo;
  if (st->n == 0) return GRAY_OK;
  InitArgs A;
  A.x = st->x_dev; A.k = st->k_dev; A.status = st->status_dev; A.steps = st->steps_dev;
  A.n = st->n; A.p0 = p0; A.seed = seed;
  A.a = a; A.r_obs = r_obs; A.W = W; A.R_lo = R_lo;
  const double inc = inc_deg * 3.14159265358979323846 / 180.0;
  A.sin_i = sin(inc); A.cos_i = cos(inc);
  A.nx = (unsigned long long)(nx > 0 ? nx : 1); A.ny = (unsigned long long)(ny > 0 ? ny : 1);
  const unsigned long long blocks = (st->n + 255) / 256;
  if (blocks > 0x7fffffffull) { set_error("n too large"); return GRAY_ERR_ARG; }
  const bool f32 = st->prec == GRAY_F32;
  if (pixels == GRAY_PIXELS_POLAR) {
    if (f32) init_kernel<float, GRAY_PIXELS_POLAR><<<(unsigned)blocks, 256, 0, stream>>>(A);
    else init_kernel<double, GRAY_PIXELS_POLAR><<<(unsigned)blocks, 256, 0, stream>>>(A);
  } else if (pixels == GRAY_PIXELS_GRID) {
    if (f32) init_kernel<float, GRAY_PIXELS_GRID><<<(unsigned)blocks, 256, 0, stream>>>(A);
    else init_kernel<double, GRAY_PIXELS_GRID><<<(unsigned)blocks, 256, 0, stream>>>(A);
  } else {
    if (f32) init_kernel<float, GRAY_PIXELS_RANDOM><<<(unsigned)blocks, 256, 0, stream>>>(A);
    else init_kernel<double, GRAY_PIXELS_RANDOM><<<(unsigned)blocks, 256, 0, stream>>>(A);
  }
  GRAY_CUDA(cudaGetLastError());
  return GRAY_OK;
}

}  // namespace gray

extern "C" {

int gray_init_rays(gray_state* state, double a, double r_obs, double inc_deg, double half_width,
                   int32_t nx, int32_t ny, uint64_t p0, void* cuda_stream) {
  return gray::init_common(state, a, r_obs, inc_deg, half_width, GRAY_PIXELS_GRID, nx, ny, 0, p0,
                           (cudaStream_t)cuda_stream);
}

int gray_init_rays_polar(gray_state* state, double a, double r_obs, double inc_deg, double R_lo, double R_hi,
                         int32_t n_R, int32_t n_theta, uint64_t p0, void* cuda_stream) {
  return gray::init_common(state, a, r_obs, inc_deg, R_hi, GRAY_PIXELS_POLAR, n_R, n_theta, 0, p0,
                           (cudaStream_t)cuda_stream, R_lo);
}

int gray_init_rays_random(gray_state* state, double a, double r_obs, double inc_deg, double half_width,
                          uint64_t seed, uint64_t p0, void* cuda_stream) {
  return gray::init_common(state, a, r_obs, inc_deg, half_width, GRAY_PIXELS_RANDOM, 0, 0, seed, p0,
                           (cudaStream_t)cuda_stream);
}

}  // extern "C"
