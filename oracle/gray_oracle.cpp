// gray_oracle.cpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE (see gray_oracle.hpp).
//
// C entry points (ctypes) around the templates of gray_oracle.hpp: single-call
// probes used by the pins, a batch tracer that splits rays statically across
// std::threads (the timed CPU baseline), the shadow statistics of paper eqs.
// (6)-(8), and the operation tally.  Build: python oracle/build.py
#include "gray_oracle.hpp"

#include <algorithm>
#include <cstring>
#include <thread>
#include <vector>

namespace go = gray_oracle;

// ------------------------------------------------------------ counting scalar
// A double that counts the floating-point operations applied to it, for the
// per-photon-step operation tally.  add/sub = 1 each,
// mul = 1, div = 1, sqrt/sin/cos = 1 each; negation, fabs, comparisons and
// copies are recorded separately and not counted as flops.
namespace gray_oracle {
struct Tally { uint64_t add = 0, mul = 0, div = 0, sqrt_ = 0, sin_ = 0, cos_ = 0, other = 0; };
static thread_local Tally g_tally;
struct Counted {
  double v;
  Counted() : v(0) {}
  Counted(double x) : v(x) {}
  Counted(int x) : v(x) {}
};
inline Counted operator+(Counted a, Counted b) { ++g_tally.add; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { ++g_tally.add; return Counted(a.v - b.v); }
inline Counted operator*(Counted a, Counted b) { ++g_tally.mul; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { ++g_tally.div; return Counted(a.v / b.v); }
inline Counted operator-(Counted a) { ++g_tally.other; return Counted(-a.v); }
inline bool operator<(Counted a, Counted b) { ++g_tally.other; return a.v < b.v; }
inline bool operator>(Counted a, Counted b) { ++g_tally.other; return a.v > b.v; }
inline Counted sin(Counted a) { ++g_tally.sin_; return Counted(std::sin(a.v)); }
inline Counted cos(Counted a) { ++g_tally.cos_; return Counted(std::cos(a.v)); }
inline Counted sqrt(Counted a) { ++g_tally.sqrt_; return Counted(std::sqrt(a.v)); }
inline Counted fabs(Counted a) { ++g_tally.other; return Counted(std::fabs(a.v)); }
}  // namespace gray_oracle

static const double kPi = 3.14159265358979323846;

extern "C" {

double gray_oracle_horizon(double a) { return go::horizon(a); }

void gray_oracle_metric(double a, double r, double th, double* g16) {
  double g[4][4];
  go::metric(a, r, th, g);
  std::memcpy(g16, g, sizeof g);
}

void gray_oracle_christoffel(double a, double r, double th, double* G64) {
  double G[4][4][4];
  go::christoffel(a, r, th, G);
  std::memcpy(G64, G, sizeof G);
}

void gray_oracle_rhs(double a, const double* y, double* dy) { go::rhs(a, y, dy); }

void gray_oracle_rhs_reduced(double a, double E, double L, const double* y6, double* dy6) {
  go::rhs_reduced(a, E, L, y6, dy6);
}

void gray_oracle_killing_velocities(double a, double E, double L, double r, double th, double* kt, double* kp) {
  go::killing_velocities(a, E, L, r, th, kt, kp);
}

void gray_oracle_invariants(double a, const double* y, double* inv4) { go::invariants(a, y, inv4); }

void gray_oracle_pixel_grid(double W, int64_t nx, int64_t ny, uint64_t p, double* alpha, double* beta) {
  go::pixel_grid(W, nx, ny, p, alpha, beta);
}

void gray_oracle_pixel_polar(double R_lo, double R_hi, int64_t n_R, int64_t n_theta, uint64_t p, double* alpha,
                             double* beta) {
  go::pixel_polar(R_lo, R_hi, n_R, n_theta, p, alpha, beta);
}

void gray_oracle_pixel_random(uint64_t seed, uint64_t p, double W, double* alpha, double* beta) {
  go::pixel_random(seed, p, W, alpha, beta);
}

void gray_oracle_init_ray(double a, double r_obs, double inc_deg, double alpha, double beta, double* y) {
  go::init_ray(a, r_obs, inc_deg * kPi / 180.0, alpha, beta, y);
}

double gray_oracle_step_size(double a, const double* y, double h, int rule) {
  return go::step_size(a, y, h, rule);
}

void gray_oracle_rk4_step(double a, double* y, double dl) { go::rk4_step(a, y, dl); }

void gray_oracle_remap_theta(double* y) { go::remap_theta(y); }

// Integrate one ray from state y (in/out).  See gray_oracle::integrate.
int gray_oracle_integrate(double a, double* y, double h, double r_capture, double r_escape, int rule,
                          uint32_t max_steps, int64_t force_steps, uint32_t* steps, double xi_eps,
                          int stop_at_equator, int system) {
  go::StepParams sp{h, r_capture, r_escape, rule, xi_eps, stop_at_equator, system};
  return go::integrate(a, y, sp, max_steps, force_steps, steps);
}

// Trace a batch: initialise (O1-O3) and integrate (O5-O7) the photons whose
// indices are idx[0..n_idx) (idx == NULL: photons 0..n_idx-1).
//   nx > 0  : grid workload, nx x ny pixel centres over [-W, W]^2
//   nx == 0 : random workload keyed by (seed, photon index)
//   nx < 0  : polar grid of -nx radii in (polar_R_lo, W) x ny angles in [0, pi] (gray_oracle::pixel_polar)
//   capture radius = cap_factor * r_h if cap_factor > 0, else r_h + horizon_delta
//   init_f32 != 0 : the initial state is rounded to fp32 before integrating (what
//                   the fp32 build stores; the integration itself stays double)
//   force_steps   : NULL, or per ray a step count to take regardless of the tests
//                   (< 0: normal termination)
//   xi_eps > 0    : the paper's pole treatment (gray_oracle::advance)
//   stop_at_equator: the grid-projection workload (gray_oracle::equator_land)
// Outputs (any may be NULL): y0 (n x 8), y (n x 8), status (n), steps (n).
// Rays are split statically and contiguously across n_threads std::threads.
int gray_oracle_trace(double a, double r_obs, double inc_deg, double W, int64_t nx, int64_t ny,
                      uint64_t seed, const uint64_t* idx, uint64_t n_idx, double h, double cap_factor,
                      double esc_factor, double horizon_delta, int rule, uint32_t max_steps,
                      int init_f32, const int64_t* force_steps, int n_threads, double* y0_out,
                      double* y_out, int32_t* status_out, uint32_t* steps_out, double xi_eps, int stop_at_equator,
                      double polar_R_lo, int system) {
  if (n_threads < 1) n_threads = 1;
  double rh = go::horizon(a);
  go::StepParams sp{h, cap_factor > 0 ? cap_factor * rh : rh + horizon_delta, esc_factor * r_obs, rule, xi_eps,
                    stop_at_equator, system};
  double inc = inc_deg * kPi / 180.0;
  auto work = [&](uint64_t lo, uint64_t hi) {
    for (uint64_t j = lo; j < hi; ++j) {
      uint64_t p = idx ? idx[j] : j;
      double al, be, y[8];
      if (nx < 0) go::pixel_polar(polar_R_lo, W, -nx, ny, p, &al, &be);
      else if (nx > 0) go::pixel_grid(W, nx, ny, p, &al, &be);
      else go::pixel_random(seed, p, W, &al, &be);
      go::init_ray(a, r_obs, inc, al, be, y);
      if (init_f32)
        for (int i = 0; i < 8; ++i) y[i] = (double)(float)y[i];
      if (y0_out) std::memcpy(y0_out + 8 * j, y, sizeof y);
      uint32_t steps = 0;
      int st = go::integrate(a, y, sp, max_steps, force_steps ? force_steps[j] : -1, &steps);
      if (y_out) std::memcpy(y_out + 8 * j, y, sizeof y);
      if (status_out) status_out[j] = st;
      if (steps_out) steps_out[j] = steps;
    }
  };
  if (n_threads == 1) { work(0, n_idx); return 0; }
  std::vector<std::thread> pool;
  for (int t = 0; t < n_threads; ++t) {
    uint64_t lo = n_idx * (uint64_t)t / (uint64_t)n_threads;
    uint64_t hi = n_idx * (uint64_t)(t + 1) / (uint64_t)n_threads;
    pool.emplace_back(work, lo, hi);
  }
  for (auto& th : pool) th.join();
  return 0;
}

int gray_oracle_hardware_threads(void) { return (int)std::thread::hardware_concurrency(); }

// Shadow statistics from a capture map (paper eqs. 6-8,
// P:176-193).  captured[row*nx+col] != 0 marks a captured pixel of the nx x ny
// grid over [-W, W]^2.
//   out[0] area         = N_captured * dalpha * dbeta
//   out[1], out[2]      = mean (alpha, beta) of captured pixel centres
//   out[3], out[4]      = alpha_min, alpha_max: outer edges of the extreme captured columns
//   out[5] D            = |alpha_min + alpha_max| / 2                     (eq. 6)
//   out[6] <R>, out[7] A: over n_angles spokes about the image origin at
//                         vartheta_k = 2 pi (k + 1/2) / n_angles, R measured from
//                         ((alpha_min + alpha_max)/2, 0)                  (eqs. 7-8)
//   out[8]              = number of captured pixels
//   radius[k]           = rho(vartheta_k): marching outwards in steps of half a pixel,
//                         the mid-point between the last sample whose nearest pixel is
//                         captured and the first whose nearest pixel is not (0 if the
//                         origin pixel is not captured; the image edge if never left).
void gray_oracle_shadow_stats(const uint8_t* captured, int64_t nx, int64_t ny, double W,
                              int32_t n_angles, double* radius, double* out) {
  double da = 2.0 * W / (double)nx, db = 2.0 * W / (double)ny;
  uint64_t ncap = 0;
  double sa = 0, sb = 0;
  int64_t cmin = nx, cmax = -1;
  for (int64_t row = 0; row < ny; ++row)
    for (int64_t col = 0; col < nx; ++col)
      if (captured[row * nx + col]) {
        ++ncap;
        sa += -W + ((double)col + 0.5) * da;
        sb += -W + ((double)row + 0.5) * db;
        cmin = std::min(cmin, col);
        cmax = std::max(cmax, col);
      }
  out[8] = (double)ncap;
  out[0] = (double)ncap * da * db;
  out[1] = ncap ? sa / (double)ncap : 0.0;
  out[2] = ncap ? sb / (double)ncap : 0.0;
  double amin = ncap ? -W + (double)cmin * da : 0.0;
  double amax = ncap ? -W + (double)(cmax + 1) * da : 0.0;
  out[3] = amin; out[4] = amax;
  out[5] = std::fabs(amin + amax) / 2.0;
  double centre = (amin + amax) / 2.0;
  double delta = std::min(da, db) / 2.0;
  std::vector<double> R(n_angles > 0 ? n_angles : 0);
  for (int32_t k = 0; k < n_angles; ++k) {
    double vt = 2.0 * kPi * ((double)k + 0.5) / (double)n_angles;
    double cv = std::cos(vt), sv = std::sin(vt);
    double rho = 0.0;
    for (int64_t j = 0;; ++j) {
      double q = (double)j * delta;
      int64_t col = (int64_t)std::floor((q * cv + W) / da);
      int64_t row = (int64_t)std::floor((q * sv + W) / db);
      bool inside = col >= 0 && col < nx && row >= 0 && row < ny;
      if (!inside) { rho = ((double)j - 0.5) * delta; break; }
      if (!captured[row * nx + col]) { rho = j == 0 ? 0.0 : ((double)j - 0.5) * delta; break; }
    }
    if (radius) radius[k] = rho;
    double x = rho * cv - centre, yv = rho * sv;
    R[k] = std::sqrt(x * x + yv * yv);
  }
  double mean = 0;
  for (double v : R) mean += v;
  mean = n_angles > 0 ? mean / n_angles : 0.0;
  double var = 0;
  for (double v : R) var += (v - mean) * (v - mean);
  var = n_angles > 0 ? var / n_angles : 0.0;
  out[6] = mean;
  out[7] = 2.0 * std::sqrt(var);
}

// Photon-ring statistics on the paper's polar grid (eqs. 6-10; NEXT-4).  captured[k*n_R+j] != 0 marks a
// captured ray at angle vartheta_k = k pi / (n_theta - 1), radius cell j of (R_lo, R_hi).
//   radius[k] = ring radius on spoke k: the outer edge of the outermost captured cell (R_lo if none is captured).
//               Scanning from the outside keeps the outline insensitive to a stray non-captured ray inside the
//               shadow (the axis spoke vartheta = pi/2 of the paper's grid has alpha = 0: its rays run through the
//               pole exactly, the degenerate case of Boyer-Lindquist coordinates, R20)
//   out[0], out[1] = alpha_min = -radius[n_theta-1], alpha_max = radius[0]  (the ring meets the alpha axis there)
//   out[2] D (eq. 6); with R = [(alpha_0 - c)^2 + beta_0^2]^(1/2) about the ring centre c = (alpha_min + alpha_max)/2
//   out[3] <R> (eq. 7), out[4] A (eq. 8): the integrals over [0, 2 pi] are twice those over [0, pi] (the image is
//   symmetric under beta -> -beta), evaluated by the trapezoidal rule on the n_theta angles.
//   bridge_axis != 0 (n_theta odd): the radius of the middle spoke vartheta = pi/2 is replaced by the mean of its two
//               neighbours before anything else is computed (and returned so in radius[]).
void gray_oracle_ring_polar(const uint8_t* captured, int64_t n_R, int64_t n_theta, double R_lo, double R_hi,
                            int bridge_axis, double* radius, double* out) {
  double dR = (R_hi - R_lo) / (double)n_R;
  std::vector<double> rad(n_theta), R(n_theta);
  for (int64_t k = 0; k < n_theta; ++k) {
    int64_t j = n_R;
    while (j > 0 && !captured[k * n_R + j - 1]) --j;
    rad[k] = R_lo + (double)j * dR;
  }
  if (bridge_axis && n_theta >= 3 && (n_theta % 2) == 1) {
    int64_t m = (n_theta - 1) / 2;
    rad[m] = 0.5 * (rad[m - 1] + rad[m + 1]);
  }
  if (radius)
    for (int64_t k = 0; k < n_theta; ++k) radius[k] = rad[k];
  double amax = rad[0], amin = -rad[n_theta - 1];
  double c = (amin + amax) / 2.0;
  for (int64_t k = 0; k < n_theta; ++k) {
    double vt = (double)k * (kPi / (double)(n_theta - 1));
    double x = rad[k] * std::cos(vt) - c, y = rad[k] * std::sin(vt);
    R[k] = std::sqrt(x * x + y * y);
  }
  auto trapz_mean = [&](const std::vector<double>& f) {
    double sum = 0;
    for (int64_t k = 0; k < n_theta; ++k) sum += (k == 0 || k == n_theta - 1 ? 0.5 : 1.0) * f[k];
    return sum / (double)(n_theta - 1);
  };
  double mean = trapz_mean(R);
  std::vector<double> dev(n_theta);
  for (int64_t k = 0; k < n_theta; ++k) dev[k] = (R[k] - mean) * (R[k] - mean);
  out[0] = amin; out[1] = amax; out[2] = std::fabs(amin + amax) / 2.0; out[3] = mean;
  out[4] = 2.0 * std::sqrt(trapz_mean(dev));
}

// Operation tally of one photon-step (step size + RK4 step + remap) at state y.
// counts = { add/sub, mul, div, sqrt, sin, cos, other(neg, fabs, compare) }.
void gray_oracle_op_tally(double a, const double* y, double h, int rule, uint64_t* counts7) {
  using go::Counted;
  Counted yc[8];
  for (int i = 0; i < 8; ++i) yc[i] = Counted(y[i]);
  go::g_tally = go::Tally();
  Counted dl = go::step_size(Counted(a), yc, Counted(h), rule);
  go::rk4_step(Counted(a), yc, dl);
  go::remap_theta(yc);
  const go::Tally& t = go::g_tally;
  counts7[0] = t.add; counts7[1] = t.mul; counts7[2] = t.div; counts7[3] = t.sqrt_;
  counts7[4] = t.sin_; counts7[5] = t.cos_; counts7[6] = t.other;
}

// The same tally for either system (0 = full as above, 1 = reduced: step size + rk4_step_reduced, whose four stages and
// final state each rebuild k^t, k^phi with killing_velocities, + remap).  E and L of the ray are formed once per ray
// (integrate()), not per step, and are not counted.  Bookkeeping only: no arithmetic of the method changes.
void gray_oracle_op_tally_system(double a, const double* y, double h, int rule, int system, uint64_t* counts7) {
  using go::Counted;
  if (system != go::SYS_REDUCED) { gray_oracle_op_tally(a, y, h, rule, counts7); return; }
  double inv[4];
  go::invariants(a, y, inv);
  Counted yc[8];
  for (int i = 0; i < 8; ++i) yc[i] = Counted(y[i]);
  go::g_tally = go::Tally();
  Counted dl = go::step_size(Counted(a), yc, Counted(h), rule);
  go::rk4_step_reduced(Counted(a), Counted(inv[0]), Counted(inv[1]), yc, dl);
  go::remap_theta(yc);
  const go::Tally& t = go::g_tally;
  counts7[0] = t.add; counts7[1] = t.mul; counts7[2] = t.div; counts7[3] = t.sqrt_;
  counts7[4] = t.sin_; counts7[5] = t.cos_; counts7[6] = t.other;
}

}  // extern "C"
