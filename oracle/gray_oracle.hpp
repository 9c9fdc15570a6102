// gray_oracle.hpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, scalar CPU statement of the GRay photon-geodesic hot path
// (Chan, Psaltis & Özel, arXiv 1303.5057; PAPER.md = P:<line>).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may use it.  It shares no code with paper_1303_5057_b200/csrc (the CUDA path)
// and is written the way the formulas are printed, in double precision, with no
// blocking, fusion or reordering, so it can be checked against the text by eye.
//
// Everything is templated on the scalar type T only so that the same lines can
// be run once with a counting scalar (the operation tally).
//
// Units G = c = M = 1.  State y[8] = (t, r, theta, phi, k^t, k^r, k^theta, k^phi).
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
//   metric + Christoffels : Ricci-flatness and metric compatibility by finite
//                           differences; a=0 -> Schwarzschild symbols
//   rhs                   : d/dlambda of E, L_z, Q, null norm = 0 to round-off
//   init                  : null, E=1, (xi,eta) -> Bardeen impact parameters
//   rk4 + step rule       : one step and a whole arc against an independent
//                           adaptive integrator (scipy DOP853) at 5th / 4th
//                           order under step halving; eq. (2) branch values
//   integrate             : sqrt(27) circle (a=0), quartic radial-potential
//                           classifier (Kerr), Schwarzschild deflection
//                           quadrature, reflection / spin-flip symmetries,
//                           the face-on critical radius next to P:91's value
//   pole treatment        : advance() with xi_eps > 0 (paper P:103-107): ONE step against
//                           y_old + (dl/9) rhs(y_old) / the RK4 result formed in numpy from
//                           the pinned rhs, step_size, metric (branch by xi from the metric;
//                           the 9 from the paper's text); whole rays next to the spin axis
//                           against the exact classifier
//   equatorial projection : a = 0 line of nodes and orbit integral (phi, r at the
//                           crossing to 2e-6); Kerr: invariants at the landed state,
//                           reflection symmetry
//   reduced system        : killing_velocities / rhs_reduced against the full rhs;
//                           classifiers; E, L_z to rounding; step halving
//   polar grid, ring stats: exact disc; Bardeen curve sampled on the same spokes;
//                           the paper's fits eqs. 11-14 (soft)
//   shadow statistics     : Bardeen closed-form curve (area, alpha extent, D,
//                           <R>, A), an exact synthetic disc, paper eqs. 11-14
//   Kerr rays off the equator: final (r, theta, phi) of CAPTURED and ESCAPED rays, and the equatorial
//                           crossing (r, phi) of stop_at_equator, against Carter's separated first-order
//                           equations in Mino time integrated by DOP853 (error falls 16x per step halving)
// Parity unpinned (GPU-vs-oracle only): which branch of the EQ2 step rule's min() individual steps of a
// whole trajectory take (the two branch values themselves are pinned by hand).
#pragma once
#include <cmath>
#include <cstdint>

namespace gray_oracle {

enum Status : int { LIVE = 0, CAPTURED = 1, ESCAPED = 2, BAD = 3, EQUATOR = 4 };
enum StepRule : int { STEP_REL = 0, STEP_EQ2 = 1 };
enum System : int { SYS_FULL = 0, SYS_REDUCED = 1 };

// ---------------------------------------------------------------- geometry
// Kerr metric in Boyer-Lindquist coordinates (the spacetime of P:75; r_bh there
// is r_h here).  g[mu][nu], index order (t, r, theta, phi).
template <class T>
void metric(T a, T r, T th, T g[4][4]) {
  T s = sin(th), c = cos(th);
  T Sigma = r * r + a * a * c * c;
  T Delta = r * r - T(2) * r + a * a;
  for (int m = 0; m < 4; ++m)
    for (int n = 0; n < 4; ++n) g[m][n] = T(0);
  g[0][0] = -(T(1) - T(2) * r / Sigma);
  g[0][3] = g[3][0] = -T(2) * a * r * s * s / Sigma;
  g[1][1] = Sigma / Delta;
  g[2][2] = Sigma;
  g[3][3] = (r * r + a * a + T(2) * a * a * r * s * s / Sigma) * s * s;
}

// Horizon radius r_bh = 1 + sqrt(1 - a^2).
template <class T>
T horizon(T a) { return T(1) + sqrt(T(1) - a * a); }

// The 20 independent non-zero Christoffel symbols of the Kerr metric
// ("equations (9)-(12)" of Psaltis & Johannsen 2012 are the geodesic
// equations built from these).  G[mu][al][be], symmetric in
// the lower pair; both orderings are filled in.
template <class T>
void christoffel(T a, T r, T th, T G[4][4][4]) {
  for (int m = 0; m < 4; ++m)
    for (int al = 0; al < 4; ++al)
      for (int be = 0; be < 4; ++be) G[m][al][be] = T(0);
  T s = sin(th), c = cos(th);
  T a2 = a * a, a3 = a2 * a, r2 = r * r, s2 = s * s, s3 = s2 * s, c2 = c * c;
  T Sigma = r2 + a2 * c2;
  T Delta = r2 - T(2) * r + a2;
  T P = r2 - a2 * c2;
  T rho = r2 + a2;
  T A = rho * rho - a2 * Delta * s2;
  T Sigma2 = Sigma * Sigma, Sigma3 = Sigma2 * Sigma;
  enum { t = 0, R = 1, h = 2, p = 3 };
  auto set = [&](int m, int al, int be, T v) { G[m][al][be] = v; G[m][be][al] = v; };
  set(t, t, R, rho * P / (Sigma2 * Delta));
  set(t, t, h, -T(2) * a2 * r * s * c / Sigma2);
  set(t, R, p, -a * s2 * (P * rho + T(2) * r2 * Sigma) / (Sigma2 * Delta));
  set(t, h, p, T(2) * a3 * r * s3 * c / Sigma2);
  set(R, t, t, Delta * P / Sigma3);
  set(R, t, p, -a * s2 * Delta * P / Sigma3);
  set(R, R, R, r / Sigma - (r - T(1)) / Delta);
  set(R, R, h, -a2 * s * c / Sigma);
  set(R, h, h, -r * Delta / Sigma);
  set(R, p, p, -Delta * s2 * (r * Sigma2 - a2 * s2 * P) / Sigma3);
  set(h, t, t, -T(2) * a2 * r * s * c / Sigma3);
  set(h, t, p, T(2) * a * r * rho * s * c / Sigma3);
  set(h, R, R, a2 * s * c / (Sigma * Delta));
  set(h, R, h, r / Sigma);
  set(h, h, h, -a2 * s * c / Sigma);
  set(h, p, p, -s * c * (A * Sigma + T(2) * a2 * r * s2 * rho) / Sigma3);
  set(p, t, R, a * P / (Sigma2 * Delta));
  set(p, t, h, -T(2) * a * r * c / (s * Sigma2));
  set(p, R, p, (r * Sigma * (Sigma - T(2) * r) - a2 * s2 * P) / (Sigma2 * Delta));
  set(p, h, p, (c / s) * (Sigma2 + T(2) * a2 * r * s2) / Sigma2);
}

// Right-hand side of the second-order geodesic equations written as a first
// order system ("the second-order geodesic equations are integrated";
// P:75): dx^mu/dlambda = k^mu, dk^mu/dlambda = -Gamma^mu_{al be} k^al k^be.
// Only the 20 non-zero symbols are touched, off-diagonal ones counted twice,
// the sub-expressions of christoffel() shared (this is the formulation whose
// operations the tally counts).
template <class T>
void rhs(T a, const T y[8], T dy[8]) {
  T r = y[1], th = y[2];
  T kt = y[4], kr = y[5], kh = y[6], kp = y[7];
  T s = sin(th), c = cos(th);
  T a2 = a * a, r2 = r * r, s2 = s * s, c2 = c * c, sc = s * c;
  T Sigma = r2 + a2 * c2;
  T Delta = r2 - T(2) * r + a2;
  T P = r2 - a2 * c2;
  T rho = r2 + a2;
  T A = rho * rho - a2 * Delta * s2;
  T iS = T(1) / Sigma, iD = T(1) / Delta, cot = c / s;
  T iS2 = iS * iS, iS3 = iS2 * iS;
  T Sigma2 = Sigma * Sigma;
  T a2sc = a2 * sc;
  T ar = a * r;

  T G_t_tr = rho * P * iS2 * iD;
  T G_t_th = -T(2) * a2sc * r * iS2;
  T G_t_rp = -a * s2 * (P * rho + T(2) * r2 * Sigma) * iS2 * iD;
  T G_t_hp = -a * s2 * G_t_th;                       // = 2 a^3 r s^3 c / Sigma^2
  T G_r_tt = Delta * P * iS3;
  T G_r_tp = -a * s2 * G_r_tt;
  T G_r_rr = r * iS - (r - T(1)) * iD;
  T G_r_rh = -a2sc * iS;
  T G_r_hh = -r * Delta * iS;
  T G_r_pp = -Delta * s2 * (r * Sigma2 - a2 * s2 * P) * iS3;
  T G_h_tt = -T(2) * a2sc * r * iS3;
  T G_h_tp = T(2) * ar * rho * sc * iS3;
  T G_h_rr = a2sc * iS * iD;
  T G_h_rh = r * iS;
  T G_h_hh = G_r_rh;                                 // = -a^2 s c / Sigma
  T G_h_pp = -sc * (A * Sigma + T(2) * a2 * r * s2 * rho) * iS3;
  T G_p_tr = a * P * iS2 * iD;
  T G_p_th = -T(2) * ar * cot * iS2;
  T G_p_rp = (r * Sigma * (Sigma - T(2) * r) - a2 * s2 * P) * iS2 * iD;
  T G_p_hp = cot * (Sigma2 + T(2) * a2 * r * s2) * iS2;

  dy[0] = kt; dy[1] = kr; dy[2] = kh; dy[3] = kp;
  dy[4] = -T(2) * (G_t_tr * kt * kr + G_t_th * kt * kh + G_t_rp * kr * kp + G_t_hp * kh * kp);
  dy[5] = -(G_r_tt * kt * kt + T(2) * G_r_tp * kt * kp + G_r_rr * kr * kr +
            T(2) * G_r_rh * kr * kh + G_r_hh * kh * kh + G_r_pp * kp * kp);
  dy[6] = -(G_h_tt * kt * kt + T(2) * G_h_tp * kt * kp + G_h_rr * kr * kr +
            T(2) * G_h_rh * kr * kh + G_h_hh * kh * kh + G_h_pp * kp * kp);
  dy[7] = -T(2) * (G_p_tr * kt * kr + G_p_th * kt * kh + G_p_rp * kr * kp + G_p_hp * kh * kp);
}

// Constants of motion and the null norm from a state.
// inv = { E = -k_t, L_z = k_phi, Q (Carter), null = g k k / (g_tt k^t k^t) }.
// The last one is the paper's xi + 1 (eq. 4).
template <class T>
void invariants(T a, const T y[8], T inv[4]) {
  T g[4][4];
  metric(a, y[1], y[2], g);
  T kt = y[4], kr = y[5], kh = y[6], kp = y[7];
  T E = -(g[0][0] * kt + g[0][3] * kp);
  T L = g[3][3] * kp + g[0][3] * kt;
  T kth_low = g[2][2] * kh;
  T s = sin(y[2]), c = cos(y[2]);
  T Q = kth_low * kth_low + c * c * (L * L / (s * s) - a * a * E * E);
  T norm = g[0][0] * kt * kt + T(2) * g[0][3] * kt * kp + g[1][1] * kr * kr +
           g[2][2] * kh * kh + g[3][3] * kp * kp;
  inv[0] = E; inv[1] = L; inv[2] = Q; inv[3] = norm / (g[0][0] * kt * kt);
}

// ------------------------------------------------------------ reduced system
// NEXT-3 of SURVEY §8(f) (R0, R21).  The notation of the paper's eqs. (2) and (4) (dt/dlambda' and
// dphi/dlambda' appear as velocities, the remap flips k_theta only) suggests that GRay itself integrates the system of
// Psaltis & Johannsen (2012) in which the two Killing constants E = -k_t and L_z = k_phi are used to ELIMINATE k^t
// and k^phi: t and phi obey first-order equations, r and theta second-order ones.  Written out from the metric:
//   k^t   = -g^tt E + g^tphi L,   k^phi = -g^tphi E + g^phiphi L          (inverse Kerr metric, textbook)
//         = (A E - 2 a r L) / (Sigma Delta),   (2 a r E + (Sigma - 2r) L / s^2) / (Sigma Delta),
//           A = (r^2 + a^2)^2 - a^2 Delta s^2
//   dr/dl = k^r, dtheta/dl = k^theta, and dk^r/dl, dk^theta/dl by the same Christoffel contraction as rhs(),
//   evaluated with those k^t, k^phi.
// State y6 = (t, r, theta, phi, k^r, k^theta); E and L are constants of the ray taken from its initial state.
template <class T>
void killing_velocities(T a, T E, T L, T r, T th, T* kt, T* kp) {
  T s = sin(th);
  T a2 = a * a, r2 = r * r, s2 = s * s;
  T c = cos(th);
  T Sigma = r2 + a2 * c * c;
  T Delta = r2 - T(2) * r + a2;
  T rho = r2 + a2;
  T A = rho * rho - a2 * Delta * s2;
  *kt = (A * E - T(2) * a * r * L) / (Sigma * Delta);
  *kp = (T(2) * a * r * E + (Sigma - T(2) * r) * L / s2) / (Sigma * Delta);
}

template <class T>
void rhs_reduced(T a, T E, T L, const T y6[6], T dy6[6]) {
  T y[8], dy[8];
  y[0] = y6[0]; y[1] = y6[1]; y[2] = y6[2]; y[3] = y6[3]; y[5] = y6[4]; y[6] = y6[5];
  killing_velocities(a, E, L, y6[1], y6[2], &y[4], &y[7]);
  rhs(a, y, dy);                        // dy[4], dy[7] (the equations that were eliminated) are not used
  dy6[0] = y[4]; dy6[1] = y[5]; dy6[2] = y[6]; dy6[3] = y[7]; dy6[4] = dy[5]; dy6[5] = dy[6];
}

// One classical RK4 step of the reduced system on the full 8-component state: E, L are taken from y (invariants()),
// the six evolving components are stepped, and k^t, k^phi of the result are rebuilt from the constants.
template <class T>
void rk4_step_reduced(T a, T E, T L, T y[8], T dl) {
  T y6[6] = {y[0], y[1], y[2], y[3], y[5], y[6]};
  T k1[6], k2[6], k3[6], k4[6], w[6];
  rhs_reduced(a, E, L, y6, k1);
  for (int i = 0; i < 6; ++i) w[i] = y6[i] + T(0.5) * dl * k1[i];
  rhs_reduced(a, E, L, w, k2);
  for (int i = 0; i < 6; ++i) w[i] = y6[i] + T(0.5) * dl * k2[i];
  rhs_reduced(a, E, L, w, k3);
  for (int i = 0; i < 6; ++i) w[i] = y6[i] + dl * k3[i];
  rhs_reduced(a, E, L, w, k4);
  for (int i = 0; i < 6; ++i) y6[i] = y6[i] + dl * (k1[i] + T(2) * k2[i] + T(2) * k3[i] + k4[i]) / T(6);
  y[0] = y6[0]; y[1] = y6[1]; y[2] = y6[2]; y[3] = y6[3]; y[5] = y6[4]; y[6] = y6[5];
  killing_velocities(a, E, L, y[1], y[2], &y[4], &y[7]);
}

// --------------------------------------------------------- image plane (O1-O3)
// Pixel centres of an nx x ny grid over [-W, W]^2; photon index p = row*nx+col,
// beta (row) slow.  ("grid spacing"; reading R1.)
inline void pixel_grid(double W, int64_t nx, int64_t ny, uint64_t p, double* alpha, double* beta) {
  uint64_t col = p % (uint64_t)nx, row = p / (uint64_t)nx;
  *alpha = -W + ((double)col + 0.5) * (2.0 * W / (double)nx);
  *beta = -W + ((double)row + 0.5) * (2.0 * W / (double)ny);
}

// Polar image-plane grid of the paper's photon-ring study ("a grid of 6000 x 181 rays in the polar
// domain (1.5, 7.5) x [0, pi]"; NEXT-4).  Reading (R20): the open radial interval is sampled at the n_R
// cell centres, the closed angular interval at n_theta equally spaced angles including both ends; photon index
// p = k n_R + j (angle slow); alpha = R cos(vartheta), beta = R sin(vartheta) (eqs. 9-10).
inline void pixel_polar(double R_lo, double R_hi, int64_t n_R, int64_t n_theta, uint64_t p, double* alpha, double* beta) {
  uint64_t j = p % (uint64_t)n_R, k = p / (uint64_t)n_R;
  double R = R_lo + ((double)j + 0.5) * ((R_hi - R_lo) / (double)n_R);
  double vt = (double)k * (3.14159265358979323846 / (double)(n_theta - 1));
  *alpha = R * cos(vt);
  *beta = R * sin(vt);
}

// Stateless counter-based pixel generator for the throughput workload (C4):
// a 64-bit mix of (seed, p); two 24-bit integers u, v from it; the pixel is the
// fp32 rounding of (2u + 1 - 2^24) W 2^-24.  (DESIGN.md input recipe.)
inline uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
inline void pixel_random(uint64_t seed, uint64_t p, double W, double* alpha, double* beta) {
  uint64_t z = mix64(mix64(seed) ^ p);
  int64_t u = (int64_t)(z >> 40);              // top 24 bits
  int64_t v = (int64_t)((z >> 16) & 0xFFFFFF); // next 24 bits
  double fa = (double)(2 * u + 1 - (1 << 24)) * W * (1.0 / 16777216.0);
  double fb = (double)(2 * v + 1 - (1 << 24)) * W * (1.0 / 16777216.0);
  *alpha = (double)(float)fa;
  *beta = (double)(float)fb;
}

// Image-plane point (alpha, beta) of an observer at (r_obs, inclination i) to the
// initial photon state ("initial conditions ... as in Psaltis & Johannsen
// (2012)", image plane at r = 1000 M; readings R2-R4):
//   pixel position  = r_obs o + alpha yhat + beta bhat,   o = (sin i, 0, cos i),
//                     bhat = (-cos i, 0, sin i)   (flat-space mapping)
//   photon momentum = along +o (it is travelling to the observer),
//   k^t             = positive root of g_mu_nu k^mu k^nu = 0,
//   then all four components divided by E = -k_t so that E = 1.
template <class T>
void init_ray(T a, T r_obs, T inc_rad, T alpha, T beta, T y[8]) {
  T si = sin(inc_rad), ci = cos(inc_rad);
  T x = r_obs * si - beta * ci;
  T yy = alpha;
  T z = r_obs * ci + beta * si;
  T r = sqrt(x * x + yy * yy + z * z);
  T q = sqrt(x * x + yy * yy);          // distance from the spin axis, r sin(theta)
  T th = atan2(q, z);                   // (not acos(z / r): near the axis acos loses half the digits; reading R23)
  T ph = atan2(yy, x);
  T s = sin(th), c = cos(th);
  T kr = r_obs / r;
  T kh = (si * c * cos(ph) - ci * s) / r;
  T kp = -si * sin(ph) / (r * s);
  // a pixel exactly on the spin axis (face-on observer, alpha = beta = 0) has no azimuth; the direction o is then
  // parallel to the axis and its theta and phi components vanish in the limit (reading R23)
  if (q == T(0)) { kh = T(0); kp = T(0); }
  T g[4][4];
  metric(a, r, th, g);
  // g_tt kt^2 + 2 g_tp kp kt + C = 0 with C the spatial part
  T C = g[1][1] * kr * kr + g[2][2] * kh * kh + g[3][3] * kp * kp;
  T B = g[0][3] * kp;
  T kt = (-B - sqrt(B * B - g[0][0] * C)) / g[0][0];   // g_tt < 0: the positive root
  T E = -(g[0][0] * kt + g[0][3] * kp);
  y[0] = T(0); y[1] = r; y[2] = th; y[3] = ph;
  y[4] = kt / E; y[5] = kr / E; y[6] = kh / E; y[7] = kp / E;
}

// ------------------------------------------------------------- stepping (O5-O7)
// Step size, evaluated at the start of a step and frozen over its four stages.
// Negative: the ray is traced backwards from the observer.
//   REL: dlambda = -h r                          (BASELINE.json configs)
//   EQ2: paper eq. (2), with its Delta := h and k normalised so E = 1:
//        dlambda = -min( h / (|k^r|/r + |k^theta| + |k^phi|),
//                        (r - r_h) / (2 |k^r|) )
template <class T>
T step_size(T a, const T y[8], T h, int rule) {
  T r = y[1];
  if (rule == STEP_REL) return -h * r;
  T d1 = h / (fabs(y[5]) / r + fabs(y[6]) + fabs(y[7]));
  T d2 = (r - horizon(a)) / (T(2) * fabs(y[5]));
  return -(d1 < d2 ? d1 : d2);
}

// One classical 4th-order Runge-Kutta step, stages at 0, 1/2, 1/2, 1,
// weights 1/6, 1/3, 1/3, 1/6, on all eight components.
template <class T>
void rk4_step(T a, T y[8], T dl) {
  T k1[8], k2[8], k3[8], k4[8], w[8];
  rhs(a, y, k1);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + T(0.5) * dl * k1[i];
  rhs(a, w, k2);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + T(0.5) * dl * k2[i];
  rhs(a, w, k3);
  for (int i = 0; i < 8; ++i) w[i] = y[i] + dl * k3[i];
  rhs(a, w, k4);
  for (int i = 0; i < 8; ++i)
    y[i] = y[i] + dl * (k1[i] + T(2) * k2[i] + T(2) * k3[i] + k4[i]) / T(6);
}

// theta-domain remap, paper eq. (3).
template <class T>
void remap_theta(T y[8]) {
  const T pi = T(3.14159265358979323846);
  if (y[2] > pi) { y[2] = T(2) * pi - y[2]; y[3] = y[3] + pi; y[6] = -y[6]; }
  else if (y[2] < T(0)) { y[2] = -y[2]; y[3] = y[3] - pi; y[6] = -y[6]; }
}

struct StepParams {
  double h;            // paper's Delta ~ 1/32
  double r_capture;    // captured when r <  r_capture  (1.01 r_h in the configs; r_h + delta in P:79)
  double r_escape;     // escaped  when r >  r_escape   (1.01 r_obs)
  int rule;            // StepRule
  double xi_eps = 0.0; // > 0: the paper's production pole treatment with epsilon = xi_eps, see integrate()
  int stop_at_equator = 0;  // != 0: the grid-projection workload, see equator_land()
  int system = SYS_FULL;    // SYS_REDUCED: see rhs_reduced()
  double E = 1.0, L = 0.0;  // SYS_REDUCED: constants of the ray being integrated (filled by integrate())
};

// Status of a state after a full step: non-finite -> BAD,
// r < r_capture -> CAPTURED, r > r_escape -> ESCAPED, else LIVE.
inline int classify_state(const double y[8], const StepParams& sp) {
  for (int i = 0; i < 8; ++i)
    if (!std::isfinite(y[i])) return BAD;
  if (y[1] < sp.r_capture) return CAPTURED;
  if (y[1] > sp.r_escape) return ESCAPED;
  return LIVE;
}

// The paper's production pole treatment (NEXT-1 of SURVEY §8(f)): "monitor the quantity xi [eq. 4]
// which should always remain equal to -1.  If |xi + 1| > epsilon, for some small parameter epsilon ~ 1e-3 ...
// we re-integrate the inaccurate step by falling back to the 1st-order forward Euler scheme with a smaller
// time step dlambda'/9".  xi + 1 is invariants()[3] (the null norm over g_tt (k^t)^2).  Reading (R18):
// the test is applied to the state an RK4 step produced; on failure that step is discarded and replaced by ONE
// forward Euler step of dlambda/9 from the state before it, which is not tested itself; a non-finite xi fails
// the test.  One step (RK4 or its Euler replacement) counts as one step.
inline void advance(double a, double y[8], const StepParams& sp, const double* forced_dl = nullptr) {
  double dl = forced_dl ? *forced_dl : step_size(a, y, sp.h, sp.rule);
  if (sp.system == SYS_REDUCED) {         // E, L of the ray: carried by the caller in sp_E, sp_L (set by integrate())
    rk4_step_reduced(a, sp.E, sp.L, y, dl);
    return;
  }
  if (!(sp.xi_eps > 0.0)) { rk4_step(a, y, dl); return; }
  double y_old[8], inv[4];
  for (int i = 0; i < 8; ++i) y_old[i] = y[i];
  rk4_step(a, y, dl);
  invariants(a, y, inv);
  if (!(fabs(inv[3]) <= sp.xi_eps)) {
    double f[8];
    rhs(a, y_old, f);
    for (int i = 0; i < 8; ++i) y[i] = y_old[i] + (dl / 9.0) * f[i];
  }
}

// The paper's first benchmark (Fig. 3; NEXT-2 of SURVEY §8(f)): project the image-plane grid
// onto the equatorial plane, i.e. follow each ray until it first reaches theta = pi/2.  Reading (R19):
// a step crosses the plane if its start lies on one side (theta <= pi/2 counts as the upper side) and its end
// strictly on the other.  The ray is then landed on the plane with two Newton iterations, each an ordinary step
// (same scheme, counted like any step) whose size is dlambda = -(theta - pi/2) / k^theta instead of the step
// rule; the state after the second one is the result (theta within ~1e-9 of pi/2, all eight components fourth
// order accurate).  During the landing the termination tests are not applied.
inline bool equator_crossed(double th_old, const double y[8]) {
  const double half_pi = 1.57079632679489661923;
  return th_old <= half_pi ? (y[2] > half_pi) : (y[2] < half_pi);
}
inline void equator_land(double a, double y[8], const StepParams& sp, uint32_t* steps) {
  const double half_pi = 1.57079632679489661923;
  for (int it = 0; it < 2; ++it) {
    double dl = -(y[2] - half_pi) / y[6];
    advance(a, y, sp, &dl);
    ++*steps;
  }
}

// Integrate one ray until it is captured, escapes, goes non-finite, (optionally) reaches the equatorial plane,
// or has taken max_steps steps in total.  Test order: BAD, CAPTURED, EQUATOR, ESCAPED.  *steps is the running
// step counter (in/out), so a call can resume an earlier one.  If force_steps >= 0 the tests are ignored and
// exactly that many further steps are taken (the equal-step-count protocol, reading R11); the
// returned status is then that of the last state.
inline int integrate(double a, double y[8], const StepParams& sp_in, uint32_t max_steps,
                     int64_t force_steps, uint32_t* steps) {
  StepParams sp = sp_in;
  if (sp.system == SYS_REDUCED) {
    double inv[4];
    invariants(a, y, inv);
    sp.E = inv[0]; sp.L = inv[1];
  }
  if (force_steps >= 0) {
    for (int64_t n = 0; n < force_steps; ++n) {
      advance(a, y, sp);
      remap_theta(y);
      ++*steps;
    }
    return classify_state(y, sp);
  }
  int st = LIVE;
  while (*steps < max_steps) {
    double th_old = y[2];
    advance(a, y, sp);
    remap_theta(y);
    ++*steps;
    st = classify_state(y, sp);
    if (sp.stop_at_equator && (st == LIVE || st == ESCAPED) && equator_crossed(th_old, y)) {
      equator_land(a, y, sp, steps);
      st = classify_state(y, sp) == BAD ? BAD : EQUATOR;
    }
    if (st != LIVE) break;
  }
  return st;
}

}  // namespace gray_oracle
