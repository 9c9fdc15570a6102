// gray_integrate.cu — the integrator kernel of libgray and gray_integrate() (include/gray.h).
//
// One photon per lane of a vector type V (gray_vec.cuh): float / double = one photon per thread, f2 = two
// fp32 photons per thread in packed FFMA2 / FMUL2 / FADD2 instructions.  A photon's 8-component state
// stays in registers from the moment it is loaded until it terminates ("GRay integrates each geodesic
// for many steps in a single data load", P:81 fn 5).  What differs from the paper's fixed grid of
// 64-thread blocks: the kernel is persistent (148 SMs x resident blocks) and a lane whose
// photon has terminated is refilled from a device-side queue, so a warp never idles on its slowest
// ray; HBM is touched once per photon on load and once on retirement, with 16-byte vector accesses.
#include "gray_internal.h"
#include "gray_math.cuh"

namespace gray {

template <typename S> struct Vec4T;
template <> struct Vec4T<float> { using type = float4; };
template <> struct Vec4T<double> { using type = double4; };

// Resume records (gray_state.resume_dev, gray.h): integers and bit patterns travel in scalar slots of the batch's
// precision; they are only loaded, stored and compared, never computed with.
__device__ __forceinline__ float bits_to_scalar(unsigned long long b, float) { return __uint_as_float((unsigned int)b); }
__device__ __forceinline__ double bits_to_scalar(unsigned long long b, double) { return __longlong_as_double((long long)b); }
__device__ __forceinline__ unsigned long long scalar_bits(float v) { return __float_as_uint(v); }
__device__ __forceinline__ unsigned long long scalar_bits(double v) { return (unsigned long long)__double_as_longlong(v); }
constexpr unsigned long long kResumeMagic = 0x47524159ull;       // "GRAY"
// Key word of a resume record: the magic mixed with the bits of the four stored k^mu and with the system (full / reduced)
// that wrote the record, in the width of the scalar.  A record is only taken back by a call that finds the very k it was
// written next to and integrates the same system: a caller who edits k (say, reverses a ray), or who switches
// GRAY_SYS_FULL <-> GRAY_SYS_REDUCED between calls, gets the photon rebuilt from (x, k) instead of stale compensation
// terms or stale constants E, L.
__device__ __forceinline__ unsigned long long resume_key(float kt, float kr, float kh, float kp, bool red) {
  unsigned int h = (unsigned int)kResumeMagic ^ (red ? 0x52454455u : 0u);      // "REDU"
  const unsigned int w[4] = {__float_as_uint(kt), __float_as_uint(kr), __float_as_uint(kh), __float_as_uint(kp)};
#pragma unroll
  for (int i = 0; i < 4; ++i) { h = (h ^ w[i]) * 0x9e3779b1u; h ^= h >> 15; }
  return h;
}
__device__ __forceinline__ unsigned long long resume_key(double kt, double kr, double kh, double kp, bool red) {
  unsigned long long h = kResumeMagic ^ (red ? 0x5245445500000000ull : 0ull);
  const unsigned long long w[4] = {scalar_bits(kt), scalar_bits(kr), scalar_bits(kh), scalar_bits(kp)};
#pragma unroll
  for (int i = 0; i < 4; ++i) { h = (h ^ w[i]) * 0xff51afd7ed558ccdull; h ^= h >> 33; }
  return h;
}

template <typename V>
struct IntegrateArgs {
  using S = typename VT<V>::S;
  typename Vec4T<S>::type* x;
  typename Vec4T<S>::type* k;
  uint8_t* status;
  uint32_t* steps;
  typename Vec4T<S>::type* resume;   // gray_state.resume_dev: 4 vectors per photon, or NULL
  unsigned long long n;
  uint32_t max_steps;
  int refill_interval;
  int stop_eq;               // gray_step_params.stop_at_equator
  int reduced;               // gray_step_params.system == GRAY_SYS_REDUCED
  Workspace* ws;
  Consts<V> K;
};

#ifndef GRAY_BLOCK
#define GRAY_BLOCK 128
#endif
#ifndef GRAY_STEP_UNROLL
#define GRAY_STEP_UNROLL 2     // RK4 steps per trip of the inner loop of the full-system kernels (refill_interval is rounded up to a
                               // multiple)
#endif
#ifndef GRAY_F2_MIN_BLOCKS
#define GRAY_F2_MIN_BLOCKS 4
#endif
constexpr int kBlock = GRAY_BLOCK;
template <typename V> struct Tune;
template <> struct Tune<float> { static constexpr int min_blocks = 4; };    // <= 128 registers/thread
template <> struct Tune<f2> { static constexpr int min_blocks = GRAY_F2_MIN_BLOCKS; };   // 4 x 128 threads: <= 128 registers/thread
#ifndef GRAY_F64_MIN_BLOCKS
#define GRAY_F64_MIN_BLOCKS 4
#endif
// 4 x 128 threads: <= 128 registers/thread, no spills; measured 3.81e10 photon-steps/s against 3.75e10 with 3 blocks (the
// compiler's own choice of 142 registers) and 3.71e10 with 5
template <> struct Tune<double> { static constexpr int min_blocks = GRAY_F64_MIN_BLOCKS; };

__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <typename V, int RULE, int SCHED, bool FROZEN, bool XI, bool EQ, bool RED>
__global__ void __launch_bounds__(kBlock, Tune<V>::min_blocks)
integrate_kernel(const __grid_constant__ IntegrateArgs<V> A) {
  using S = typename VT<V>::S;
  constexpr int N = VT<V>::N;
  constexpr unsigned FULL = 0xffffffffu;
  // RK4 steps per trip of the inner loop.  Measured on B200: pairs help the full system (+1.3 % fp32, +0.8 % with the xi
  // monitor, +0.3 % fp64) and cost the reduced system (-8 %) and the frozen peak-rate kernel (-1.5 %)
  constexpr int UN = (FROZEN || RED) ? 1 : GRAY_STEP_UNROLL;
  const int lane = threadIdx.x & 31;
  const Consts<V>& K = A.K;

  V y[8], comp[8];
  int mirrored[N];
  unsigned long long idx[N];
  uint32_t nst[N], nst0[N], iss[N];
  int fstat[N];
  int landing[N];            // stop_at_equator: 0 = cruising, 1 / 2 = before the first / second Newton step onto the plane
  bool lnd = false;          // any slot of this thread landing
  bool have[N];
  // Which sine / cosine the first stage of a step uses (gray_math.cuh rk4_step FOLD) is a function of the step rule and
  // of stop_at_equator only, so that every kernel variant of a rule does the same arithmetic per photon: under eq. (2)
  // without landing steps the folded polynomial always (1); otherwise (REL steps are not bounded in theta, landing steps
  // sit beyond pi/2) the polynomial for every photon within its range, photon by photon (2; float builds).
  constexpr int FOLD = (RULE == GRAY_STEP_EQ2 && !EQ) ? 1 : (sizeof(S) == 4 ? 2 : 0);
  bool fold_ok = false;      // FOLD == 2: every photon this thread is advancing within the folded polynomial's range?
  auto fold_check = [&](const bool use[N]) {
    if (FOLD != 2) return;
    S th[N];
    vunpack(y[2], th);
    fold_ok = true;
#pragma unroll
    for (int l = 0; l < N; ++l) fold_ok &= !use[l] || (th[l] >= fold_lo<S>() && th[l] <= fold_hi<S>());
  };
  bool exhausted = (SCHED == GRAY_SCHED_STATIC);
  unsigned long long c_steps = 0;
  unsigned int c_done = 0, c_live = 0, c_iter = 0, c_fallback = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) { y[i] = K.one; comp[i] = K.zero; }
#pragma unroll
  for (int l = 0; l < N; ++l) { have[l] = false; landing[l] = 0; mirrored[l] = 0; idx[l] = 0; nst[l] = nst0[l] = iss[l] = 0; fstat[l] = GRAY_LIVE; }

  // HBM -> registers: photon want[l] into slot l (for the slots with want[l] < n), if it is live and has steps
  // left.  (t, r, theta, phi), k^mu -> the kernel's variables (gray_math.cuh): d = r - r_+ and theta folded into
  // [0, pi/2].  The state is taken apart into scalars, the slots are filled under their own conditions, and it is
  // put together again unconditionally: a packed value is never half-updated inside a branch.
  auto take = [&](const unsigned long long want[N]) {
    S ys[8][N], cs[8][N];
#pragma unroll
    for (int i = 0; i < 8; ++i) { vunpack(y[i], ys[i]); vunpack(comp[i], cs[i]); }
#pragma unroll
    for (int l = 0; l < N; ++l) {
      const unsigned long long p = want[l];
      if (p >= A.n) continue;
      const uint8_t st = A.status[p];
      const uint32_t s = A.steps[p];
      if (st != GRAY_LIVE) continue;
      if (s >= A.max_steps) { ++c_live; continue; }
      const typename Vec4T<S>::type xv = A.x[p], kv = A.k[p];
      S th = xv.z, kh = kv.z, ph = xv.w;
      int m = 0;
      {
        // eq. (3) first (a state uploaded by the caller may carry a polar angle outside [0, pi]; one stored by this
        // library never does), then the fold into [0, pi/2]: the first-stage sine / cosine is fitted on the folded range
        S unused0 = S(0), unused1 = S(0);
        remap_theta(th, ph, kh, unused0, unused1, m, true);
      }
      ys[0][l] = xv.x; ys[1][l] = xv.y - vget(K.rp, 0); ys[2][l] = th; ys[3][l] = ph;
      ys[4][l] = kv.x; ys[5][l] = kv.y; ys[6][l] = kh; ys[7][l] = kv.w;
#pragma unroll
      for (int i = 0; i < 8; ++i) cs[i][l] = S(0);
      // A photon left LIVE by an earlier call that wrote a resume record (gray.h): if the record belongs to exactly
      // this stored state (same r, theta bits, same step count, same k and same system through resume_key), the
      // kernel's own variables - d, the folded theta, the compensation terms, E and L of the reduced system - are
      // taken from it, and the continuation is bit-identical to an uninterrupted run.  Otherwise they are rebuilt
      // from (x, k) as above.
      bool resumed = false;
      if (A.resume != nullptr) {
        const typename Vec4T<S>::type r3 = A.resume[4 * p + 3];
        if (scalar_bits(r3.x) == scalar_bits(xv.y) && scalar_bits(r3.y) == scalar_bits(xv.z) &&
            scalar_bits(r3.z) == (unsigned long long)s && scalar_bits(r3.w) == resume_key(kv.x, kv.y, kv.z, kv.w, RED)) {
          const typename Vec4T<S>::type r0 = A.resume[4 * p], r1 = A.resume[4 * p + 1], r2 = A.resume[4 * p + 2];
          const unsigned long long flags = scalar_bits(r2.w);
          m = (int)(flags & 1ull);
          ys[1][l] = r0.x; ys[2][l] = r0.y;
          ys[6][l] = m ? sneg(kv.z) : kv.z;
          cs[1][l] = r1.x; cs[2][l] = r1.y; cs[3][l] = r1.z; cs[4][l] = r1.w;
          cs[5][l] = r2.x; cs[6][l] = r2.y; cs[7][l] = r2.z;
          if (RED) { ys[4][l] = r0.z; ys[7][l] = r0.w; }
          resumed = true;
        }
      }
      if (RED) {
        // reduced system: the slots of k^t, k^phi carry the constants E, L of the photon, their compensation
        // slots -a E, -a L (rk4_step_reduced)
        if (!resumed) {
          S E, L;
          killing_constants(vget(K.a, 0), vget(K.rp, 0), ys[1][l], th, kv.x, kv.w, E, L);
          ys[4][l] = E; ys[7][l] = L;
        }
        cs[4][l] = vneg(vmul(vget(K.a, 0), ys[4][l])); cs[7][l] = vneg(vmul(vget(K.a, 0), ys[7][l]));
      }
      mirrored[l] = m;
      idx[l] = p;
      nst[l] = nst0[l] = iss[l] = s;
      fstat[l] = GRAY_LIVE;
      landing[l] = 0;
      have[l] = true;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) { vpack(y[i], ys[i]); vpack(comp[i], cs[i]); }
  };
  // registers -> HBM
  auto retire = [&](int l, int st) {
    typename Vec4T<S>::type xv, kv;
    const S th = vget(y[2], l), kh = vget(y[6], l);
    xv.x = vget(y[0], l); xv.y = vget(y[1], l) + vget(K.rp, 0); xv.z = mirrored[l] ? pi_minus(th) : th; xv.w = vget(y[3], l);
    kv.x = vget(y[4], l); kv.y = vget(y[5], l); kv.z = mirrored[l] ? sneg(kh) : kh; kv.w = vget(y[7], l);
    if (RED) killing_velocities(vget(K.a, 0), vget(K.rp, 0), vget(K.rpm, 0), vget(y[1], l), th, vget(y[4], l), vget(y[7], l), kv.x, kv.w);
    const unsigned long long p = idx[l];
    A.x[p] = xv;
    A.k[p] = kv;
    A.status[p] = (uint8_t)st;
    A.steps[p] = nst[l];
    if (A.resume != nullptr && st == GRAY_LIVE) {
      // resume record of a photon stopped at max_steps (read back by take()): the kernel's own variables, tagged with
      // the stored (r, theta) bits and the step count they belong to
      typename Vec4T<S>::type r0, r1, r2, r3;
      r0.x = vget(y[1], l); r0.y = th; r0.z = RED ? vget(y[4], l) : S(0); r0.w = RED ? vget(y[7], l) : S(0);
      r1.x = vget(comp[1], l); r1.y = vget(comp[2], l); r1.z = vget(comp[3], l); r1.w = RED ? S(0) : vget(comp[4], l);
      r2.x = vget(comp[5], l); r2.y = vget(comp[6], l); r2.z = RED ? S(0) : vget(comp[7], l);
      r2.w = bits_to_scalar(mirrored[l] ? 1ull : 0ull, S(0));
      r3.x = xv.y; r3.y = xv.z; r3.z = bits_to_scalar((unsigned long long)nst[l], S(0)); r3.w = bits_to_scalar(resume_key(kv.x, kv.y, kv.z, kv.w, RED), S(0));
      A.resume[4 * p] = r0; A.resume[4 * p + 1] = r1; A.resume[4 * p + 2] = r2; A.resume[4 * p + 3] = r3;
    }
    c_steps += nst[l] - nst0[l];
    if (st == GRAY_LIVE) ++c_live; else ++c_done;
    have[l] = false;
  };

  if (SCHED == GRAY_SCHED_STATIC) {
    unsigned long long want[N];
#pragma unroll
    for (int l = 0; l < N; ++l) want[l] = ((unsigned long long)blockIdx.x * N + l) * kBlock + threadIdx.x;
    take(want);
    fold_check(have);
  }

  for (;;) {
    if (SCHED == GRAY_SCHED_REFILL && !exhausted) {
      unsigned need[N];
      int cnt = 0;
#pragma unroll
      for (int l = 0; l < N; ++l) { need[l] = __ballot_sync(FULL, !have[l]); cnt += __popc(need[l]); }
      if (cnt) {
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(&A.ws->queue_head, (unsigned long long)cnt);
        base = __shfl_sync(FULL, base, 0);
        unsigned long long want[N];
        int off = 0;
#pragma unroll
        for (int l = 0; l < N; ++l) {
          want[l] = have[l] ? ~0ull : base + off + __popc(need[l] & ((1u << lane) - 1u));
          off += __popc(need[l]);
        }
        take(want);
        fold_check(have);
        if (base + cnt >= A.n) exhausted = true;
      }
    }
    bool any = false;
#pragma unroll
    for (int l = 0; l < N; ++l) any |= have[l];
    if (!__any_sync(FULL, any)) {
      if (exhausted) break;
      continue;
    }
    for (int it2 = 0; it2 < A.refill_interval; it2 += UN)
#pragma unroll
    for (int un = 0; un < UN; ++un) {
      // A thread whose slots are all empty costs its warp nothing either way.  The float builds let it step its stale
      // registers (nothing of it is ever stored) instead of testing for it at every step: +2 % on B200; the double build
      // keeps the test (-0.7 % without)
      any = sizeof(S) == 4;
#pragma unroll
      for (int l = 0; l < N; ++l) any |= have[l];
      if (any) {
        V dl = RED ? K.zero : step_size<V, RULE>(K, y[1], y[5], y[6], y[7]);
        if (EQ && lnd) {
          // landing on the equatorial plane: a Newton step dlambda = -(theta - pi/2) / k^theta instead of the rule
          S dls[N], ths[N], khs[N];
          vunpack(dl, dls); vunpack(y[2], ths); vunpack(y[6], khs);
#pragma unroll
          for (int l = 0; l < N; ++l)
            if (landing[l]) dls[l] = -(ths[l] - S(1.57079632679489661923)) / khs[l];
          vpack(dl, dls);
        }
        if (!FROZEN) {
          bool rej[N];
          if (RED) rk4_step_reduced<RULE>(K, y, comp);
          else rk4_step<XI, FOLD>(K, y, comp, dl, rej, nullptr, fold_ok);
          if (XI) {
#pragma unroll
            for (int l = 0; l < N; ++l) c_fallback += (rej[l] && have[l]) ? 1u : 0u;
          }
          const V z = RED ? vfma(K.zero, y[6], vmul(K.zero, y[5])) : nonfinite_probe(K, y);
          const V r = y[1];                       // the tests compare heights above the horizon (Consts::r_cap, r_esc)
          // Bookkeeping.  Common case first, with one branch for the whole thread: every slot's theta still in
          // [0, pi/2] (no eq. (3) remap, no fold) and no slot finished.
          S th[N], rr[N], zz[N];
          vunpack(y[2], th); vunpack(r, rr); vunpack(z, zz);
          bool out_of_fold = false;
#pragma unroll
          for (int l = 0; l < N; ++l) out_of_fold |= !(th[l] >= S(0) && th[l] <= S(1.57079632679489661923));
          const bool slow = out_of_fold || (EQ && lnd);
          bool start[N];
#pragma unroll
          for (int l = 0; l < N; ++l) start[l] = false;
          if (slow) {
            // eq. (3) remap and the fold, on the scalars of every slot (a slot without a photon carries junk,
            // which is remapped too and never stored), then the packed values are rebuilt unconditionally.
            // stop_at_equator: a photon that crosses the plane is not folded but landed on it.
            S ph[N], kh[N], c2[N], c6[N];
            vunpack(y[3], ph); vunpack(y[6], kh); vunpack(comp[2], c2); vunpack(comp[6], c6);
#pragma unroll
            for (int l = 0; l < N; ++l) {
              const bool fold = !(EQ && have[l]);
              const bool over = remap_theta(th[l], ph[l], kh[l], c2[l], c6[l], mirrored[l], fold);
              start[l] = !fold && over && landing[l] == 0;
            }
            vpack(y[2], th); vpack(y[3], ph); vpack(y[6], kh); vpack(comp[2], c2); vpack(comp[6], c6);
            fold_check(have);
          } else if (FOLD == 2) fold_ok = true;
          bool fin[N], any_fin = false;
#pragma unroll
          for (int l = 0; l < N; ++l) {
            ++nst[l];
            const bool bad_or_captured = !(zz[l] == S(0) && rr[l] >= K.r_cap);
            bool f = have[l] && (bad_or_captured || !(rr[l] <= K.r_esc) || nst[l] >= A.max_steps);
            if (EQ && slow) {
              if (landing[l] == 2) f = have[l];                              // second Newton step done: on the plane
              else if (landing[l] == 1) { landing[l] = 2; f = false; }
              else if (start[l] && !bad_or_captured) { landing[l] = 1; f = false; }
            }
            fin[l] = f;
            any_fin |= f;
          }
          if (any_fin) {
#pragma unroll
            for (int l = 0; l < N; ++l)
              if (fin[l]) {
                int st = state_status(zz[l], rr[l], K.r_cap, K.r_esc);
                if (EQ && landing[l] == 2) st = zz[l] == S(0) ? GRAY_EQUATOR : GRAY_BAD;
                landing[l] = 0;
                retire(l, st);
              }
          }
          if (EQ && (slow || any_fin)) {
            lnd = false;
#pragma unroll
            for (int l = 0; l < N; ++l) lnd |= landing[l] != 0;
          }
        } else {
          // Peak-rate case (gray.h `frozen`): every slot executes the whole step; a slot whose photon has finished
          // takes it with dlambda = 0 (no stage leaves its state) and its increments are replaced by its own
          // residuals, so its state stays exactly as it is whatever the right-hand sides evaluate to there.
          bool adv[N];
          S dls[N];
          vunpack(dl, dls);
#pragma unroll
          for (int l = 0; l < N; ++l) {
            adv[l] = have[l] && fstat[l] == GRAY_LIVE;
            dls[l] = adv[l] ? dls[l] : S(0);
          }
          vpack(dl, dls);
          bool rej[N];
          rk4_step<false, FOLD, true>(K, y, comp, dl, rej, adv, fold_ok);
          const V z = nonfinite_probe(K, y);
          const V r = y[1];
          S th[N], zz[N], rr[N];
          vunpack(y[2], th); vunpack(z, zz); vunpack(r, rr);
          bool out_of_fold = false;
#pragma unroll
          for (int l = 0; l < N; ++l) out_of_fold |= adv[l] && !(th[l] >= S(0) && th[l] <= S(1.57079632679489661923));
          if (out_of_fold) {
            S ph[N], kh[N], c2[N], c6[N];
            vunpack(y[3], ph); vunpack(y[6], kh); vunpack(comp[2], c2); vunpack(comp[6], c6);
#pragma unroll
            for (int l = 0; l < N; ++l)
              if (adv[l]) remap_theta(th[l], ph[l], kh[l], c2[l], c6[l], mirrored[l], true);
            vpack(y[2], th); vpack(y[3], ph); vpack(y[6], kh); vpack(comp[2], c2); vpack(comp[6], c6);
            fold_check(adv);
          } else if (FOLD == 2) fold_ok = true;            // every advancing photon is inside [0, pi/2]; the others do not matter
#pragma unroll
          for (int l = 0; l < N; ++l) {
            if (have[l]) {
              const int st = state_status(zz[l], rr[l], K.r_cap, K.r_esc);
              nst[l] += adv[l] ? 1u : 0u;
              fstat[l] = adv[l] ? st : fstat[l];
              ++iss[l];
              if (iss[l] == A.max_steps) retire(l, fstat[l]);
            }
          }
        }
      }
    }
    c_iter += (A.refill_interval + UN - 1) / UN * UN;
  }

  c_steps = warp_sum(c_steps);
  const unsigned long long done = warp_sum((unsigned long long)c_done);
  const unsigned long long live = warp_sum((unsigned long long)c_live);
  const unsigned long long fb = XI ? warp_sum((unsigned long long)c_fallback) : 0ull;
  if (lane == 0) {
    if (c_steps) atomicAdd(&A.ws->photon_steps, c_steps);
    if (c_iter) atomicAdd(&A.ws->issued_steps, (unsigned long long)(32 * N) * c_iter);
    if (done) atomicAdd(&A.ws->photons_done, done);
    if (live) atomicAdd(&A.ws->photons_live, live);
    if (XI && fb) atomicAdd(&A.ws->fallback_steps, fb);
  }
}

template <typename V, int RULE, int SCHED, bool FROZEN, bool XI, bool EQ, bool RED = false>
static int launch(const IntegrateArgs<V>& A, cudaStream_t stream) {
  auto kern = integrate_kernel<V, RULE, SCHED, FROZEN, XI, EQ, RED>;
  constexpr unsigned long long per_block = (unsigned long long)kBlock * VT<V>::N;
  unsigned long long blocks_needed = (A.n + per_block - 1) / per_block;
  unsigned int grid;
  if (SCHED == GRAY_SCHED_STATIC) {
    if (blocks_needed > 0x7fffffffull) { set_error("n too large for the static schedule"); return GRAY_ERR_ARG; }
    grid = (unsigned int)blocks_needed;
  } else {
    int occ = 0;
    GRAY_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kBlock, 0));
    if (occ < 1) occ = 1;
    const unsigned long long resident = (unsigned long long)sm_count() * occ;
    grid = (unsigned int)(blocks_needed < resident ? blocks_needed : resident);
  }
  kern<<<grid, kBlock, 0, stream>>>(A);
  GRAY_CUDA(cudaGetLastError());
  return GRAY_OK;
}

template <typename V, int RULE, int SCHED>
static int dispatch_frozen(const IntegrateArgs<V>& A, bool frozen, cudaStream_t s) {
  if (A.reduced) return launch<V, RULE, SCHED, false, false, false, true>(A, s);
  if (frozen) return launch<V, RULE, SCHED, true, false, false>(A, s);
  if (A.stop_eq) return A.K.xi_eps > 0 ? launch<V, RULE, SCHED, false, true, true>(A, s) : launch<V, RULE, SCHED, false, false, true>(A, s);
  return A.K.xi_eps > 0 ? launch<V, RULE, SCHED, false, true, false>(A, s) : launch<V, RULE, SCHED, false, false, false>(A, s);
}
template <typename V, int RULE>
static int dispatch_sched(const IntegrateArgs<V>& A, int sched, bool frozen, cudaStream_t s) {
  return sched == GRAY_SCHED_STATIC ? dispatch_frozen<V, RULE, GRAY_SCHED_STATIC>(A, frozen, s)
                                    : dispatch_frozen<V, RULE, GRAY_SCHED_REFILL>(A, frozen, s);
}

template <typename V>
static int integrate(const gray_state* st, uint64_t n, uint32_t max_steps, const gray_step_params* p,
                     Workspace* ws, cudaStream_t stream) {
  using S = typename VT<V>::S;
  IntegrateArgs<V> A;
  A.x = (typename Vec4T<S>::type*)st->x_dev;
  A.k = (typename Vec4T<S>::type*)st->k_dev;
  A.status = st->status_dev;
  A.steps = st->steps_dev;
  A.resume = (typename Vec4T<S>::type*)st->resume_dev;
  A.n = n;
  A.max_steps = max_steps;
  A.refill_interval = p->refill_interval > 0 ? p->refill_interval : 8;
  A.stop_eq = p->stop_at_equator != 0;
  A.reduced = p->system == GRAY_SYS_REDUCED;
  const double a = st->a, rh = 1.0 + sqrt(1.0 - a * a);
  A.K = make_consts<V>(a, p->h, p->r_capture_factor > 0.0 ? p->r_capture_factor * rh : rh + p->horizon_delta,
                       p->r_escape_factor * st->r_obs, p->xi_epsilon);
  A.ws = ws;
  const bool frozen = p->frozen != 0;
  return p->rule == GRAY_STEP_EQ2 ? dispatch_sched<V, GRAY_STEP_EQ2>(A, p->schedule, frozen, stream)
                                  : dispatch_sched<V, GRAY_STEP_REL>(A, p->schedule, frozen, stream);
}

}  // namespace gray

extern "C" {

int gray_integrate(gray_state* state, uint64_t n_photons, uint32_t max_steps, const gray_step_params* params,
                   void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  using namespace gray;
  int rc = check_state(state, true);
  if (rc) return rc;
  if (!params) { set_error("params is NULL"); return GRAY_ERR_ARG; }
  if (n_photons > state->n) { set_error("n_photons (%llu) exceeds state.n (%llu)", (unsigned long long)n_photons, (unsigned long long)state->n); return GRAY_ERR_ARG; }
  if (params->rule != GRAY_STEP_REL && params->rule != GRAY_STEP_EQ2) { set_error("bad step rule %d", params->rule); return GRAY_ERR_ARG; }
  if (params->schedule != GRAY_SCHED_REFILL && params->schedule != GRAY_SCHED_STATIC) { set_error("bad schedule %d", params->schedule); return GRAY_ERR_ARG; }
  if (params->refill_interval < 0) { set_error("refill_interval must be >= 0"); return GRAY_ERR_ARG; }
  if (!(params->xi_epsilon >= 0.0)) { set_error("xi_epsilon must be >= 0"); return GRAY_ERR_DOMAIN; }
  if (params->xi_epsilon > 0.0 && params->frozen) { set_error("xi_epsilon > 0 is not available together with frozen"); return GRAY_ERR_UNSUPPORTED; }
  if (params->stop_at_equator && params->frozen) { set_error("stop_at_equator is not available together with frozen"); return GRAY_ERR_UNSUPPORTED; }
  if (params->system != GRAY_SYS_FULL && params->system != GRAY_SYS_REDUCED) { set_error("bad system %d", params->system); return GRAY_ERR_ARG; }
  if (params->system == GRAY_SYS_REDUCED && (params->frozen || params->stop_at_equator || params->xi_epsilon > 0.0)) {
    set_error("the reduced system is not available together with frozen, stop_at_equator or xi_epsilon");
    return GRAY_ERR_UNSUPPORTED;
  }
  if (params->photons_per_thread < 0 || params->photons_per_thread > 2) { set_error("photons_per_thread must be 0 (default), 1 or 2"); return GRAY_ERR_ARG; }
  if (params->photons_per_thread == 2 && state->prec != GRAY_F32) { set_error("photons_per_thread = 2 (packed FP32 instructions) needs GRAY_F32"); return GRAY_ERR_UNSUPPORTED; }
  if (params->rule == GRAY_STEP_EQ2 && params->h > 0.2) {
    // under eq. (2) a step moves theta by at most h; the folded first-stage sine / cosine covers [-0.2, pi/2 + 0.2]
    set_error("h = %g: GRAY_STEP_EQ2 supports 0 < h <= 0.2 (the paper's Delta ~ 1/32, P:79)", params->h);
    return GRAY_ERR_DOMAIN;
  }
  if (!(params->h > 0.0) || !(params->r_escape_factor > 0.0) || params->r_capture_factor < 0.0 ||
      (params->r_capture_factor == 0.0 && !(params->horizon_delta >= 0.0))) {
    set_error("step parameters out of domain (h > 0, r_escape_factor > 0, r_capture_factor >= 0, horizon_delta >= 0)");
    return GRAY_ERR_DOMAIN;
  }
  rc = check_workspace(workspace_dev, workspace_bytes);
  if (rc) return rc;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  Workspace* ws = (Workspace*)workspace_dev;
  GRAY_CUDA(cudaMemsetAsync(ws, 0, 256, stream));   // queue head and gray_counters
  if (n_photons == 0 || max_steps == 0) return GRAY_OK;
  if (state->prec == GRAY_F64) return integrate<double>(state, n_photons, max_steps, params, ws, stream);
  return params->photons_per_thread == 1 ? integrate<float>(state, n_photons, max_steps, params, ws, stream)
                                         : integrate<f2>(state, n_photons, max_steps, params, ws, stream);
}

int gray_integrate_counters(const void* workspace_dev, gray_counters* counters_host, void* cuda_stream) {
  using namespace gray;
  if (!counters_host) { set_error("counters_host is NULL"); return GRAY_ERR_ARG; }
  int rc = check_workspace(workspace_dev, sizeof(Workspace));
  if (rc) return rc;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const Workspace* ws = (const Workspace*)workspace_dev;
  unsigned long long c[5];
  GRAY_CUDA(cudaMemcpyAsync(c, &ws->photon_steps, sizeof c, cudaMemcpyDeviceToHost, stream));
  GRAY_CUDA(cudaStreamSynchronize(stream));
  counters_host->photon_steps = c[0];
  counters_host->issued_steps = c[1];
  counters_host->photons_done = c[2];
  counters_host->photons_live = c[3];
  counters_host->fallback_steps = c[4];
  return GRAY_OK;
}

}  // extern "C"
