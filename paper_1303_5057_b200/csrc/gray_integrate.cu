// gray_integrate.cu — the integrator kernel of libgray and gray_integrate() (include/gray.h).
//
// One photon per thread, its 8-component state in registers from the moment it is loaded until it
// terminates ("GRay integrates each geodesic for many steps in a single data load", P:81 fn 5).
// What differs from the paper's fixed grid of 64-thread blocks: the kernel is persistent
// (148 SMs x resident blocks) and a lane whose photon has terminated is refilled from a device-side
// queue, so a warp never idles on its slowest ray; HBM is touched once per photon on load and once
// on retirement, with 16-byte vector accesses.
#include "gray_internal.h"
#include "gray_math.cuh"

namespace gray {

template <typename T> struct Vec4T;
template <> struct Vec4T<float> { using type = float4; };
template <> struct Vec4T<double> { using type = double4; };

template <typename T>
struct IntegrateArgs {
  typename Vec4T<T>::type* x;
  typename Vec4T<T>::type* k;
  uint8_t* status;
  uint32_t* steps;
  unsigned long long n;
  uint32_t max_steps;
  int refill_interval;
  KerrConst<T> K;
  Workspace* ws;
};

constexpr int kBlock = 128;
template <typename T> struct Tune;
template <> struct Tune<float> { static constexpr int min_blocks = 4; };    // <= 128 registers/thread
template <> struct Tune<double> { static constexpr int min_blocks = 2; };   // <= 255 registers/thread

// HBM -> registers: (t, r, theta, phi), k^mu -> the kernel's variables (gray_math.cuh): d = r - r_+ and
// theta folded into [0, pi/2].
template <typename T>
__device__ __forceinline__ void load_photon(const IntegrateArgs<T>& A, unsigned long long p, T y[8], int& mirrored) {
  const typename Vec4T<T>::type xv = A.x[p], kv = A.k[p];
  y[0] = xv.x; y[1] = xv.y - A.K.rp; y[2] = xv.z; y[3] = xv.w;
  y[4] = kv.x; y[5] = kv.y; y[6] = kv.z; y[7] = kv.w;
  mirrored = 0;
  if (y[2] > T(1.57079632679489661923)) {
    y[2] = pi_minus(y[2]);
    y[6] = -y[6];
    mirrored = 1;
  }
}

template <typename T>
__device__ __forceinline__ void store_photon(const IntegrateArgs<T>& A, unsigned long long p, const T y[8],
                                             int mirrored, int st, uint32_t nst) {
  typename Vec4T<T>::type xv, kv;
  xv.x = y[0]; xv.y = y[1] + A.K.rp; xv.z = mirrored ? pi_minus(y[2]) : y[2]; xv.w = y[3];
  kv.x = y[4]; kv.y = y[5]; kv.z = mirrored ? -y[6] : y[6]; kv.w = y[7];
  A.x[p] = xv;
  A.k[p] = kv;
  A.status[p] = (uint8_t)st;
  A.steps[p] = nst;
}

__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <typename T, int RULE, int SCHED, bool FROZEN>
__global__ void __launch_bounds__(kBlock, Tune<T>::min_blocks)
integrate_kernel(const __grid_constant__ IntegrateArgs<T> A) {
  constexpr unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const KerrConst<T> K = A.K;

  T y[8], comp[8];
  int mirrored = 0;
  unsigned long long idx = 0;
  uint32_t nst = 0, nst0 = 0, iss = 0;
  int fstat = GRAY_LIVE;
  bool have = false;
  bool exhausted = (SCHED == GRAY_SCHED_STATIC);
  unsigned long long c_steps = 0;
  unsigned int c_done = 0, c_live = 0, c_iter = 0;

  // take photon p if it is live and has steps left
  auto take = [&](unsigned long long p) {
    const uint8_t st = A.status[p];
    const uint32_t s = A.steps[p];
    if (st != GRAY_LIVE) return;
    if (s >= A.max_steps) { ++c_live; return; }
    load_photon(A, p, y, mirrored);
#pragma unroll
    for (int i = 0; i < 8; ++i) comp[i] = T(0);
    idx = p;
    nst = nst0 = iss = s;
    fstat = GRAY_LIVE;
    have = true;
  };
  auto retire = [&](int st) {
    store_photon(A, idx, y, mirrored, st, nst);
    c_steps += nst - nst0;
    if (st == GRAY_LIVE) ++c_live; else ++c_done;
    have = false;
  };

  if (SCHED == GRAY_SCHED_STATIC) {
    const unsigned long long p = (unsigned long long)blockIdx.x * kBlock + threadIdx.x;
    if (p < A.n) take(p);
  }

  for (;;) {
    if (SCHED == GRAY_SCHED_REFILL && !exhausted) {
      const unsigned need = __ballot_sync(FULL, !have);
      if (need) {
        const int cnt = __popc(need), leader = __ffs(need) - 1;
        unsigned long long base = 0;
        if (lane == leader) base = atomicAdd(&A.ws->queue_head, (unsigned long long)cnt);
        base = __shfl_sync(FULL, base, leader);
        if (!have) {
          const unsigned long long p = base + __popc(need & ((1u << lane) - 1u));
          if (p < A.n) take(p);
        }
        if (base + cnt >= A.n) exhausted = true;
      }
    }
    if (!__any_sync(FULL, have)) {
      if (exhausted) break;
      continue;
    }
    for (int it = 0; it < A.refill_interval; ++it) {
      if (have) {
        const T dl = step_size<T, RULE>(K, y);
        if (!FROZEN) {
          rk4_step(K, y, comp, dl);
          remap_theta(y, comp, mirrored);
          ++nst;
          const int st = state_status(K, y);
          if (st != GRAY_LIVE || nst == A.max_steps) retire(st);
        } else {
          T z[8], zc[8];
          int zm = mirrored;
#pragma unroll
          for (int i = 0; i < 8; ++i) { z[i] = y[i]; zc[i] = comp[i]; }
          rk4_step(K, z, zc, dl);
          remap_theta(z, zc, zm);
          const int st = state_status(K, z);
          const bool adv = (fstat == GRAY_LIVE);
#pragma unroll
          for (int i = 0; i < 8; ++i) { y[i] = adv ? z[i] : y[i]; comp[i] = adv ? zc[i] : comp[i]; }
          mirrored = adv ? zm : mirrored;
          nst += adv ? 1u : 0u;
          fstat = adv ? st : fstat;
          ++iss;
          if (iss == A.max_steps) retire(fstat);
        }
      }
    }
    c_iter += A.refill_interval;
  }

  c_steps = warp_sum(c_steps);
  const unsigned long long done = warp_sum((unsigned long long)c_done);
  const unsigned long long live = warp_sum((unsigned long long)c_live);
  if (lane == 0) {
    if (c_steps) atomicAdd(&A.ws->photon_steps, c_steps);
    if (c_iter) atomicAdd(&A.ws->issued_steps, 32ull * c_iter);
    if (done) atomicAdd(&A.ws->photons_done, done);
    if (live) atomicAdd(&A.ws->photons_live, live);
  }
}

template <typename T, int RULE, int SCHED, bool FROZEN>
static int launch(const IntegrateArgs<T>& A, cudaStream_t stream) {
  auto kern = integrate_kernel<T, RULE, SCHED, FROZEN>;
  unsigned long long blocks_needed = (A.n + kBlock - 1) / kBlock;
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

template <typename T, int RULE, int SCHED>
static int dispatch_frozen(const IntegrateArgs<T>& A, bool frozen, cudaStream_t s) {
  return frozen ? launch<T, RULE, SCHED, true>(A, s) : launch<T, RULE, SCHED, false>(A, s);
}
template <typename T, int RULE>
static int dispatch_sched(const IntegrateArgs<T>& A, int sched, bool frozen, cudaStream_t s) {
  return sched == GRAY_SCHED_STATIC ? dispatch_frozen<T, RULE, GRAY_SCHED_STATIC>(A, frozen, s)
                                    : dispatch_frozen<T, RULE, GRAY_SCHED_REFILL>(A, frozen, s);
}

template <typename T>
static int integrate(const gray_state* st, uint64_t n, uint32_t max_steps, const gray_step_params* p,
                     Workspace* ws, cudaStream_t stream) {
  IntegrateArgs<T> A;
  A.x = (typename Vec4T<T>::type*)st->x_dev;
  A.k = (typename Vec4T<T>::type*)st->k_dev;
  A.status = st->status_dev;
  A.steps = st->steps_dev;
  A.n = n;
  A.max_steps = max_steps;
  A.refill_interval = p->refill_interval > 0 ? p->refill_interval : 8;
  const double a = st->a, root = sqrt(1.0 - a * a), rh = 1.0 + root;
  A.K.a = (T)a;
  A.K.a2 = (T)(a * a);
  A.K.rp = (T)rh;
  A.K.rpm = (T)(2.0 * root);
  A.K.h = (T)p->h;
  A.K.r_cap = (T)(p->r_capture_factor > 0.0 ? p->r_capture_factor * rh : rh + p->horizon_delta);
  A.K.r_esc = (T)(p->r_escape_factor * st->r_obs);
  A.ws = ws;
  const bool frozen = p->frozen != 0;
  return p->rule == GRAY_STEP_EQ2 ? dispatch_sched<T, GRAY_STEP_EQ2>(A, p->schedule, frozen, stream)
                                  : dispatch_sched<T, GRAY_STEP_REL>(A, p->schedule, frozen, stream);
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
  return state->prec == GRAY_F32 ? integrate<float>(state, n_photons, max_steps, params, ws, stream)
                                 : integrate<double>(state, n_photons, max_steps, params, ws, stream);
}

int gray_integrate_counters(const void* workspace_dev, gray_counters* counters_host, void* cuda_stream) {
  using namespace gray;
  if (!counters_host) { set_error("counters_host is NULL"); return GRAY_ERR_ARG; }
  int rc = check_workspace(workspace_dev, sizeof(Workspace));
  if (rc) return rc;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const Workspace* ws = (const Workspace*)workspace_dev;
  unsigned long long c[4];
  GRAY_CUDA(cudaMemcpyAsync(c, &ws->photon_steps, sizeof c, cudaMemcpyDeviceToHost, stream));
  GRAY_CUDA(cudaStreamSynchronize(stream));
  counters_host->photon_steps = c[0];
  counters_host->issued_steps = c[1];
  counters_host->photons_done = c[2];
  counters_host->photons_live = c[3];
  return GRAY_OK;
}

}  // extern "C"
