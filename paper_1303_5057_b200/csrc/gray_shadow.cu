// gray_shadow.cu — gray_classify and gray_shadow_edge (include/gray.h): capture map, status counts and
// the shadow / photon-ring statistics of paper eqs. (6)-(8), from the per-photon status.
#include "gray_internal.h"

#include <mutex>

namespace gray {

__device__ __forceinline__ unsigned int warp_sum_u32(unsigned int v) { return __reduce_add_sync(0xffffffffu, v); }

// status -> capture flags + histogram of the GRAY_N_STATUS statuses (bytes outside 0 .. GRAY_N_STATUS-1 are counted
// nowhere).  16 photons per thread per iteration when the buffers allow 16-byte accesses; the bytes of a word are
// compared four at a time (__vcmpeq4).
__global__ void __launch_bounds__(256) classify_kernel(const uint8_t* __restrict__ status, uint8_t* __restrict__ cmap,
                                                       unsigned long long n, int vec_ok, Workspace* ws) {
  unsigned int c[GRAY_N_STATUS];
#pragma unroll
  for (int q = 0; q < GRAY_N_STATUS; ++q) c[q] = 0;
  const unsigned long long tid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long nthreads = (unsigned long long)gridDim.x * blockDim.x;
  const unsigned long long nvec = vec_ok ? n / 16 : 0;
  for (unsigned long long v = tid; v < nvec; v += nthreads) {
    const uint4 w = ((const uint4*)status)[v];
    const unsigned int in[4] = {w.x, w.y, w.z, w.w};
    unsigned int out[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
#pragma unroll
      for (int s = 0; s < GRAY_N_STATUS; ++s) c[s] += __popc(__vcmpeq4(in[q], 0x01010101u * (unsigned int)s)) >> 3;
      out[q] = __vcmpeq4(in[q], 0x01010101u * (unsigned int)GRAY_CAPTURED) & 0x01010101u;
    }
    if (cmap) ((uint4*)cmap)[v] = make_uint4(out[0], out[1], out[2], out[3]);
  }
  for (unsigned long long p = nvec * 16 + tid; p < n; p += nthreads) {
    const unsigned int s = status[p];
#pragma unroll
    for (int q = 0; q < GRAY_N_STATUS; ++q) c[q] += (s == (unsigned int)q) ? 1u : 0u;
    if (cmap) cmap[p] = (s == GRAY_CAPTURED) ? 1 : 0;
  }
#pragma unroll
  for (int q = 0; q < GRAY_N_STATUS; ++q) {
    const unsigned int t = warp_sum_u32(c[q]);
    if ((threadIdx.x & 31) == 0 && t) atomicAdd(&ws->counts[q], (unsigned long long)t);
  }
}

// captured pixels: count, sums of column / row indices (exact integers), extreme columns
__global__ void __launch_bounds__(256) shadow_reduce_kernel(const uint8_t* __restrict__ status, unsigned long long n,
                                                            unsigned int nx, Workspace* ws) {
  unsigned long long cnt = 0, sc = 0, sr = 0;
  unsigned int cmin = 0xffffffffu, cmax = 0;
  const unsigned long long nthreads = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long p = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += nthreads) {
    if (status[p] == GRAY_CAPTURED) {
      const unsigned int col = (unsigned int)(p % nx), row = (unsigned int)(p / nx);
      ++cnt; sc += col; sr += row;
      cmin = min(cmin, col); cmax = max(cmax, col);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    sc += __shfl_xor_sync(0xffffffffu, sc, o);
    sr += __shfl_xor_sync(0xffffffffu, sr, o);
  }
  cmin = __reduce_min_sync(0xffffffffu, cmin);
  cmax = __reduce_max_sync(0xffffffffu, cmax);
  if ((threadIdx.x & 31) == 0 && cnt) {
    atomicAdd(&ws->n_captured, cnt);
    atomicAdd(&ws->sum_col, sc);
    atomicAdd(&ws->sum_row, sr);
    atomicMin(&ws->min_col, cmin);
    atomicMax(&ws->max_col, cmax);
  }
}

struct EdgeArgs {
  const uint8_t* status;
  long long nx, ny;
  double W;
  int n_angles;
  double* radius;
  Workspace* ws;
};

// rho(vartheta): march outwards from the image origin in half-pixel steps until the pixel under the
// sample is not captured (or the image ends); the edge is the mid-point of the last two samples.
// One warp per spoke: its lanes look at 32 consecutive samples at a time and the first one that stops the march is
// found by ballot (the samples do not depend on each other, only the stopping rule does).
constexpr int kMaxSpokesInShared = 5120;        // radii of up to this many spokes are kept in shared memory (40 KB)
__device__ double spoke_radius_warp(const EdgeArgs& A, double da, double db, double delta, double cv, double sv) {
  const int lane = threadIdx.x & 31;
  for (long long j0 = 0;; j0 += 32) {
    const long long j = j0 + lane;
    const double q = (double)j * delta;
    const long long col = (long long)floor((q * cv + A.W) / da);
    const long long row = (long long)floor((q * sv + A.W) / db);
    const bool inside = col >= 0 && col < A.nx && row >= 0 && row < A.ny;
    const bool stop = !inside || A.status[row * A.nx + col] != GRAY_CAPTURED;
    const unsigned m = __ballot_sync(0xffffffffu, stop);
    if (m) {
      const long long js = j0 + (__ffs(m) - 1);
      const bool in_s = (__ballot_sync(0xffffffffu, inside) >> (__ffs(m) - 1)) & 1u;
      return (!in_s || js > 0) ? ((double)js - 0.5) * delta : 0.0;
    }
  }
}

__device__ double block_sum(double v, double* sh) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
  return t;
}

// one block: spokes (a warp each), then eqs. (6)-(8)
__global__ void __launch_bounds__(1024) shadow_edge_kernel(const __grid_constant__ EdgeArgs A) {
  __shared__ double sh[32];
  __shared__ double rho_sh[kMaxSpokesInShared];
  Workspace* ws = A.ws;
  const double da = 2.0 * A.W / (double)A.nx, db = 2.0 * A.W / (double)A.ny;
  const double delta = fmin(da, db) / 2.0;
  const unsigned long long ncap = ws->n_captured;
  const double amin = ncap ? -A.W + (double)ws->min_col * da : 0.0;
  const double amax = ncap ? -A.W + (double)(ws->max_col + 1) * da : 0.0;
  const double centre = (amin + amax) / 2.0;
  const double two_pi = 2.0 * 3.14159265358979323846;
  const int warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5, lane = threadIdx.x & 31;
  // R_k = distance of the edge point on spoke k from the ring's centre; the spoke's rho from shared memory if it is there
  auto R_of = [&](int k, double rho) {
    const double vt = two_pi * ((double)k + 0.5) / (double)A.n_angles;
    double sv, cv;
    sincos(vt, &sv, &cv);
    const double x = rho * cv - centre, y = rho * sv;
    return sqrt(x * x + y * y);
  };
  auto rho_of = [&](int k) {                       // called by whole warps
    const double vt = two_pi * ((double)k + 0.5) / (double)A.n_angles;
    double sv, cv;
    sincos(vt, &sv, &cv);
    return spoke_radius_warp(A, da, db, delta, cv, sv);
  };
  double sumR = 0.0;
  for (int k = warp; k < A.n_angles; k += n_warps) {
    const double rho = rho_of(k);
    if (lane == 0) {
      if (k < kMaxSpokesInShared) rho_sh[k] = rho;
      if (A.radius) A.radius[k] = rho;
      sumR += R_of(k, rho);
    }
  }
  const double mean = A.n_angles > 0 ? block_sum(sumR, sh) / (double)A.n_angles : 0.0;     // (block_sum synchronises)
  double var = 0.0;
  for (int k = warp; k < A.n_angles; k += n_warps) {
    const double rho = k < kMaxSpokesInShared ? rho_sh[k] : rho_of(k);
    if (lane == 0) {
      const double d = R_of(k, rho) - mean;
      var += d * d;
    }
  }
  var = A.n_angles > 0 ? block_sum(var, sh) / (double)A.n_angles : 0.0;
  if (threadIdx.x == 0) {
    ws->stats[0] = (double)ncap * da * db;
    ws->stats[1] = ncap ? -A.W + ((double)ws->sum_col / (double)ncap + 0.5) * da : 0.0;
    ws->stats[2] = ncap ? -A.W + ((double)ws->sum_row / (double)ncap + 0.5) * db : 0.0;
    ws->stats[3] = amin;
    ws->stats[4] = amax;
    ws->stats[5] = fabs(amin + amax) / 2.0;
    ws->stats[6] = mean;
    ws->stats[7] = 2.0 * sqrt(var);
  }
}

// Photon ring on the paper's polar grid (gray_ring_polar in gray.h; eqs. 6-10).  One block; a warp per
// spoke finds the outermost captured cell, then eqs. (6)-(8) by block reductions (trapezoidal rule).
struct RingArgs {
  const uint8_t* status;
  long long n_R, n_theta;
  double R_lo, R_hi;
  int bridge_axis;
  double* radius;
  Workspace* ws;
};

// outer edge of the outermost captured cell of spoke k, by a whole warp: the lanes share the cells, the largest captured
// index wins
__device__ double ring_radius_raw_warp(const RingArgs& A, long long k) {
  const uint8_t* row = A.status + k * A.n_R;
  long long best = 0;
  for (long long j = threadIdx.x & 31; j < A.n_R; j += 32)
    if (row[j] == GRAY_CAPTURED) best = j + 1;
  for (int o = 16; o > 0; o >>= 1) {
    const long long other = __shfl_xor_sync(0xffffffffu, best, o);
    best = other > best ? other : best;
  }
  return A.R_lo + (double)best * ((A.R_hi - A.R_lo) / (double)A.n_R);
}

__global__ void __launch_bounds__(1024) ring_polar_kernel(const __grid_constant__ RingArgs A) {
  __shared__ double sh[32];
  __shared__ double raw_sh[kMaxSpokesInShared];
  const double pi = 3.14159265358979323846;
  const int warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5, lane = threadIdx.x & 31;
  const long long mid = (A.n_theta - 1) / 2;
  const bool has_axis = A.n_theta >= 3 && (A.n_theta % 2) == 1;
  for (long long k = warp; k < A.n_theta && k < kMaxSpokesInShared; k += n_warps) {
    const double r = ring_radius_raw_warp(A, k);
    if (lane == 0) raw_sh[k] = r;
  }
  __syncthreads();
  auto raw_of = [&](long long k) { return k < kMaxSpokesInShared ? raw_sh[k] : ring_radius_raw_warp(A, k); };   // whole warps
  auto radius_of = [&](long long k) {
    if (A.bridge_axis && has_axis && k == mid) return 0.5 * (raw_of(k - 1) + raw_of(k + 1));      // the axis spoke (gray.h)
    return raw_of(k);
  };
  const double amax = radius_of(0), amin = -radius_of(A.n_theta - 1);
  const double centre = (amin + amax) / 2.0;
  const double step = pi / (double)(A.n_theta - 1);
  auto R_of = [&](long long k, double rho) {
    double sv, cv;
    sincos((double)k * step, &sv, &cv);
    const double x = rho * cv - centre, y = rho * sv;
    return sqrt(x * x + y * y);
  };
  double sum = 0.0;
  for (long long k = warp; k < A.n_theta; k += n_warps) {
    const double rho = radius_of(k);
    if (lane == 0) {
      if (A.radius) A.radius[k] = rho;
      sum += ((k == 0 || k == A.n_theta - 1) ? 0.5 : 1.0) * R_of(k, rho);
    }
  }
  const double mean = block_sum(sum, sh) / (double)(A.n_theta - 1);
  double var = 0.0;
  for (long long k = warp; k < A.n_theta; k += n_warps) {
    const double rho = radius_of(k);
    if (lane == 0) {
      const double d = R_of(k, rho) - mean;
      var += ((k == 0 || k == A.n_theta - 1) ? 0.5 : 1.0) * d * d;
    }
  }
  var = block_sum(var, sh) / (double)(A.n_theta - 1);
  // the axis spoke (vartheta = pi/2, n_theta odd), reported whether or not it is bridged: its radius as traced, the
  // radius used, and how many of its rays did not end CAPTURED or ESCAPED (gray.h)
  double lost = 0.0;
  if (has_axis)
    for (long long j = threadIdx.x; j < A.n_R; j += blockDim.x) {
      const uint8_t st = A.status[mid * A.n_R + j];
      lost += (st != GRAY_CAPTURED && st != GRAY_ESCAPED) ? 1.0 : 0.0;
    }
  lost = block_sum(lost, sh);
  const double axis_raw = has_axis ? raw_of(mid) : 0.0, axis_used = has_axis ? radius_of(mid) : 0.0;     // (every warp, uniformly)
  if (threadIdx.x == 0) {
    A.ws->stats[0] = amin;
    A.ws->stats[1] = amax;
    A.ws->stats[2] = fabs(amin + amax) / 2.0;
    A.ws->stats[3] = mean;
    A.ws->stats[4] = 2.0 * sqrt(var);
    A.ws->stats[5] = axis_raw;
    A.ws->stats[6] = axis_used;
    A.ws->stats[7] = lost;
  }
}

static unsigned int reduce_grid(unsigned long long n, unsigned long long per_thread) {
  unsigned long long blocks = (n / per_thread + 255) / 256 + 1;
  const unsigned long long cap = (unsigned long long)sm_count() * 16;
  if (blocks > cap) blocks = cap;
  return (unsigned int)(blocks ? blocks : 1);
}

// ------------------------------------------------------------------ gray_shadow_edge_noalloc (gray.h)
// The scratch memory of gray_shadow_edge, for callers that cannot hand the library a device workspace because they have
// no way to allocate one: the reduction cells of the Workspace and one radius per spoke live in a file-scope device
// array.  The driver reserves it on every GPU that loads libgray, from the moment the module is loaded until the
// process ends, so it is kept small: 512 B + 8 B x GRAY_NOALLOC_MAX_ANGLES = 128.5 KB.
struct NoAllocScratch {
  Workspace ws;                              // sum_col .. n_captured and stats[] are used, as in gray_shadow_edge
  double rho[GRAY_NOALLOC_MAX_ANGLES];       // rho(vartheta_k) between the two passes of the statistics kernel
};
static __device__ __align__(256) unsigned long long noalloc_scratch[(sizeof(NoAllocScratch) + 7) / 8];

// shadow_edge_kernel with the radii of ALL spokes kept in the scratch array between the mean (eq. 7) and the variance
// (eq. 8) pass, instead of the first 5120 in shared memory and the rest marched a second time.  Same arithmetic in the
// same order, so the results are those of shadow_edge_kernel.  Every rho[k], k < n_angles, is written in the first pass
// before the second reads it (by the same lane), so what an earlier call left there is never seen.
__global__ void __launch_bounds__(1024) shadow_edge_scratch_kernel(const __grid_constant__ EdgeArgs A, double* __restrict__ rho_scratch) {
  __shared__ double sh[32];
  Workspace* ws = A.ws;
  const double da = 2.0 * A.W / (double)A.nx, db = 2.0 * A.W / (double)A.ny;
  const double delta = fmin(da, db) / 2.0;
  const unsigned long long ncap = ws->n_captured;
  const double amin = ncap ? -A.W + (double)ws->min_col * da : 0.0;
  const double amax = ncap ? -A.W + (double)(ws->max_col + 1) * da : 0.0;
  const double centre = (amin + amax) / 2.0;
  const double two_pi = 2.0 * 3.14159265358979323846;
  const int warp = threadIdx.x >> 5, n_warps = blockDim.x >> 5, lane = threadIdx.x & 31;
  auto R_of = [&](int k, double rho) {
    const double vt = two_pi * ((double)k + 0.5) / (double)A.n_angles;
    double sv, cv;
    sincos(vt, &sv, &cv);
    const double x = rho * cv - centre, y = rho * sv;
    return sqrt(x * x + y * y);
  };
  double sumR = 0.0;
  for (int k = warp; k < A.n_angles; k += n_warps) {
    const double vt = two_pi * ((double)k + 0.5) / (double)A.n_angles;
    double sv, cv;
    sincos(vt, &sv, &cv);
    const double rho = spoke_radius_warp(A, da, db, delta, cv, sv);
    if (lane == 0) {
      rho_scratch[k] = rho;
      if (A.radius) A.radius[k] = rho;
      sumR += R_of(k, rho);
    }
  }
  const double mean = A.n_angles > 0 ? block_sum(sumR, sh) / (double)A.n_angles : 0.0;     // (block_sum synchronises)
  double var = 0.0;
  for (int k = warp; k < A.n_angles; k += n_warps) {
    if (lane == 0) {
      const double d = R_of(k, rho_scratch[k]) - mean;
      var += d * d;
    }
  }
  var = A.n_angles > 0 ? block_sum(var, sh) / (double)A.n_angles : 0.0;
  if (threadIdx.x == 0) {
    ws->stats[0] = (double)ncap * da * db;
    ws->stats[1] = ncap ? -A.W + ((double)ws->sum_col / (double)ncap + 0.5) * da : 0.0;
    ws->stats[2] = ncap ? -A.W + ((double)ws->sum_row / (double)ncap + 0.5) * db : 0.0;
    ws->stats[3] = amin;
    ws->stats[4] = amax;
    ws->stats[5] = fabs(amin + amax) / 2.0;
    ws->stats[6] = mean;
    ws->stats[7] = 2.0 * sqrt(var);
  }
}

// Device address of noalloc_scratch on the current device.  In host code the name `noalloc_scratch` is only the
// runtime's handle for the symbol, not memory a kernel could use: the address has to be asked for, once per device
// (each GPU has its own copy of the array), with that device current.
constexpr int kNoAllocMaxDevices = 64;
static std::mutex g_noalloc_mutex;
static NoAllocScratch* g_noalloc_ptr[kNoAllocMaxDevices];
static int noalloc_scratch_on_current_device(NoAllocScratch** out) {
  int dev = -1;
  GRAY_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoAllocMaxDevices) { set_error("gray_shadow_edge_noalloc: device ordinal %d is not below %d", dev, kNoAllocMaxDevices); return GRAY_ERR_UNSUPPORTED; }
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    GRAY_CUDA(cudaGetSymbolAddress(&p, noalloc_scratch));
    if (!p || ((uintptr_t)p & 255)) { set_error("gray_shadow_edge_noalloc: the runtime gave no usable address for the static scratch array"); return GRAY_ERR_CUDA; }
    g_noalloc_ptr[dev] = (NoAllocScratch*)p;
  }
  *out = g_noalloc_ptr[dev];
  return GRAY_OK;
}

}  // namespace gray

extern "C" {

int gray_classify(const gray_state* state, uint8_t* capture_map_dev, uint64_t counts_host[GRAY_N_STATUS], void* workspace_dev,
                  size_t workspace_bytes, void* cuda_stream) {
  using namespace gray;
  int rc = check_state(state, false);
  if (rc) return rc;
  if (!counts_host) { set_error("counts_host is NULL"); return GRAY_ERR_ARG; }
  rc = check_workspace(workspace_dev, workspace_bytes);
  if (rc) return rc;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  Workspace* ws = (Workspace*)workspace_dev;
  GRAY_CUDA(cudaMemsetAsync(&ws->counts[0], 0, sizeof ws->counts, stream));
  if (state->n) {
    const int vec_ok = (((uintptr_t)state->status_dev & 15) == 0) && (!capture_map_dev || ((uintptr_t)capture_map_dev & 15) == 0);
    classify_kernel<<<reduce_grid(state->n, 16), 256, 0, stream>>>(state->status_dev, capture_map_dev, state->n, vec_ok, ws);
    GRAY_CUDA(cudaGetLastError());
  }
  unsigned long long c[GRAY_N_STATUS];
  GRAY_CUDA(cudaMemcpyAsync(c, &ws->counts[0], sizeof c, cudaMemcpyDeviceToHost, stream));
  GRAY_CUDA(cudaStreamSynchronize(stream));
  for (int q = 0; q < GRAY_N_STATUS; ++q) counts_host[q] = c[q];
  return GRAY_OK;
}

int gray_shadow_edge(const gray_state* state, int32_t n_angles, double* radius_dev, gray_shadow_stats* stats_host,
                     void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  using namespace gray;
  int rc = check_state(state, true);
  if (rc) return rc;
  if (!stats_host || n_angles < 0) { set_error("stats_host is NULL or n_angles < 0"); return GRAY_ERR_ARG; }
  if (state->pixels != GRAY_PIXELS_GRID || state->p0 != 0 || state->nx <= 0 || state->ny <= 0 ||
      state->n != (uint64_t)state->nx * (uint64_t)state->ny) {
    set_error("gray_shadow_edge needs a full grid image (pixels = GRID, p0 = 0, n = nx * ny)");
    return GRAY_ERR_ARG;
  }
  rc = check_workspace(workspace_dev, workspace_bytes);
  if (rc) return rc;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  Workspace* ws = (Workspace*)workspace_dev;
  // sum_col .. n_captured; min_col must start at the maximum
  GRAY_CUDA(cudaMemsetAsync(&ws->sum_col, 0, (char*)&ws->pad3[0] - (char*)&ws->sum_col, stream));
  GRAY_CUDA(cudaMemsetAsync(&ws->min_col, 0xff, sizeof ws->min_col, stream));
  shadow_reduce_kernel<<<reduce_grid(state->n, 4), 256, 0, stream>>>(state->status_dev, state->n, (unsigned int)state->nx, ws);
  GRAY_CUDA(cudaGetLastError());
  EdgeArgs A;
  A.status = state->status_dev; A.nx = state->nx; A.ny = state->ny; A.W = state->half_width;
  A.n_angles = n_angles; A.radius = radius_dev; A.ws = ws;
  shadow_edge_kernel<<<1, 1024, 0, stream>>>(A);
  GRAY_CUDA(cudaGetLastError());
  double s[8];
  unsigned long long ncap = 0;
  GRAY_CUDA(cudaMemcpyAsync(s, &ws->stats[0], sizeof s, cudaMemcpyDeviceToHost, stream));
  GRAY_CUDA(cudaMemcpyAsync(&ncap, &ws->n_captured, sizeof ncap, cudaMemcpyDeviceToHost, stream));
  GRAY_CUDA(cudaStreamSynchronize(stream));
  stats_host->area = s[0]; stats_host->centroid_alpha = s[1]; stats_host->centroid_beta = s[2];
  stats_host->alpha_min = s[3]; stats_host->alpha_max = s[4]; stats_host->D = s[5];
  stats_host->R_mean = s[6]; stats_host->A = s[7];
  stats_host->n_captured = ncap;
  return GRAY_OK;
}

int gray_ring_polar(const gray_state* state, int32_t bridge_axis, double* radius_dev, gray_ring_stats* stats_host,
                    void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  using namespace gray;
  int rc = check_state(state, true);
  if (rc) return rc;
  if (!stats_host) { set_error("stats_host is NULL"); return GRAY_ERR_ARG; }
  if (state->pixels != GRAY_PIXELS_POLAR || state->p0 != 0 || state->nx <= 0 || state->ny < 2 ||
      state->n != (uint64_t)state->nx * (uint64_t)state->ny) {
    set_error("gray_ring_polar needs a full polar image (pixels = POLAR, p0 = 0, n = n_R * n_theta)");
    return GRAY_ERR_ARG;
  }
  rc = check_workspace(workspace_dev, workspace_bytes);
  if (rc) return rc;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  Workspace* ws = (Workspace*)workspace_dev;
  RingArgs A;
  A.status = state->status_dev; A.n_R = state->nx; A.n_theta = state->ny;
  A.R_lo = state->r_lo; A.R_hi = state->half_width; A.bridge_axis = bridge_axis; A.radius = radius_dev; A.ws = ws;
  ring_polar_kernel<<<1, 1024, 0, stream>>>(A);
  GRAY_CUDA(cudaGetLastError());
  double s[8];
  GRAY_CUDA(cudaMemcpyAsync(s, &ws->stats[0], sizeof s, cudaMemcpyDeviceToHost, stream));
  GRAY_CUDA(cudaStreamSynchronize(stream));
  stats_host->alpha_min = s[0]; stats_host->alpha_max = s[1]; stats_host->D = s[2];
  stats_host->R_mean = s[3]; stats_host->A = s[4];
  stats_host->axis_radius_traced = s[5]; stats_host->axis_radius_used = s[6]; stats_host->axis_rays_lost = (uint64_t)s[7];
  return GRAY_OK;
}

int gray_noalloc_max_angles(void) { return GRAY_NOALLOC_MAX_ANGLES; }

// gray_shadow_edge without a caller-supplied workspace (gray.h).  Nothing in here allocates or frees: argument checks,
// one address look-up the first time a device is seen, two memsets, two kernels, two small copies to the caller's host
// struct, one stream synchronisation.
int gray_shadow_edge_noalloc(const gray_state* state, int32_t n_angles, double* radius_dev, gray_shadow_stats* stats_host,
                             void* cuda_stream) {
  using namespace gray;
  int rc = check_state(state, true);
  if (rc) return rc;
  if (!stats_host || n_angles < 0) { set_error("stats_host is NULL or n_angles < 0"); return GRAY_ERR_ARG; }
  if (n_angles > GRAY_NOALLOC_MAX_ANGLES) {
    set_error("gray_shadow_edge_noalloc: n_angles = %d is more than the %d spokes the static scratch array holds "
              "(GRAY_NOALLOC_MAX_ANGLES); use gray_shadow_edge with a workspace of your own for more", (int)n_angles,
              (int)GRAY_NOALLOC_MAX_ANGLES);
    return GRAY_ERR_ARG;
  }
  if (state->pixels != GRAY_PIXELS_GRID || state->p0 != 0 || state->nx <= 0 || state->ny <= 0 ||
      state->n != (uint64_t)state->nx * (uint64_t)state->ny) {
    set_error("gray_shadow_edge_noalloc needs a full grid image (pixels = GRID, p0 = 0, n = nx * ny)");
    return GRAY_ERR_ARG;
  }
  NoAllocScratch* scratch = nullptr;
  rc = noalloc_scratch_on_current_device(&scratch);
  if (rc) return rc;
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  Workspace* ws = &scratch->ws;
  // the array still holds the previous call's sums: the cells the reduction adds into start at zero, min_col at the maximum
  GRAY_CUDA(cudaMemsetAsync(&ws->sum_col, 0, (char*)&ws->pad3[0] - (char*)&ws->sum_col, stream));
  GRAY_CUDA(cudaMemsetAsync(&ws->min_col, 0xff, sizeof ws->min_col, stream));
  shadow_reduce_kernel<<<reduce_grid(state->n, 4), 256, 0, stream>>>(state->status_dev, state->n, (unsigned int)state->nx, ws);
  GRAY_CUDA(cudaGetLastError());
  EdgeArgs A;
  A.status = state->status_dev; A.nx = state->nx; A.ny = state->ny; A.W = state->half_width;
  A.n_angles = n_angles; A.radius = radius_dev; A.ws = ws;
  shadow_edge_scratch_kernel<<<1, 1024, 0, stream>>>(A, scratch->rho);
  GRAY_CUDA(cudaGetLastError());
  double s[8];
  unsigned long long ncap = 0;
  GRAY_CUDA(cudaMemcpyAsync(s, &ws->stats[0], sizeof s, cudaMemcpyDeviceToHost, stream));
  GRAY_CUDA(cudaMemcpyAsync(&ncap, &ws->n_captured, sizeof ncap, cudaMemcpyDeviceToHost, stream));
  GRAY_CUDA(cudaStreamSynchronize(stream));
  stats_host->area = s[0]; stats_host->centroid_alpha = s[1]; stats_host->centroid_beta = s[2];
  stats_host->alpha_min = s[3]; stats_host->alpha_max = s[4]; stats_host->D = s[5];
  stats_host->R_mean = s[6]; stats_host->A = s[7];
  stats_host->n_captured = ncap;
  return GRAY_OK;
}

}  // extern "C"
