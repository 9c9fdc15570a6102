// gray_api.cu — error reporting, argument checks, workspace size, device facts and the FMA-peak
// microbenchmark of libgray (include/gray.h).
#include <stdarg.h>
#include <string.h>

#include "gray_internal.h"

namespace gray {

static thread_local char g_err[512] = "";

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
}

int cuda_fail(cudaError_t e, const char* what) {
  set_error("CUDA error %d (%s) in %s", (int)e, cudaGetErrorString(e), what);
  return GRAY_ERR_CUDA;
}

int check_state(const gray_state* st, bool need_image_fields) {
  if (!st) { set_error("state is NULL"); return GRAY_ERR_ARG; }
  if (st->prec != GRAY_F32 && st->prec != GRAY_F64) { set_error("state.prec must be GRAY_F32 or GRAY_F64"); return GRAY_ERR_ARG; }
  if (st->n == 0) return GRAY_OK;   // empty batch: nothing is dereferenced
  if (!st->x_dev || !st->k_dev || !st->status_dev || !st->steps_dev) { set_error("state has a NULL device pointer"); return GRAY_ERR_ARG; }
  if (((uintptr_t)st->x_dev & 15) || ((uintptr_t)st->k_dev & 15)) { set_error("state.x_dev / k_dev must be 16-byte aligned"); return GRAY_ERR_ARG; }
  if ((uintptr_t)st->steps_dev & 3) { set_error("state.steps_dev must be 4-byte aligned"); return GRAY_ERR_ARG; }
  if (need_image_fields) {
    if (!(st->a > -1.0 && st->a < 1.0) || !(st->r_obs > 0.0)) { set_error("state image-plane fields are not initialised (call gray_init_rays first)"); return GRAY_ERR_ARG; }
  }
  return GRAY_OK;
}

int check_workspace(const void* ws, size_t bytes) {
  if (!ws || bytes < sizeof(Workspace)) { set_error("workspace is NULL or smaller than gray_workspace_bytes() = %zu", sizeof(Workspace)); return GRAY_ERR_WORKSPACE; }
  if ((uintptr_t)ws & 15) { set_error("workspace must be 16-byte aligned"); return GRAY_ERR_WORKSPACE; }
  return GRAY_OK;
}

int sm_count() {
  static int n = 0;
  if (n == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) n = 0;
  }
  return n;
}

// Register-only FMA throughput: 16 independent accumulators per thread, 2 FMAs each per round.
template <typename T>
__global__ void __launch_bounds__(256) fma_peak_kernel(int iters, T seed, T* sink) {
  T acc[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) acc[i] = seed + T(i) + T(threadIdx.x) * T(1e-3);
  const T m = T(0.999), b = seed * T(1e-7);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = acc[i] * m + b;
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = acc[i] * b + m;
  }
  T s = T(0);
#pragma unroll
  for (int i = 0; i < 16; ++i) s += acc[i];
  if (s == T(-12345.678)) sink[0] = s;   // never true; keeps the loop alive
}

template <typename T>
static int fma_peak(int iters, double* out, cudaStream_t stream) {
  const int sms = sm_count();
  if (sms <= 0) { set_error("no CUDA device"); return GRAY_ERR_CUDA; }
  const int blocks = sms * 8, threads = 256;
  T* sink = nullptr;
  GRAY_CUDA(cudaMalloc(&sink, sizeof(T)));   // 8 bytes of scratch for the benchmark only
  cudaEvent_t e0, e1;
  GRAY_CUDA(cudaEventCreate(&e0));
  GRAY_CUDA(cudaEventCreate(&e1));
  fma_peak_kernel<T><<<blocks, threads, 0, stream>>>(iters / 8 + 1, T(1.5), sink);   // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, stream);
    fma_peak_kernel<T><<<blocks, threads, 0, stream>>>(iters, T(1.5), sink);
    cudaEventRecord(e1, stream);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) { cudaFree(sink); return cuda_fail(e, "fma_peak_kernel"); }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  const double flops = 2.0 * 32.0 * (double)iters * (double)blocks * (double)threads;
  *out = flops / (best * 1e-3);
  return GRAY_OK;
}

}  // namespace gray

extern "C" {

const char* gray_last_error(void) { return gray::g_err; }
const char* gray_version(void) { return "libgray 0.1 (sm_100a)"; }

size_t gray_workspace_bytes(uint64_t) { return sizeof(gray::Workspace); }

int gray_device_info(int32_t* sm_count_host, int32_t* sm_clock_khz_host) {
  int dev = 0, sms = 0, khz = 0;
  GRAY_CUDA(cudaGetDevice(&dev));
  GRAY_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  GRAY_CUDA(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
  if (sm_count_host) *sm_count_host = sms;
  if (sm_clock_khz_host) *sm_clock_khz_host = khz;
  return GRAY_OK;
}

int gray_fma_peak(int32_t prec, int32_t iters, double* flops_per_s_host, void* cuda_stream) {
  if (!flops_per_s_host || iters <= 0) { gray::set_error("gray_fma_peak: bad arguments"); return GRAY_ERR_ARG; }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (prec == GRAY_F32) return gray::fma_peak<float>(iters, flops_per_s_host, s);
  if (prec == GRAY_F64) return gray::fma_peak<double>(iters, flops_per_s_host, s);
  gray::set_error("gray_fma_peak: bad precision");
  return GRAY_ERR_ARG;
}

}  // extern "C"
