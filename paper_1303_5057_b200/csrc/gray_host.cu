// gray_host.cu — gray_integrate_host (include/gray.h): host buffers in, host buffers out, chunks
// double-buffered over two streams so PCIe copies overlap the integrator kernel.
#include "gray_internal.h"

#include <mutex>

namespace gray {

struct Slot {
  char* x; char* k; uint32_t* steps; uint8_t* status; Workspace* ws;
  cudaStream_t stream;
  unsigned long long* c;     // counters of the chunk last run on this slot (pinned host staging)
  bool in_flight;            // a chunk has been enqueued on this slot and not drained yet
};

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

static size_t slot_bytes(uint64_t chunk, int prec) {
  const size_t vec = (prec == GRAY_F32 ? 16 : 32);
  return align256(chunk * vec) * 2 + align256(chunk * 4) + align256(chunk) + align256(sizeof(Workspace));
}

// The two copy / compute streams, the event that orders them after the caller's stream and the pinned staging of the
// counters are created once per device, on the first call, and kept for the life of the process (they are not
// device memory: 80 bytes of pinned host memory and three driver handles).  Calls are serialised by a mutex.
struct HostPath {
  bool ready = false;
  cudaStream_t stream[2] = {nullptr, nullptr};
  cudaEvent_t caller_done = nullptr;
  unsigned long long* pinned = nullptr;
};
static std::mutex g_host_mutex;
static HostPath g_host_path[64];

static int host_path(HostPath** out) {
  int dev = 0;
  GRAY_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) { set_error("gray_integrate_host: device index %d out of range", dev); return GRAY_ERR_CUDA; }
  HostPath& H = g_host_path[dev];
  if (!H.ready) {
    HostPath T;
    cudaError_t e = cudaHostAlloc(&T.pinned, 10 * sizeof(unsigned long long), cudaHostAllocDefault);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&T.stream[0], cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&T.stream[1], cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&T.caller_done, cudaEventDisableTiming);
    if (e != cudaSuccess) {
      if (T.caller_done) cudaEventDestroy(T.caller_done);
      for (int s = 0; s < 2; ++s) if (T.stream[s]) cudaStreamDestroy(T.stream[s]);
      if (T.pinned) cudaFreeHost(T.pinned);
      return cuda_fail(e, "gray_integrate_host: creating streams / pinned staging");
    }
    T.ready = true;
    H = T;
  }
  *out = &H;
  return GRAY_OK;
}

}  // namespace gray

extern "C" {

size_t gray_host_scratch_bytes(uint64_t chunk, int32_t prec) { return 2 * gray::slot_bytes(chunk, prec); }

int gray_integrate_host(const void* x_in_host, const void* k_in_host, void* x_out_host, void* k_out_host,
                        uint8_t* status_host, uint32_t* steps_host, uint64_t n, int32_t prec, double a, double r_obs,
                        uint32_t max_steps, const gray_step_params* params, uint64_t chunk, void* scratch_dev,
                        size_t scratch_bytes, gray_counters* counters_host, void* cuda_stream) {
  using namespace gray;
  if (prec != GRAY_F32 && prec != GRAY_F64) { set_error("bad precision"); return GRAY_ERR_ARG; }
  if (!params) { set_error("params is NULL"); return GRAY_ERR_ARG; }
  if (counters_host) *counters_host = gray_counters{0, 0, 0, 0, 0};
  if (n == 0) return GRAY_OK;
  if (!x_in_host || !k_in_host || !x_out_host || !k_out_host || !status_host || !steps_host) { set_error("NULL host buffer"); return GRAY_ERR_ARG; }
  if (chunk == 0) { set_error("chunk must be positive"); return GRAY_ERR_ARG; }
  if (chunk > n) chunk = n;
  if (!scratch_dev || ((uintptr_t)scratch_dev & 255) || scratch_bytes < gray_host_scratch_bytes(chunk, prec)) {
    set_error("scratch_dev is NULL, not 256-byte aligned or smaller than gray_host_scratch_bytes()");
    return GRAY_ERR_WORKSPACE;
  }
  std::lock_guard<std::mutex> lock(g_host_mutex);
  HostPath* H = nullptr;
  int rc = host_path(&H);
  if (rc) return rc;
  // everything the caller has enqueued on its stream so far (e.g. the kernel that produced scratch_dev's previous
  // contents, or a copy into the host inputs) comes before the first copy in
  GRAY_CUDA(cudaEventRecord(H->caller_done, (cudaStream_t)cuda_stream));
  const size_t vec = (prec == GRAY_F32 ? 16 : 32);
  Slot slot[2];
  char* base = (char*)scratch_dev;
  for (int s = 0; s < 2; ++s) {
    char* p = base + s * slot_bytes(chunk, prec);
    slot[s].x = p; p += align256(chunk * vec);
    slot[s].k = p; p += align256(chunk * vec);
    slot[s].steps = (uint32_t*)p; p += align256(chunk * 4);
    slot[s].status = (uint8_t*)p; p += align256(chunk);
    slot[s].ws = (Workspace*)p;
    slot[s].c = H->pinned + 5 * s;
    slot[s].stream = H->stream[s];
    slot[s].in_flight = false;
    GRAY_CUDA(cudaStreamWaitEvent(slot[s].stream, H->caller_done, 0));
  }
  gray_counters total = {0, 0, 0, 0, 0};
  // wait for the chunk in flight on slot s (if any) and add its counters; each chunk is drained exactly once
  auto drain = [&](int s, bool count) -> int {
    if (!slot[s].in_flight) return GRAY_OK;
    slot[s].in_flight = false;
    cudaError_t e = cudaStreamSynchronize(slot[s].stream);
    if (e != cudaSuccess) return cuda_fail(e, "gray_integrate_host: cudaStreamSynchronize");
    if (count) {
      total.photon_steps += slot[s].c[0]; total.issued_steps += slot[s].c[1];
      total.photons_done += slot[s].c[2]; total.photons_live += slot[s].c[3];
      total.fallback_steps += slot[s].c[4];
    }
    return GRAY_OK;
  };
  uint64_t chunk_index = 0;
  for (uint64_t lo = 0; lo < n && rc == GRAY_OK; lo += chunk, ++chunk_index) {
    const int s = (int)(chunk_index & 1);
    const uint64_t m = (n - lo < chunk) ? n - lo : chunk;
    Slot& S = slot[s];
    rc = drain(s, true);
    if (rc) break;
    S.in_flight = true;          // from here on something may be enqueued on the slot's stream
    cudaError_t e;
    e = cudaMemcpyAsync(S.x, (const char*)x_in_host + lo * vec, m * vec, cudaMemcpyHostToDevice, S.stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(S.k, (const char*)k_in_host + lo * vec, m * vec, cudaMemcpyHostToDevice, S.stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(S.status, GRAY_LIVE, m, S.stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(S.steps, 0, m * 4, S.stream);
    if (e != cudaSuccess) { rc = cuda_fail(e, "gray_integrate_host: copy in"); break; }
    gray_state st;
    st.x_dev = S.x; st.k_dev = S.k; st.status_dev = S.status; st.steps_dev = S.steps;
    st.n = m; st.prec = prec; st.pixels = GRAY_PIXELS_GRID;
    st.a = a; st.r_obs = r_obs; st.inc_deg = 0; st.half_width = 0; st.nx = st.ny = 0; st.seed = 0; st.p0 = lo; st.r_lo = 0; st.resume_dev = nullptr;
    rc = gray_integrate(&st, m, max_steps, params, S.ws, sizeof(Workspace), S.stream);
    if (rc) break;
    e = cudaMemcpyAsync((char*)x_out_host + lo * vec, S.x, m * vec, cudaMemcpyDeviceToHost, S.stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync((char*)k_out_host + lo * vec, S.k, m * vec, cudaMemcpyDeviceToHost, S.stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(status_host + lo, S.status, m, cudaMemcpyDeviceToHost, S.stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(steps_host + lo, S.steps, m * 4, cudaMemcpyDeviceToHost, S.stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(S.c, &S.ws->photon_steps, 5 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, S.stream);
    if (e != cudaSuccess) { rc = cuda_fail(e, "gray_integrate_host: copy out"); break; }
  }
  // epilogue: whatever is still in flight, in order; after an error the counters of incomplete chunks are not added
  for (int q = 0; q < 2; ++q) {
    const int s = (int)((chunk_index + q) & 1);
    const int r2 = drain(s, rc == GRAY_OK);
    if (rc == GRAY_OK) rc = r2;
  }
  if (counters_host) *counters_host = total;
  return rc;
}

}  // extern "C"
