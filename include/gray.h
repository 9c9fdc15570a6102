/* gray.h — C ABI of libgray: photon null geodesics in Kerr spacetime on one B200 (sm_100a).
 *
 * The hot path of GRay (Chan, Psaltis & Ozel, arXiv 1303.5057; P:<n> = PAPER.md line n):
 * "integrate the second-order geodesic equations" for very many independent photons
 * with a 4th-order Runge-Kutta scheme from an image plane at r = 1000 M
 * until each ray reaches the horizon r_bh = 1 + sqrt(1 - a^2) or
 * leaves; then read the shadow / photon ring off the capture map (eqs. 6-8).
 *
 * Conventions
 *   units           G = c = M = 1 (lengths in gravitational radii)
 *   coordinates     Boyer-Lindquist (t, r, theta, phi); state of a photon = x^mu and k^mu = dx^mu/dlambda
 *   memory          every pointer named *_dev is DEVICE memory owned by the caller (PyTorch tensors in
 *                   the Python binding); the library never allocates, frees or keeps it.  Pointers
 *                   named *_host are HOST memory owned by the caller.  Exceptions, stated where they occur:
 *                   gray_integrate_host keeps two streams and 80 bytes of pinned staging per device; the two
 *                   microbenchmarks gray_fma_peak / gray_packed_peak allocate and free a few KB while they run;
 *                   gray_shadow_edge_noalloc takes no workspace and uses a 128.5 KB array built into the library.
 *   layout          structure of arrays of 16-byte-aligned 4-vectors: x[p] = (t, r, theta, phi),
 *                   k[p] = (k^t, k^r, k^theta, k^phi); float4 for GRAY_F32, 4 doubles for GRAY_F64.
 *   stream          `cuda_stream` is a cudaStream_t passed as void* (NULL = the default stream).  All
 *                   work is enqueued on it.  Functions that return values to *_host pointers
 *                   synchronise that stream before returning and say so below; the others are
 *                   asynchronous.
 *   errors          every function returns GRAY_OK (0) or a negative gray_status and never throws or
 *                   exits; gray_last_error() gives a thread-local message.  Argument errors are
 *                   detected before any launch.  A ray whose state goes non-finite is data, not an
 *                   error: its status becomes GRAY_BAD.
 *   no fallback     there is no CPU path: without a CUDA device every compute entry point returns
 *                   GRAY_ERR_CUDA.
 */
#ifndef GRAY_H_
#define GRAY_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define GRAY_API __attribute__((visibility("default")))
#else
#define GRAY_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  GRAY_OK = 0,
  GRAY_ERR_ARG = -1,         /* null / misaligned pointer, size mismatch, bad enum                  */
  GRAY_ERR_DOMAIN = -2,      /* |a| >= 1, r_obs <= 0, half_width <= 0, h <= 0, inclination out of [0,180] */
  GRAY_ERR_WORKSPACE = -3,   /* workspace missing or smaller than gray_workspace_bytes()            */
  GRAY_ERR_CUDA = -4,        /* CUDA runtime error (message in gray_last_error)                     */
  GRAY_ERR_UNSUPPORTED = -5
} gray_status;

typedef enum { GRAY_F32 = 0, GRAY_F64 = 1 } gray_prec;

/* Step-size rule, evaluated at the start of each step and frozen over its four stages; negative
 * because rays are traced backwards from the observer.
 *   GRAY_STEP_REL  dlambda = -h r                              (BASELINE.json configs, literal)
 *   GRAY_STEP_EQ2  dlambda = -min( h / (|k^r|/r + |k^theta| + |k^phi|), (r - r_bh) / (2 |k^r|) )
 *                  paper eq. (2), with its Delta := h ~ 1/32                          */
typedef enum { GRAY_STEP_REL = 0, GRAY_STEP_EQ2 = 1 } gray_step_rule;

/* Which equations gray_integrate advances (R0, R21).
 *   GRAY_SYS_FULL     all eight: dx^mu/dl = k^mu, dk^mu/dl = -Gamma^mu_ab k^a k^b                  (BASELINE north_star)
 *   GRAY_SYS_REDUCED  the Killing constants E = -k_t and L = k_phi, taken from the photon's state when it is
 *                     loaded, eliminate k^t and k^phi: t and phi obey first-order equations with k^t, k^phi from
 *                     the inverse metric, r and theta the same second-order ones (what the paper's own notation
 *                     suggests GRay integrates).  The stored state keeps all eight components.  */
typedef enum { GRAY_SYS_FULL = 0, GRAY_SYS_REDUCED = 1 } gray_system;

typedef enum { GRAY_LIVE = 0, GRAY_CAPTURED = 1, GRAY_ESCAPED = 2, GRAY_BAD = 3,
               GRAY_EQUATOR = 4 /* reached theta = pi/2 (stop_at_equator only) */ } gray_ray_status;
#define GRAY_N_STATUS 5   /* number of gray_ray_status values = length of gray_classify's counts_host */

/* How photons are mapped to threads by gray_integrate.
 *   GRAY_SCHED_REFILL  persistent warps; a lane whose photon has terminated fetches the next live
 *                      photon from a device-side queue, so warps stay full (in-register stream
 *                      compaction driven by __ballot_sync masks).  Default.
 *   GRAY_SCHED_STATIC  photon p on thread p for the whole call, a warp leaves when all its lanes are
 *                      done (the paper's fixed grid; kept for comparison).
 * Per-photon results are bit-identical for both and for any refill_interval.                       */
typedef enum { GRAY_SCHED_REFILL = 0, GRAY_SCHED_STATIC = 1 } gray_schedule;

typedef enum { GRAY_PIXELS_GRID = 0, GRAY_PIXELS_RANDOM = 1, GRAY_PIXELS_POLAR = 2 } gray_pixels;

/* A batch of photons.  The caller fills the four pointers, n and prec; gray_init_rays* fills the
 * rest (the description of the image plane), which gray_integrate / gray_classify /
 * gray_shadow_edge read.  x and k must be 16-byte aligned.                                          */
typedef struct {
  void* x_dev;            /* n x 4 scalars (t, r, theta, phi)                                        */
  void* k_dev;            /* n x 4 scalars (k^t, k^r, k^theta, k^phi)                                */
  uint8_t* status_dev;    /* n x gray_ray_status                                                     */
  uint32_t* steps_dev;    /* n x RK4 steps taken so far                                              */
  uint64_t n;             /* photons held by these buffers                                           */
  int32_t prec;           /* gray_prec                                                               */
  int32_t pixels;         /* gray_pixels                                                             */
  double a;               /* spin, |a| < 1                                                    */
  double r_obs;           /* distance of the image plane, 1000 M in the paper               */
  double inc_deg;         /* observer inclination i in degrees from the spin axis            */
  double half_width;      /* image plane covers alpha, beta in [-half_width, half_width]             */
  int32_t nx, ny;         /* grid workload: pixels per row (alpha, fast) and rows (beta, slow)       */
  uint64_t seed;          /* random workload: key of the counter-based pixel generator               */
  uint64_t p0;            /* global index of photon 0 of this batch (sharding across GPUs / chunks)  */
  double r_lo;            /* polar workload: inner radius of the image-plane annulus (outer = half_width) */
  void* resume_dev;       /* optional (may be NULL): n x 16 scalars of `prec`, 16-byte aligned, caller-owned.
                             gray_integrate writes a record here for every photon it leaves GRAY_LIVE at
                             max_steps and reads it back when a later call takes that photon up again; see
                             gray_integrate.  Need not be initialised.                                   */
} gray_state;

/* Image plane -> initial photon states ("initial conditions ... as in Psaltis & Johannsen
 * (2012)"; readings R1-R4).  One thread per photon, fp64 arithmetic, rounded to
 * state->prec on store.  Photon j of the batch is global photon p = p0 + j:
 *   grid    pixel centre alpha = -W + (col + 1/2) 2W/nx, beta = -W + (row + 1/2) 2W/ny,
 *           col = p mod nx, row = p / nx; requires p0 + n <= nx * ny
 *   random  (alpha, beta) from the stateless generator of DESIGN.md keyed by (seed, p)
 *   position  r_obs o + alpha yhat + beta bhat,  o = (sin i, 0, cos i), bhat = (-cos i, 0, sin i)
 *   momentum  along +o, k^t from the null condition g_mu_nu k^mu k^nu = 0, normalised to E = -k_t = 1
 * A pixel exactly on the spin axis (inc_deg = 0 or 180 and alpha = beta = 0) gets theta = 0 or pi and
 * k^theta = k^phi = 0 (the limit); Boyer-Lindquist coordinates cannot carry such a ray and gray_integrate
 * ends it GRAY_BAD on its first step.
 * Writes x, k, status = GRAY_LIVE, steps = 0 and the image-plane fields of *state.  Asynchronous.
 * Errors: GRAY_ERR_ARG, GRAY_ERR_DOMAIN (also when half_width is so large that a pixel starts
 * outside 1.01 r_obs), GRAY_ERR_CUDA.                                                               */
GRAY_API int gray_init_rays(gray_state* state, double a, double r_obs, double inc_deg, double half_width,
                   int32_t nx, int32_t ny, uint64_t p0, void* cuda_stream);
GRAY_API int gray_init_rays_random(gray_state* state, double a, double r_obs, double inc_deg, double half_width,
                          uint64_t seed, uint64_t p0, void* cuda_stream);

/* The paper's polar image-plane grid (photon-ring study: "6000 x 181 rays in the polar domain
 * (1.5, 7.5) x [0, pi]"; reading R20).  Photon p of the image: j = p mod n_R, k = p / n_R,
 *   R_j = R_lo + (j + 1/2) (R_hi - R_lo) / n_R,  vartheta_k = k pi / (n_theta - 1),
 *   alpha = R cos(vartheta), beta = R sin(vartheta)  (eqs. 9-10).
 * Everything else as gray_init_rays (state->nx = n_R, ny = n_theta, half_width = R_hi, r_lo = R_lo).
 * Requires n_theta >= 2, 0 <= R_lo < R_hi, p0 + n <= n_R * n_theta.                                  */
GRAY_API int gray_init_rays_polar(gray_state* state, double a, double r_obs, double inc_deg, double R_lo, double R_hi,
                         int32_t n_R, int32_t n_theta, uint64_t p0, void* cuda_stream);

typedef struct {
  double h;                  /* step parameter, the paper's Delta ~ 1/32; > 0, and <= 0.2 with GRAY_STEP_EQ2 */
  double r_capture_factor;   /* captured when r < factor * r_bh (configs: 1.01); if 0, the paper's    */
  double horizon_delta;      /*   r < r_bh + horizon_delta (delta ~ 1e-6) is used instead       */
  double r_escape_factor;    /* escaped when r > factor * r_obs (configs: 1.01)                       */
  int32_t rule;              /* gray_step_rule                                                        */
  int32_t schedule;          /* gray_schedule                                                         */
  int32_t refill_interval;   /* REFILL: RK4 steps between looks at the termination mask (>= 1; 0 = default 8; the full-system
                                kernels take their steps in pairs and round odd values up) */
  int32_t frozen;            /* peak-rate case of BASELINE config 4 (reading R17): every
                                live photon is stepped until its counter reaches max_steps with no
                                early exit; once a test fires its state, status and step count are
                                frozen by select while the arithmetic continues                      */
  int32_t photons_per_thread; /* 0 = default (2 for GRAY_F32, 1 for GRAY_F64); 2 = two photons per thread
                                advanced together by the packed sm_100a FP32 instructions (FFMA2 /
                                FMUL2 / FADD2, GRAY_F32 only); 1 = one photon per thread, scalar
                                instructions.  Per-photon results are bit-identical for 1 and 2.       */
  int32_t stop_at_equator;   /* != 0: the paper's grid-projection workload: a photon stops when it
                                first reaches the equatorial plane.  A step crosses the plane if its start lies
                                on one side (theta <= pi/2 is the upper side) and its end strictly on the other;
                                unless that end state is BAD or CAPTURED, the photon is then landed on the plane
                                by two Newton iterations - ordinary, counted steps of size
                                dlambda = -(theta - pi/2) / k^theta - and gets status GRAY_EQUATOR; the stored
                                state is the one after the second (theta within rounding of pi/2).  Test
                                order: BAD, CAPTURED, EQUATOR, ESCAPED.  The landing steps are taken even when they pass
                                max_steps (by at most 2), as the crossing step itself decides the status.
                                Not available together with `frozen`.                                 */
  double xi_epsilon;         /* > 0: the paper's production pole treatment: after every RK4 step
                                xi of eq. (4) is evaluated at the new state; if |xi + 1| > xi_epsilon (the
                                paper's epsilon ~ 1e-3) or xi is not finite, the step is discarded and
                                re-integrated from the old state as ONE forward Euler step of dlambda / 9,
                                which is not tested itself (reading R18).  0 = off.  Not available
                                together with `frozen`.                                               */
  int32_t system;            /* gray_system; GRAY_SYS_REDUCED excludes frozen, stop_at_equator, xi_epsilon  */
  int32_t reserved;          /* must be 0                                                             */
} gray_step_params;

/* Bytes of device workspace gray_integrate / gray_classify / gray_shadow_edge need (queue head and
 * counters; independent of n today, the argument is kept for layouts that are not).                */
GRAY_API size_t gray_workspace_bytes(uint64_t n);

/* Integrate photons 0 .. n_photons-1 of the batch (n_photons <= state->n) whose status is GRAY_LIVE:
 * repeat { dlambda by the step rule; one classical RK4 step of the 8 equations dx^mu/dlambda = k^mu,
 * dk^mu/dlambda = -Gamma^mu_ab k^a k^b; theta remap of eq. (3); steps += 1; tests in the
 * order non-finite -> GRAY_BAD, r < r_capture -> GRAY_CAPTURED, r > r_escape -> GRAY_ESCAPED } until a
 * test fires or steps == max_steps (the photon then stays GRAY_LIVE and a later call resumes it).  The
 * stored state is the first one that satisfies a test.  x, k, status, steps are updated in place.
 * Resuming (the paper's interactive mode takes "a few steps" per call, P:81 fn 5).  Inside the kernel a photon
 * is carried in variables that the stored (t, r, theta, phi; k) do not hold exactly: the height above the horizon
 * d = r - r_bh, the polar angle folded into [0, pi/2], and (GRAY_F32) the compensation terms of the state update.
 *   state->resume_dev != NULL  these are saved for every photon left LIVE (64 B per photon in fp32, 128 B in fp64)
 *                              and restored by the next call if the record still matches the stored r, theta, k^mu
 *                              and step count bit for bit and was written for the same `system`: any sequence of
 *                              calls with the same parameters then gives results BIT-IDENTICAL to one uninterrupted
 *                              call.  A photon whose stored r, theta, any k^mu or step count the caller has edited,
 *                              or that the previous call advanced with the other gray_system, is re-read from
 *                              (x, k) like a fresh one (an edit of t or phi alone keeps the record: they feed nothing
 *                              back, and the edited value is the one integrated on).
 *   state->resume_dev == NULL  each interruption rounds r and theta once and drops the compensation: results agree
 *                              with the uninterrupted call to rounding error amplified along the ray (within the
 *                              tolerances of the build, tests/test_gpu_parity.py), not bit for bit.
 * Asynchronous.  Counters of the call are left in the workspace for gray_integrate_counters().
 * Errors: GRAY_ERR_ARG, GRAY_ERR_DOMAIN, GRAY_ERR_WORKSPACE, GRAY_ERR_CUDA.                         */
GRAY_API int gray_integrate(gray_state* state, uint64_t n_photons, uint32_t max_steps,
                   const gray_step_params* params, void* workspace_dev, size_t workspace_bytes,
                   void* cuda_stream);

typedef struct {
  uint64_t photon_steps;     /* RK4 steps that advanced a live photon (the unit of BASELINE's metric)  */
  uint64_t issued_steps;     /* lane-steps issued by warps, including idle and frozen lanes            */
  uint64_t photons_done;     /* photons this call brought to CAPTURED / ESCAPED / BAD                  */
  uint64_t photons_live;     /* photons this call left LIVE at max_steps                               */
  uint64_t fallback_steps;   /* steps re-integrated by the xi monitor (xi_epsilon > 0)                 */
} gray_counters;

/* Counters of the last gray_integrate on this workspace.  Synchronises the stream.                  */
GRAY_API int gray_integrate_counters(const void* workspace_dev, gray_counters* counters_host, void* cuda_stream);

/* Per-pixel capture flags (capture_map[p] = 1 iff status[p] == GRAY_CAPTURED, else 0; may be NULL)
 * and the number of photons in each gray_ray_status: counts_host[s], s = GRAY_LIVE .. GRAY_EQUATOR
 * (GRAY_N_STATUS = 5 entries; a status byte outside that range is counted nowhere, so the counts sum
 * to n exactly when every byte is a valid status).  Synchronises the stream.                        */
GRAY_API int gray_classify(const gray_state* state, uint8_t* capture_map_dev, uint64_t counts_host[GRAY_N_STATUS],
                  void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* Shadow / photon-ring statistics of a grid image (reading R13):
 *   area = N_captured dalpha dbeta; centroid = mean (alpha, beta) of captured pixel centres;
 *   alpha_min / alpha_max = outer edges of the extreme captured columns; D = |alpha_min + alpha_max| / 2
 *   (eq. 6); rho(vartheta_k), k = 0 .. n_angles-1, vartheta_k = 2 pi (k + 1/2) / n_angles about the image
 *   origin: marching outwards in steps of half a pixel, the mid-point between the last sample whose
 *   pixel is captured and the first whose pixel is not; R_k = distance of that point from
 *   ((alpha_min + alpha_max)/2, 0); R_mean = mean R_k (eq. 7); A = 2 std R_k (eq. 8).                */
typedef struct {
  double area, centroid_alpha, centroid_beta, alpha_min, alpha_max, D, R_mean, A;
  uint64_t n_captured;
} gray_shadow_stats;

/* Requires a full grid batch (pixels == GRAY_PIXELS_GRID, p0 == 0, n == nx * ny).  radius_dev
 * (n_angles doubles) may be NULL.  Synchronises the stream.                                         */
GRAY_API int gray_shadow_edge(const gray_state* state, int32_t n_angles, double* radius_dev,
                     gray_shadow_stats* stats_host, void* workspace_dev, size_t workspace_bytes,
                     void* cuda_stream);

/* gray_shadow_edge for callers that cannot allocate device memory, and so have no workspace_dev to pass.
 *
 * Who that is: code that runs on a GPU whose memory it does not manage.  A plug-in inside a host program (a
 * visualisation tool, a simulation that calls libgray in situ) is typically handed its device buffers and forbidden
 * cudaMalloc, because the host program gave the whole device to its own pool; a worker inside a fixed memory slice
 * (MIG, an MPS limit, a scheduler's quota) that the photon buffers already fill has nothing left to ask for; and a
 * frame loop like the paper's interactive mode cannot afford cudaMalloc / cudaFree, which stall every stream of
 * the device while they run.  Every other entry point of this header expects such a caller to have set a workspace
 * aside in advance; this one needs none.
 *
 * What it computes: exactly gray_shadow_edge (same statistics, same radius_dev[k], eqs. 6-8), from the
 * same inputs (state: a full grid batch) into the same outputs (radius_dev, optional; stats_host).  The scratch memory
 * the computation needs - the reduction cells and one radius per spoke - is an array built into libgray's device
 * image: 512 B + 8 B x GRAY_NOALLOC_MAX_ANGLES = 128.5 KB, which every GPU that loads the library holds from then
 * until the process exits, used or not.  That is why the limit is modest: n_angles > GRAY_NOALLOC_MAX_ANGLES
 * (also returned by gray_noalloc_max_angles()) is refused with GRAY_ERR_ARG and a message that says so, before
 * anything is launched; gray_shadow_edge with a workspace has no such limit.
 *
 * The call performs no cudaMalloc, cudaFree, cudaHostAlloc, stream / event creation or any other allocating
 * runtime or library routine: argument checks, two cudaMemsetAsync, two kernels, two 64-byte copies into
 * *stats_host, one cudaStreamSynchronize.
 *
 * First call on a device: the library asks the runtime where that device's copy of the array lives
 * (cudaGetSymbolAddress, checked; each GPU has its own copy, so this is done once per device, with the device the
 * caller has made current) and remembers the answer.  That look-up is a set-up step, not stream work: make the first
 * call on each device early - before any stream capture is begun on it - and from then on the call only enqueues.
 *
 * One array per GPU, shared by every call: it still holds what the previous call left.  The cells that must start
 * from zero (the sums, the captured count, the extreme columns) are cleared on `cuda_stream` at the start of each
 * call and every spoke's radius is written before it is read, so consecutive calls on one stream, or calls
 * separated by a synchronisation, are independent of each other.  Two calls of one process that can run on the
 * same GPU at the same time (different streams, different host threads) write the same cells and RACE: serialise
 * them yourself.  Another process has loaded its own copy of the array and does not interfere.
 * Synchronises the stream.  Errors: GRAY_ERR_ARG (as gray_shadow_edge, or n_angles over the limit),
 * GRAY_ERR_UNSUPPORTED (device ordinal >= 64), GRAY_ERR_CUDA.                                           */
#define GRAY_NOALLOC_MAX_ANGLES 16384
GRAY_API int gray_noalloc_max_angles(void);
GRAY_API int gray_shadow_edge_noalloc(const gray_state* state, int32_t n_angles, double* radius_dev,
                             gray_shadow_stats* stats_host, void* cuda_stream);

/* Photon-ring statistics of a polar image (eqs. 6-10).  radius[k] = ring radius on spoke k: the outer
 * edge of the outermost captured cell (R_lo if none is captured).  alpha_max = radius[0], alpha_min = -radius[n_theta - 1]; D = |alpha_min + alpha_max| / 2
 * (eq. 6); R = [(alpha_0 - c)^2 + beta_0^2]^(1/2) about the ring centre c = (alpha_min + alpha_max)/2; R_mean (eq. 7)
 * and A (eq. 8) with the integrals over [0, pi] (the image is symmetric under beta -> -beta) by the trapezoidal
 * rule on the n_theta spokes.  bridge_axis != 0 (n_theta odd): the middle spoke vartheta = pi/2 has alpha = 0, its rays
 * run through the spin axis, the degenerate case of Boyer-Lindquist coordinates in which the second-order equations
 * lose rays even with the xi monitor (R20); its radius is then replaced by the mean of its two neighbours
 * before the statistics are formed; what the spoke's own rays gave is reported next to it (axis_radius_traced,
 * axis_rays_lost), so a caller sees an interpolated value for what it is.  Requires a full polar batch.  radius_dev
 * (n_theta doubles) may be NULL.  Synchronises the stream.                                                                             */
typedef struct {
  double alpha_min, alpha_max, D, R_mean, A;
  double axis_radius_traced;   /* n_theta odd: ring radius on the axis spoke vartheta = pi/2 as the rays gave it ...        */
  double axis_radius_used;     /* ... and the one the statistics used (the neighbours' mean if bridge_axis, else the same)  */
  uint64_t axis_rays_lost;     /* rays of that spoke that ended neither CAPTURED nor ESCAPED (BAD, or LIVE at the cap)     */
} gray_ring_stats;
GRAY_API int gray_ring_polar(const gray_state* state, int32_t bridge_axis, double* radius_dev, gray_ring_stats* stats_host,
                    void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* End-to-end variant with HOST buffers (bench.py's `e2e` figure).  n photons whose initial states are
 * x_in_host / k_in_host (n x 4 scalars of `prec`, status LIVE, steps 0 implied) are streamed through
 * the GPU in chunks of `chunk` photons on two internal streams, so that the host->device copy of one
 * chunk and the device->host copy of another overlap the integration of a third: copy in, gray_integrate
 * semantics with (a, r_obs, params, max_steps), copy out.  Results: x_out_host, k_out_host (may alias the
 * inputs), status_host (n bytes), steps_host (n).  Host buffers should be pinned (cudaHostAlloc /
 * torch pin_memory) for the copies to be asynchronous.  scratch_dev must hold
 * gray_host_scratch_bytes(chunk, prec) bytes of device memory, 256-byte aligned.  counters_host (may be
 * NULL) receives the summed gray_counters.  Synchronous: returns when every result is in host memory.
 * Ordering: the internal streams start after everything enqueued so far on `cuda_stream` (NULL = the default
 * stream), so inputs or scratch written by earlier work on that stream are safe.  The two streams, one event and
 * 80 bytes of pinned host staging are created on the first call on a device and kept for the life of the process
 * (the only resources the library ever keeps); concurrent calls are serialised.  After an error every chunk
 * already enqueued is still waited for before the function returns, and counters_host holds the chunks completed. */
GRAY_API size_t gray_host_scratch_bytes(uint64_t chunk, int32_t prec);
GRAY_API int gray_integrate_host(const void* x_in_host, const void* k_in_host, void* x_out_host, void* k_out_host,
                        uint8_t* status_host, uint32_t* steps_host, uint64_t n, int32_t prec, double a,
                        double r_obs, uint32_t max_steps, const gray_step_params* params, uint64_t chunk,
                        void* scratch_dev, size_t scratch_bytes, gray_counters* counters_host, void* cuda_stream);

/* Register-only FFMA (GRAY_F32) or DFMA (GRAY_F64) microbenchmark: the measured CUDA-core peak the
 * integrator's rate is divided by.  Runs `iters` dependent-chain-free FMA rounds
 * on every SM, times them with CUDA events on the stream, returns FLOP/s (FMA = 2).  Synchronises.
 * Allocates 8 bytes of device memory (cudaMalloc) for the duration of the call and frees them.      */
GRAY_API int gray_fma_peak(int32_t prec, int32_t iters, double* flops_per_s_host, void* cuda_stream);

/* Packed FP32 (FFMA2 / FMUL2 / FADD2, the instructions of the GRAY_F32 integrator) register-only microbenchmark,
 * 16 warps per SM like the integrator: the rate at which the FP32 pipe retires packed instructions depends on how
 * many distinct register pairs an instruction reads (register-file bandwidth), which bounds the integrator below
 * the FFMA peak.
 *   mix 0  FFMA2 x <- x * m + c with loop-invariant m, c
 *   mix 1  FFMA2 reading three different, changing register pairs
 *   mix 2  round 1's instruction mix: 50 % FMUL2, 37.5 % FFMA2 (three pairs), 12.5 % FADD2
 *   mix 3  FMUL2 reading two changing pairs            mix 4  FFMA2 x <- x * x' + x (two distinct pairs)
 *   mix 5  the full-system integrator's packed instructions as they stand (per 16: 7 FMUL2, 3 FFMA2 with three pairs,
 *          3 FFMA2 with two pairs and a launch constant, 2 FADD2, 1 FADD2 with a constant)
 *   mix 6  mix 5 plus the other instructions the integrator issues beside them (per 16 packed: ~1.2 MUFU.RCP and
 *          ~5 integer / select / move instructions): the rate the integrator's loop can reach at best
 * Returns packed fp32 lane-operations per second (one packed instruction = 2 per thread; multiply by 2 for FMA flops of
 * mix 0 / 1 / 4); the extra instructions of mix 6 are not counted.
 * Synchronises.  Allocates 8 KB of device memory (cudaMalloc) for the duration of the call and frees them.   */
GRAY_API int gray_packed_peak(int32_t mix, int32_t iters, double* lane_ops_per_s_host, void* cuda_stream);

/* Device facts used by the benchmark: SM count and SM clock (kHz) reported by the runtime.         */
GRAY_API int gray_device_info(int32_t* sm_count_host, int32_t* sm_clock_khz_host);

GRAY_API const char* gray_last_error(void);   /* thread-local, valid until the next call on this thread       */
GRAY_API const char* gray_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GRAY_H_ */
