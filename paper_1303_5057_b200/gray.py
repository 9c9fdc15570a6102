"""ctypes binding of libgray (include/gray.h): argument marshalling only.

Function names are those of the C ABI.  Device buffers are torch tensors owned by the caller
(`PhotonBatch` allocates them with torch.empty); the stream is torch's current CUDA stream.
"""
import ctypes as C
import os

import torch

GRAY_F32, GRAY_F64 = 0, 1
STEP_REL, STEP_EQ2 = 0, 1
SYS_FULL, SYS_REDUCED = 0, 1
LIVE, CAPTURED, ESCAPED, BAD, EQUATOR = 0, 1, 2, 3, 4
N_STATUS = 5
SCHED_REFILL, SCHED_STATIC = 0, 1
PIXELS_GRID, PIXELS_RANDOM, PIXELS_POLAR = 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


class GrayError(RuntimeError):
    pass


class _State(C.Structure):
    _fields_ = [("x_dev", C.c_void_p), ("k_dev", C.c_void_p), ("status_dev", C.c_void_p), ("steps_dev", C.c_void_p),
                ("n", C.c_uint64), ("prec", C.c_int32), ("pixels", C.c_int32), ("a", C.c_double),
                ("r_obs", C.c_double), ("inc_deg", C.c_double), ("half_width", C.c_double), ("nx", C.c_int32),
                ("ny", C.c_int32), ("seed", C.c_uint64), ("p0", C.c_uint64), ("r_lo", C.c_double), ("resume_dev", C.c_void_p)]


class _StepParams(C.Structure):
    _fields_ = [("h", C.c_double), ("r_capture_factor", C.c_double), ("horizon_delta", C.c_double),
                ("r_escape_factor", C.c_double), ("rule", C.c_int32), ("schedule", C.c_int32),
                ("refill_interval", C.c_int32), ("frozen", C.c_int32), ("photons_per_thread", C.c_int32),
                ("stop_at_equator", C.c_int32), ("xi_epsilon", C.c_double), ("system", C.c_int32), ("reserved", C.c_int32)]


class _Counters(C.Structure):
    _fields_ = [("photon_steps", C.c_uint64), ("issued_steps", C.c_uint64), ("photons_done", C.c_uint64),
                ("photons_live", C.c_uint64), ("fallback_steps", C.c_uint64)]


class _RingStats(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("alpha_min", "alpha_max", "D", "R_mean", "A", "axis_radius_traced", "axis_radius_used")] + \
               [("axis_rays_lost", C.c_uint64)]


class _ShadowStats(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("area", "centroid_alpha", "centroid_beta", "alpha_min", "alpha_max", "D",
                                           "R_mean", "A")] + [("n_captured", C.c_uint64)]


def lib_path():
    return os.path.join(_HERE, "libgray.so")


def lib():
    """Load libgray.so (built in-tree by `python -m paper_1303_5057_b200.build`).  Raises if it is missing."""
    global _LIB
    if _LIB is None:
        path = lib_path()
        if not os.path.exists(path):
            raise GrayError(f"{path} not found: build it with `python -m paper_1303_5057_b200.build` "
                            "(there is no CPU fallback)")
        L = C.CDLL(path)
        vp, u64, i32, dbl = C.c_void_p, C.c_uint64, C.c_int32, C.c_double
        L.gray_init_rays.argtypes = [C.POINTER(_State), dbl, dbl, dbl, dbl, i32, i32, u64, vp]
        L.gray_init_rays_polar.argtypes = [C.POINTER(_State), dbl, dbl, dbl, dbl, dbl, i32, i32, u64, vp]
        L.gray_ring_polar.argtypes = [C.POINTER(_State), i32, vp, C.POINTER(_RingStats), vp, C.c_size_t, vp]
        L.gray_init_rays_random.argtypes = [C.POINTER(_State), dbl, dbl, dbl, dbl, u64, u64, vp]
        L.gray_workspace_bytes.argtypes = [u64]
        L.gray_workspace_bytes.restype = C.c_size_t
        L.gray_integrate.argtypes = [C.POINTER(_State), u64, C.c_uint32, C.POINTER(_StepParams), vp, C.c_size_t, vp]
        L.gray_integrate_counters.argtypes = [vp, C.POINTER(_Counters), vp]
        L.gray_classify.argtypes = [C.POINTER(_State), vp, C.POINTER(u64), vp, C.c_size_t, vp]
        L.gray_shadow_edge.argtypes = [C.POINTER(_State), i32, vp, C.POINTER(_ShadowStats), vp, C.c_size_t, vp]
        L.gray_shadow_edge_noalloc.argtypes = [C.POINTER(_State), i32, vp, C.POINTER(_ShadowStats), vp]
        L.gray_shadow_edge_noalloc.restype = C.c_int
        L.gray_noalloc_max_angles.argtypes = []
        L.gray_noalloc_max_angles.restype = C.c_int
        L.gray_host_scratch_bytes.argtypes = [u64, i32]
        L.gray_host_scratch_bytes.restype = C.c_size_t
        L.gray_integrate_host.argtypes = [vp, vp, vp, vp, vp, vp, u64, i32, dbl, dbl, C.c_uint32, C.POINTER(_StepParams),
                                          u64, vp, C.c_size_t, C.POINTER(_Counters), vp]
        L.gray_fma_peak.argtypes = [i32, i32, C.POINTER(dbl), vp]
        L.gray_packed_peak.argtypes = [i32, i32, C.POINTER(dbl), vp]
        L.gray_device_info.argtypes = [C.POINTER(i32), C.POINTER(i32)]
        L.gray_last_error.restype = C.c_char_p
        L.gray_version.restype = C.c_char_p
        for name in ("gray_init_rays", "gray_init_rays_random", "gray_init_rays_polar", "gray_ring_polar", "gray_integrate", "gray_integrate_counters",
                     "gray_classify", "gray_shadow_edge", "gray_fma_peak", "gray_packed_peak", "gray_device_info", "gray_integrate_host"):
            getattr(L, name).restype = C.c_int
        _LIB = L
    return _LIB


def _check(rc):
    if rc != 0:
        raise GrayError(f"libgray error {rc}: {lib().gray_last_error().decode()}")


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


class StepParams:
    """gray_step_params (include/gray.h).  Defaults: the BASELINE configs' h, capture and escape radii."""

    def __init__(self, h=1.0 / 32, r_capture_factor=1.01, horizon_delta=1e-6, r_escape_factor=1.01, rule=STEP_EQ2,
                 schedule=SCHED_REFILL, refill_interval=0, frozen=False, photons_per_thread=0, xi_epsilon=0.0, stop_at_equator=False,
                 system=SYS_FULL):
        self.c = _StepParams(h, r_capture_factor, horizon_delta, r_escape_factor, rule, schedule, refill_interval,
                             int(bool(frozen)), photons_per_thread, int(bool(stop_at_equator)), xi_epsilon, system, 0)


class PhotonBatch:
    """Caller-owned device buffers of a gray_state: x, k (n x 4), status (n, uint8), steps (n, int32 bits of
    a uint32) and the workspace.  Memory comes from torch; nothing else does."""

    def __init__(self, n, prec=GRAY_F32, device="cuda", resumable=False):
        if not torch.cuda.is_available():
            raise GrayError("no CUDA device: libgray has no CPU path")
        dt = torch.float32 if prec == GRAY_F32 else torch.float64
        self.n, self.prec = int(n), prec
        self.x = torch.empty((self.n, 4), dtype=dt, device=device)
        self.k = torch.empty((self.n, 4), dtype=dt, device=device)
        self.status = torch.empty((self.n,), dtype=torch.uint8, device=device)
        self.steps = torch.empty((self.n,), dtype=torch.int32, device=device)
        self.workspace = torch.zeros((gray_workspace_bytes(self.n),), dtype=torch.uint8, device=device)
        # gray_state.resume_dev (include/gray.h): makes interrupted gray_integrate calls bit-identical to one call
        self.resume = torch.empty((self.n, 16), dtype=dt, device=device) if resumable else None
        self.c = _State(self.x.data_ptr(), self.k.data_ptr(), self.status.data_ptr(), self.steps.data_ptr(),
                        self.n, prec, 0, 0.0, 0.0, 0.0, 0.0, 0, 0, 0, 0, 0.0,
                        self.resume.data_ptr() if resumable else None)

    def set_image_plane(self, a, r_obs, inc_deg, half_width, nx=0, ny=0, seed=0, p0=0, pixels=PIXELS_GRID):
        """Describe the image plane without running gray_init_rays (for states uploaded by the caller)."""
        self.c.a, self.c.r_obs, self.c.inc_deg, self.c.half_width = a, r_obs, inc_deg, half_width
        self.c.nx, self.c.ny, self.c.seed, self.c.p0, self.c.pixels = nx, ny, seed, p0, pixels


def _slice(self, lo, hi):
    """A batch over photons lo .. hi-1 of this one, sharing its buffers (its own workspace and image-plane fields): several
    images that differ only in what gray_integrate does not read (inclination, pixel grid) can be initialised slice by slice,
    integrated in ONE launch over the parent batch, and evaluated slice by slice."""
    lo, hi = int(lo), int(hi)
    if not 0 <= lo <= hi <= self.n:
        raise GrayError("slice out of range")
    v = object.__new__(PhotonBatch)
    v.n, v.prec = hi - lo, self.prec
    v.x, v.k, v.status, v.steps = self.x[lo:hi], self.k[lo:hi], self.status[lo:hi], self.steps[lo:hi]
    v.workspace = torch.zeros_like(self.workspace)
    v.resume = self.resume[lo:hi] if self.resume is not None else None
    v.c = _State(v.x.data_ptr(), v.k.data_ptr(), v.status.data_ptr(), v.steps.data_ptr(), v.n, v.prec, self.c.pixels,
                 self.c.a, self.c.r_obs, self.c.inc_deg, self.c.half_width, self.c.nx, self.c.ny, self.c.seed, self.c.p0 + lo,
                 self.c.r_lo, v.resume.data_ptr() if v.resume is not None else None)
    return v


PhotonBatch.slice = _slice


def gray_workspace_bytes(n):
    return int(lib().gray_workspace_bytes(int(n)))


def gray_version():
    return lib().gray_version().decode()


def gray_init_rays(batch, a, r_obs, inc_deg, half_width, nx, ny, p0=0):
    _check(lib().gray_init_rays(C.byref(batch.c), a, r_obs, inc_deg, half_width, nx, ny, p0, _stream()))


def gray_init_rays_polar(batch, a, r_obs, inc_deg, R_lo, R_hi, n_R, n_theta, p0=0):
    _check(lib().gray_init_rays_polar(C.byref(batch.c), a, r_obs, inc_deg, R_lo, R_hi, n_R, n_theta, p0, _stream()))


def gray_ring_polar(batch, radius=None, bridge_axis=False):
    """Returns the gray_ring_stats as a dict; fills radius (float64 tensor of n_theta) if given."""
    s = _RingStats()
    _check(lib().gray_ring_polar(C.byref(batch.c), int(bool(bridge_axis)), _ptr(radius), C.byref(s), _ptr(batch.workspace),
                                 batch.workspace.numel(), _stream()))
    return {k: getattr(s, k) for k, _ in _RingStats._fields_}


def gray_init_rays_random(batch, a, r_obs, inc_deg, half_width, seed, p0=0):
    _check(lib().gray_init_rays_random(C.byref(batch.c), a, r_obs, inc_deg, half_width, seed, p0, _stream()))


def gray_integrate(batch, n_photons=None, max_steps=20000, params=None):
    params = params or StepParams()
    n = batch.n if n_photons is None else int(n_photons)
    _check(lib().gray_integrate(C.byref(batch.c), n, max_steps, C.byref(params.c), _ptr(batch.workspace),
                                batch.workspace.numel(), _stream()))


def gray_integrate_counters(batch):
    c = _Counters()
    _check(lib().gray_integrate_counters(_ptr(batch.workspace), C.byref(c), _stream()))
    return dict(photon_steps=c.photon_steps, issued_steps=c.issued_steps, photons_done=c.photons_done,
                photons_live=c.photons_live, fallback_steps=c.fallback_steps)


def gray_classify(batch, capture_map=None):
    """Returns counts[5] (LIVE, CAPTURED, ESCAPED, BAD, EQUATOR); fills capture_map (uint8 tensor of n) if given."""
    counts = (C.c_uint64 * N_STATUS)()
    _check(lib().gray_classify(C.byref(batch.c), _ptr(capture_map), counts, _ptr(batch.workspace),
                               batch.workspace.numel(), _stream()))
    return [int(v) for v in counts]


def gray_shadow_edge(batch, n_angles, radius=None):
    """Returns the gray_shadow_stats as a dict; fills radius (float64 tensor of n_angles) if given."""
    s = _ShadowStats()
    _check(lib().gray_shadow_edge(C.byref(batch.c), n_angles, _ptr(radius), C.byref(s), _ptr(batch.workspace),
                                  batch.workspace.numel(), _stream()))
    return {k: getattr(s, k) for k, _ in _ShadowStats._fields_}


def gray_noalloc_max_angles():
    """Most spokes gray_shadow_edge_noalloc accepts (GRAY_NOALLOC_MAX_ANGLES of include/gray.h)."""
    return int(lib().gray_noalloc_max_angles())


def gray_shadow_edge_noalloc(batch, n_angles, radius=None):
    """gray_shadow_edge for a caller that may not allocate device memory (a plug-in whose host program owns the
    GPU's memory pool, a worker whose memory slice is already full, a frame loop that cannot stall on cudaMalloc):
    batch.workspace is NOT used, the scratch memory is an array built into libgray.so (include/gray.h has the details:
    at most gray_noalloc_max_angles() spokes, one call at a time per GPU, first call on a device does a one-off address
    look-up).  Same results as gray_shadow_edge: the stats as a dict; fills radius (float64 tensor of n_angles) if given."""
    s = _ShadowStats()
    _check(lib().gray_shadow_edge_noalloc(C.byref(batch.c), n_angles, _ptr(radius), C.byref(s), _stream()))
    return {k: getattr(s, k) for k, _ in _ShadowStats._fields_}


def gray_host_scratch_bytes(chunk, prec=GRAY_F32):
    return int(lib().gray_host_scratch_bytes(int(chunk), prec))


def gray_integrate_host(x_in, k_in, x_out, k_out, status, steps, a, r_obs, max_steps=20000, params=None,
                        chunk=1 << 24, scratch=None):
    """Host tensors in (x_in, k_in: n x 4, pinned), host tensors out; `scratch` is a device uint8 tensor of
    gray_host_scratch_bytes(chunk, prec) bytes.  Returns the summed counters."""
    params = params or StepParams()
    n = x_in.shape[0]
    prec = GRAY_F32 if x_in.dtype == torch.float32 else GRAY_F64
    for t in (x_in, k_in, x_out, k_out, status, steps):
        if t.is_cuda or not t.is_contiguous():
            raise GrayError("gray_integrate_host takes contiguous HOST tensors")
    c = _Counters()
    _check(lib().gray_integrate_host(_ptr(x_in), _ptr(k_in), _ptr(x_out), _ptr(k_out), _ptr(status), _ptr(steps), n,
                                     prec, a, r_obs, max_steps, C.byref(params.c), chunk, _ptr(scratch),
                                     scratch.numel(), C.byref(c), _stream()))
    return dict(photon_steps=c.photon_steps, issued_steps=c.issued_steps, photons_done=c.photons_done,
                photons_live=c.photons_live, fallback_steps=c.fallback_steps)


def gray_fma_peak(prec=GRAY_F32, iters=4096):
    v = C.c_double()
    _check(lib().gray_fma_peak(prec, iters, C.byref(v), _stream()))
    return v.value


def gray_packed_peak(mix, iters=2048):
    """fp32 lane-operations/s of the packed-instruction microbenchmark (include/gray.h)."""
    v = C.c_double()
    _check(lib().gray_packed_peak(mix, iters, C.byref(v), _stream()))
    return v.value


def gray_device_info():
    sms, khz = C.c_int32(), C.c_int32()
    _check(lib().gray_device_info(C.byref(sms), C.byref(khz)))
    return sms.value, khz.value


def trace_image(a, inc_deg, half_width, nx, ny, r_obs=1000.0, prec=GRAY_F32, max_steps=20000, params=None,
                n_angles=0):
    """Convenience: init + integrate + classify (+ shadow statistics) of one grid image; four C-ABI calls."""
    b = PhotonBatch(nx * ny, prec)
    gray_init_rays(b, a, r_obs, inc_deg, half_width, nx, ny)
    gray_integrate(b, max_steps=max_steps, params=params)
    cmap = torch.empty((ny, nx), dtype=torch.uint8, device=b.x.device)
    counts = gray_classify(b, cmap)
    out = dict(batch=b, capture_map=cmap, counts=counts, counters=gray_integrate_counters(b))
    if n_angles:
        radius = torch.empty((n_angles,), dtype=torch.float64, device=b.x.device)
        out["stats"] = gray_shadow_edge(b, n_angles, radius)
        out["radius"] = radius
    return out
