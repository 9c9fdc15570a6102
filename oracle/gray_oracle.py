"""ctypes binding of oracle/libgray_oracle.so.  TEST INFRASTRUCTURE ONLY.

Argument marshalling only; all arithmetic is in gray_oracle.hpp / gray_oracle.cpp.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

LIVE, CAPTURED, ESCAPED, BAD, EQUATOR = 0, 1, 2, 3, 4
STEP_REL, STEP_EQ2 = 0, 1
SYS_FULL, SYS_REDUCED = 0, 1

_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.gray_oracle_horizon.restype = C.c_double
        L.gray_oracle_horizon.argtypes = [C.c_double]
        L.gray_oracle_metric.argtypes = [C.c_double] * 3 + [_dp]
        L.gray_oracle_christoffel.argtypes = [C.c_double] * 3 + [_dp]
        L.gray_oracle_rhs.argtypes = [C.c_double, _dp, _dp]
        L.gray_oracle_rhs_reduced.argtypes = [C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.gray_oracle_killing_velocities.argtypes = [C.c_double] * 5 + [_dp, _dp]
        L.gray_oracle_invariants.argtypes = [C.c_double, _dp, _dp]
        L.gray_oracle_pixel_grid.argtypes = [C.c_double, C.c_int64, C.c_int64, C.c_uint64, _dp, _dp]
        L.gray_oracle_pixel_random.argtypes = [C.c_uint64, C.c_uint64, C.c_double, _dp, _dp]
        L.gray_oracle_pixel_polar.argtypes = [C.c_double, C.c_double, C.c_int64, C.c_int64, C.c_uint64, _dp, _dp]
        L.gray_oracle_init_ray.argtypes = [C.c_double] * 5 + [_dp]
        L.gray_oracle_step_size.restype = C.c_double
        L.gray_oracle_step_size.argtypes = [C.c_double, _dp, C.c_double, C.c_int]
        L.gray_oracle_rk4_step.argtypes = [C.c_double, _dp, C.c_double]
        L.gray_oracle_remap_theta.argtypes = [_dp]
        L.gray_oracle_integrate.restype = C.c_int
        L.gray_oracle_integrate.argtypes = [C.c_double, _dp, C.c_double, C.c_double, C.c_double, C.c_int,
                                            C.c_uint32, C.c_int64, C.POINTER(C.c_uint32), C.c_double, C.c_int, C.c_int]
        L.gray_oracle_trace.restype = C.c_int
        L.gray_oracle_trace.argtypes = [C.c_double] * 4 + [C.c_int64, C.c_int64, C.c_uint64, C.c_void_p,
                                                            C.c_uint64, C.c_double, C.c_double, C.c_double,
                                                            C.c_double, C.c_int, C.c_uint32, C.c_int,
                                                            C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                                                            C.c_void_p, C.c_void_p, C.c_double, C.c_int, C.c_double, C.c_int]
        L.gray_oracle_hardware_threads.restype = C.c_int
        L.gray_oracle_shadow_stats.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_double, C.c_int32,
                                               C.c_void_p, C.c_void_p]
        L.gray_oracle_ring_polar.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_int,
                                             C.c_void_p, C.c_void_p]
        L.gray_oracle_op_tally.argtypes = [C.c_double, _dp, C.c_double, C.c_int, C.POINTER(C.c_uint64)]
        L.gray_oracle_op_tally_system.argtypes = [C.c_double, _dp, C.c_double, C.c_int, C.c_int, C.POINTER(C.c_uint64)]
        _lib = L
    return _lib


def _vec(y, n):
    y = np.ascontiguousarray(y, dtype=np.float64)
    assert y.shape == (n,)
    return y


def horizon(a):
    return lib().gray_oracle_horizon(float(a))


def metric(a, r, th):
    g = np.zeros((4, 4))
    lib().gray_oracle_metric(a, r, th, g.ctypes.data_as(_dp))
    return g


def christoffel(a, r, th):
    G = np.zeros((4, 4, 4))
    lib().gray_oracle_christoffel(a, r, th, G.ctypes.data_as(_dp))
    return G


def rhs(a, y):
    y = _vec(y, 8)
    dy = np.zeros(8)
    lib().gray_oracle_rhs(a, y.ctypes.data_as(_dp), dy.ctypes.data_as(_dp))
    return dy


def rhs_reduced(a, E, L, y6):
    y6 = _vec(y6, 6)
    dy = np.zeros(6)
    lib().gray_oracle_rhs_reduced(a, E, L, y6.ctypes.data_as(_dp), dy.ctypes.data_as(_dp))
    return dy


def killing_velocities(a, E, L, r, th):
    kt, kp = C.c_double(), C.c_double()
    lib().gray_oracle_killing_velocities(a, E, L, r, th, C.byref(kt), C.byref(kp))
    return kt.value, kp.value


def invariants(a, y):
    """(E, L_z, Q, null) of a state."""
    y = _vec(y, 8)
    inv = np.zeros(4)
    lib().gray_oracle_invariants(a, y.ctypes.data_as(_dp), inv.ctypes.data_as(_dp))
    return inv


def pixel_grid(W, nx, ny, p):
    al, be = C.c_double(), C.c_double()
    lib().gray_oracle_pixel_grid(W, nx, ny, p, C.byref(al), C.byref(be))
    return al.value, be.value


def pixel_random(seed, p, W):
    al, be = C.c_double(), C.c_double()
    lib().gray_oracle_pixel_random(seed, p, W, C.byref(al), C.byref(be))
    return al.value, be.value


def init_ray(a, r_obs, inc_deg, alpha, beta):
    y = np.zeros(8)
    lib().gray_oracle_init_ray(a, r_obs, inc_deg, alpha, beta, y.ctypes.data_as(_dp))
    return y


def step_size(a, y, h, rule):
    y = _vec(y, 8)
    return lib().gray_oracle_step_size(a, y.ctypes.data_as(_dp), h, rule)


def rk4_step(a, y, dl):
    y = _vec(y, 8).copy()
    lib().gray_oracle_rk4_step(a, y.ctypes.data_as(_dp), dl)
    return y


def remap_theta(y):
    y = _vec(y, 8).copy()
    lib().gray_oracle_remap_theta(y.ctypes.data_as(_dp))
    return y


def integrate(a, y, h, r_capture, r_escape, rule, max_steps, force_steps=-1, steps=0, xi_eps=0.0, stop_at_equator=False,
              system=SYS_FULL):
    """Integrate one ray; returns (y, status, steps)."""
    y = _vec(y, 8).copy()
    st = C.c_uint32(steps)
    status = lib().gray_oracle_integrate(a, y.ctypes.data_as(_dp), h, r_capture, r_escape, rule, max_steps,
                                         force_steps, C.byref(st), xi_eps, int(bool(stop_at_equator)), system)
    return y, status, st.value


def hardware_threads():
    return lib().gray_oracle_hardware_threads()


def trace(a, r_obs, inc_deg, W, nx=0, ny=0, seed=0, idx=None, n=None, h=1.0 / 32, cap_factor=1.01,
          esc_factor=1.01, horizon_delta=1e-6, rule=STEP_EQ2, max_steps=20000, init_f32=False,
          force_steps=None, threads=1, want_y0=True, xi_eps=0.0, stop_at_equator=False, polar=None, system=SYS_FULL):
    """Initialise and integrate a batch of photons; see gray_oracle_trace in gray_oracle.cpp.
    polar = (R_lo, R_hi, n_R, n_theta) selects the paper's polar image-plane grid (W, nx, ny are then ignored).

    Returns dict(y0, y, status, steps).
    """
    R_lo = 0.0
    if polar is not None:
        R_lo, W, n_R, ny = polar
        nx = -int(n_R)
    if idx is not None:
        idx = np.ascontiguousarray(idx, dtype=np.uint64)
        n = idx.size
    elif n is None:
        n = abs(nx) * ny
    y0 = np.zeros((n, 8)) if want_y0 else None
    y = np.zeros((n, 8))
    status = np.zeros(n, dtype=np.int32)
    steps = np.zeros(n, dtype=np.uint32)
    if force_steps is not None:
        force_steps = np.ascontiguousarray(force_steps, dtype=np.int64)
        assert force_steps.size == n
    lib().gray_oracle_trace(a, r_obs, inc_deg, W, nx, ny, seed,
                            idx.ctypes.data if idx is not None else None, n, h, cap_factor, esc_factor,
                            horizon_delta, rule, max_steps, int(bool(init_f32)),
                            force_steps.ctypes.data if force_steps is not None else None, threads,
                            y0.ctypes.data if y0 is not None else None, y.ctypes.data,
                            status.ctypes.data, steps.ctypes.data, xi_eps, int(bool(stop_at_equator)), R_lo, system)
    return dict(y0=y0, y=y, status=status, steps=steps)


def shadow_stats(captured, W, n_angles):
    """captured: (ny, nx) uint8.  Returns (stats dict, radius[n_angles])."""
    captured = np.ascontiguousarray(captured, dtype=np.uint8)
    ny, nx = captured.shape
    radius = np.zeros(n_angles)
    out = np.zeros(9)
    lib().gray_oracle_shadow_stats(captured.ctypes.data, nx, ny, W, n_angles, radius.ctypes.data,
                                   out.ctypes.data)
    keys = ["area", "centroid_alpha", "centroid_beta", "alpha_min", "alpha_max", "D", "R_mean", "A",
            "n_captured"]
    return dict(zip(keys, out.tolist())), radius


def ring_polar(captured, R_lo, R_hi, bridge_axis=False):
    """captured: (n_theta, n_R) uint8.  Returns (dict(alpha_min, alpha_max, D, R_mean, A), radius[n_theta])."""
    captured = np.ascontiguousarray(captured, dtype=np.uint8)
    n_theta, n_R = captured.shape
    radius = np.zeros(n_theta)
    out = np.zeros(5)
    lib().gray_oracle_ring_polar(captured.ctypes.data, n_R, n_theta, R_lo, R_hi, int(bool(bridge_axis)), radius.ctypes.data,
                                 out.ctypes.data)
    return dict(zip(["alpha_min", "alpha_max", "D", "R_mean", "A"], out.tolist())), radius


def pixel_polar(R_lo, R_hi, n_R, n_theta, p):
    al, be = C.c_double(), C.c_double()
    lib().gray_oracle_pixel_polar(R_lo, R_hi, n_R, n_theta, p, C.byref(al), C.byref(be))
    return al.value, be.value


def op_tally(a, y, h, rule, system=SYS_FULL):
    """Operation counts of one photon-step: dict(add, mul, div, sqrt, sin, cos, other)."""
    y = _vec(y, 8)
    c = (C.c_uint64 * 7)()
    lib().gray_oracle_op_tally_system(a, y.ctypes.data_as(_dp), h, rule, system, c)
    return dict(zip(["add", "mul", "div", "sqrt", "sin", "cos", "other"], [int(v) for v in c]))
