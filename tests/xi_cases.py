"""States for the one-step pins of the paper's xi monitor (eq. 4; reading R18), shared by the
oracle pin (-m "not gpu") and the GPU parity test.  Only the oracle's separately pinned pieces are used here
(metric, rhs, step_size, rk4_step, remap_theta); the expected result of the fallback is formed in numpy."""
import numpy as np

import golden_values
import oracle as o

GOLD = golden_values.load()
A_SPIN = 0.9
H = GOLD["step_parameter"]
EPS = GOLD["xi_epsilon"]
NINE = GOLD["euler_fraction"]          # "a smaller time step dlambda'/9"


def xi_plus_one(a, y):
    """eq. (4) + 1 = g_mu_nu k^mu k^nu / (g_tt (k^t)^2), from the (pinned) metric."""
    g = o.metric(a, y[1], y[2])
    k = y[4:8]
    return float(k @ g @ k) / float(g[0, 0] * k[0] * k[0])


def base_states():
    """Null states on rays of a Kerr image, some steps in (r between ~3 and ~30, Christoffels far from trivial)."""
    out = []
    for al, be, nsteps in ((4.0, 3.0, 330), (-6.5, 1.0, 300), (2.0, -7.0, 280), (7.0, 6.0, 310), (-3.0, -2.5, 340)):
        y0 = o.init_ray(A_SPIN, 1000.0, 60.0, al, be)
        y, _, _ = o.integrate(A_SPIN, y0, H, 0.0, 1e9, o.STEP_EQ2, 10 ** 6, force_steps=nsteps)
        assert 1.5 < y[1] < 60.0 and abs(xi_plus_one(A_SPIN, y)) < 1e-5
        out.append(y)
    return out


def off_shell(y, delta):
    """The same state with k^t scaled by (1 + delta): g k k / (g_tt k^t k^t) moves to ~2 delta."""
    z = y.copy()
    z[4] *= 1.0 + delta
    return z


def expected_one_step(a, y, rule=o.STEP_EQ2):
    """(accepted RK4 result, Euler dl/9 fallback, xi + 1 of the RK4 result, dl), each theta-remapped (eq. 3)."""
    dl = o.step_size(a, y, H, rule)
    rk = o.rk4_step(a, y, dl)
    eu = y + (dl / NINE) * o.rhs(a, y)
    return o.remap_theta(rk), o.remap_theta(eu), xi_plus_one(a, rk), dl


def paper_pole_rays():
    """The paper's own pole test ray (spin 0.99, r0 cos(theta0) = 1000 M, r0 sin(theta0) = 4.833605 M, phi0 = 0) and
    its neighbours, as (alpha, beta) on the face-on (i = 0) image plane at r = 1000 M, where r0 cos(theta0) = r_obs,
    r0 sin(theta0) = (alpha^2 + beta^2)^(1/2) and phi0 = atan2(alpha, -beta).  Every one lies INSIDE the face-on
    critical radius 4.838284 M (test_pole_ray_value_printed_in_paper_is_the_face_on_critical_radius), by 0.1 % to
    0.4 %: the exact answer is CAPTURED ("eventually hit the event horizon").
      0  the printed ray itself, phi0 = 0          1  the same ray at phi0 = 90 deg (axisymmetry: the same trajectory)
      2  (3.0, -3.79): radius 4.833746             3  radius 4.82"""
    R = GOLD["pole_ray_impact"]
    return np.array([(0.0, -R), (R, 0.0), (3.0, -3.79), (0.0, -4.82)])
