"""Pins for the oracle's image-plane initialiser, step rules, RK4 step and theta remap."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle as o


def test_pixel_grid_centres():
    # pixel centres, beta slow (reading R1)
    assert o.pixel_grid(10.0, 64, 64, 0) == (-10 + 10 / 64, -10 + 10 / 64)
    assert o.pixel_grid(10.0, 64, 32, 65) == (-10 + 1.5 * 20 / 64, -10 + 1.5 * 20 / 32)
    al = [o.pixel_grid(12.0, 8, 4, p) for p in range(32)]
    assert np.isclose(np.mean([x for x, _ in al]), 0) and np.isclose(np.mean([y for _, y in al]), 0)


def test_pixel_random_is_uniform_and_fp32_exact():
    W = 15.0
    pts = np.array([o.pixel_random(20130322, p, W) for p in range(20000)])
    assert np.all(np.abs(pts) < W)
    assert np.all(pts == pts.astype(np.float32).astype(np.float64))     # exactly representable in fp32
    assert abs(pts.mean()) < 0.3 and abs(pts.std() - 2 * W / np.sqrt(12)) < 0.15
    assert abs(np.corrcoef(pts[:, 0], pts[:, 1])[0, 1]) < 0.03
    assert o.pixel_random(20130322, 7, W) == o.pixel_random(20130322, 7, W)
    assert o.pixel_random(1, 7, W) != o.pixel_random(2, 7, W)
    h, _ = np.histogram(pts[:, 0], bins=10, range=(-W, W))
    assert h.min() > 1700 and h.max() < 2300


@pytest.mark.parametrize("a,inc", [(0.0, 60.0), (0.7, 45.0), (0.9, 60.0), (0.99, 90.0), (0.5, 5.0)])
def test_init_ray_null_E1_and_bardeen_impact_parameters(a, inc):
    i = np.deg2rad(inc)
    worst = np.zeros(2)
    for al, be in [(3.0, 4.0), (-7.5, 0.3), (0.2, -9.0), (9.9, 9.9), (-0.01, 0.01)]:
        y = o.init_ray(a, 1000.0, inc, al, be)
        E, L, Q, null = o.invariants(a, y)
        assert abs(null) < 1e-14 and abs(E - 1) < 1e-13
        assert y[0] == 0 and y[4] > 0 and y[5] > 0          # future-directed, moving outwards to the observer
        # k^t = 1/(1 - 2/r) to leading order at r = 1000
        assert abs(y[4] - 1 / (1 - 2 / y[1])) < 1e-5
        # Cartesian position of the pixel: r_obs o + alpha yhat + beta bhat
        x = y[1] * np.sin(y[2]) * np.cos(y[3]); yy = y[1] * np.sin(y[2]) * np.sin(y[3]); z = y[1] * np.cos(y[2])
        assert np.allclose([x, yy, z], [1000 * np.sin(i) - be * np.cos(i), al, 1000 * np.cos(i) + be * np.sin(i)],
                           atol=1e-9)
        # Bardeen's impact parameters for an observer at infinity: xi = -alpha sin i,
        # eta = beta^2 + (alpha^2 - a^2) cos^2 i; finite-distance corrections O(1/r_obs) (reading R3)
        worst = np.maximum(worst, [abs(L + al * np.sin(i)), abs(Q - (be ** 2 + (al ** 2 - a ** 2) * np.cos(i) ** 2))])
    assert worst[0] < 3e-2 and worst[1] < 0.35, worst


def test_init_ray_for_observers_on_and_next_to_the_spin_axis():
    # Reading R23.  For i = 0 and i = 0.1 deg the polar angle of a pixel is ~ rho / r_obs ~ 1e-3: theta from atan2 keeps
    # r sin(theta) - the quantity every 1 / sin(theta) of the right-hand side divides by - to rounding (acos(z / r)
    # would lose half the digits there); the state stays null with E = 1; and the central pixel of the face-on image
    # (no azimuth: o is parallel to the axis) gets theta = 0, k^theta = k^phi = 0, all finite.
    a = 0.9
    for inc in (0.0, 0.1, 179.9, 180.0):
        i = np.deg2rad(inc)
        for al, be in ((3.0, 4.0), (-0.5, 0.002), (1e-3, -2e-3), (4.833605, 0.0)):
            y = o.init_ray(a, 1000.0, inc, al, be)
            X, Y, Z = 1000 * np.sin(i) - be * np.cos(i), al, 1000 * np.cos(i) + be * np.sin(i)
            q = np.hypot(X, Y)
            assert abs(y[1] * np.sin(y[2]) - q) <= 4e-16 * 1000.0          # a few ulp of r, i.e. 1e-13 relative at q = 5
            assert abs(y[1] * np.cos(y[2]) - Z) <= 4e-13 and abs(y[3] - np.arctan2(Y, X)) <= 1e-15
            E, L, Q, null = o.invariants(a, y)
            assert abs(null) < 1e-14 and abs(E - 1) < 1e-13
            # velocity parallel to the observer's axis, in Cartesian components (curvature corrections ~ 1/r_obs)
            r, th, ph, kr, kh, kp = y[1], y[2], y[3], y[5], y[6], y[7]
            vz = kr * np.cos(th) - r * kh * np.sin(th)
            vq = kr * np.sin(th) + r * kh * np.cos(th)
            assert abs(vz / np.hypot(vz, vq) - np.cos(i)) < 1e-2 and abs(r * kp * np.sin(th)) < 2e-3
    for inc, th0 in ((0.0, 0.0), (180.0, np.pi)):
        y = o.init_ray(a, 1000.0, inc, 0.0, 0.0)
        assert np.all(np.isfinite(y)) and y[1] == 1000.0 and abs(y[2] - th0) < 2e-13 and y[6] == 0.0 and y[7] == 0.0
        assert abs(o.invariants(a, y)[0] - 1) < 1e-13


def test_init_ray_direction_is_parallel_to_observer_axis():
    # flat-space limit (r_obs huge): the Cartesian velocity of every pixel's photon is (sin i, 0, cos i)
    a, inc, robs = 0.0, 35.0, 1e7
    i = np.deg2rad(inc)
    for al, be in [(5.0, -3.0), (-8.0, 8.0)]:
        y = o.init_ray(a, robs, inc, al, be)
        r, th, ph, kr, kh, kp = y[1], y[2], y[3], y[5], y[6], y[7]
        vx = kr * np.sin(th) * np.cos(ph) + r * kh * np.cos(th) * np.cos(ph) - r * kp * np.sin(th) * np.sin(ph)
        vy = kr * np.sin(th) * np.sin(ph) + r * kh * np.cos(th) * np.sin(ph) + r * kp * np.sin(th) * np.cos(ph)
        vz = kr * np.cos(th) - r * kh * np.sin(th)
        assert np.allclose([vx, vy, vz], [np.sin(i), 0.0, np.cos(i)], atol=1e-6)


def test_step_size_rules():
    a = 0.9
    y = o.init_ray(a, 1000.0, 60.0, 3.0, 4.0)
    h = 1 / 32
    assert o.step_size(a, y, h, o.STEP_REL) == -h * y[1]
    # far field: eq. (2) -> h r / |k^r|; the horizon limiter is inactive
    d = o.step_size(a, y, h, o.STEP_EQ2)
    assert d < 0 and abs(d / (-h * y[1] / abs(y[5])) - 1) < 1e-2
    # near the horizon with a large radial velocity the second branch of eq. (2) wins
    rh = o.horizon(a)
    y2 = np.array([0, rh + 0.01, 1.2, 0, 50.0, -3.0, 0.01, 0.2])
    assert np.isclose(o.step_size(a, y2, h, o.STEP_EQ2), -(0.01) / (2 * 3.0))
    # angular terms: pure theta motion
    y3 = np.array([0, 10.0, 1.2, 0, 1.0, 0.0, 0.25, 0.0])
    assert np.isclose(o.step_size(a, y3, h, o.STEP_EQ2), -h / 0.25)
    y3[7] = -0.75
    assert np.isclose(o.step_size(a, y3, h, o.STEP_EQ2), -h / 1.0)


def test_remap_theta_eq3():
    # paper eq. (3)
    y = np.array([1.0, 5.0, np.pi + 0.1, 0.3, 1, 2, 3, 4.0])
    z = o.remap_theta(y)
    assert np.allclose(z, [1.0, 5.0, np.pi - 0.1, 0.3 + np.pi, 1, 2, -3, 4.0])
    y[2] = -0.2
    z = o.remap_theta(y)
    assert np.allclose(z, [1.0, 5.0, 0.2, 0.3 - np.pi, 1, 2, -3, 4.0])
    y[2] = 1.0
    assert np.array_equal(o.remap_theta(y), y)
    # the remapped point is the same point of space with the same Cartesian velocity
    def cart(y):
        r, th, ph = y[1:4]
        return np.array([r * np.sin(th) * np.cos(ph), r * np.sin(th) * np.sin(ph), r * np.cos(th)])
    y = np.array([0, 5.0, -0.05, 0.3, 1, 0.1, 0.2, 0.3])
    assert np.allclose(cart(y), cart(o.remap_theta(y)))
    eps = 1e-6
    v0 = (cart(y + eps * np.r_[y[4:], 0, 0, 0, 0]) - cart(y)) / eps
    z = o.remap_theta(y)
    v1 = (cart(z + eps * np.r_[z[4:], 0, 0, 0, 0]) - cart(z)) / eps
    assert np.allclose(v0, v1, atol=1e-5)


def _reference_flow(a, y0, lam):
    """High-accuracy solution of the same ODE (oracle rhs, pinned in test_oracle_geometry) by an
    independent adaptive integrator."""
    sol = solve_ivp(lambda t, y: o.rhs(a, y), (0.0, lam), y0, method="DOP853", rtol=1e-13, atol=1e-15)
    return sol.y[:, -1]


def test_rk4_step_is_fourth_order_against_adaptive_integrator():
    # one step of size dl has local error C dl^5; halving dl must reduce it 32x.  A wrong weight
    # or stage position lowers the order and fails this.
    a = 0.9
    y0 = np.array([0, 6.0, 1.1, 0.2, 1.6, -0.7, 0.05, 0.11])
    errs = []
    for dl in (-0.4, -0.2, -0.1):
        y1 = o.rk4_step(a, y0, dl)
        errs.append(np.abs(y1 - _reference_flow(a, y0, dl)).max())
    assert 24 < errs[0] / errs[1] < 42 and 24 < errs[1] / errs[2] < 42, errs
    assert errs[2] < 1e-6


def test_integration_converges_at_fourth_order_with_step_halving():
    # global error after integrating a fixed affine distance falls 16x per halving of h.
    # REL rule: dlambda_n = -h r_n, so the affine distance is not fixed; use forced step counts
    # and compare with the adaptive integrator run to the same total lambda.
    a = 0.9
    y0 = o.init_ray(a, 50.0, 60.0, 4.0, 5.5)
    errs = []
    for h, n in ((1 / 16, 40), (1 / 32, 80), (1 / 64, 160)):
        y = y0.copy()
        lam = 0.0
        for _ in range(n):
            dl = o.step_size(a, y, h, o.STEP_REL)
            lam += dl
            y = o.rk4_step(a, y, dl)
        errs.append(np.abs(y - _reference_flow(a, y0, lam))[1:].max())
    assert 11 < errs[0] / errs[1] < 22 and 11 < errs[1] / errs[2] < 22, errs


def test_invariant_drift_halves_at_fourth_order():
    # north_star: "step-halving convergence at 4th order on tiny inputs"
    a = 0.9
    drift = []
    for h in (1 / 16, 1 / 32, 1 / 64, 1 / 128):
        res = o.trace(a, 1000.0, 60.0, 10.0, 4, 4, h=h, rule=o.STEP_EQ2)
        esc = res["status"] == o.ESCAPED
        assert esc.sum() >= 8
        d = 0.0
        for y0, y in zip(res["y0"][esc], res["y"][esc]):
            i0, i1 = o.invariants(a, y0), o.invariants(a, y)
            d = max(d, abs(i1[1] - i0[1]) / abs(i0[1]), abs(i1[2] - i0[2]) / abs(i0[2]))
        drift.append(d)
    ratios = [drift[k] / drift[k + 1] for k in range(3)]
    assert all(10 < r < 24 for r in ratios), (drift, ratios)


def test_integrate_counts_steps_and_resumes():
    a = 0.7
    y0 = o.init_ray(a, 1000.0, 45.0, 6.0, -7.0)
    rh = o.horizon(a)
    full, st, n = o.integrate(a, y0, 1 / 32, 1.01 * rh, 1010.0, o.STEP_EQ2, 20000)
    assert st == o.ESCAPED and 300 < n < 2000
    # stopping at a cap leaves the ray LIVE and resuming reproduces the uninterrupted run exactly
    part, st1, n1 = o.integrate(a, y0, 1 / 32, 1.01 * rh, 1010.0, o.STEP_EQ2, 100)
    assert st1 == o.LIVE and n1 == 100
    rest, st2, n2 = o.integrate(a, part, 1 / 32, 1.01 * rh, 1010.0, o.STEP_EQ2, 20000, steps=n1)
    assert st2 == st and n2 == n and np.array_equal(rest, full)
    # force_steps ignores the tests
    forced, _, n3 = o.integrate(a, y0, 1 / 32, 1.01 * rh, 1010.0, o.STEP_EQ2, 20000, force_steps=n)
    assert n3 == n and np.array_equal(forced, full)
    # the first state that satisfies a test is the stored one: one step earlier r was inside
    prev, _, _ = o.integrate(a, y0, 1 / 32, 1.01 * rh, 1010.0, o.STEP_EQ2, 20000, force_steps=n - 1)
    assert prev[1] <= 1010.0 < full[1]
