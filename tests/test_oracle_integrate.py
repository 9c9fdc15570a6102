"""Pins for the oracle's whole-ray integration and shadow statistics (-m "not gpu")."""
import numpy as np
import pytest

import closed_forms as cf
import golden_values
import oracle as o
import xi_cases

GOLD = golden_values.load()


def _grid(W, nx, ny):
    al = -W + (np.arange(nx) + 0.5) * 2 * W / nx
    be = -W + (np.arange(ny) + 0.5) * 2 * W / ny
    A, B = np.meshgrid(al, be)          # beta slow
    return A.ravel(), B.ravel()


def test_schwarzschild_critical_impact_parameter_sqrt27():
    # BASELINE config C1: a = 0, i = 60 deg, 64 x 64 over +-10 M; captured <=> sqrt(alpha^2 + beta^2) < sqrt(27)
    res = o.trace(0.0, 1000.0, 60.0, 10.0, 64, 64, rule=o.STEP_EQ2, threads=4)
    al, be = _grid(10.0, 64, 64)
    b = np.hypot(al, be)
    cap = res["status"] == o.CAPTURED
    assert np.all(np.isin(res["status"], (o.CAPTURED, o.ESCAPED)))
    bad = cap != (b < np.sqrt(27.0))
    assert np.all(np.abs(b[bad] / np.sqrt(27.0) - 1) < 0.01)
    assert bad.sum() == 0       # measured: the paper's eq. (2) rule classifies every C1 pixel correctly


def test_rel_rule_misclassifies_as_design_md_states():
    # DESIGN.md reading R5: the configs' literal rule dlambda = -h r, tested after full steps only,
    # jumps the band [r_h, 1.01 r_h] and misclassifies pixels deep inside the shadow.  This test
    # documents the failure (it is the reason the physical checks run with eq. (2)).
    res = o.trace(0.0, 1000.0, 60.0, 10.0, 64, 64, rule=o.STEP_REL, threads=4)
    al, be = _grid(10.0, 64, 64)
    b = np.hypot(al, be)
    bad = (res["status"] == o.CAPTURED) != (b < np.sqrt(27.0))
    assert 20 < bad.sum() < 400
    assert np.any(b[bad] < 0.9 * np.sqrt(27.0))


@pytest.mark.parametrize("a,inc,W", [(0.9, 60.0, 10.0), (0.99, 90.0, 12.0), (0.7, 45.0, 15.0), (0.5, 5.0, 10.0)])
def test_kerr_capture_matches_radial_potential_classifier(a, inc, W):
    # exact per-ray classifier independent of the integrator: (xi, eta) of the initial state and
    # the roots of the radial quartic
    n = 48
    res = o.trace(a, 1000.0, inc, W, n, n, rule=o.STEP_EQ2, threads=4)
    exact = np.zeros(n * n, dtype=bool)
    for p, y0 in enumerate(res["y0"]):
        E, L, Q, _ = o.invariants(a, y0)
        exact[p] = cf.captured_exact(a, L / E, Q / E ** 2)
    cap = res["status"] == o.CAPTURED
    assert np.all(np.isin(res["status"], (o.CAPTURED, o.ESCAPED)))
    al, be = _grid(W, n, n)
    rho_c = cf.bardeen_rho(a, inc, np.arctan2(be, al))
    bad = cap != exact
    assert np.all(np.abs(np.hypot(al, be)[bad] / rho_c[bad] - 1) < 0.01)
    assert bad.mean() <= 1e-3
    # and the exact classifier itself agrees with the Bardeen curve away from the edge
    far = np.abs(np.hypot(al, be) / rho_c - 1) > 0.01
    assert np.array_equal(exact[far], (np.hypot(al, be) < rho_c)[far])


def test_schwarzschild_deflection_matches_orbit_integral():
    # a = 0, observer in the equatorial plane, beta = 0: the ray stays at theta = pi/2 and its total
    # sweep in phi between the radii actually used is the textbook orbit integral
    for alpha in (5.4, 6.0, 8.0, 14.0):
        y0 = o.init_ray(0.0, 1000.0, 90.0, alpha, 0.0)
        rh = 2.0
        y, st, n = o.integrate(0.0, y0, 1 / 32, 1.01 * rh, 1010.0, o.STEP_EQ2, 20000)
        assert st == o.ESCAPED
        assert abs(y[2] - np.pi / 2) < 1e-12
        E, L, _, _ = o.invariants(0.0, y0)
        b = abs(L / E)
        exact = cf.schwarzschild_dphi(b, y0[1], y[1])
        # traced backwards: phi decreases for L < 0 ... compare magnitudes of the sweep
        got = abs(y[3] - y0[3])
        assert abs(got - exact) < 2e-5 * exact, (alpha, got, exact)
        assert exact > np.pi            # light bending: more than a straight line's pi


def test_reflection_symmetries():
    # equatorial reflection: (i, beta) -> (180 - i, -beta) maps theta -> pi - theta
    a = 0.9
    for al, be in [(4.0, 3.0), (-6.0, 2.0), (2.0, -1.0)]:
        y1, s1, n1 = o.integrate(a, o.init_ray(a, 1000.0, 60.0, al, be), 1 / 32, 1.01 * o.horizon(a), 1010.0, o.STEP_EQ2, 20000)
        y2, s2, n2 = o.integrate(a, o.init_ray(a, 1000.0, 120.0, al, -be), 1 / 32, 1.01 * o.horizon(a), 1010.0, o.STEP_EQ2, 20000)
        assert s1 == s2 and n1 == n2
        assert np.allclose(y1[[1, 3]], y2[[1, 3]], rtol=1e-9, atol=1e-9) and np.isclose(y1[2], np.pi - y2[2], atol=1e-9)
        # spin flip: (a, alpha) -> (-a, -alpha) mirrors phi
        y3, s3, n3 = o.integrate(-a, o.init_ray(-a, 1000.0, 60.0, -al, be), 1 / 32, 1.01 * o.horizon(a), 1010.0, o.STEP_EQ2, 20000)
        assert s1 == s3 and n1 == n3
        assert np.allclose(y1[[1, 2]], y3[[1, 2]], rtol=1e-9, atol=1e-9) and np.isclose(y1[3], -y3[3], atol=1e-8)


def test_a0_rotation_invariance():
    # Schwarzschild: with the REL rule (dlambda depends on r only) the radial motion depends on
    # sqrt(alpha^2 + beta^2) only, up to the coordinate dependence of the RK4 truncation error,
    # which must fall as h^4
    spread = []
    for h in (1 / 32, 1 / 64):
        out = []
        for ang in (0.3, 1.4, 2.9, 4.4):
            y, s, n = o.integrate(0.0, o.init_ray(0.0, 1000.0, 60.0, 7.0 * np.cos(ang), 7.0 * np.sin(ang)),
                                  h, 2.02, 1010.0, o.STEP_REL, 20000)
            out.append((y[1], s, n))
        assert all(s == o.ESCAPED for _, s, _ in out)
        assert len({n for _, _, n in out}) == 1
        spread.append(max(abs(r - out[0][0]) for r, _, _ in out) / out[0][0])
    assert spread[0] < 2e-4 and spread[1] < spread[0] / 8, spread


def test_conservation_along_rays():
    # E, L_z, Q and the null norm between the first and last state (north_star); truncation-limited
    # at h = 1/32 (reading R12)
    a = 0.9
    res = o.trace(a, 1000.0, 60.0, 10.0, 16, 16, rule=o.STEP_EQ2)
    esc = res["status"] == o.ESCAPED
    d = []
    for y0, y in zip(res["y0"][esc], res["y"][esc]):
        i0, i1 = o.invariants(a, y0), o.invariants(a, y)
        d.append([abs(i1[0] - 1), abs(i1[1] - i0[1]) / max(abs(i0[1]), 0.1), abs(i1[2] - i0[2]) / abs(i0[2]), abs(i1[3])])
    d = np.array(d)
    assert np.median(d, axis=0).max() < 1e-6 and d.max() < 2e-4, (np.median(d, axis=0), d.max(axis=0))


def test_pole_ray_value_printed_in_paper_is_the_face_on_critical_radius():
    # r0 sin(theta0) = 4.833605 M for a = 0.99 "passes both the south and north poles ...
    # and eventually hit[s] the event horizon": a ray parallel to the spin axis with L_z = 0 on the
    # critical curve.  Closed form: xi(r_p) = 0, radius = sqrt(eta(r_p) + a^2).
    from scipy.optimize import brentq
    a = GOLD["pole_ray_spin"]
    pro, ret = cf.photon_orbit_radii(a)
    rp = brentq(lambda r: cf.xi_eta(a, r)[0], pro, ret)
    radius = np.sqrt(cf.xi_eta(a, rp)[1] + a * a)
    # the printed value lies 0.1 % inside that radius (4.838284): the ray winds "a couple times"
    # and is captured, as P:93 says
    assert 0 < radius - GOLD["pole_ray_impact"] < 1.1e-3 * radius
    assert abs(radius - 4.838284) < 1e-6
    # the oracle's nearly face-on (i = 1 deg) shadow edge brackets the closed-form curve, whose
    # radius there is that value to 0.2 %: rays 1 % inside are captured, 1 % outside escape.
    # (alpha = 0 exactly is avoided: such rays have |L_z| < 1e-5 and hit the pole failure the
    # paper describes; its cure is SURVEY 8(f) NEXT-1.)
    for ang in (0.0, 0.8, 2.0, np.pi):
        rc = cf.bardeen_rho(a, 1.0, ang)
        assert abs(rc / GOLD["pole_ray_impact"] - 1) < 3e-2
        for f, want in ((0.99, o.CAPTURED), (1.01, o.ESCAPED)):
            y0 = o.init_ray(a, GOLD["image_plane_radius"], 1.0, f * rc * np.cos(ang), f * rc * np.sin(ang))
            _, st, _ = o.integrate(a, y0, GOLD["step_parameter"], 1.01 * o.horizon(a), 1010.0, o.STEP_EQ2, 20000)
            assert st == want


def _paper_fit(a, inc_deg):
    R0 = sum(c * a ** k for k, c in enumerate(GOLD["fit_R0_coeffs"]))
    c1 = GOLD["fit_R1_coeffs"]
    R1 = (c1[0] - c1[1] / ((a - c1[2]) ** 2 + c1[3])) * 1e-3
    ph = GOLD["fit_R_phase"]
    R = R0 + R1 * np.cos(np.deg2rad(ph[0] * inc_deg - ph[1]))
    ca = GOLD["fit_A0_coeffs"]
    A0 = ca[0] * a ** ca[1] + ca[2] * a ** ca[3] + ca[4] * a ** ca[5]
    cn = GOLD["fit_n_coeffs"]
    n = cn[0] * (1 - a) ** cn[1] + cn[2] * (1 - a) ** cn[3]
    return R, A0 * np.sin(np.deg2rad(inc_deg)) ** n


@pytest.mark.parametrize("a,inc", [(0.0, 60.0), (0.9, 60.0), (0.99, 90.0)])
def test_shadow_stats_against_bardeen_and_paper_fits(a, inc):
    # eqs. (6)-(8) of the paper evaluated on the oracle's capture map vs the closed-form curve
    n, W = 96, 10.0
    res = o.trace(a, 1000.0, inc, W, n, n, rule=o.STEP_EQ2, threads=4, want_y0=False)
    cmap = (res["status"] == o.CAPTURED).reshape(n, n).astype(np.uint8)
    st, radius = o.shadow_stats(cmap, W, 360)
    ex = cf.bardeen_stats(a, inc)
    px = 2 * W / n
    assert abs(st["area"] - ex["area"]) < 0.012 * ex["area"]
    assert abs(st["alpha_min"] - ex["alpha_min"]) < px and abs(st["alpha_max"] - ex["alpha_max"]) < px
    assert abs(st["D"] - ex["D"]) < px
    assert abs(st["R_mean"] - ex["R_mean"]) < 0.5 * px
    # pixelisation adds ~px/sqrt(12) of scatter to every spoke radius, i.e. ~0.58 px to A = 2 std(R)
    assert abs(st["A"] - ex["A"]) < 0.8 * px
    assert abs(st["centroid_beta"]) < 1e-9 or abs(st["centroid_beta"]) < px
    vt = 2 * np.pi * (np.arange(360) + 0.5) / 360
    assert np.max(np.abs(radius - cf.bardeen_rho(a, inc, vt))) < 1.1 * px
    # the paper's fitting formulae, eqs. (11)-(14): soft (they are fits)
    Rf, Af = _paper_fit(a, inc)
    assert abs(ex["R_mean"] - Rf) < 0.04 and abs(ex["A"] - Af) < 0.03
    assert abs(st["R_mean"] - Rf) < 0.04 + 0.5 * px


def test_shadow_stats_on_synthetic_disc():
    # exact geometry: a disc of radius 3 centred at (1, 0)
    n, W = 400, 8.0
    al, be = _grid(W, n, n)
    cmap = (np.hypot(al - 1.0, be) < 3.0).reshape(n, n).astype(np.uint8)
    st, radius = o.shadow_stats(cmap, W, 720)
    px = 2 * W / n
    assert abs(st["area"] - np.pi * 9) < 0.01 * np.pi * 9
    assert abs(st["centroid_alpha"] - 1.0) < 1e-3 and abs(st["centroid_beta"]) < 1e-9
    assert abs(st["alpha_min"] + 2.0) < px and abs(st["alpha_max"] - 4.0) < px
    assert abs(st["D"] - 1.0) < px and abs(st["R_mean"] - 3.0) < 0.5 * px and st["A"] < px
    vt = 2 * np.pi * (np.arange(720) + 0.5) / 720
    rho = np.cos(vt) + np.sqrt(9 - np.sin(vt) ** 2)        # boundary of the disc seen from the origin
    assert np.max(np.abs(radius - rho)) < 1.5 * px
    # empty map
    st0, r0 = o.shadow_stats(np.zeros((8, 8), np.uint8), 1.0, 16)
    assert st0["area"] == 0 and st0["n_captured"] == 0 and np.all(r0 == 0)


def test_op_tally_is_stable_and_plausible():
    a = 0.7
    y = o.init_ray(a, 1000.0, 45.0, 3.0, 4.0)
    t = o.op_tally(a, y, 1 / 32, o.STEP_REL)
    t2 = o.op_tally(a, o.init_ray(a, 1000.0, 45.0, -9.0, 1.0), 1 / 32, o.STEP_REL)
    assert t == t2                                   # straight-line code: state-independent
    assert t["sin"] == 4 and t["cos"] == 4           # four RHS evaluations per RK4 step
    flops = t["add"] + t["mul"] + t["div"] + t["sqrt"] + t["sin"] + t["cos"]
    assert 600 < flops < 900
    te = o.op_tally(a, y, 1 / 32, o.STEP_EQ2)
    assert te["div"] > t["div"] and te["sqrt"] == 1


def test_pole_treatment_xi_monitor_cures_the_pole_failures():
    # NEXT-1.  Pin: the exact radial-potential classifier (independent of any integrator).  Rays of the
    # pixel column next to the spin axis of a face-on-ish image (a = 0.8, i = 5 deg, 1024 x 1024 over +-10 M),
    # well inside the shadow: plain RK4 "kicks" some of them "back to infinity" at the pole; with the xi
    # monitor of eq. (4) at epsilon = 1e-3 every one is captured, as the paper reports for its own
    # 3e8 trajectories.
    a, inc, W, nx = 0.8, 5.0, 10.0, 1024
    cols, rows = np.arange(511, 514), np.arange(284, 308)
    idx = (cols[None, :] + nx * rows[:, None]).ravel().astype(np.uint64)
    plain = o.trace(a, 1000.0, inc, W, nx, nx, idx=idx, rule=o.STEP_EQ2, threads=8)
    inv = np.array([o.invariants(a, v) for v in plain["y0"]])
    exact = np.array([cf.captured_exact(a, L / E, Q / E ** 2) for E, L, Q, _ in inv])
    assert exact.all()                                                  # every ray of the strip is inside the shadow
    assert np.sum(plain["status"] == o.ESCAPED) >= 3                    # the failure
    cured = o.trace(a, 1000.0, inc, W, nx, nx, idx=idx, rule=o.STEP_EQ2, threads=8, xi_eps=1e-3)
    assert np.all(cured["status"] == o.CAPTURED)                        # the cure
    # away from the pole the monitor never fires: identical results
    idx2 = (np.arange(200, 216)[None, :] + nx * np.arange(500, 504)[:, None]).ravel().astype(np.uint64)
    p2 = o.trace(a, 1000.0, inc, W, nx, nx, idx=idx2, rule=o.STEP_EQ2)
    c2 = o.trace(a, 1000.0, inc, W, nx, nx, idx=idx2, rule=o.STEP_EQ2, xi_eps=1e-3)
    esc = p2["status"] == o.ESCAPED
    assert esc.any() and np.array_equal(p2["y"][esc], c2["y"][esc]) and np.array_equal(p2["steps"][esc], c2["steps"][esc])


def test_paper_pole_test_ray_of_fig2():
    # P:91-107, Fig. 2 ("regression on the P:91 test ray").  The printed ray starts at
    # r0 cos(theta0) = 1000 M, r0 sin(theta0) = 4.833605 M, phi0 = 0 above a spin 0.99 hole and "passes both the south
    # and north poles"; the red (monitored) trajectory "eventually hit[s] the event horizon", the blue (plain RK4) one
    # "is kicked back to infinity".  What the oracle must and does reproduce:
    a, r_obs = GOLD["pole_ray_spin"], GOLD["pole_ray_height"]
    rays = xi_cases.paper_pole_rays()
    y0 = np.array([o.init_ray(a, r_obs, 0.0, al, be) for al, be in rays])
    assert abs(y0[0, 1] * np.cos(y0[0, 2]) - r_obs) < 1e-9 and abs(y0[0, 1] * np.sin(y0[0, 2]) - GOLD["pole_ray_impact"]) < 1e-10
    assert y0[0, 3] == 0.0 and abs(y0[1, 3] - np.pi / 2) < 1e-15
    inv = np.array([o.invariants(a, v) for v in y0])
    assert np.max(np.abs(inv[:, 1])) < 1e-7                                   # L_z = g_t_phi k^t ~ -5e-8: rays through the axis
    assert all(cf.captured_exact(a, L / E, Q / E ** 2) for E, L, Q, _ in inv)   # the exact answer: captured
    run = lambda y, eps: o.integrate(a, y, GOLD["step_parameter"], 1.01 * o.horizon(a), 1.01 * r_obs, o.STEP_EQ2, 20000,
                                     xi_eps=eps)
    # (i) the south pole is passed first, then the north pole: theta leaves [0, pi] above, later below (plain steps
    # written out with the pinned pieces; the remap of eq. (3) folds it back)
    y, crossings = y0[0].copy(), []
    for _ in range(1100):
        y = o.rk4_step(a, y, o.step_size(a, y, GOLD["step_parameter"], o.STEP_EQ2))
        if y[2] > np.pi or y[2] < 0.0:
            crossings.append("S" if y[2] > np.pi else "N")
        y = o.remap_theta(y)
    assert crossings[:2] == ["S", "N"], crossings
    # (ii) with the monitor (epsilon = 1e-3) every one of the rays is captured, after a couple of windings
    mon = [run(v, GOLD["xi_epsilon"]) for v in y0]
    assert all(st == o.CAPTURED for _, st, _ in mon)
    assert mon[0][2] == mon[1][2] and mon[0][2] > 2000                        # phi0 does not matter; > 2 windings' worth of steps
    # (iii) without it, the blue trajectory: neighbours 3e-5 and 3e-3 M away are kicked back to infinity, although
    # they too lie inside the critical radius (the printed ray itself survives the poles in this implementation)
    plain = [run(v, 0.0) for v in y0]
    assert [st for _, st, _ in plain] == [o.CAPTURED, o.CAPTURED, o.ESCAPED, o.ESCAPED]
    assert abs(plain[2][0][1] - 1.01 * r_obs) < 0.1 * r_obs                   # ... all the way out


def test_xi_monitor_fallback_is_one_euler_step_of_a_ninth_from_the_old_state():
    # P:103-107 / reading R18, pinned step by step: after ONE step with xi_eps > 0 the state is
    #   the RK4 result                              if |xi + 1| <= eps at the RK4 result,
    #   y_old + (dlambda / 9) rhs(y_old)             otherwise
    # (theta-remapped, one step counted either way), with xi + 1 formed here from the metric, the Euler step formed
    # here in numpy from the separately pinned rhs / step_size, and 9 read from the paper's text (golden).
    import xi_cases as xc
    a, eps = xc.A_SPIN, xc.EPS
    assert xc.NINE == 9.0
    taken = {"rk4": 0, "euler": 0}
    for y in xc.base_states():
        for delta in (0.0, 1e-4, 3e-4, 4.5e-4, 5.5e-4, 8e-4, 2e-3, 1e-2, -4.5e-4, -5.5e-4, -5e-3):
            z = xc.off_shell(y, delta)
            rk, eu, xi1, dl = xc.expected_one_step(a, z)
            if abs(abs(xi1) - eps) < 1e-9:
                continue
            got, status, steps = o.integrate(a, z, xc.H, 0.0, 1e9, o.STEP_EQ2, 1, xi_eps=eps)
            assert steps == 1 and status == o.LIVE
            want = eu if abs(xi1) > eps else rk
            taken["euler" if abs(xi1) > eps else "rk4"] += 1
            assert np.array_equal(got, want), (delta, xi1)
            if abs(xi1) > eps:
                # what a plausible misreading would give is far from rounding distance: Euler with dl/3, Euler with
                # the NEW state's derivative, Euler from the new state, or keeping the RK4 step
                scale = np.maximum(np.abs(want), 1.0)
                alts = [z + (dl / 3.0) * o.rhs(a, z), z + (dl / 9.0) * o.rhs(a, rk), rk + (dl / 9.0) * o.rhs(a, rk), rk,
                        z + dl * o.rhs(a, z)]
                for alt in alts:
                    assert np.max(np.abs(o.remap_theta(alt) - want) / scale) > 1e-6
            # with the monitor off the RK4 step is kept whatever xi is
            off, _, _ = o.integrate(a, z, xc.H, 0.0, 1e9, o.STEP_EQ2, 1, xi_eps=0.0)
            assert np.array_equal(off, rk)
    assert taken["rk4"] >= 15 and taken["euler"] >= 15, taken
    # same under the configs' literal rule, and the fallback is not re-tested: a second step starts from the Euler state
    z = xc.off_shell(xc.base_states()[0], 1e-2)
    rk, eu, xi1, dl = xc.expected_one_step(a, z, rule=o.STEP_REL)
    got, _, steps = o.integrate(a, z, xc.H, 0.0, 1e9, o.STEP_REL, 1, xi_eps=eps)
    assert abs(xi1) > eps and np.array_equal(got, eu)
    two, _, steps = o.integrate(a, z, xc.H, 0.0, 1e9, o.STEP_EQ2, 2, xi_eps=eps)
    _, eu1, _, _ = xc.expected_one_step(a, z)
    rk2, eu2, xi2, _ = xc.expected_one_step(a, eu1)
    assert steps == 2 and np.array_equal(two, eu2 if abs(xi2) > eps else rk2)


def test_equatorial_projection_schwarzschild_node_line_and_orbit_integral():
    # NEXT-2: follow rays to the equatorial plane.  Pins for a = 0, where the motion is planar:
    # (i) the plane of the orbit contains the origin, the observer direction o and the pixel offset, so its line of
    # nodes with the equatorial plane - hence phi at the crossing - is pure geometry; (ii) the crossing radius
    # follows from the textbook orbit integral  psi = int du / sqrt(1/b^2 - u^2 (1 - 2u))  over the in-plane
    # angle psi between the starting point and the node.
    from scipy import integrate as sint, optimize
    a, inc_deg, r_obs = 0.0, 60.0, 1000.0
    inc = np.radians(inc_deg)
    o_hat = np.array([np.sin(inc), 0.0, np.cos(inc)])
    b_hat = np.array([-np.cos(inc), 0.0, np.sin(inc)])
    y_hat = np.array([0.0, 1.0, 0.0])
    checked = 0
    for al, be in [(6.0, 9.0), (-8.0, 7.0), (3.0, 9.5), (-9.0, 4.0), (9.5, 9.5)]:
        y0 = o.init_ray(a, r_obs, inc_deg, al, be)
        y, st, n = o.integrate(a, y0, 1 / 32, 1.01 * 2.0, 1.01 * r_obs, o.STEP_EQ2, 20000, stop_at_equator=True)
        assert st == o.EQUATOR and abs(y[2] - np.pi / 2) < 1e-8
        X0 = r_obs * o_hat + al * y_hat + be * b_hat
        nrm = np.cross(o_hat, al * y_hat + be * b_hat)
        node = np.cross([0.0, 0.0, 1.0], nrm)
        node /= np.linalg.norm(node)
        hit = np.array([np.cos(y[3]), np.sin(y[3]), 0.0])
        s = np.sign(hit @ node)
        assert abs(np.cross(hit, node)[2]) < 2e-6                           # (i) phi on the line of nodes
        psi = np.arccos(np.clip((X0 / np.linalg.norm(X0)) @ (s * node), -1, 1))
        E, L, Q, _ = o.invariants(a, y0)
        b = np.sqrt(Q + L * L) / E                                            # total angular momentum / energy
        f = lambda u: 1.0 / (b * b) - u * u * (1.0 - 2.0 * u)
        u0 = 1.0 / y0[1]
        um = optimize.brentq(f, 0.5 / b, 1.0 / 3.0, xtol=1e-16)
        def leg(uc):      # in-plane angle between u = uc and the periapsis u = um; u = um - s^2 removes the end-point singularity
            g = lambda t: 2.0 * t / np.sqrt(max(f(um - t * t), 1e-300))
            return sint.quad(g, 0.0, np.sqrt(um - uc), epsabs=1e-13, epsrel=1e-13, limit=400)[0]

        if psi <= leg(u0):                                                    # node reached on the way in
            uc = optimize.brentq(lambda u: leg(u0) - leg(u) - psi, u0, um, xtol=1e-15)
        else:                                                                 # ... or on the way out
            uc = optimize.brentq(lambda u: leg(u) - (psi - leg(u0)), 1e-9, um, xtol=1e-15)
        assert abs(y[1] - 1.0 / uc) < 2e-6 / uc, (al, be, y[1], 1.0 / uc)     # (ii) crossing radius
        checked += 1
    assert checked == 5


def test_equatorial_projection_kerr_invariants_and_symmetry():
    # Kerr: the reported crossing state conserves E, L_z and Q to the scheme's truncation error, the
    # map is symmetric under (i, beta) -> (180 - i, -beta), and rays aimed inside the shadow are still CAPTURED
    # unless they reach the plane first.  Beyond this the Kerr crossing radius is parity-unpinned.
    a = 0.95
    for al, be in [(5.0, 8.0), (-7.0, 6.0), (9.0, -9.0)]:
        y0 = o.init_ray(a, 1000.0, 60.0, al, be)
        y, st, n = o.integrate(a, y0, 1 / 32, 1.01 * o.horizon(a), 1010.0, o.STEP_EQ2, 20000, stop_at_equator=True)
        assert st == o.EQUATOR
        i0, i1 = o.invariants(a, y0), o.invariants(a, y)
        assert abs(y[2] - np.pi / 2) < 1e-8
        assert np.all(np.abs(np.array(i1[:3]) - np.array(i0[:3])) < 2e-5 * np.maximum(1.0, np.abs(i0[:3])))
        y2, st2, n2 = o.integrate(a, o.init_ray(a, 1000.0, 120.0, al, -be), 1 / 32, 1.01 * o.horizon(a), 1010.0, o.STEP_EQ2,
                                  20000, stop_at_equator=True)
        assert st2 == o.EQUATOR and n2 == n and np.allclose(y[[1, 3]], y2[[1, 3]], rtol=1e-9, atol=1e-9)
    r = o.trace(a, 1000.0, 60.0, 10.0, 32, 32, rule=o.STEP_EQ2, stop_at_equator=True, threads=8)
    assert set(np.unique(r["status"])) == {o.CAPTURED, o.EQUATOR}
    plain = o.trace(a, 1000.0, 60.0, 10.0, 32, 32, rule=o.STEP_EQ2, threads=8)
    assert np.all(plain["status"][r["status"] == o.CAPTURED] == o.CAPTURED)   # captured without touching the plane


def test_polar_grid_and_ring_statistics_on_a_synthetic_disc():
    # NEXT-4: polar grid geometry, and eqs. (6)-(10) on an exact shape: a disc of radius 3 centred at (1, 0)
    # has alpha_min = -2, alpha_max = 4, D = 1, R = 3 on every spoke, A = 0.
    R_lo, R_hi, n_R, n_th = 1.5, 7.5, 6000, 181
    al, be = o.pixel_polar(R_lo, R_hi, n_R, n_th, 0)
    assert abs(al - 1.5005) < 1e-12 and be == 0.0
    al, be = o.pixel_polar(R_lo, R_hi, n_R, n_th, 90 * n_R + 2999)
    assert abs(al) < 1e-12 and abs(be - (1.5 + 2999.5e-3)) < 1e-12           # vartheta = pi/2, mid radius
    al, be = o.pixel_polar(R_lo, R_hi, n_R, n_th, 180 * n_R + 5999)
    assert abs(al + 7.4995) < 1e-12 and abs(be) < 1e-12                         # vartheta = pi, outermost cell
    vt = np.pi * np.arange(n_th) / (n_th - 1)
    Rc = R_lo + (np.arange(n_R) + 0.5) * (R_hi - R_lo) / n_R
    A_, B_ = Rc[None, :] * np.cos(vt)[:, None], Rc[None, :] * np.sin(vt)[:, None]
    disc = (np.hypot(A_ - 1.0, B_) < 3.0).astype(np.uint8)
    st, radius = o.ring_polar(disc, R_lo, R_hi)
    exact = np.cos(vt) + np.sqrt(9.0 - np.sin(vt) ** 2)
    assert np.max(np.abs(radius - exact)) <= 1.0e-3 + 1e-12                     # one radial cell
    assert abs(st["alpha_min"] + 2) < 1e-3 and abs(st["alpha_max"] - 4) < 1e-3 and abs(st["D"] - 1) < 1e-3
    assert abs(st["R_mean"] - 3) < 1e-3 and st["A"] < 1.5e-3


@pytest.mark.parametrize("a,inc", [(0.9, 60.0), (1 - 10 ** (-10 / 5), 90.0), (0.6019, 0.0)])
def test_polar_ring_study_against_bardeen_and_paper_fits(a, inc):
    # the paper's photon-ring study on a coarser polar grid (600 x 37), with the xi monitor as in the
    # paper; i = 0 needs it: every ray of a face-on image has L_z = 0 and passes over the pole
    R_lo, R_hi, n_R, n_th = 1.5, 7.5, 600, 37
    res = o.trace(a, 1000.0, inc, 0, polar=(R_lo, R_hi, n_R, n_th), rule=o.STEP_EQ2, xi_eps=1e-3, threads=8, want_y0=False)
    assert not np.any(res["status"] == o.BAD) and not np.any(res["status"] == o.LIVE)
    cap = (res["status"] == o.CAPTURED).reshape(n_th, n_R).astype(np.uint8)
    st, radius = o.ring_polar(cap, R_lo, R_hi)
    ex, rho = cf.bardeen_ring_polar(a, inc, n_th)
    dR = (R_hi - R_lo) / n_R
    assert np.max(np.abs(radius - rho)) < 1.0 * dR
    for k in ("alpha_min", "alpha_max", "D", "R_mean"):
        assert abs(st[k] - ex[k]) < dR, k
    assert abs(st["A"] - ex["A"]) < dR
    Rf, Af = _paper_fit(a, inc)                                                # eqs. (11)-(14): soft, they are fits
    assert abs(st["R_mean"] - Rf) < 0.04 and abs(st["A"] - Af) < 0.04


def _random_null_state(rng, a):
    r, th = rng.uniform(2.5, 50.0), rng.uniform(0.2, np.pi - 0.2)
    kr, kh, kp = rng.normal(size=3) * np.array([1.0, 1.0 / r, 1.0 / (r * np.sin(th))])
    g = o.metric(a, r, th)
    C = g[1, 1] * kr * kr + g[2, 2] * kh * kh + g[3, 3] * kp * kp
    B = g[0, 3] * kp
    kt = (-B - np.sqrt(B * B - g[0, 0] * C)) / g[0, 0]
    return np.array([0.0, r, th, rng.uniform(-3, 3), kt, kr, kh, kp])


def test_reduced_system_is_the_full_system_with_the_killing_constants_eliminated():
    # NEXT-3.  Pin: the full right-hand side (itself pinned by the conservation laws): at any state, k^t and k^phi
    # rebuilt from E = -k_t and L_z = k_phi are the state's own, and the r, theta accelerations coincide.
    rng = np.random.default_rng(5)
    for a in (0.0, 0.5, 0.99):
        for _ in range(50):
            y = _random_null_state(rng, a)
            E, L, Q, _n = o.invariants(a, y)
            kt, kp = o.killing_velocities(a, E, L, y[1], y[2])
            assert abs(kt - y[4]) <= 1e-12 * abs(y[4]) and abs(kp - y[7]) <= 1e-12 * max(abs(y[7]), abs(y[4]) / y[1] ** 2)
            d6 = o.rhs_reduced(a, E, L, y[[0, 1, 2, 3, 5, 6]])
            d8 = o.rhs(a, y)
            scale = np.abs(d8).max()
            assert np.all(np.abs(d6 - d8[[0, 1, 2, 3, 5, 6]]) <= 1e-12 * np.maximum(np.abs(d8[[0, 1, 2, 3, 5, 6]]), scale * 1e-3))


def test_reduced_system_integration_classifies_conserves_and_converges_to_the_full_system():
    R = o.SYS_REDUCED
    # a = 0: the sqrt(27) circle; Kerr: the exact radial-potential classifier
    for a, inc, W in [(0.0, 60.0, 10.0), (0.9, 60.0, 10.0)]:
        n = 24
        res = o.trace(a, 1000.0, inc, W, n, n, rule=o.STEP_EQ2, threads=8, system=R)
        al = -W + (np.arange(n) + 0.5) * 2 * W / n
        A_, B_ = np.meshgrid(al, al)
        rho_c = cf.bardeen_rho(a, inc, np.arctan2(B_, A_).ravel()) if a else np.full(n * n, np.sqrt(27.0))
        band = np.abs(np.hypot(A_, B_).ravel() / rho_c - 1) < 0.01
        inv = np.array([o.invariants(a, v) for v in res["y0"]])
        exact = np.array([cf.captured_exact(a, L / E, Q / E ** 2) for E, L, Q, _ in inv])
        assert np.all(((res["status"] == o.CAPTURED) == exact) | band)
        inv1 = np.array([o.invariants(a, v) for v in res["y"]])
        esc = res["status"] == o.ESCAPED
        # E and L_z are constants of the reduced system: conserved to rounding, not to truncation
        assert np.max(np.abs(inv1[esc, 0] - inv[esc, 0])) < 1e-12 and np.max(np.abs(inv1[esc, 1] - inv[esc, 1])) < 1e-11
        assert np.max(np.abs(inv1[esc, 2] - inv[esc, 2]) / np.maximum(np.abs(inv[esc, 2]), 0.1)) < 1e-4      # Q: truncation
    # step halving: Q drift and the distance to the full system's solution both fall ~16x per halving
    a = 0.9
    y0 = o.init_ray(a, 1000.0, 60.0, 6.0, 5.0)
    Q0 = o.invariants(a, y0)[2]
    dq, dist = [], []
    for h in (1 / 16, 1 / 32, 1 / 64):
        nsteps = int(round(300 * (1 / 16) / h))
        yr = o.integrate(a, y0, h, 1.0, 1e9, o.STEP_REL, 10 ** 6, force_steps=nsteps, system=R)[0]
        yf = o.integrate(a, y0, h, 1.0, 1e9, o.STEP_REL, 10 ** 6, force_steps=nsteps)[0]
        dq.append(abs(o.invariants(a, yr)[2] - Q0))
        dist.append(np.max(np.abs(yr[1:4] - yf[1:4])))
    assert 10 < dq[0] / dq[1] < 40 and 10 < dq[1] / dq[2] < 40, dq                 # 4th order or better
    assert 10 < dist[0] / dist[1] < 40 and 10 < dist[1] / dist[2] < 40, dist


def test_captured_rays_final_state_schwarzschild_orbit_integral():
    # The final state of CAPTURED rays (stopped at r < 1.01 r_h) pinned for a = 0: an equatorial ray (i = 90 deg,
    # beta = 0) with impact parameter b < sqrt(27) has no turning point, and phi swept from the start to the final
    # radius is the textbook integral  int_{u0}^{uf} du / sqrt(1/b^2 - u^2 (1 - 2u)),  u = 1/r.
    from scipy import integrate as sint
    a = 0.0
    for al in (1.0, 3.0, 4.5, 5.1):
        y0 = o.init_ray(a, 1000.0, 90.0, al, 0.0)
        y, st, n = o.integrate(a, y0, 1 / 32, 1.01 * 2.0, 1010.0, o.STEP_EQ2, 20000)
        assert st == o.CAPTURED and 2.0 < y[1] < 2.02 and abs(y[2] - np.pi / 2) < 1e-12
        E, L, Q, _ = o.invariants(a, y0)
        b = abs(L) / E
        f = lambda u: 1.0 / (b * b) - u * u * (1.0 - 2.0 * u)
        exact = sint.quad(lambda u: 1.0 / np.sqrt(f(u)), 1.0 / y0[1], 1.0 / y[1], epsabs=1e-13, epsrel=1e-13, limit=400)[0]
        assert abs(abs(y[3] - y0[3]) - exact) < 2e-5 * exact, (al, abs(y[3] - y0[3]), exact)
        # and the radial momentum there follows from the null condition with the conserved E, L
        kr_exact = np.sqrt(E * E - (1 - 2 / y[1]) * L * L / y[1] ** 2)   # > 0: r grows with lambda, the ray is traced backwards
        assert abs(y[5] - kr_exact) < 2e-2 * kr_exact               # the last steps next to the coordinate singularity: ~1 %


def test_equatorial_kerr_rays_against_the_bardeen_1972_quadrature():
    # Kerr pin for whole trajectories, captured ones included: a ray in the equatorial plane (i = 90 deg, beta = 0)
    # stays there, and with E = -k_t, L = k_phi (textbook, Bardeen, Press & Teukolsky 1972)
    #     dphi/dl = [(1 - 2/r) L + (2a/r) E] / Delta,      (dr/dl)^2 = E^2 + (a^2 E^2 - L^2)/r^2 + 2 (L - a E)^2 / r^3,
    # so phi along a ray without a turning point is a quadrature in r.  Checked for rays captured on the prograde and on
    # the retrograde side (frame dragging reverses dphi/dl of the latter near the horizon).
    from scipy import integrate as sint
    a = 0.9
    rh = o.horizon(a)
    checked = 0
    for al in (-2.5, -1.0, 1.0, 3.0, 5.5):
        y0 = o.init_ray(a, 1000.0, 90.0, al, 0.0)
        y, st, n = o.integrate(a, y0, 1 / 32, 1.01 * rh, 1010.0, o.STEP_EQ2, 20000)
        assert abs(y[2] - np.pi / 2) < 1e-12
        if st != o.CAPTURED:
            continue
        E, L, Q, _ = o.invariants(a, y0)
        dphi = lambda r: ((1 - 2 / r) * L + 2 * a * E / r) / (r * r - 2 * r + a * a)
        rdot = lambda r: np.sqrt(E * E + (a * a * E * E - L * L) / r ** 2 + 2 * (L - a * E) ** 2 / r ** 3)
        sweep = sint.quad(lambda r: dphi(r) / rdot(r), y[1], y0[1], epsabs=1e-13, epsrel=1e-13, limit=800)[0]
        got = y0[3] - y[3]                      # the physical photon runs from the hole (y) out to the observer (y0)
        assert abs(got - sweep) < 5e-5 * max(1.0, abs(sweep)), (al, got, sweep)
        assert abs(y[5] - rdot(y[1])) < 2e-2 * rdot(y[1])
        checked += 1
    assert checked >= 4


# ---- whole Kerr trajectories off the equatorial plane, against Carter's separated first-order equations ----------
def _carter_flow(a, y0, events):
    """The same geodesic from a different formulation: Carter's (1968) separated equations in Mino time tau
    (dlambda = Sigma dtau) for the covariant momenta, with the constants E = -p_t, L = p_phi of the initial state:
        dr/dtau = Delta p_r,      dp_r/dtau  = -(r - 1) p_r^2 + 2 r E R0 / Delta - (r - 1) R0^2 / Delta^2,   R0 = (r^2 + a^2) E - a L,
        dth/dtau = p_th,          dp_th/dtau = (L/s - a E s)(L c / s^2 + a E c),
        dphi/dtau = a R0 / Delta - a E + L / s^2
    (no Christoffel symbols, no second-order equations), integrated by scipy's DOP853 at 1e-13 towards negative tau
    (the oracle steps dlambda < 0) until `events` (terminal) fires.  Returns the solve_ivp result."""
    from scipy.integrate import solve_ivp
    E, L, _, _ = o.invariants(a, y0)
    r, th = y0[1], y0[2]
    Sg, Dl = r * r + (a * np.cos(th)) ** 2, r * r - 2 * r + a * a
    z0 = np.array([r, th, y0[3], Sg / Dl * y0[5], Sg * y0[6]])

    def f(tau, z):
        r, th, ph, pr, pt = z
        s, c = np.sin(th), np.cos(th)
        Dl = r * r - 2 * r + a * a
        R0 = (r * r + a * a) * E - a * L
        return [Dl * pr, pt, a * R0 / Dl - a * E + L / (s * s),
                -(r - 1) * pr * pr + 2 * r * E * R0 / Dl - (r - 1) * R0 * R0 / (Dl * Dl),
                (L / s - a * E * s) * (L * c / (s * s) + a * E * c)]

    guard = lambda tau, z: z[0] - 1.003 * o.horizon(a)      # the equations are singular on the horizon: stop short of it
    guard.terminal = True
    return solve_ivp(f, (0.0, -1e3), z0, method="DOP853", rtol=1e-13, atol=1e-14, events=[events, guard])


def test_kerr_rays_off_the_equator_against_carters_separated_equations():
    # The final state of whole Kerr (a != 0) trajectories away from the equatorial plane, CAPTURED ones (stopped at the
    # first step below 1.01 r_h) and ESCAPED ones: the oracle's final (r, theta, phi) must lie on the geodesic that
    # Carter's first-order equations give for the same initial state - theta and phi compared where that solution
    # reaches the oracle's final radius - to the RK4 scheme's truncation error, which falls ~16x when h is halved.
    a = 0.9
    rh = o.horizon(a)
    seen = {o.CAPTURED: 0, o.ESCAPED: 0}
    for inc, al, be in [(60.0, 1.0, 2.0), (60.0, -1.5, -3.0), (30.0, 2.0, 1.0), (75.0, 0.5, -2.5), (60.0, 6.0, 5.0), (45.0, -7.0, 3.0),
                        (60.0, 3.5, 6.5)]:
        y0 = o.init_ray(a, 1000.0, inc, al, be)
        errs = []
        for h in (1 / 32, 1 / 64):
            y, st, n = o.integrate(a, y0, h, 1.01 * rh, 1010.0, o.STEP_EQ2, 40000)
            assert st in seen
            if st == o.CAPTURED:
                ev = lambda tau, z, rf=y[1]: z[0] - rf            # inward all the way: the first crossing of r_f
                ev.direction = 0
            else:
                ev = lambda tau, z, rf=y[1]: z[0] - rf if tau < -1e-6 else -1.0      # outbound crossing, after the periapsis
                ev.direction = 0
            ev.terminal = True
            sol = _carter_flow(a, y0, ev)
            assert sol.status == 1 and len(sol.y_events[0]) == 1, (inc, al, be, st)
            rE, thE, phE = sol.y_events[0][0][:3]
            assert abs(rE - y[1]) < 1e-9 * y[1]
            errs.append(max(abs(y[2] - thE), abs(y[3] - phE)))
        seen[st] += 1
        assert errs[0] < 1e-5, (inc, al, be, st, errs)                       # h = 1/32: the scheme's truncation error
        assert errs[1] < errs[0] / 10, (inc, al, be, st, errs)      # and it falls at ~4th order
    assert seen[o.CAPTURED] >= 3 and seen[o.ESCAPED] >= 3, seen


def test_equatorial_projection_kerr_crossing_against_carters_separated_equations():
    # The Kerr equatorial-plane crossing of stop_at_equator (R19): (r, phi) of the landed state against the point where
    # the solution of Carter's first-order equations first reaches theta = pi/2.
    a = 0.95
    for inc, al, be in [(60.0, 5.0, 8.0), (60.0, -7.0, 6.0), (60.0, 9.0, -9.0), (30.0, 2.0, 9.0), (80.0, -3.0, 4.0)]:
        y0 = o.init_ray(a, 1000.0, inc, al, be)
        ev = lambda tau, z: z[1] - np.pi / 2
        ev.terminal, ev.direction = True, 0
        sol = _carter_flow(a, y0, ev)
        assert sol.status == 1 and len(sol.y_events[0]) == 1
        rE, _, phE = sol.y_events[0][0][:3]
        errs = []
        for h in (1 / 32, 1 / 64):
            y, st, n = o.integrate(a, y0, h, 1.01 * o.horizon(a), 1010.0, o.STEP_EQ2, 40000, stop_at_equator=True)
            assert st == o.EQUATOR and abs(y[2] - np.pi / 2) < 1e-8
            errs.append(max(abs(y[1] - rE) / rE, abs(y[3] - phE)))
        assert errs[0] < 1e-5, (inc, al, be, errs)
        assert errs[1] < errs[0] / 6 or errs[1] < 2e-8, (inc, al, be, errs)
