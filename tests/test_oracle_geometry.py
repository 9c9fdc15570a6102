"""Pins for the oracle's metric, Christoffel symbols, RHS and invariants (-m "not gpu").

None of these compares the oracle with a retyped copy of its own formula: they use what the
mathematics fixes (Kerr is a vacuum solution; the connection is metric-compatible; geodesic
motion conserves E, L_z, Q and the norm; a = 0 is Schwarzschild).
"""
import numpy as np
import pytest

import oracle as o

RNG = np.random.default_rng(1303_5057)
POINTS = [(a, r, th) for a in (0.0, 0.3, 0.9, 0.99) for r, th in ((2.7, 0.4), (6.0, 1.3), (40.0, 2.5))]


def test_metric_textbook_facts():
    # det g = -Sigma^2 sin^2(theta);  g_tt g_phiphi - g_tphi^2 = -Delta sin^2(theta);
    # g^rr = Delta/Sigma vanishes at r_bh = 1 + sqrt(1 - a^2)
    for a, r, th in POINTS:
        g = o.metric(a, r, th)
        Sigma = r * r + a * a * np.cos(th) ** 2
        Delta = r * r - 2 * r + a * a
        assert np.allclose(g, g.T)
        assert np.isclose(np.linalg.det(g), -Sigma ** 2 * np.sin(th) ** 2, rtol=1e-12)
        assert np.isclose(g[0, 0] * g[3, 3] - g[0, 3] ** 2, -Delta * np.sin(th) ** 2, rtol=1e-12)
    for a in (0.0, 0.5, 0.99):
        rh = o.horizon(a)
        assert np.isclose(rh, 1 + np.sqrt(1 - a * a))
        g = o.metric(a, rh * (1 + 1e-9), 1.0)
        assert 1.0 / g[1, 1] < 1e-8       # g^rr -> 0 at the horizon


def test_metric_asymptotically_flat_and_schwarzschild():
    g = o.metric(0.0, 10.0, 1.1)
    assert np.allclose(np.diag(g), [-(1 - 0.2), 1 / (1 - 0.2), 100.0, 100.0 * np.sin(1.1) ** 2])
    assert g[0, 3] == 0.0
    g = o.metric(0.9, 1e6, 0.7)
    assert np.allclose(np.diag(g) / [-1, 1, 1e12, 1e12 * np.sin(0.7) ** 2], 1.0, atol=1e-5)
    # frame dragging: g_tphi -> -2 J sin^2(theta) / r with J = a M
    assert np.isclose(g[0, 3], -2 * 0.9 * np.sin(0.7) ** 2 / 1e6, rtol=1e-6)


def _dmetric(a, r, th, eps=1e-5):
    """d g / d x^c by 4th-order central differences, c in (r, theta)."""
    dg = np.zeros((4, 4, 4))
    for c, (dr, dth) in ((1, (eps * r, 0.0)), (2, (0.0, eps))):
        h = dr + dth
        dg[c] = (-o.metric(a, r + 2 * dr, th + 2 * dth) + 8 * o.metric(a, r + dr, th + dth)
                 - 8 * o.metric(a, r - dr, th - dth) + o.metric(a, r - 2 * dr, th - 2 * dth)) / (12 * h)
    return dg


def test_christoffel_from_metric_derivatives():
    # Gamma^m_ab = 1/2 g^{mn} (d_a g_nb + d_b g_na - d_n g_ab), the definition, with numerical
    # derivatives of the (independently pinned) metric
    for a, r, th in POINTS:
        g = o.metric(a, r, th)
        gi = np.linalg.inv(g)
        dg = _dmetric(a, r, th)
        ref = np.zeros((4, 4, 4))
        for m in range(4):
            for al in range(4):
                for be in range(4):
                    ref[m, al, be] = 0.5 * sum(gi[m, n] * (dg[al][n, be] + dg[be][n, al] - dg[n][al, be])
                                               for n in range(4))
        G = o.christoffel(a, r, th)
        assert np.allclose(G, ref, rtol=1e-7, atol=1e-9), (a, r, th)
        assert np.allclose(G, G.transpose(0, 2, 1))
        # exactly the 20 independent non-zero symbols when a != 0
        nz = sum(1 for m in range(4) for al in range(4) for be in range(al, 4) if G[m, al, be] != 0.0)
        assert nz == (20 if a != 0 else 9)


def test_christoffel_schwarzschild_textbook():
    r, th = 7.0, 0.9
    G = o.christoffel(0.0, r, th)
    f = 1 - 2 / r
    t, R, h, p = 0, 1, 2, 3
    assert np.isclose(G[t, t, R], 1 / (r * r * f))
    assert np.isclose(G[R, t, t], f / (r * r))
    assert np.isclose(G[R, R, R], -1 / (r * r * f))
    assert np.isclose(G[R, h, h], -(r - 2))
    assert np.isclose(G[R, p, p], -(r - 2) * np.sin(th) ** 2)
    assert np.isclose(G[h, R, h], 1 / r) and np.isclose(G[p, R, p], 1 / r)
    assert np.isclose(G[h, p, p], -np.sin(th) * np.cos(th))
    assert np.isclose(G[p, h, p], np.cos(th) / np.sin(th))


def test_kerr_is_ricci_flat():
    # R_ab = d_c G^c_ab - d_b G^c_ac + G^c_cd G^d_ab - G^c_bd G^d_ac = 0 (vacuum).  A wrong sign,
    # power or factor in any symbol breaks this.
    def dG(a, r, th, eps=1e-4):
        d = np.zeros((4, 4, 4, 4))
        for c, (dr, dth) in ((1, (eps * r, 0.0)), (2, (0.0, eps))):
            h = dr + dth
            d[c] = (-o.christoffel(a, r + 2 * dr, th + 2 * dth) + 8 * o.christoffel(a, r + dr, th + dth)
                    - 8 * o.christoffel(a, r - dr, th - dth) + o.christoffel(a, r - 2 * dr, th - 2 * dth)) / (12 * h)
        return d
    for a, r, th in [(0.9, 3.0, 0.8), (0.99, 2.0, 1.9), (0.5, 8.0, 0.3)]:
        G = o.christoffel(a, r, th)
        d = dG(a, r, th)
        Ric = (np.einsum("ccab->ab", d) - np.einsum("bcac->ab", d)
               + np.einsum("ccd,dab->ab", G, G) - np.einsum("cbd,dac->ab", G, G))
        scale = np.abs(np.einsum("ccd,dab->ab", G, G)).max()
        assert np.abs(Ric).max() < 1e-8 * max(scale, 1.0), (a, r, th, np.abs(Ric).max())


def _random_null_state(a):
    r = RNG.uniform(1.2 * o.horizon(a), 30.0)
    th = RNG.uniform(0.15, np.pi - 0.15)
    kr, kh, kp = RNG.normal(size=3) * [1.0, 1.0 / r, 1.0 / r]
    g = o.metric(a, r, th)
    C = g[1, 1] * kr ** 2 + g[2, 2] * kh ** 2 + g[3, 3] * kp ** 2
    B = g[0, 3] * kp
    kt = (-B - np.sqrt(B * B - g[0, 0] * C)) / g[0, 0] if g[0, 0] < 0 else None
    if kt is None:
        return _random_null_state(a)
    return np.array([0.3, r, th, 1.0, kt, kr, kh, kp])


def test_rhs_matches_full_contraction():
    # rhs() uses shared sub-expressions; the plain 4x4x4 contraction with christoffel() (pinned
    # above against the metric's derivatives) must give the same accelerations
    for a in (0.0, 0.7, 0.99):
        for _ in range(20):
            y = _random_null_state(a)
            G = o.christoffel(a, y[1], y[2])
            acc = -np.einsum("mab,a,b->m", G, y[4:], y[4:])
            dy = o.rhs(a, y)
            assert np.allclose(dy[:4], y[4:], rtol=0, atol=0)
            assert np.allclose(dy[4:], acc, rtol=1e-11, atol=1e-13)


def test_rhs_conserves_invariants_locally():
    # d/dlambda (E, L_z, Q, g k k) = 0 along the flow of rhs(): central difference along the flow,
    # no integrator involved (SURVEY 8(c) "local conservation")
    for a in (0.0, 0.5, 0.9, 0.99):
        for _ in range(25):
            y = _random_null_state(a)
            dy = o.rhs(a, y)
            eps = 1e-5 * y[1]
            # second-order Taylor step along the flow in both directions (error O(eps^3) cancels to O(eps^2) in the difference)
            d2p = o.rhs(a, y + 0.5 * eps * dy)
            d2m = o.rhs(a, y - 0.5 * eps * dy)
            ip = o.invariants(a, y + eps * d2p)
            im = o.invariants(a, y - eps * d2m)
            i0 = o.invariants(a, y)
            scale = np.array([abs(i0[0]), abs(i0[1]) + 1, abs(i0[2]) + 1, 1.0])
            drift = np.abs(ip - im) / (2 * eps) / scale
            # compare with the size of a non-conserved quantity's derivative, |dk/dlambda|/|k|
            ref = np.abs(dy[4:]).max() / np.abs(y[4:]).max()
            assert np.all(drift[:3] < 1e-6 * max(ref, 1e-3) + 1e-9), (a, y, drift, ref)
            assert abs(i0[3]) < 1e-12          # the state is null


def test_invariants_equatorial_closed_form():
    # a = 0, equatorial circular-ish state: E = (1 - 2/r) k^t, L = r^2 k^phi, Q = r^4 (k^theta)^2
    r = 9.0
    y = np.array([0, r, np.pi / 2, 0, 1.3, 0.1, 0.02, 0.05])
    E, L, Q, _ = o.invariants(0.0, y)
    assert np.isclose(E, (1 - 2 / r) * 1.3) and np.isclose(L, r * r * 0.05)
    assert np.isclose(Q, (r * r * 0.02) ** 2)
    # Kerr equatorial: L = g_phiphi k^phi + g_tphi k^t with g_phiphi = r^2 + a^2 + 2 a^2 / r
    a = 0.8
    E, L, Q, _ = o.invariants(a, y)
    assert np.isclose(L, (r * r + a * a + 2 * a * a / r) * 0.05 - 2 * a / r * 1.3)
    assert np.isclose(E, (1 - 2 / r) * 1.3 + 2 * a / r * 0.05)
