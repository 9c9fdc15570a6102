"""Closed forms the oracle (and then the CUDA path) are pinned against.  Test harness only.

Nothing here is used by the oracle or the product; these are the textbook results of Kerr photon
orbits (Bardeen 1973) written independently in numpy, in the notation of SURVEY.md App. A.4:
  xi  = L_z / E,  eta = Q / E^2,
  spherical photon orbits at radius r_p:
      xi(r_p)  = -[r_p^2 (r_p - 3) + a^2 (r_p + 1)] / [a (r_p - 1)]
      eta(r_p) = r_p^3 [4 a^2 - r_p (r_p - 3)^2] / [a^2 (r_p - 1)^2]
  image-plane curve at inclination i:  alpha = -xi / sin i,
      beta = +-sqrt(eta + a^2 cos^2 i - xi^2 cot^2 i)
  radial potential R(r) = r^4 + (a^2 - xi^2 - eta) r^2 + 2 [eta + (xi - a)^2] r - a^2 eta.
"""
import numpy as np
from scipy import integrate, optimize


def horizon(a):
    return 1.0 + np.sqrt(1.0 - a * a)


def photon_orbit_radii(a):
    """Prograde and retrograde equatorial circular photon orbits."""
    pro = 2.0 * (1.0 + np.cos(2.0 / 3.0 * np.arccos(-a)))
    ret = 2.0 * (1.0 + np.cos(2.0 / 3.0 * np.arccos(a)))
    return pro, ret


def xi_eta(a, rp):
    xi = -(rp * rp * (rp - 3.0) + a * a * (rp + 1.0)) / (a * (rp - 1.0))
    eta = rp ** 3 * (4.0 * a * a - rp * (rp - 3.0) ** 2) / (a * a * (rp - 1.0) ** 2)
    return xi, eta


def bardeen_curve(a, inc_deg, n=200001):
    """Upper half (beta >= 0) of the critical curve, ordered by increasing alpha.

    Returns alpha[], beta[].  a = 0 gives the circle of radius sqrt(27).
    """
    i = np.deg2rad(inc_deg)
    if a == 0.0:
        t = np.linspace(np.pi, 0.0, n)
        return np.sqrt(27.0) * np.cos(t), np.sqrt(27.0) * np.sin(t)
    pro, ret = photon_orbit_radii(a)

    def radicand(rp):
        xi, eta = xi_eta(a, rp)
        return eta + a * a * np.cos(i) ** 2 - xi * xi / np.tan(i) ** 2

    # end points: beta = 0.  The radicand is positive between two roots inside [pro, ret].
    rmid = optimize.minimize_scalar(lambda x: -radicand(x), bounds=(pro, ret), method="bounded",
                                    options=dict(xatol=1e-14)).x
    lo = optimize.brentq(radicand, pro - 1e-12 if radicand(pro - 1e-12) < 0 else pro * (1 - 1e-9), rmid,
                         xtol=1e-15) if radicand(pro) < 0 else pro
    hi = optimize.brentq(radicand, rmid, ret, xtol=1e-15) if radicand(ret) < 0 else ret
    # cluster the samples at the end points, where beta ~ sqrt(distance)
    t = 0.5 * (1.0 - np.cos(np.linspace(0.0, np.pi, n)))
    rp = lo + (hi - lo) * t
    xi, eta = xi_eta(a, rp)
    alpha = -xi / np.sin(i)
    beta = np.sqrt(np.maximum(radicand(rp), 0.0))
    beta[0] = 0.0
    beta[-1] = 0.0
    return alpha, beta


def bardeen_rho(a, inc_deg, vartheta):
    """Radius of the critical curve along the spoke at polar angle vartheta about the image origin.
    Symmetries: i -> 180 - i leaves the curve unchanged (it depends on sin i and cos^2 i); a -> -a mirrors alpha."""
    if inc_deg > 90.0:
        inc_deg = 180.0 - inc_deg
    if a < 0.0:
        return bardeen_rho(-a, inc_deg, np.pi - np.asarray(vartheta, dtype=float))
    al, be = bardeen_curve(a, inc_deg)
    ang = np.arctan2(be, al)          # pi ... 0, decreasing along the curve
    rho = np.hypot(al, be)
    vt = np.mod(np.asarray(vartheta, dtype=float), 2 * np.pi)
    vt = np.where(vt > np.pi, 2 * np.pi - vt, vt)   # the curve is symmetric in beta
    return np.interp(vt, ang[::-1], rho[::-1])


def bardeen_stats(a, inc_deg, n_angles=3600):
    """area, alpha_min, alpha_max, D (eq. 6), <R> (eq. 7), A (eq. 8) of the critical curve.

    <R>, A with the spoke angle about the image origin and R from (centre, 0), uniform weights
    (reading R13), centre = (alpha_min + alpha_max)/2 (signed).
    """
    al, be = bardeen_curve(a, inc_deg)
    area = 2.0 * integrate.trapezoid(be, al)
    amin, amax = al[0], al[-1]
    centre = 0.5 * (amin + amax)
    vt = 2 * np.pi * (np.arange(n_angles) + 0.5) / n_angles
    rho = bardeen_rho(a, inc_deg, vt)
    R = np.hypot(rho * np.cos(vt) - centre, rho * np.sin(vt))
    return dict(area=area, alpha_min=amin, alpha_max=amax, D=abs(centre), R_mean=R.mean(),
                A=2.0 * R.std())


def captured_exact(a, xi, eta):
    """A photon arriving from infinity with (xi, eta) is captured iff R(r) has no real root
    outside the horizon (no radial turning point)."""
    coeffs = [1.0, 0.0, a * a - xi * xi - eta, 2.0 * (eta + (xi - a) ** 2), -a * a * eta]
    roots = np.roots(coeffs)
    real = roots[np.abs(roots.imag) < 1e-9 * np.maximum(1.0, np.abs(roots.real))].real
    return not np.any(real > horizon(a) * (1 + 1e-12))


def sin_theta_min(a, xi, eta):
    """Sine of the smallest polar angle a photon with (xi, eta), eta >= 0, can reach: the root of
    Theta(theta) = eta + a^2 cos^2(theta) - xi^2 cot^2(theta) = 0.  With u = cos^2(theta):
    a^2 u^2 + (eta + xi^2 - a^2) u - eta = 0, u_max its non-negative root."""
    B = eta + xi * xi - a * a
    u = 2.0 * eta / (B + np.sqrt(B * B + 4.0 * a * a * eta))
    return np.sqrt(np.clip(1.0 - u, 0.0, 1.0))


def schwarzschild_dphi(b, r_start, r_end):
    """|change of phi| of a Schwarzschild (M = 1) photon of impact parameter b > sqrt(27) that
    comes in from r_start, turns at r_min and goes out to r_end (textbook orbit integral,
    u = 1/r:  dphi/du = 1/sqrt(1/b^2 - u^2 (1 - 2u)))."""
    f = lambda u: 1.0 / (b * b) - u * u * (1.0 - 2.0 * u)
    # turning point: the largest u below 1/3 where f = 0
    um = optimize.brentq(f, 1.0 / b * 0.5, 1.0 / 3.0, xtol=1e-16)

    def leg(u0):
        # u = um - s^2 removes the inverse-square-root end-point singularity
        g = lambda s: 2.0 * s / np.sqrt(max(f(um - s * s), 1e-300))
        val, _ = integrate.quad(g, 0.0, np.sqrt(um - u0), epsabs=1e-13, epsrel=1e-13, limit=400)
        return val

    return leg(1.0 / r_start) + leg(1.0 / r_end)


def bardeen_ring_polar(a, inc_deg, n_theta=181):
    """The paper's ring statistics (eqs. 6-10) of the closed-form critical curve, sampled like the paper's
    polar grid: spokes vartheta_k = k pi / (n_theta - 1) about the image origin, R about the ring centre
    ((alpha_min + alpha_max)/2, 0), integrals over [0, pi] by the trapezoidal rule.  i = 0 and a = 0 are the circles
    sqrt(eta(xi = 0) + a^2) and sqrt(27)."""
    vt = np.pi * np.arange(n_theta) / (n_theta - 1)
    if a == 0.0:
        rho = np.full(n_theta, np.sqrt(27.0))
    elif inc_deg == 0.0:
        lo, hi = photon_orbit_radii(a)
        rp = optimize.brentq(lambda r: xi_eta(a, r)[0], lo, hi, xtol=1e-15)
        rho = np.full(n_theta, np.sqrt(xi_eta(a, rp)[1] + a * a))
    else:
        rho = bardeen_rho(a, inc_deg, vt)
    amax, amin = rho[0], -rho[-1]
    c = 0.5 * (amin + amax)
    R = np.hypot(rho * np.cos(vt) - c, rho * np.sin(vt))
    w = np.ones(n_theta)
    w[0] = w[-1] = 0.5
    mean = np.sum(w * R) / (n_theta - 1)
    A = 2.0 * np.sqrt(np.sum(w * (R - mean) ** 2) / (n_theta - 1))
    return dict(alpha_min=amin, alpha_max=amax, D=abs(c), R_mean=mean, A=A), rho
