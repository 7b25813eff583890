"""Pins of the oracle's Q-point Gauss-Legendre rule for the t-integral of eq. (24) (PAPER.md:152-168,
eq. (25)-(28)).  CPU only.

What would fail if it were wrong:
  nodes/weights            -> numpy's leggauss mapped to [0, 1]
  A_i, B_i, C_i of (26)-(28) or the prefactor of (24)
                           -> the closed-form (arctan) segment integrals of the flux-tube profile, eq. (68)
  the rule itself          -> convergence order h^(2Q) on a subdivided polygon against its exact line integral,
                              and against the flux through a square (Stokes, eq. (19)-(20)) by dblquad
  Q = 1                    -> the midpoint rule of wlo_loop_phase_spin (already pinned in test_oracle_loop.py)
  weights not summing to 1 -> the uniform-field shoelace area, any Q
"""
import numpy as np
import pytest
from scipy import integrate

from oracle import wl_oracle as o


def _rand_loop(rng, N, scale=0.6):
    y = rng.normal(size=(N, 2)) * scale
    return y - y.mean(0)


def _subdivide(poly, k):
    """Every segment of the closed polygon cut into k collinear pieces: the same curve, k times the points."""
    pts = []
    n = len(poly)
    for i in range(n):
        a, b = poly[i], poly[(i + 1) % n]
        for j in range(k):
            pts.append(a + (b - a) * j / k)
    return np.array(pts)


@pytest.mark.parametrize("Q", [1, 2, 3])
def test_nodes_and_weights_are_gauss_legendre_on_0_1(Q):
    t, w = o.gauss_legendre_01(Q)
    x, wx = np.polynomial.legendre.leggauss(Q)
    assert np.allclose(t, 0.5 * (x + 1.0), rtol=0, atol=1e-15)
    assert np.allclose(w, 0.5 * wx, rtol=0, atol=1e-15)
    # exact for polynomials of degree 2Q - 1 in t, not for degree 2Q
    for d in range(2 * Q):
        assert abs(np.sum(w * t ** d) - 1.0 / (d + 1)) < 1e-15
    assert abs(np.sum(w * t ** (2 * Q)) - 1.0 / (2 * Q + 1)) > 1e-4


def test_bad_order_is_rejected():
    y = _rand_loop(np.random.default_rng(0), 8)
    for Q in (0, 4, -1):
        with pytest.raises(ValueError):
            o.loop_phase_spin_q(o.SECH2, [1.0, 1.0], y, 1.0, 0.0, 0.0, Q)


def test_Q1_is_the_midpoint_rule():
    """rho_i^2(1/2) = A + B + C/4 = |(x_i + x_{i+1})/2|^2 and x^i y^{i+1} - y^i x^{i+1} = m x d: same numbers
    up to rounding; the spin sum is the same expression and must agree bit for bit."""
    rng = np.random.default_rng(11)
    for prof, par in [(o.SECH2, [1.3, 0.7]), (o.FLUXTUBE, [10.0, 1.0]), (o.UNIFORM, [2.0])]:
        for N in (3, 4, 17, 256):
            y = _rand_loop(rng, N)
            for T, cx, cy in [(0.01, 0.0, 0.0), (1.0, 0.4, -0.3), (9.0, 2.0, 1.0)]:
                p0, s0 = o.loop_phase_spin(prof, par, y, T, cx, cy)
                p1, s1 = o.loop_phase_spin_q(prof, par, y, T, cx, cy, 1)
                assert abs(p1 - p0) <= 2e-13 * max(1.0, abs(p0))
                assert s1 == s0


@pytest.mark.parametrize("Q", [1, 2, 3])
def test_uniform_field_gives_the_shoelace_area_for_every_Q(Q):
    """eq. (19)-(20): phase = eB x area for any quadrature whose weights sum to one (g is constant)."""
    rng = np.random.default_rng(12)
    y = _rand_loop(rng, 100)
    area = 0.5 * np.sum(y[:, 0] * np.roll(y[:, 1], -1) - y[:, 1] * np.roll(y[:, 0], -1))
    for T, cx, cy in [(0.5, 0.0, 0.0), (4.0, 3.0, -1.0)]:
        ph, sp = o.loop_phase_spin_q(o.UNIFORM, [1.7], y, T, cx, cy, Q)
        assert abs(ph - 1.7 * T * area) < 1e-12 * max(1.0, abs(1.7 * T * area))
        assert abs(sp - 1.7 * T) < 1e-13 * 1.7 * T


def _fluxtube_polygon_exact(F, lam, x):
    """Exact e oint A.dr round the closed polygon x[n][2] for eq. (68): per segment, eq. (24) with
    f/rho^2 = 1/(lam^2 + rho^2) and rho^2(t) = A + 2Bt + Ct^2 (eq. (25)):
    int_0^1 dt/(a + 2Bt + Ct^2) = [atan((Ct + B)/sqrt(D))]_0^1/sqrt(D),  a = lam^2 + A,  D = aC - B^2 > 0."""
    xn = np.roll(x, -1, axis=0)
    d = xn - x
    A = np.sum(x * x, 1)
    B = np.sum(x * d, 1)
    Cc = np.sum(d * d, 1)
    a = lam * lam + A
    D = a * Cc - B * B
    sD = np.sqrt(D)
    integral = (np.arctan((Cc + B) / sD) - np.arctan(B / sD)) / sD
    cross = x[:, 0] * xn[:, 1] - x[:, 1] * xn[:, 0]
    return F * np.sum(cross * integral)


@pytest.mark.parametrize("Q", [1, 2, 3])
def test_converges_to_the_exact_polygon_integral_with_order_2Q(Q):
    """where the segment integrals can be done analytically the result is exact; the numerical
    rule must approach it.  Subdividing the segments leaves the curve (and the exact integral) unchanged and
    shrinks h, so the error of the Q-point rule falls like h^(2Q)."""
    rng = np.random.default_rng(13)
    F, lam = 10.0, 1.0
    poly = _rand_loop(rng, 12, scale=1.2)
    T, cx, cy = 1.0, 0.3, -0.2
    exact = _fluxtube_polygon_exact(F, lam, poly + np.array([cx, cy]))
    errs = []
    for k in (8, 16, 32):                      # h well below lambda: the asymptotic regime
        ph, _ = o.loop_phase_spin_q(o.FLUXTUBE, [F, lam], _subdivide(poly, k), T, cx, cy, Q)
        errs.append(abs(ph - exact))
    orders = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert errs[2] < errs[1] < errs[0]
    assert abs(orders[1] - 2 * Q) < 0.6, (errs, orders)
    # and a higher order is closer at the same points
    if Q > 1:
        fine = _subdivide(poly, 8)
        lower, _ = o.loop_phase_spin_q(o.FLUXTUBE, [F, lam], fine, T, cx, cy, Q - 1)
        here, _ = o.loop_phase_spin_q(o.FLUXTUBE, [F, lam], fine, T, cx, cy, Q)
        assert abs(here - exact) < 0.1 * abs(lower - exact)


@pytest.mark.parametrize("eB0,lam,centre", [(1.0, 1.0, (0.0, 0.0)), (1.0, 1.0, (0.9, 0.4)), (2.0, 0.5, (0.2, -0.1))])
def test_stokes_sech2_flux_through_a_square(eB0, lam, centre):
    """eq. (19)-(20) for the sech^2 profile: the line integral round a square is e x flux (dblquad of b alone).
    Order h^(2Q) again, and a COARSE polygon at Q = 3 beats a 4x finer one at Q = 1."""
    side, T = 2.0, 1.0
    cx, cy = centre
    flux, _ = integrate.dblquad(
        lambda yy, xx: o.field_b(o.SECH2, [eB0, lam], np.hypot(xx, yy))[0],
        cx - side / 2, cx + side / 2, cy - side / 2, cy + side / 2, epsabs=1e-13, epsrel=1e-13)
    corners = (np.array([[0, 0], [1, 0], [1, 1], [0, 1]], dtype=float) - 0.5) * side
    err = {}
    for Q in (1, 2, 3):
        for k in (4, 8, 16):
            ph, _ = o.loop_phase_spin_q(o.SECH2, [eB0, lam], _subdivide(corners, k), T, cx, cy, Q)
            err[Q, k] = abs(ph - flux)
    for Q in (1, 2):
        assert abs(np.log2(err[Q, 8] / err[Q, 16]) - 2 * Q) < 0.7, err
    assert err[3, 16] < 1e-7 * abs(flux) + 1e-12
    assert err[3, 4] < err[1, 16]
    assert err[2, 4] < err[1, 8]


def test_segment_through_the_axis_is_finite():
    """rho_i^2(t) can round below zero where a segment passes through the axis; the result must stay finite
    and equal the limit g(0)."""
    y = np.array([[-1.0, 0.0], [1.0, 0.0], [1.0, 1.0], [-1.0, 1.0]])
    for Q in (1, 2, 3):
        ph, sp = o.loop_phase_spin_q(o.SECH2, [1.0, 1.0], y, 1.0, 0.0, 0.0, Q)
        assert np.isfinite(ph) and np.isfinite(sp)
    # a degenerate loop back and forth through the axis encloses nothing: phase 0
    y = np.array([[-1.0, 0.0], [1.0, 0.0]])
    for Q in (1, 2, 3):
        ph, _ = o.loop_phase_spin_q(o.SECH2, [3.0, 0.5], y, 2.0, 0.0, 0.0, Q)
        assert abs(ph) < 1e-15


@pytest.mark.parametrize("Q", [1, 2, 3])
def test_ensemble_call_is_the_single_loop_call_entry_by_entry(Q):
    loops = o.generate_loops(21, 12, 16)
    T = np.array([0.05, 1.0, 4.0])
    rho = np.array([0.0, 0.7, 2.0])
    phi = np.array([0.0, 1.0, -2.5])
    par = [1.2, 0.8]
    res = o.evaluate_quadrature(o.SECH2, par, loops, T, rho, phi, n_groups=3, per_loop=True, Q=Q)
    for l in (0, 5, 11):
        for t in range(3):
            for r in range(3):
                ph, sp = o.loop_phase_spin_q(o.SECH2, par, loops[l], T[t], rho[r] * np.cos(phi[r]),
                                             rho[r] * np.sin(phi[r]), Q)
                assert res["phase"][l, t, r] == ph and res["spin"][l, t, r] == sp
                assert abs(res["W"][l, t, r] - np.cos(ph) * np.cosh(sp)) <= 4e-16 * np.cosh(sp)
    gs = res["W"].reshape(3, 4, 3, 3).sum(1)
    assert np.allclose(res["group_sums"], gs, rtol=1e-14, atol=0)
    assert np.allclose(res["W_mean"], res["W"].mean(0), rtol=1e-14, atol=0)
    if Q == 1:
        ref = o.evaluate(o.SECH2, par, loops, T, rho, phi, n_groups=3)
        assert np.allclose(res["group_sums"], ref["group_sums"], rtol=1e-13, atol=0)
    sc = o.evaluate_quadrature(o.SECH2, par, loops, T, rho, phi, n_groups=3, per_loop=True, Q=Q, scalar=True)
    assert np.allclose(sc["W"], np.cos(res["phase"]), rtol=0, atol=4e-16)


def test_discretisation_error_of_the_ensemble_average_shrinks_with_Q():
    """The second, independent handle on the discretisation error that Sec. IV.A asks for: on the same
    N-point ensemble the spread between Q = 2 and Q = 3 is far smaller than between Q = 1 and Q = 2."""
    loops = o.generate_loops(22, 256, 32)
    T = np.array([1.0, 3.0])
    rho = np.array([0.0, 1.0])
    W = [o.evaluate_quadrature(o.FLUXTUBE, [10.0, 1.0], loops, T, rho, None, Q=Q, scalar=True)["W_mean"]
         for Q in (1, 2, 3)]
    d12 = np.abs(W[0] - W[1]).max()
    d23 = np.abs(W[1] - W[2]).max()
    assert d23 < 0.2 * d12, (d12, d23)
