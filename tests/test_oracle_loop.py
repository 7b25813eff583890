"""Pins for the oracle's per-loop phase / spin / W (eq. (8), (18), (21)-(24), (31)-(33)).

Deterministic pins, one loop at a time:
  P1  zero field  ->  W == 1 exactly                                    (north_star)
  P2  uniform field: phase == eB T x shoelace area of the unit loop, any x_cm
      (eq. (19)-(20)); spin == eB T exactly            (eq. (31))
  Stokes for the sech^2 profile: on a finely subdivided square the midpoint line
      integral -> e x flux through the square, the flux computed by 2-D quadrature
      of b alone (eq. (19)-(20))
  spin sum on a circle: (T/N) sum_i B(x_i) = T x angular mean of B     (eq. (31)-(33))
  P6  lambda -> infinity: sech^2 -> uniform with eB = eB0
  P9  exact invariances: cyclic relabelling, reversal, mirror, joint rotation (A13)
"""
import numpy as np
import pytest
from scipy import integrate

from oracle import wl_oracle as o


def _rand_loop(rng, N):
    y = rng.normal(size=(N, 2)) * 0.4
    return y - y.mean(0)


def _shoelace(y):
    z = np.roll(y, -1, axis=0)
    return 0.5 * np.sum(y[:, 0] * z[:, 1] - y[:, 1] * z[:, 0])


def test_zero_field_gives_W_exactly_one():
    rng = np.random.default_rng(0)
    loops = np.stack([_rand_loop(rng, 32) for _ in range(8)])
    T = np.array([0.01, 1.0, 30.0])
    rho = np.array([0.0, 0.7, 5.0])
    for prof, par in [(o.UNIFORM, [0.0]), (o.SECH2, [0.0, 1.0]), (o.SECH2, [0.0, 0.1])]:
        r = o.evaluate(prof, par, loops, T, rho, n_groups=2, per_loop=True)
        assert np.all(r["W"] == 1.0) and np.all(r["phase"] == 0.0) and np.all(r["spin"] == 0.0)
        assert np.all(r["W_mean"] == 1.0) and np.all(r["group_sums"] == 4.0)


@pytest.mark.parametrize("N", [3, 4, 17, 256])
def test_uniform_phase_is_eBT_times_shoelace_area(N):
    rng = np.random.default_rng(N)
    y = _rand_loop(rng, N)
    area = _shoelace(y)
    for eB in [1.0, -2.5]:
        for T in [0.01, 1.0, 5.0]:
            for (cx, cy) in [(0.0, 0.0), (2.0, 0.0), (-1.3, 0.4), (2 * np.cos(2.0), 2 * np.sin(2.0))]:
                ph, sp = o.loop_phase_spin(o.UNIFORM, [eB], y, T, cx, cy)
                assert abs(ph - eB * T * area) < 5e-14 * max(1.0, abs(eB * T)) * (1 + cx * cx + cy * cy)
                assert abs(sp - eB * T) < 1e-15 * N * abs(eB * T)


def test_orientation_and_unit_square():
    # counter-clockwise unit square has area +1: phase = +eB T  (sign convention A5)
    sq = np.array([[0.0, 0.0], [1.0, 0.0], [1.0, 1.0], [0.0, 1.0]]) - 0.5
    ph, sp = o.loop_phase_spin(o.UNIFORM, [2.0], sq, 3.0, 0.3, -0.2)
    assert abs(ph - 6.0) < 1e-14 and abs(sp - 6.0) < 1e-14
    ph, _ = o.loop_phase_spin(o.UNIFORM, [2.0], sq[::-1].copy(), 3.0, 0.3, -0.2)
    assert abs(ph + 6.0) < 1e-14


def _subdivided_square(side, per_edge):
    c = np.array([[0, 0], [1, 0], [1, 1], [0, 1]], dtype=float) * side - side / 2
    pts = []
    for k in range(4):
        a, b = c[k], c[(k + 1) % 4]
        for j in range(per_edge):
            pts.append(a + (b - a) * j / per_edge)
    return np.array(pts)


@pytest.mark.parametrize("eB0,lam,centre", [(1.0, 1.0, (0.0, 0.0)), (1.0, 1.0, (0.9, 0.4)),
                                            (10.0, 0.1, (0.05, 0.0)), (2.0, 0.5, (3.0, -1.0))])
def test_stokes_sech2_line_integral_converges_to_flux(eB0, lam, centre):
    """eq. (19)-(20): e oint A.dx = e x flux.  Midpoint rule on collinear sub-segments
    converges O(h^2) to the exact line integral, so two refinements extrapolate."""
    side, T = 1.0, 1.0                       # x = x_cm + sqrt(T) y with T = 1
    cx, cy = centre
    flux, _ = integrate.dblquad(
        lambda yy, xx: o.field_b(o.SECH2, [eB0, lam], np.hypot(xx, yy))[0],
        cx - side / 2, cx + side / 2, cy - side / 2, cy + side / 2, epsabs=1e-12, epsrel=1e-12)
    ph = [o.loop_phase_spin(o.SECH2, [eB0, lam], _subdivided_square(side, n), T, cx, cy)[0]
          for n in (200, 400)]
    richardson = ph[1] + (ph[1] - ph[0]) / 3.0
    assert abs(ph[1] - flux) < 2e-4 * max(1.0, abs(flux))
    assert abs(richardson - flux) < 1e-7 * max(1.0, abs(flux))


def test_T_scaling_of_the_loop():
    # eq. (8): x = x_cm + sqrt(T) y.  A side-1 square at T = 4 is the side-2 square at T = 1.
    sq = _subdivided_square(1.0, 8)
    p4, s4 = o.loop_phase_spin(o.SECH2, [1.3, 0.8], sq, 4.0, 0.2, 0.1)
    p1, s1 = o.loop_phase_spin(o.SECH2, [1.3, 0.8], 2.0 * sq, 1.0, 0.2, 0.1)
    assert abs(p4 - p1) < 1e-14
    assert abs(s4 - 4.0 * s1) < 1e-13     # spin = (T/N) sum: same points, T four times larger


def test_spin_on_a_circle_is_T_times_angular_mean_of_B():
    # eq. (31)-(33): e int_0^T B dtau -> (T/N) sum_i eB(x_i).  Points on a circle of radius R
    # about c: periodic trapezoid rule, spectrally accurate against quad of b alone.
    N, R, T = 512, 0.8, 2.5
    th = 2 * np.pi * np.arange(N) / N
    y = R / np.sqrt(T) * np.stack([np.cos(th), np.sin(th)], 1)
    for (eB0, lam, cx) in [(1.0, 1.0, 0.0), (1.0, 1.0, 1.1), (10.0, 0.1, 0.75)]:
        _, sp = o.loop_phase_spin(o.SECH2, [eB0, lam], y, T, cx, 0.0)
        mean_b, _ = integrate.quad(
            lambda t: o.field_b(o.SECH2, [eB0, lam], np.hypot(cx + R * np.cos(t), R * np.sin(t)))[0],
            0, 2 * np.pi, epsabs=1e-13, epsrel=1e-13, limit=400)
        assert abs(sp - T * mean_b / (2 * np.pi)) < 1e-10


def test_large_lambda_limit_reduces_to_uniform():
    rng = np.random.default_rng(5)
    y = _rand_loop(rng, 64)
    for T, cx, cy in [(0.5, 0.0, 0.0), (3.0, 1.0, -2.0)]:
        pu, su = o.loop_phase_spin(o.UNIFORM, [1.4], y, T, cx, cy)
        ps, ss = o.loop_phase_spin(o.SECH2, [1.4, 1e5], y, T, cx, cy)
        # corrections are O((rho/lambda)^2) ~ 1e-9
        assert abs(pu - ps) < 1e-8 and abs(su - ss) < 1e-8
        assert abs(pu - ps) > 0 or abs(su - ss) > 0      # and it is not the same code path


def test_invariances_exact_to_rounding():
    rng = np.random.default_rng(7)
    y = _rand_loop(rng, 48)
    par, T, rho = [1.0, 0.7], 2.0, 1.3
    p0, s0 = o.loop_phase_spin(o.SECH2, par, y, T, rho, 0.0)
    # cyclic relabelling of the points
    p, s = o.loop_phase_spin(o.SECH2, par, np.roll(y, 11, axis=0), T, rho, 0.0)
    assert abs(p - p0) < 1e-13 and abs(s - s0) < 1e-13
    # reversed orientation: phase flips sign, spin unchanged, W unchanged (A5)
    p, s = o.loop_phase_spin(o.SECH2, par, y[::-1].copy(), T, rho, 0.0)
    assert abs(p + p0) < 1e-13 and abs(s - s0) < 1e-13
    # mirror y -> -y with x_cm on the x axis
    p, s = o.loop_phase_spin(o.SECH2, par, y * np.array([1.0, -1.0]), T, rho, 0.0)
    assert abs(p + p0) < 1e-13 and abs(s - s0) < 1e-13
    # joint rotation of the loop and x_cm about the axis (A13)
    a = 0.83
    R = np.array([[np.cos(a), -np.sin(a)], [np.sin(a), np.cos(a)]])
    p, s = o.loop_phase_spin(o.SECH2, par, y @ R.T, T, rho * np.cos(a), rho * np.sin(a))
    assert abs(p - p0) < 1e-13 and abs(s - s0) < 1e-13


def test_uniform_field_W_does_not_depend_on_x_cm():
    # gauge shift integrates to zero round a closed loop; config 2's 8 angles
    rng = np.random.default_rng(8)
    loops = np.stack([_rand_loop(rng, 128) for _ in range(16)])
    phi = 2 * np.pi * np.arange(8) / 8
    r = o.evaluate(o.UNIFORM, [1.0], loops, np.array([0.1, 1.0, 5.0]), np.full(8, 2.0), phi,
                   n_groups=4, per_loop=True)
    assert np.max(np.abs(r["W"] - r["W"][:, :, :1])) < 1e-11


def test_evaluate_matches_single_loop_entry_and_combines_cos_cosh():
    rng = np.random.default_rng(9)
    loops = np.stack([_rand_loop(rng, 16) for _ in range(6)])
    T = np.array([0.3, 2.0])
    rho = np.array([0.0, 0.5, 1.5])
    phi = np.array([0.0, 1.0, -2.0])
    r = o.evaluate(o.SECH2, [1.0, 1.0], loops, T, rho, phi, n_groups=3, per_loop=True)
    for l in range(6):
        for t in range(2):
            for k in range(3):
                p, s = o.loop_phase_spin(o.SECH2, [1.0, 1.0], loops[l], T[t],
                                         rho[k] * np.cos(phi[k]), rho[k] * np.sin(phi[k]))
                assert r["phase"][l, t, k] == p and r["spin"][l, t, k] == s
                assert abs(r["W"][l, t, k] - np.cos(p) * np.cosh(s)) < 1e-15 * np.cosh(s)   # eq. (18)
    # eq. (60): contiguous groups in generation order; eq. (61)-(62): mean of group means == mean
    gs = r["W"].reshape(3, 2, 2, 3).sum(1)
    assert np.max(np.abs(gs - r["group_sums"])) < 1e-14
    assert np.max(np.abs(r["W_mean"] - r["W"].mean(0))) < 1e-14
