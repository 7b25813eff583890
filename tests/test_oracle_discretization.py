"""Pins for the oracle's discretisation estimate (Sec. IV.A, eq. (48)-(52), PAPER.md:269-304;
SURVEY.md section 8(f) NEXT-2; reading A15).

  * which points form the three interleaved sub-worldlines (circle = every other point, box / triangle =
    the remaining points alternately, Fig. 2) and the weights of eq. (48)-(50): uniform field, where every
    sub-worldline integral is eB T x its polygon area (eq. (19)-(20)) -- areas by numpy's own shoelace;
  * level N/2 is the ordinary evaluation of the every-other-point ensemble, and the
    levels N/4 and N follow from the ordinary per-loop phases / spins of the strided ensembles
    (evaluate() is pinned in tests/test_oracle_loop.py, test_oracle_ensemble.py);
  * level N/2 in a uniform field has the exact finite-N average of pin P3 with N/2 points;
  * eq. (51) is the parabola in 1/N through the three levels: exact for a + b/N + c/N^2; eq. (52).
"""
import numpy as np
import pytest

from oracle import wl_oracle as o
from test_oracle_ensemble import _finite_N_uniform


def _area(y):
    yn = np.roll(y, -1, axis=1)
    return 0.5 * np.sum(y[:, :, 0] * yn[:, :, 1] - y[:, :, 1] * yn[:, :, 0], axis=1)


def test_sub_worldlines_and_weights_in_a_uniform_field():
    n_loops, N, eB = 24, 64, 1.3
    y = o.generate_loops(3, n_loops, N)
    T, rho = np.array([0.4, 2.0, 5.0]), np.array([0.0, 1.7])
    gs, W = o.evaluate_discretization(o.UNIFORM, [eB], y, T, rho, n_groups=4, per_loop=True)
    Ac, Ab, At = _area(y[:, 0::2]), _area(y[:, 1::4]), _area(y[:, 3::4])
    x = eB * T[None, :, None] * np.ones((n_loops, 1, len(rho)))
    ph = lambda A: eB * T[None, :, None] * A[:, None, None] * np.ones((1, 1, len(rho)))
    want = np.stack([np.cos(0.5 * ph(At) + 0.5 * ph(Ab)) * np.cosh(x),                       # eq. (48)
                     np.cos(ph(Ac)) * np.cosh(x),                                             # eq. (49)
                     np.cos(0.5 * ph(Ac) + 0.25 * ph(Ab) + 0.25 * ph(At)) * np.cosh(x)])     # eq. (50)
    assert np.max(np.abs(W - want) / np.abs(want)) < 1e-12
    assert np.max(np.abs(gs - W.reshape(3, 4, 6, len(T), len(rho)).sum(2))) < 1e-12
    # the three sub-worldlines are different polygons, and a wrong assignment is visible
    assert np.min(np.abs(Ab - At)) > 1e-6 and np.min(np.abs(Ac - Ab)) > 1e-6
    s = o.evaluate_discretization(o.UNIFORM, [eB], y, T, rho, n_groups=4, per_loop=True, scalar=True)[1]
    assert np.max(np.abs(s - want / np.cosh(x))) < 1e-12


@pytest.mark.parametrize("profile,params", [(o.SECH2, [2.0, 0.7]), (o.FLUXTUBE, [3.0, 1.1])])
def test_levels_from_the_ordinary_evaluation_of_the_strided_ensembles(profile, params):
    n_loops, N = 16, 128
    y = o.generate_loops(4, n_loops, N)
    T, rho, phi = np.array([0.3, 1.5]), np.array([0.0, 0.8, 2.5]), np.array([0.0, 1.0, 4.0])
    gs, W = o.evaluate_discretization(profile, params, y, T, rho, phi, n_groups=2, per_loop=True)
    c = o.evaluate(profile, params, y[:, 0::2], T, rho, phi, n_groups=2, per_loop=True)
    b = o.evaluate(profile, params, y[:, 1::4], T, rho, phi, n_groups=2, per_loop=True)
    t = o.evaluate(profile, params, y[:, 3::4], T, rho, phi, n_groups=2, per_loop=True)
    assert np.array_equal(W[1], c["W"]) and np.array_equal(gs[1], c["group_sums"])            # eq. (49)
    w4 = np.cos(0.5 * t["phase"] + 0.5 * b["phase"]) * np.cosh(0.5 * t["spin"] + 0.5 * b["spin"])
    wN = (np.cos(0.5 * c["phase"] + 0.25 * b["phase"] + 0.25 * t["phase"])
          * np.cosh(0.5 * c["spin"] + 0.25 * b["spin"] + 0.25 * t["spin"]))
    assert np.max(np.abs(W[0] - w4)) < 1e-13 * np.abs(w4).max()
    assert np.max(np.abs(W[2] - wN)) < 1e-13 * np.abs(wN).max()


def test_level_N_over_2_has_the_exact_uniform_field_average():
    n_loops, N = 1 << 14, 32
    y = o.generate_loops(27, n_loops, N)
    T = np.array([0.5, 2.0])
    gs = o.evaluate_discretization(o.UNIFORM, [1.0], y, T, np.array([0.0]), n_groups=64)
    mean, err = o.finalize(gs[1], n_loops)
    for t, x in enumerate(T):
        assert abs(mean[t, 0] - _finite_N_uniform(x, N // 2)) < 4.5 * err[t, 0]
        assert abs(_finite_N_uniform(x, N // 2) - _finite_N_uniform(x, N)) > 0.2 * err[t, 0] or t == 0


def test_eq51_is_the_parabola_in_one_over_N_and_eq52():
    N = 64.0
    a, b, c = 1.7, -3.0, 11.0
    f = lambda n: a + b / n + c / n ** 2
    lev = np.array([[f(N / 4), 2.0], [f(N / 2), 2.0], [f(N), 2.0]])
    W_inf, delta = o.extrapolate(lev)
    assert abs(W_inf[0] - a) < 1e-13 and abs(W_inf[1] - 2.0) < 1e-14
    assert abs(delta[0] - abs(f(N) - a)) < 1e-13 and delta[1] < 1e-14
    # the paper's weights, eq. (51)
    e = np.eye(3)
    w = [o.extrapolate(e[:, k:k + 1])[0][0] for k in range(3)]
    assert np.allclose(w, [1.0 / 3.0, -2.0, 8.0 / 3.0], atol=1e-15)


def test_invalid_sizes():
    y = np.zeros((4, 6, 2))
    with pytest.raises(ValueError):
        o.evaluate_discretization(o.UNIFORM, [1.0], y, [1.0], [0.0])          # N % 4 != 0
    with pytest.raises(ValueError):
        o.evaluate_discretization(o.UNIFORM, [1.0], np.zeros((4, 8, 2)), [1.0], [0.0], n_groups=3)
