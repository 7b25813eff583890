"""Pins for the oracle's effective-action integrals (eq. (12), (44)-(47), (69)-(70); PAPER.md:89-92, 234-255,
417, 472, 488-495; reading A16).

  * eq. (44), (45): mpmath Taylor coefficients of the exact constant-field integrands built from eq. (42),
    (43); the [0, a] integral against mpmath quadrature of the exact integrand;
  * proper-time nodes and Simpson weights: with the exact constant-field <W> (eq. (42)/(43)) fed in as
    group sums, small-T part + Simpson part == adaptive quadrature of the exact integrand over [0, inf);
  * Simpson is exact for cubics in x (radial integral: for cubics in rho);
  * eq. (69): with <W> = eB(rho) T coth(eB(rho) T) the two integrals reproduce the LCF action of the
    flux-tube profile of eq. (68), by scipy's 2-D adaptive quadrature;
  * linearity in the group sums, and the group statistics of PAPER.md:417 through finalize().
"""
import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

from oracle import wl_oracle as o

mp.mp.dps = 30


def _I_exact(T, b, m2, scalar):
    """The exact constant-field integrand from eq. (42)/(43); Laurent series of coth / csch for x < 0.2
    (Bernoulli numbers), where the closed form cancels."""
    x = b * T
    if x < 0.2:
        br = (7 * x ** 4 / 360 - 31 * x ** 6 / 15120 + 127 * x ** 8 / 604800 - 73 * x ** 10 / 3421440) if scalar \
            else (-x ** 4 / 45 + 2 * x ** 6 / 945 - x ** 8 / 4725 + 2 * x ** 10 / 93555)
    else:
        br = (x / np.sinh(x) - 1 + x * x / 6) if scalar else (x / np.tanh(x) - 1 - x * x / 3)
    return np.exp(-m2 * T) / T ** 3 * br


@pytest.mark.parametrize("scalar", [False, True])
def test_small_T_expansions_eq44_eq45(scalar):
    b, m2 = mp.mpf("1.7"), mp.mpf("0.8")

    def I(T):
        x = b * T
        br = (x / mp.sinh(x) - 1 + x * x / 6) if scalar else (x * mp.coth(x) - 1 - x * x / 3)
        return mp.exp(-m2 * T) / T ** 3 * br

    with mp.workdps(80):                               # the bracket cancels to O(T^4) before the 1/T^3
        for a in (0.05, 0.1):
            exact = mp.quad(I, [mp.mpf(10) ** -6, mp.mpf(a) / 2, mp.mpf(a)])      # [0, 1e-6] holds 1e-12 of it
            got = o.small_T_integral(float(b), float(m2), a, scalar)
            # the expansion stops at T^4: the neglected O(T^5) term integrates to O(a^6)
            assert abs(got - float(exact)) < 0.05 * float(b) ** 8 * a ** 6
            assert abs(got / float(exact) - 1) < 1e-4
        # leading coefficient: -(eB)^4/45 (fermion), 7 (eB)^4/360 (scalar)
        lead = float((mp.mpf(7) / 360 if scalar else -mp.mpf(1) / 45) * b ** 4)
        small = [o.small_T_integral(float(b), float(m2), t, scalar) for t in (1e-3, 2e-3)]
        assert abs(small[0] / (lead * 1e-6 / 2) - 1) < 2e-3 and abs(small[1] / small[0] / 4 - 1) < 2e-3


def test_proper_time_nodes_follow_the_papers_mapping():
    a, Tmax, n = 0.05, 1.3, 16
    T = o.proper_time_nodes(a, Tmax, n)
    x = 1.0 / (1.0 + T / Tmax)
    xa = 1.0 / (1.0 + a / Tmax)
    assert T[0] == a and np.all(np.diff(T) > 0)
    assert np.max(np.abs(x - xa * (n - np.arange(n)) / n)) < 1e-15
    with pytest.raises(ValueError):
        o.proper_time_nodes(a, Tmax, 7)


@pytest.mark.parametrize("scalar", [False, True])
@pytest.mark.parametrize("eB,m2", [(1.0, 1.0), (3.0, 1.0), (0.5, 0.25)])
def test_density_with_exact_constant_field_W_equals_quadrature(scalar, eB, m2):
    a, n = 0.05, 400
    Tmax = 3.0 / eB if eB > 1 else 1.0
    T = o.proper_time_nodes(a, Tmax, n)
    rho = np.array([0.0, 1.0])
    x = eB * T
    W = x / np.sinh(x) if scalar else x / np.tanh(x)               # eq. (43) / (42)
    G, per_group = 3, 5
    gs = np.repeat((W * per_group)[None, :, None], G, axis=0) * np.ones((1, 1, len(rho)))
    d = o.action_density(o.UNIFORM, [eB], gs, G * per_group, T, rho, m2, a, Tmax, scalar=scalar)
    want, _ = integrate.quad(_I_exact, 0.0, np.inf, args=(eB, m2, scalar), epsabs=1e-14, epsrel=1e-12, limit=500)
    assert d.shape == (G, 2)
    assert np.max(np.abs(d - want)) < 2e-7 * abs(want) + 1e-12
    # a coarser rule is still close (Simpson, h^4), and not identical (the nodes matter)
    T2 = o.proper_time_nodes(a, Tmax, n // 2)
    W2 = (eB * T2) / np.sinh(eB * T2) if scalar else (eB * T2) / np.tanh(eB * T2)
    gs2 = np.repeat((W2 * per_group)[None, :, None], G, axis=0) * np.ones((1, 1, len(rho)))
    d2 = o.action_density(o.UNIFORM, [eB], gs2, G * per_group, T2, rho, m2, a, Tmax, scalar=scalar)
    assert np.max(np.abs(d2 - want)) < 1e-5 * abs(want)
    T8 = o.proper_time_nodes(a, Tmax, 8)
    W8 = (eB * T8) / np.sinh(eB * T8) if scalar else (eB * T8) / np.tanh(eB * T8)
    gs8 = np.repeat((W8 * per_group)[None, :, None], G, axis=0) * np.ones((1, 1, len(rho)))
    d8 = o.action_density(o.UNIFORM, [eB], gs8, G * per_group, T8, rho, m2, a, Tmax, scalar=scalar)
    assert 1e-7 * abs(want) < np.max(np.abs(d8 - want)) < 0.2 * abs(want)


def test_radial_simpson_is_exact_for_cubics_and_has_the_1_over_4pi():
    rho = np.linspace(0.0, 2.0, 9)
    dens = np.stack([1.0 + 0 * rho, rho ** 2 - 0.3 * rho])        # rho * density is a cubic at most
    got = o.action_radial(dens, rho)
    want = np.array([2.0 ** 2 / 2, 2.0 ** 4 / 4 - 0.3 * 2.0 ** 3 / 3]) / (4 * np.pi)
    assert np.max(np.abs(got - want)) < 1e-15
    with pytest.raises(ValueError):
        o.action_radial(dens[:, :8], rho[:8])


def test_lcf_action_of_the_flux_tube_eq69():
    """eq. (69): feeding <W> = eB(rho) T coth(eB(rho) T) reproduces the LCF effective action
    of the profile of eq. (68) (lambda = 10 lambda_e, script-F = 10: the case of Fig. 12)."""
    F, lam, m2, a, Tmax, n = 10.0, 10.0, 1.0, 0.05, 1.0, 200
    par = [F, lam]
    rho = np.linspace(0.0, 60.0, 241)
    T = o.proper_time_nodes(a, Tmax, n)
    b = o.field_b(o.FLUXTUBE, par, rho)
    x = b[None, :] * T[:, None]
    W = np.where(x > 1e-8, x / np.tanh(np.maximum(x, 1e-300)), 1.0)
    gs = W[None] * 4.0                                             # G = 1, four loops in the group
    dens = o.action_density(o.FLUXTUBE, par, gs, 4, T, rho, m2, a, Tmax)
    act = o.action_radial(dens, rho)[0]
    f = lambda Tt, r: r * _I_exact(Tt, 2 * F * lam ** 2 / (lam ** 2 + r ** 2) ** 2, m2, False)
    want, _ = integrate.dblquad(f, 0.0, 60.0, 0.0, np.inf, epsabs=1e-12, epsrel=1e-9)
    assert abs(act - want / (4 * np.pi)) < 1e-5 * abs(want / (4 * np.pi))
    assert act < 0                                                  # the fermion term lowers the action


def test_group_statistics_of_the_integral():
    """the integral is done per group; its error is the SEM of the group values."""
    n_loops, N, G = 512, 64, 16
    a, Tmax, n = 0.05, 1.0, 20
    T = o.proper_time_nodes(a, Tmax, n)
    rho = np.array([0.0, 1.0, 2.0])
    par = [1.0, 1.0]
    y = o.generate_loops(12, n_loops, N)
    r = o.evaluate(o.SECH2, par, y, T, rho, n_groups=G)
    d = o.action_density(o.SECH2, par, r["group_sums"], n_loops, T, rho, 1.0, a, Tmax)
    mean, err = o.finalize(d[:, None, :], G)                       # one "loop" per group value
    assert np.max(np.abs(mean[0] - d.mean(0))) < 1e-15
    assert np.max(np.abs(err[0] - d.std(0, ddof=1) / np.sqrt(G))) < 1e-15
    # linear in the group sums: the density of the whole ensemble is the mean of the group densities
    whole = o.action_density(o.SECH2, par, r["group_sums"].sum(0, keepdims=True), n_loops, T, rho, 1.0, a, Tmax)
    assert np.max(np.abs(whole[0] - d.mean(0))) < 1e-13
