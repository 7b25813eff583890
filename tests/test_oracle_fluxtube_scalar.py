"""Pins for the oracle's flux-tube profile (eq. (68)) and scalar-QED output
(W = cos(phase), the paper's Wsscal).  SURVEY.md section 8(f) NEXT-1.

  * eq. (14)/(15) with f_lambda = rho^2/(lambda^2+rho^2): mpmath differentiation of
    f_lambda gives B; A_phi = F f/(2 pi rho); e folded as script-F = eF/2pi (eq. (17)).
  * eq. (16): total flux = F (f(inf) - f(0)) = F  <=>  rho^2 g(rho) -> script-F.
  * Stokes / eq. (13): rho^2 g(rho) = int_0^rho b(r) r dr by quadrature of b alone; and the discretised
    line integral round a square converges to the flux of b through it (eq. (19)-(20)).
  * lambda -> infinity at fixed eB = 2 script-F/lambda^2: the uniform field.
  * small T: <W> - 1 -> (eB(rho_cm) T)^2/3 (eq. (70)).
  * scalar part, uniform field, finite N: <cos(eBT A)>_N = prod_k [1 + (x cot(pi k/N)/N)^2]^(-1/2),
    whose N -> infinity limit is eq. (43) x/sinh x; at N = 4 it is 1/(1 + (x/4)^2).
  * 4-point loops by Gauss-Hermite quadrature for this profile, fermion and scalar.
"""
import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

from oracle import wl_oracle as o
from test_oracle_ensemble import _finite_N_uniform, _gauss_hermite_4pt_loops
from test_oracle_loop import _subdivided_square

mp.mp.dps = 40


@pytest.mark.parametrize("F,lam", [(10.0, 1.0), (10.0, 10.0), (0.7, 0.05)])
def test_fluxtube_profile_from_the_papers_f_lambda(F, lam):
    f = lambda r: r ** 2 / (mp.mpf(lam) ** 2 + r ** 2)                    # eq. (68)
    for rho in [1e-6, 0.01 * lam, 0.5 * lam, lam, 3.0 * lam, 200.0 * lam]:
        r = mp.mpf(rho)
        g_want = mp.mpf(F) * f(r) / r ** 2                                # e A_phi/rho, eq. (14), (17)
        b_want = mp.mpf(F) / r * mp.diff(f, r)                            # eq. (15), (17)
        assert abs(o.field_g(o.FLUXTUBE, [F, lam], rho)[0] / float(g_want) - 1) < 1e-14
        assert abs(o.field_b(o.FLUXTUBE, [F, lam], rho)[0] / float(b_want) - 1) < 1e-13
    assert abs(o.field_g(o.FLUXTUBE, [F, lam], 0.0)[0] / (F / lam ** 2) - 1) < 1e-15       # A_phi -> B(0) rho/2
    assert abs(o.field_b(o.FLUXTUBE, [F, lam], 0.0)[0] / (2 * F / lam ** 2) - 1) < 1e-15
    # eq. (16): total flux F  <=>  rho^2 g -> script-F
    assert abs(o.field_g(o.FLUXTUBE, [F, lam], 1e7 * lam)[0] * (1e7 * lam) ** 2 / F - 1) < 1e-13


@pytest.mark.parametrize("F,lam", [(10.0, 1.0), (2.0, 0.2)])
def test_fluxtube_stokes(F, lam):
    for rho in [0.05 * lam, lam, 7.0 * lam]:
        flux, _ = integrate.quad(lambda r: o.field_b(o.FLUXTUBE, [F, lam], r)[0] * r, 0.0, rho,
                                 epsabs=1e-14, epsrel=1e-13)
        assert abs(o.field_g(o.FLUXTUBE, [F, lam], rho)[0] * rho ** 2 - flux) < 2e-12 * max(1.0, flux)
    cx, cy, side = 0.7, -0.3, 1.0
    flux, _ = integrate.dblquad(lambda yy, xx: o.field_b(o.FLUXTUBE, [F, lam], np.hypot(xx, yy))[0],
                                cx - side / 2, cx + side / 2, cy - side / 2, cy + side / 2,
                                epsabs=1e-12, epsrel=1e-12)
    ph = [o.loop_phase_spin(o.FLUXTUBE, [F, lam], _subdivided_square(side, n), 1.0, cx, cy)[0] for n in (200, 400)]
    assert abs(ph[1] + (ph[1] - ph[0]) / 3.0 - flux) < 1e-7 * max(1.0, abs(flux))


def test_fluxtube_large_lambda_is_the_uniform_field():
    rng = np.random.default_rng(8)
    y = rng.normal(size=(48, 2)) * 0.3
    y -= y.mean(0)
    eB, lam = 1.4, 1e5
    for T, cx, cy in [(0.5, 0.0, 0.0), (3.0, 1.0, -2.0)]:
        pu, su = o.loop_phase_spin(o.UNIFORM, [eB], y, T, cx, cy)
        pf, sf = o.loop_phase_spin(o.FLUXTUBE, [eB * lam ** 2 / 2, lam], y, T, cx, cy)
        assert abs(pu - pf) < 1e-8 and abs(su - sf) < 1e-8


def test_fluxtube_small_T_law():
    n_loops, N = 1 << 14, 32
    y = o.generate_loops(16, n_loops, N)
    T, rho = np.array([0.02]), np.array([0.0, 0.8, 2.0])
    par = [3.0, 1.5]
    r = o.evaluate(o.FLUXTUBE, par, y, T, rho, n_groups=64)
    mean, err = o.finalize(r["group_sums"], n_loops)
    b = o.field_b(o.FLUXTUBE, par, rho)
    varA = (N - 1) * (N - 2) / (3.0 * N * N)
    want = (b * T[0]) ** 2 * 0.5 * (1.0 - varA)             # -> (eBT)^2/3 as N -> infinity
    assert np.all(np.abs((mean[0] - 1.0) - want) < 5 * err[0] + 0.1 * (b * T[0]) ** 2 / 3)


@pytest.mark.parametrize("N,n_loops", [(4, 1 << 16), (64, 1 << 14)])
def test_scalar_uniform_field_average_eq43(N, n_loops):
    y = o.generate_loops(70 + N, n_loops, N)
    T = np.array([0.1, 1.0, 3.0])
    r = o.evaluate(o.UNIFORM, [1.0], y, T, np.array([0.0, 2.0]), n_groups=64, scalar=True)
    mean, err = o.finalize(r["group_sums"], n_loops)
    for t, x in enumerate(T):
        want = _finite_N_uniform(x, N) / np.cosh(x)        # the fermion closed form without its cosh(x)
        assert np.all(np.abs(mean[t] - want) < 4.5 * err[t] + 1e-12)
        assert np.all(err[t] < 0.05 * want)
    assert abs(_finite_N_uniform(2.0, 1 << 20) / np.cosh(2.0) - 2.0 / np.sinh(2.0)) < 1e-4     # eq. (43)
    assert abs(_finite_N_uniform(2.0, 4) / np.cosh(2.0) - 1 / (1 + 0.25)) < 1e-14


def test_scalar_is_cos_of_the_fermion_runs_phase():
    y = o.generate_loops(5, 32, 64)
    T, rho = np.array([0.3, 2.0]), np.array([0.0, 1.0])
    f = o.evaluate(o.SECH2, [2.0, 0.7], y, T, rho, n_groups=4, per_loop=True)
    s = o.evaluate(o.SECH2, [2.0, 0.7], y, T, rho, n_groups=4, per_loop=True, scalar=True)
    assert np.array_equal(s["phase"], f["phase"]) and np.array_equal(s["spin"], f["spin"])
    assert np.max(np.abs(s["W"] - np.cos(f["phase"]))) < 1e-15
    assert np.max(np.abs(f["W"] - s["W"] * np.cosh(f["spin"]))) < 1e-12
    assert np.max(np.abs(s["group_sums"].sum(0) / 32 - s["W_mean"])) < 1e-14


def test_fluxtube_four_point_loops_brute_force():
    # The profile has poles at rho^2 = -lambda^2, so Gauss-Hermite converges more slowly than for
    # sech^2: at T <= 1 the 9- and 11-node rules agree to 1.5e-4 (allowed for below).
    loops, wt = _gauss_hermite_4pt_loops(11)                # 1771561 loops
    T, rho = np.array([0.5, 1.0]), np.array([0.0, 0.6])
    par = [0.5, 0.9]                                        # eB(0) = 2 F/lambda^2 = 1.23
    n_loops = 1 << 17
    y = o.generate_loops(45, n_loops, 4)
    for scalar in (False, True):
        r = o.evaluate(o.FLUXTUBE, par, loops, T, rho, n_groups=1, per_loop=True, scalar=scalar)
        gh = np.tensordot(wt, r["W"], axes=(0, 0))
        mc = o.evaluate(o.FLUXTUBE, par, y, T, rho, n_groups=128, scalar=scalar)
        mean, err = o.finalize(mc["group_sums"], n_loops)
        assert np.all(np.abs(mean - gh) < 4.5 * err + 2e-4)
        assert np.all(np.abs(gh - 1.0) > 10 * err + 2e-3)
