"""Pins for the oracle's field profile functions g(rho) = e A_phi/rho and b(rho) = e B_z.

What fixes them (none of this re-types the oracle's own formula):
  * mpmath evaluation at 50 digits of the textbook definitions
      Phi(rho) = 2 pi B0 [lambda rho tanh(rho/lambda) - lambda^2 ln cosh(rho/lambda)]
      (BASELINE.json config 1),  A_phi = Phi/(2 pi rho)  (eq. (14)),
      B = B0 sech^2(rho/lambda);
  * Stokes / eq. (13), (15): Phi(rho) = int_0^rho B(r) 2 pi r dr, by
    adaptive quadrature of b alone;
  * the limits A_phi -> B0 rho/2 (rho -> 0, config 1) and total flux 2 pi B0 lambda^2 ln 2.
"""
import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

from oracle import wl_oracle as o

mp.mp.dps = 50


def _g_mp(eB0, lam, rho):
    u = mp.mpf(rho) / mp.mpf(lam)
    Phi_over_2pi = mp.mpf(eB0) * (mp.mpf(lam) * rho * mp.tanh(u) - mp.mpf(lam) ** 2 * mp.log(mp.cosh(u)))
    A_phi = Phi_over_2pi / rho
    return A_phi / rho


@pytest.mark.parametrize("eB0,lam", [(1.0, 1.0), (10.0, 0.1), (0.3, 7.0)])
def test_sech2_g_matches_mpmath_over_the_whole_range(eB0, lam):
    # spans the series branch (u < 0.1), the switch, and u >> 1 (up to u = 500)
    us = np.concatenate([10.0 ** np.linspace(-8, -1.0001, 40), [0.0999999, 0.1, 0.1000001],
                         10.0 ** np.linspace(-0.99, 2.7, 60)])
    rho = us * lam
    got = o.field_g(o.SECH2, [eB0, lam], rho)
    want = np.array([float(_g_mp(eB0, lam, mp.mpf(float(r)))) for r in rho])
    assert np.max(np.abs(got / want - 1)) < 5e-14


@pytest.mark.parametrize("eB0,lam", [(1.0, 1.0), (10.0, 0.1)])
def test_sech2_b_matches_mpmath(eB0, lam):
    us = np.concatenate([[0.0], 10.0 ** np.linspace(-8, 2.5, 80)])
    rho = us * lam
    got = o.field_b(o.SECH2, [eB0, lam], rho)
    want = np.array([float(mp.mpf(eB0) / mp.cosh(mp.mpf(float(r)) / mp.mpf(lam)) ** 2) for r in rho])
    assert np.max(np.abs(got - want) / want) < 5e-14


def test_sech2_axis_limit_and_total_flux():
    # A_phi -> B0 rho/2 as rho -> 0 (config 1)  <=>  g(0) = eB0/2
    assert o.field_g(o.SECH2, [3.0, 0.5], 0.0)[0] == 1.5
    assert abs(o.field_g(o.SECH2, [3.0, 0.5], 1e-9)[0] - 1.5) < 1e-15
    # total flux: int_0^inf B0 sech^2(r/lambda) 2 pi r dr = 2 pi B0 lambda^2 ln 2  (textbook integral
    # int_0^inf u sech^2 u du = ln 2), so rho^2 g(rho) -> eB0 lambda^2 ln 2 for rho >> lambda
    eB0, lam, rho = 2.0, 0.25, 40.0
    flux_over_2pi = o.field_g(o.SECH2, [eB0, lam], rho)[0] * rho ** 2
    assert abs(flux_over_2pi - eB0 * lam ** 2 * np.log(2.0)) < 1e-14


@pytest.mark.parametrize("eB0,lam", [(1.0, 1.0), (10.0, 0.1)])
def test_stokes_flux_of_b_equals_rho2_g(eB0, lam):
    # eq. (13)/(15): e Phi(rho)/(2 pi) = int_0^rho b(r) r dr ; eq. (14): = rho^2 g(rho)
    for rho in [0.03 * lam, 0.5 * lam, 2.0 * lam, 9.0 * lam]:
        flux, _ = integrate.quad(lambda r: o.field_b(o.SECH2, [eB0, lam], r)[0] * r, 0.0, rho,
                                 epsabs=1e-14, epsrel=1e-13)
        assert abs(o.field_g(o.SECH2, [eB0, lam], rho)[0] * rho ** 2 - flux) < 2e-12 * max(1.0, flux)


def test_uniform_profile():
    # A = (B/2)(-y, x): A_phi = B rho/2 -> g = eB/2; b = eB (config 2)
    r = np.array([0.0, 1e-3, 1.0, 50.0])
    assert np.all(o.field_g(o.UNIFORM, [1.7], r) == 0.85)
    assert np.all(o.field_b(o.UNIFORM, [1.7], r) == 1.7)
