"""Pins for the oracle's loop generator (d-loops, eq. (10)-(11)), the ensemble average
(eq. (7)), grouping (eq. (60)-(63)) and the exact uniform-field results (eq. (42)-(43)).

  P3  uniform field at finite N: <W>_N = cosh(x) prod_{k=1}^{N-1} [1 + (x cot(pi k/N)/N)^2]^(-1/2),
      x = eBT; N -> infinity gives eq. (42) x coth x.  The product follows
      from diagonalising the area form in the Fourier modes of the discrete weight of config 1.
  P4  Var(area) = (N-1)(N-2)/(3 N^2) -> 1/3 (eq. (65))
  P5  small T: <W> - 1 -> (eB(rho_cm) T)^2/3
  P7  sampler moments: covariance of the points = pseudo-inverse of the cycle Laplacian form
  P8  4-point loops: tensor Gauss-Hermite quadrature over the 6 Gaussian modes (brute force)
  P10 eq. (63) == delete-one-group jackknife error of the mean
"""
import numpy as np
import pytest

from oracle import wl_oracle as o


def _finite_N_uniform(x, N):
    k = np.arange(1, N)
    return np.cosh(x) * np.prod(1.0 / np.sqrt(1.0 + (x / (N * np.tan(np.pi * k / N))) ** 2))


def _mode_covariance(N):
    """Per-component covariance of weight exp(-(N/4) sum |y_{i+1}-y_i|^2), sum y = 0 (config 1):
    exp(-1/2 y^T (N/2) L y), L the cycle Laplacian -> Cov = pinv((N/2) L)."""
    L = 2 * np.eye(N) - np.roll(np.eye(N), 1, 0) - np.roll(np.eye(N), -1, 0)
    return np.linalg.pinv(0.5 * N * L)


def test_finite_N_formula_has_the_papers_continuum_limit():
    # eq. (42): fermion <W> = eBT coth(eBT); eq. (43) scalar = eBT/sinh(eBT)
    for x in [0.3, 1.0, 5.0]:
        assert abs(_finite_N_uniform(x, 1 << 20) / (x / np.tanh(x)) - 1) < 1e-4
    assert abs(_finite_N_uniform(2.0, 4) - np.cosh(2.0) / (1 + (2.0 / 4) ** 2)) < 1e-14


def test_generator_is_deterministic_counter_based_and_centred():
    a = o.generate_loops(11, 8, 64)
    b = o.generate_loops(11, 8, 64)
    assert np.array_equal(a, b)
    # loop l is a pure function of (seed, l): generating a sub-range gives the same loops
    c = o.generate_loops(11, 3, 64, loop_begin=5)
    assert np.array_equal(a[5:8], c)
    assert not np.array_equal(a, o.generate_loops(12, 8, 64))
    assert np.max(np.abs(a.mean(1))) < 1e-15           # step (5): common centre of mass
    with pytest.raises(ValueError):
        o.generate_loops(1, 4, 48)                     # N must be a power of two


@pytest.mark.parametrize("N", [2, 4, 16])
def test_generator_point_covariance_matches_the_discrete_weight(N):
    n = 60000
    y = o.generate_loops(100 + N, n, N)
    C = _mode_covariance(N)
    for comp in range(2):
        S = y[:, :, comp].T @ y[:, :, comp] / n
        # entries are sample means of products of Gaussians: var = C_ii C_jj + C_ij^2
        se = np.sqrt((np.outer(np.diag(C), np.diag(C)) + C ** 2) / n)
        assert np.max(np.abs(S - C) / se) < 5.0
    cross = y[:, :, 0].T @ y[:, :, 1] / n                # x and y components independent
    assert np.max(np.abs(cross) / np.sqrt(np.outer(np.diag(C), np.diag(C)) / n)) < 5.0


def test_generator_moments_P7_and_subloop_property():
    N, n = 64, 20000
    y = o.generate_loops(3, n, N)
    var = (y ** 2).mean(axis=(0, 1))
    want = (N * N - 1) / (6.0 * N * N)
    assert np.all(np.abs(var - want) < 0.02 * want)
    step2 = ((np.roll(y, -1, 1) - y) ** 2).sum(2).mean()
    assert abs(step2 - 4.0 * (N - 1) / N ** 2) < 0.01 * 4.0 * (N - 1) / N ** 2
    # every-other-point sub-loop is an N/2 loop: compare its step moment
    # (about its own centre of mass the increments are unchanged)
    sub = y[:, ::2]
    M = N // 2
    step2s = ((np.roll(sub, -1, 1) - sub) ** 2).sum(2).mean()
    assert abs(step2s - 4.0 * (M - 1) / M ** 2) < 0.015 * 4.0 * (M - 1) / M ** 2


def test_area_variance_P4():
    N, n = 32, 40000
    y = o.generate_loops(4, n, N)
    z = np.roll(y, -1, 1)
    A = 0.5 * np.sum(y[:, :, 0] * z[:, :, 1] - y[:, :, 1] * z[:, :, 0], axis=1)
    want = (N - 1) * (N - 2) / (3.0 * N * N)
    assert abs(A.mean()) < 5 * np.sqrt(want / n)
    assert abs(A.var() - want) < 0.04 * want            # kurtosis of the sech^2 law is 4.2: se ~ 0.9 %


@pytest.mark.parametrize("N,n_loops", [(4, 1 << 16), (64, 1 << 14)])
def test_uniform_field_ensemble_average_P3(N, n_loops):
    y = o.generate_loops(20 + N, n_loops, N)
    T = np.array([0.1, 1.0, 3.0])
    G = 64
    r = o.evaluate(o.UNIFORM, [1.0], y, T, np.array([0.0, 2.0]), n_groups=G)
    mean, err = o.finalize(r["group_sums"], n_loops)
    for t, x in enumerate(T):
        want = _finite_N_uniform(x, N)
        assert np.all(np.abs(mean[t] - want) < 4.5 * err[t] + 1e-12), (x, mean[t], want, err[t])
        assert np.all(err[t] < 0.05 * want)              # the test has teeth


def test_small_T_expansion_P5():
    n_loops, N = 1 << 14, 32
    y = o.generate_loops(6, n_loops, N)
    T = np.array([0.02])
    rho = np.array([0.0, 0.8, 2.0])
    eB0, lam = 3.0, 1.0
    r = o.evaluate(o.SECH2, [eB0, lam], y, T, rho, n_groups=64)
    mean, err = o.finalize(r["group_sums"], n_loops)
    b = o.field_b(o.SECH2, [eB0, lam], rho)
    lead = (b * T[0]) ** 2 / 3.0
    # finite-N factor of the leading term: Var(area)·(1 - ...) -> use P4's exact variance for the
    # phase part and the exact spin: <W>-1 = (bT)^2/2 - (bT)^2 Var(A)/2 + O(T^3, T/lambda^2)
    varA = (N - 1) * (N - 2) / (3.0 * N * N)
    want = (b * T[0]) ** 2 * 0.5 * (1.0 - varA)
    assert np.all(np.abs((mean[0] - 1.0) - want) < 5 * err[0] + 0.1 * lead)
    assert np.all(np.abs(want / lead - 1.0) < 0.15)      # and that is the paper's (eBT)^2/3 up to 1/N


def _gauss_hermite_4pt_loops(n_nodes):
    """All 4-point loops on a tensor Gauss-Hermite grid over the 6 Gaussian modes, with weights.
    Modes of the N = 4 cycle Laplacian (eigenvalues 2, 4, 2): variance 2/(N lambda_k) per component."""
    x, w = np.polynomial.hermite_e.hermegauss(n_nodes)      # weight exp(-x^2/2)
    w = w / w.sum()
    e = np.array([[1, 0, -1, 0], [0, 1, 0, -1], [1, -1, 1, -1]], dtype=float)
    e /= np.linalg.norm(e, axis=1, keepdims=True)
    sig = np.sqrt(np.array([2 / (4 * 2.0), 2 / (4 * 2.0), 2 / (4 * 4.0)]))
    g = np.stack(np.meshgrid(*([x] * 6), indexing="ij"), -1).reshape(-1, 6)
    wt = np.prod(np.stack(np.meshgrid(*([w] * 6), indexing="ij"), -1).reshape(-1, 6), axis=1)
    yx = (g[:, :3] * sig) @ e
    yy = (g[:, 3:] * sig) @ e
    return np.stack([yx, yy], -1), wt


def test_four_point_loops_brute_force_P8():
    loops, wt = _gauss_hermite_4pt_loops(9)                 # 531441 loops
    T = np.array([0.5, 2.0])
    rho = np.array([0.0, 0.6])
    # (i) uniform field: quadrature reproduces the closed form cosh(x)/(1 + (x/4)^2)
    r = o.evaluate(o.UNIFORM, [1.0], loops, T, rho, n_groups=1, per_loop=True)
    gh = np.tensordot(wt, r["W"], axes=(0, 0))
    for t, x in enumerate(T):
        assert np.all(np.abs(gh[t] - np.cosh(x) / (1 + (x / 4) ** 2)) < 1e-6)   # 9-node quadrature error
    # (ii) sech^2 profile: quadrature == Monte Carlo over generated 4-point d-loops
    par = [1.5, 0.8]
    r = o.evaluate(o.SECH2, par, loops, T, rho, n_groups=1, per_loop=True)
    gh = np.tensordot(wt, r["W"], axes=(0, 0))
    n_loops = 1 << 17
    y = o.generate_loops(44, n_loops, 4)
    mc = o.evaluate(o.SECH2, par, y, T, rho, n_groups=128)
    mean, err = o.finalize(mc["group_sums"], n_loops)
    assert np.all(np.abs(mean - gh) < 4.5 * err)
    assert np.all(err < 0.01 * np.abs(gh))
    assert np.all(np.abs(gh - 1.0) > 20 * err)              # field-dependent, not trivially 1


def test_finalize_eq63_equals_delete_one_jackknife_P10():
    rng = np.random.default_rng(3)
    G, n_loops = 16, 16 * 40
    gs = rng.normal(size=(G, 3, 5)) * 7 + 40
    mean, err, d1 = o.finalize(gs, n_loops, delete_one=True)
    gm = gs / (n_loops / G)
    assert np.max(np.abs(mean - gm.mean(0))) < 1e-13                  # eq. (61)-(62)
    assert np.max(np.abs(err - gm.std(0, ddof=1) / np.sqrt(G))) < 1e-13   # eq. (63) via numpy
    jk = np.sqrt((G - 1) / G * ((d1 - d1.mean(0)) ** 2).sum(0))       # textbook jackknife
    assert np.max(np.abs(jk - err)) < 1e-12
    with pytest.raises(ValueError):
        o.finalize(gs, n_loops + 1)
