"""Pins of the oracle's shuffled group assignment (Sec. IV.B.3; Fig. 6, PAPER.md:380;
SURVEY.md 8(f) NEXT-4; reading A17).  CPU only.

What would fail if it were wrong:
  pi_t not a bijection / groups unequal      -> sorted(pi_t) == range(n) for awkward n
  pi_t the same for every t, or not random   -> distinctness across t and seeds, position and co-membership
                                                frequencies against their uniform expectations
  regrouping indexes the wrong loop / T      -> identity table reproduces the contiguous groups of `evaluate`
                                                (already pinned) bit for bit; a gather in numpy, entry by entry
  the mean depends on the grouping           -> eq. (61)-(62): <W> unchanged to rounding
  shuffling does not decorrelate             -> the paper's Fig. 6 claim as an inequality
"""
import numpy as np
import pytest

from oracle import wl_oracle as o


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 15, 16, 17, 63, 100, 1000, 1024, 1025, 4097])
def test_every_pi_t_is_a_bijection(n):
    perm = o.group_permutation(7, n, 5)
    assert perm.shape == (5, n) and perm.dtype == np.int64
    for t in range(5):
        assert np.array_equal(np.sort(perm[t]), np.arange(n))


def test_table_matches_the_index_function_and_is_deterministic():
    perm = o.group_permutation(123456789012345, 300, 4)
    for t in (0, 3):
        for i in (0, 1, 150, 299):
            assert perm[t, i] == o.shuffle_index(123456789012345, t, 300, i)
    assert np.array_equal(perm, o.group_permutation(123456789012345, 300, 4))


def test_depends_on_t_and_on_the_seed():
    a = o.group_permutation(1, 256, 8)
    b = o.group_permutation(2, 256, 8)
    for t in range(8):
        assert not np.array_equal(a[t], np.arange(256))
        assert not np.array_equal(a[t], b[t])
        for u in range(t):
            assert np.mean(a[t] == a[u]) < 0.05          # two random permutations share ~1/n fixed positions
    hi = o.group_permutation(1 << 40, 256, 2)           # the high key word matters too
    assert not np.array_equal(hi[0], o.group_permutation(0, 256, 2)[0])


def test_positions_are_uniform():
    """Over many T indices every loop must visit every position equally often: chi^2 of the n x n count table."""
    n, n_T = 24, 6000
    perm = o.group_permutation(99, n, n_T)
    counts = np.zeros((n, n))
    for i in range(n):
        counts[i] = np.bincount(perm[:, i], minlength=n)
    expect = n_T / n
    chi2 = np.sum((counts - expect) ** 2 / expect)
    dof = (n - 1) ** 2
    assert abs(chi2 - dof) < 6.0 * np.sqrt(2.0 * dof), (chi2, dof)


def test_pairs_share_a_group_as_often_as_chance_says():
    """P(loops a and b in the same group) = (m - 1)/(n - 1) for a uniformly random assignment (m per group)."""
    n, G, n_T = 60, 6, 4000
    m = n // G
    perm = o.group_permutation(5, n, n_T)
    pos = np.argsort(perm, axis=1)                       # pos[t][loop] = position of the loop at T index t
    grp = pos // m
    for a, b in [(0, 1), (0, 59), (17, 42), (30, 31)]:
        p = np.mean(grp[:, a] == grp[:, b])
        p0 = (m - 1) / (n - 1)
        assert abs(p - p0) < 5.0 * np.sqrt(p0 * (1 - p0) / n_T), (a, b, p, p0)


def _small_case(n_loops=96, N=16, seed=31):
    loops = o.generate_loops(seed, n_loops, N)
    T = np.array([0.3, 1.0, 2.5, 3.0])
    rho = np.array([0.0, 0.8, 1.9])
    res = o.evaluate(o.SECH2, [1.5, 0.9], loops, T, rho, None, n_groups=8, per_loop=True)
    return res, T, rho


def test_identity_table_reproduces_the_contiguous_groups_bit_for_bit():
    res, T, rho = _small_case()
    ident = np.tile(np.arange(96, dtype=np.int64), (len(T), 1))
    mean, gs = o.regroup_shuffled(res["W"], 8, ident)
    assert np.array_equal(gs, res["group_sums"])
    assert np.array_equal(mean, res["W_mean"])


def test_shuffled_group_sums_are_a_gather_of_the_per_loop_values():
    res, T, rho = _small_case()
    perm = o.group_permutation(77, 96, len(T))
    mean, gs = o.regroup_shuffled(res["W"], 8, perm)
    W = res["W"]
    for t in range(len(T)):
        members = perm[t].reshape(8, 12)                 # group g = positions [12 g, 12 g + 12)
        for g in range(8):
            want = W[members[g], t, :].sum(0)
            assert np.allclose(gs[g, t], want, rtol=1e-14, atol=0)
    # eq. (61)-(62): the mean does not depend on the grouping (rounding order only)
    assert np.allclose(mean, res["W_mean"], rtol=1e-14, atol=0)
    assert np.allclose(gs.sum(0) / 96, res["W_mean"], rtol=1e-14, atol=0)
    # a different T index uses a different membership
    assert not np.array_equal(np.sort(perm[0].reshape(8, 12), 1), np.sort(perm[1].reshape(8, 12), 1))
    # eq. (63) works unchanged on the shuffled sums
    m2, err = o.finalize(gs, 96)
    assert np.allclose(m2, mean, rtol=1e-14) and np.all(err > 0)


def test_bad_arguments():
    res, T, rho = _small_case()
    perm = o.group_permutation(1, 96, len(T))
    with pytest.raises(ValueError):
        o.regroup_shuffled(res["W"], 7, perm)            # 96 % 7 != 0: equal groups required
    with pytest.raises(ValueError):
        o.group_permutation(1, 0, 3)


def test_shuffling_removes_the_correlation_between_integrand_evaluations():
    """Fig. 6 and PAPER.md:411-417: with fixed groups the group means at two proper times are
    strongly correlated (the same worldlines sit in the same group); reshuffling the membership between the
    evaluations "produces a considerable reduction in the correlations".  Uniform field as in the figure."""
    n_loops, G = 4096, 64
    loops = o.generate_loops(41, n_loops, 64)
    T = np.array([2.5, 3.0])
    res = o.evaluate(o.UNIFORM, [1.0], loops, T, np.array([0.0]), None, n_groups=G, per_loop=True)
    fixed = res["group_sums"][:, :, 0]
    c_fixed = np.corrcoef(fixed[:, 0], fixed[:, 1])[0, 1]
    cs = []
    for seed in range(1, 9):
        _, gs = o.regroup_shuffled(res["W"], G, o.group_permutation(seed, n_loops, 2))
        cs.append(np.corrcoef(gs[:, 0, 0], gs[:, 1, 0])[0, 1])
    cs = np.array(cs)
    assert c_fixed > 0.8, c_fixed
    assert np.all(np.abs(cs) < 0.5), cs                  # 64 groups: a null correlation scatters by ~0.125
    assert abs(cs.mean()) < 0.2, cs
