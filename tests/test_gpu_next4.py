"""GPU parity of the SURVEY.md 8(f) NEXT-4 features, all through the C ABI:

  seeded evaluation        PAPER.md:576, 470   bit-identical to wl_loops_generate + wl_eval, and against the oracle
  Q-point quadrature       PAPER.md:152-168    per-loop phase / spin / W and <W> against the oracle (Q = 1, 2, 3)
  shuffled group assignment PAPER.md:411-417   membership table bit-exact against the oracle's, group sums against
                                               the oracle's regrouping, re-summation bit-exact
  bulk-copy staging        north_star          same bits as the default staging
Tolerances: north_star (tests/test_gpu_parity.py); per-loop bounds from DESIGN.md section 6.
"""
import numpy as np
import pytest
import torch

from paper_1407_7486_b200 import inputs
from test_gpu_parity import assert_mean_close, dev

pytestmark = pytest.mark.gpu

SECH2, FLUX, UNI = inputs.SECH2, inputs.FLUXTUBE, inputs.UNIFORM


@pytest.fixture(scope="module")
def api():
    from paper_1407_7486_b200 import api as _api
    return _api


@pytest.fixture(scope="module")
def o():
    from oracle import wl_oracle
    return wl_oracle


def grids(n_T, n_rho, T_max=6.0, rho_max=3.0, phi=False):
    T = np.geomspace(0.02, T_max, n_T)
    rho = np.linspace(0.0, rho_max, n_rho)
    ph = np.linspace(0.0, 5.5, n_rho) if phi else None
    return T, rho, ph


# --------------------------------------------------------------------------- seeded evaluation (NEXT-4a)

@pytest.mark.parametrize("profile,params,compute,storage,n_loops,N,nT,nr,G,phi", [
    (SECH2, (1.0, 1.0), "f64", "f64", 64, 256, 16, 16, 16, False),      # config 1's shape (128-thread tiles for FP32)
    (SECH2, (1.0, 1.0), "f32", "f64", 64, 256, 16, 16, 16, False),
    (SECH2, (1.0, 1.0), "f32", "f32", 48, 2048, 64, 64, 6, False),      # config 3's shape: P = 4, two chunks
    (SECH2, (10.0, 0.1), "f32", "f32", 16, 8192, 12, 48, 4, False),     # config 4/5's N: eight chunks, skeleton of 8
    (SECH2, (10.0, 0.1), "f64", "f32", 8, 8192, 6, 48, 2, False),       # FP64 kernel: 16 chunks of 512
    (SECH2, (1.0, 1.0), "f32", "f32", 24, 64, 9, 30, 3, True),          # phi_cm given, N below every chunk size
    (FLUX, (10.0, 1.0), "f32", "f32", 40, 1024, 33, 40, 5, False),
    (FLUX, (10.0, 1.0), "f64", "f64", 24, 512, 5, 7, 3, True),          # generic FP64 kernel (chunks of 256)
    (UNI, (1.0,), "f32", "f64", 32, 1024, 8, 8, 4, True),               # config 2's shape
    (UNI, (1.0,), "f64", "f64", 32, 2, 3, 3, 4, False),                 # N = 2: one noise point per loop
    (SECH2, (1.0, 1.0), "f32", "f32", 2048, 64, 64, 64, 4, False),      # units of 2 loops (loops_per_unit > 1)
    (SECH2, (1.0, 1.0), "f32", "f32", 8192, 16, 64, 64, 8, False),      # units of 8 loops
    (SECH2, (1.0, 1.0), "f32", "f32", 4, 65536, 8, 40, 2, False),       # the longest loop: skeleton of 64 points
    (SECH2, (1.0, 1.0), "f64", "f64", 2, 65536, 4, 40, 2, False),       # ... of 128 points (chunks of 512)
    (FLUX, (10.0, 1.0), "f64", "f32", 4, 16384, 4, 40, 2, False),       # generic FP64 kernel: chunks of 256, skeleton of 64
    (FLUX, (10.0, 1.0), "f64", "f64", 2, 65536, 3, 40, 2, False),       # ... the longest loop there: skeleton of 256 points
])
def test_seeded_equals_generate_then_eval_bit_for_bit(api, profile, params, compute, storage, n_loops, N, nT, nr, G, phi):
    T, rho, ph = grids(nT, nr, phi=phi)
    f = api.wl_field_create(profile, params)
    sdt = torch.float64 if storage == "f64" else torch.float32
    begin = 1000
    loops = api.wl_loops_generate(n_loops, N, 42, sdt, loop_begin=begin)
    m0, g0 = api.wl_eval(f, loops, dev(T), dev(rho), dev(ph), n_groups=G, compute=compute)
    m1, g1 = api.wl_eval_seeded(f, 42, n_loops, N, dev(T), dev(rho), dev(ph), n_groups=G, compute=compute,
                                storage=sdt, loop_begin=begin)
    torch.cuda.synchronize()
    assert torch.equal(g0, g1) and torch.equal(m0, m1)
    # a different seed or window is a different ensemble
    m2, g2 = api.wl_eval_seeded(f, 43, n_loops, N, dev(T), dev(rho), dev(ph), n_groups=G, compute=compute, storage=sdt,
                                loop_begin=begin)
    assert not torch.equal(g0, g2) or profile == UNI and N == 2


def test_seeded_against_the_oracle_on_the_oracles_own_loops(api, o):
    """No GPU-generated coordinate reaches the oracle here: it evaluates ITS d-loops (twin generator, agreement
    1e-12 per coordinate), so this also checks the in-kernel generator end to end."""
    n_loops, N, G = 64, 512, 8
    T, rho, _ = grids(7, 9)
    f = api.wl_field_create(SECH2, (1.0, 1.0))
    ref = o.evaluate(SECH2, (1.0, 1.0), o.generate_loops(7, n_loops, N, loop_begin=5), T, rho, None, n_groups=G)
    mean, gs = api.wl_eval_seeded(f, 7, n_loops, N, dev(T), dev(rho), None, n_groups=G, compute="f64",
                                  storage=torch.float64, loop_begin=5)
    torch.cuda.synchronize()
    assert_mean_close(mean.cpu().numpy(), ref["W_mean"], "f64")
    assert_mean_close(gs.cpu().numpy(), ref["group_sums"], "f64", scale=n_loops // G, what="group sums")


def test_seeded_per_loop_and_options(api):
    T, rho, _ = grids(5, 40)
    f = api.wl_field_create(SECH2, (1.0, 1.0))
    loops = api.wl_loops_generate(12, 1024, 9, torch.float32)
    W0, p0, s0 = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), None, compute="f32")
    W1, p1, s1 = api.wl_eval_per_loop(f, None, dev(T), dev(rho), None, compute="f32", n_loops=12, n_ppl=1024,
                                      storage=torch.float32, options=api.wl_eval_options(seed=9))
    torch.cuda.synchronize()
    assert torch.equal(W0, W1) and torch.equal(p0, p1) and torch.equal(s0, s1)
    # seeded + Q = 2 through wl_eval_opt == stored + Q = 2
    opt = api.wl_eval_options(quadrature_order=2)
    a = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=3, compute="f32", options=opt)
    b = api.wl_eval_seeded(f, 9, 12, 1024, dev(T), dev(rho), None, n_groups=3, compute="f32",
                           options=api.wl_eval_options(quadrature_order=2))
    torch.cuda.synchronize()
    assert torch.equal(a[1], b[1])


def test_seeded_rejects_what_it_cannot_do(api):
    T, rho, _ = grids(3, 3)
    f = api.wl_field_create(SECH2, (1.0, 1.0))
    for bad_N in (100, 1, 131072):
        with pytest.raises(api.WLError) as e:
            api.wl_eval_seeded(f, 1, 4, bad_N, dev(T), dev(rho), None, n_groups=2, compute="f64")
        assert e.value.status == 1


# --------------------------------------------------------------------------- quadrature order (NEXT-4b)

@pytest.mark.parametrize("Q", [1, 2, 3])
@pytest.mark.parametrize("profile,params,phi,N,nT,nr", [
    (SECH2, (1.0, 1.0), False, 256, 16, 16),          # lean kernels, 128-thread tiles in FP32
    (SECH2, (10.0, 0.1), False, 100, 40, 60),         # narrow tube, ragged N, P = 4 tiles in FP32
    (FLUX, (10.0, 1.0), False, 64, 24, 24),           # packed flux-tube kernel / generic FP64
    (SECH2, (1.3, 0.7), True, 33, 5, 11),             # phi_cm: generic kernels for Q > 1
    (UNI, (1.0,), True, 50, 4, 8),
])
def test_quadrature_per_loop_against_the_oracle(api, o, Q, profile, params, phi, N, nT, nr):
    rng = np.random.default_rng(100 * Q + N)
    n_loops = 10
    y = np.cumsum(rng.normal(size=(n_loops, N, 2)) / np.sqrt(N), axis=1)
    y -= y.mean(1, keepdims=True)                                   # rough open-ended walks: any polygon will do
    T, rho, ph = grids(nT, nr, T_max=4.0, rho_max=2.0 if params[-1] >= 0.5 or profile == UNI else 0.6, phi=phi)
    ref = o.evaluate_quadrature(profile, params, y, T, rho, ph, per_loop=True, Q=Q)
    f = api.wl_field_create(profile, params)
    opt = api.wl_eval_options(quadrature_order=Q)
    for compute, tol in (("f64", 1e-12), ("f32", 2e-5)):
        loops = torch.tensor(y, dtype=torch.float64, device="cuda")
        W, p, s = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), dev(ph), compute=compute, options=opt)
        torch.cuda.synchronize()
        p, s, W = p.cpu().numpy(), s.cpu().numpy(), W.cpu().numpy()
        assert np.max(np.abs(p - ref["phase"]) / np.maximum(1.0, np.abs(ref["phase"]))) < tol, (compute, Q)
        assert np.max(np.abs(s - ref["spin"]) / np.maximum(1.0, np.abs(ref["spin"]))) < tol
        wtol = 1e-10 if compute == "f64" else 2e-3
        assert np.max(np.abs(W - ref["W"]) / np.maximum(1.0, np.abs(ref["W"]))) < wtol


@pytest.mark.parametrize("Q", [2, 3])
def test_quadrature_ensemble_average_against_the_oracle(api, o, Q):
    c = inputs.config(1)
    T, rho, _ = c.grids()
    f = api.wl_field_create(c.profile, c.params)
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float64)
    ref = o.evaluate_quadrature(c.profile, c.params, loops.cpu().numpy(), T, rho, None, n_groups=c.n_groups, Q=Q)
    for compute in ("f64", "f32"):
        mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=c.n_groups, compute=compute,
                               options=api.wl_eval_options(quadrature_order=Q))
        torch.cuda.synchronize()
        assert_mean_close(mean.cpu().numpy(), ref["W_mean"], compute)
        assert_mean_close(gs.cpu().numpy(), ref["group_sums"], compute, scale=c.n_loops // c.n_groups, what="group sums")
    # the order matters: Q = 1 differs visibly from Q on this 256-point ensemble
    m1, _ = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=c.n_groups, compute="f64")
    assert float((m1 - mean).abs().max()) > 1e-6


def test_quadrature_order_zero_and_one_are_wl_eval(api):
    T, rho, _ = grids(6, 50)
    f = api.wl_field_create(SECH2, (1.0, 1.0))
    loops = api.wl_loops_generate(16, 128, 3, torch.float32)
    base = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=4, compute="f32")
    for q in (0, 1):
        got = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=4, compute="f32",
                          options=api.wl_eval_options(quadrature_order=q))
        assert torch.equal(base[1], got[1])
    with pytest.raises(api.WLError) as e:
        api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=4, compute="f32", options=api.wl_eval_options(quadrature_order=4))
    assert e.value.status == 1


# --------------------------------------------------------------------------- shuffled groups (NEXT-4c)

@pytest.mark.parametrize("n_loops,n_T", [(1, 3), (2, 2), (5, 4), (96, 4), (1000, 3), (4096, 5), (16385, 2)])
def test_membership_table_is_the_oracles_bit_for_bit(api, o, n_loops, n_T):
    for seed in (1, (1 << 40) + 17):
        perm = api.wl_group_permutation(seed, n_loops, n_T)
        torch.cuda.synchronize()
        assert np.array_equal(perm.cpu().numpy().astype(np.int64), o.group_permutation(seed, n_loops, n_T))


@pytest.mark.parametrize("compute", ["f64", "f32"])
def test_shuffled_group_sums(api, o, compute):
    n_loops, N, G, seed = 192, 128, 12, 77
    T, rho, _ = grids(6, 44)
    f = api.wl_field_create(SECH2, (1.5, 0.9))
    loops = api.wl_loops_generate(n_loops, N, 31, torch.float64)
    opt = api.wl_eval_options(shuffle_seed=seed)
    mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=G, compute=compute, options=opt)
    mean_u, gs_u = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=G, compute=compute)
    W, _, _ = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), None, compute=compute, want_phase_spin=False)
    torch.cuda.synchronize()
    mean, gs, W = mean.cpu().numpy(), gs.cpu().numpy(), W.cpu().numpy()
    # (i) against the oracle: its per-loop W regrouped with ITS table
    ref = o.evaluate(SECH2, (1.5, 0.9), loops.cpu().numpy(), T, rho, None, per_loop=True)
    perm = o.group_permutation(seed, n_loops, len(T))
    rmean, rgs = o.regroup_shuffled(ref["W"], G, perm)
    assert_mean_close(mean, rmean, compute)
    assert_mean_close(gs, rgs, compute, scale=n_loops // G, what="shuffled group sums")
    # (ii) membership bit-exact: re-summing the GPU's own per-loop W in the documented order gives S_g to the last
    # bit; the contiguous membership does not
    per = n_loops // G
    for t in range(len(T)):
        members = perm[t].reshape(G, per)
        for g in range(G):
            S = np.zeros(len(rho))
            for l in members[g]:
                S = S + W[l, t, :]
            assert np.array_equal(S, gs[g, t])
    assert not np.array_equal(gs, gs_u.cpu().numpy())
    # (iii) eq. (61)-(62): the mean does not care
    assert np.max(np.abs(mean - mean_u.cpu().numpy())) < 1e-12 * np.abs(mean).max()
    m2, err = api.wl_jackknife_finalize(torch.tensor(gs, device="cuda"), n_loops)
    assert np.all(err.cpu().numpy() > 0)


def test_shuffled_and_seeded_together(api):
    T, rho, _ = grids(4, 40)
    f = api.wl_field_create(SECH2, (1.0, 1.0))
    loops = api.wl_loops_generate(64, 256, 12, torch.float32)
    a = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=8, compute="f32", options=api.wl_eval_options(shuffle_seed=3))
    b = api.wl_eval_seeded(f, 12, 64, 256, dev(T), dev(rho), None, n_groups=8, compute="f32",
                           options=api.wl_eval_options(shuffle_seed=3))
    torch.cuda.synchronize()
    assert torch.equal(a[1], b[1]) and torch.equal(a[0], b[0])


# --------------------------------------------------------------------------- bulk-copy staging (row J)

@pytest.mark.parametrize("profile,params,compute,storage,N,nT,nr,phi", [
    (SECH2, (1.0, 1.0), "f32", "f32", 2048, 64, 64, False),     # the instantiated variants ...
    (SECH2, (1.0, 1.0), "f32", "f32", 2050, 40, 60, False),     # ragged last chunk
    (SECH2, (1.0, 1.0), "f32", "f64", 300, 40, 60, False),
    (SECH2, (10.0, 0.1), "f64", "f64", 1500, 16, 40, False),
    (SECH2, (10.0, 0.1), "f64", "f32", 1024, 16, 40, False),
    (UNI, (1.0,), "f32", "f64", 1024, 32, 8, True),
    (UNI, (1.0,), "f64", "f64", 1000, 32, 8, True),
    (SECH2, (1.0, 1.0), "f32", "f32", 255, 64, 64, False),      # ... and shapes it silently declines (odd N in FP32)
    (FLUX, (10.0, 1.0), "f32", "f32", 256, 64, 64, False),
])
def test_bulk_staging_gives_the_same_bits(api, profile, params, compute, storage, N, nT, nr, phi):
    T, rho, ph = grids(nT, nr, phi=phi)
    f = api.wl_field_create(profile, params)
    rng = np.random.default_rng(N)
    n_loops = 24 if N != 300 else 8193          # 8193 = 3 x 2731 loops: units of one loop; see below for longer units
    y = np.cumsum(rng.normal(size=(n_loops, N, 2)) / np.sqrt(N), axis=1)
    loops = torch.tensor(y - y.mean(1, keepdims=True), dtype=torch.float64 if storage == "f64" else torch.float32, device="cuda")
    a = api.wl_eval(f, loops, dev(T), dev(rho), dev(ph), n_groups=3, compute=compute)
    b = api.wl_eval(f, loops, dev(T), dev(rho), dev(ph), n_groups=3, compute=compute, options=api.wl_eval_options(staging=1))
    torch.cuda.synchronize()
    assert torch.equal(a[1], b[1]) and torch.equal(a[0], b[0])


def test_bulk_staging_with_units_of_several_loops(api):
    """The ring runs across the loops of a unit: 8192 loops of 16 points on a 64 x 64 grid are cut in units of 8."""
    T, rho, _ = grids(64, 64)
    f = api.wl_field_create(SECH2, (1.0, 1.0))
    loops = api.wl_loops_generate(8192, 16, 5, torch.float32)
    a = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=8, compute="f32")
    b = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=8, compute="f32", options=api.wl_eval_options(staging=1))
    torch.cuda.synchronize()
    assert torch.equal(a[1], b[1])
    loops = api.wl_loops_generate(4096, 1024, 5, torch.float64)      # 600 of its points: two chunks of 512 + 88, units of 2
    T2, rho2, _ = grids(16, 40)
    a = api.wl_eval(f, loops[:, :600].contiguous(), dev(T2), dev(rho2), None, n_groups=4, compute="f64")
    b = api.wl_eval(f, loops[:, :600].contiguous(), dev(T2), dev(rho2), None, n_groups=4, compute="f64",
                    options=api.wl_eval_options(staging=1))
    torch.cuda.synchronize()
    assert torch.equal(a[1], b[1])
