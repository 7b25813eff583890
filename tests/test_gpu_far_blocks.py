"""GPU tests of the "far block" tiers (csrc/wl_block_bounds.cuh) of the packed FP32 and the lean FP64 sech^2 kernels
(csrc/wl_terms_packed_f32.cuh, csrc/wl_terms_sech2_f64.cuh) and of the strip-wise grid walk (csrc/wl_wilson_body.cuh);
DESIGN.md section 5.

Before a block of 128 staged segments is walked, every warp bounds rho_i^2(t) from below over the block's bounding
box and picks one of six instantiations (tier 0: the axis may be near; tiers 1-5: no near-axis polynomial and a
shorter polynomial for 1 - log2(1+E)).  What must hold:

  * every tier agrees with the oracle per loop (phase, spin, W) at the FP32 bounds of DESIGN.md section 6, on grids
    and loops built so that each tier is reached, including blocks that straddle the axis inside a far warp;
  * the tier is an optimisation, not a result: the same grid points evaluated in another order (other warps, other
    neighbours, other tiers) agree to FP32 rounding;
  * the walk order of the grid touches every point exactly once for awkward (n_T, n_rho), in every tile shape.
"""
import numpy as np
import pytest
import torch

from paper_1407_7486_b200 import inputs
from test_gpu_parity import assert_mean_close, dev

pytestmark = pytest.mark.gpu

SECH2 = inputs.SECH2


@pytest.fixture(scope="module")
def api():
    from paper_1407_7486_b200 import api as _api
    return _api


@pytest.fixture(scope="module")
def o():
    from oracle import wl_oracle
    return wl_oracle


def smooth_loops(n_loops, N, seed, radius):
    """Closed loops that are NOT Brownian: a few Fourier modes, so that 128 consecutive points form a short arc with a
    tight bounding box (Brownian d-loops of a few hundred points wander over the whole loop within one block)."""
    rng = np.random.default_rng(seed)
    t = 2.0 * np.pi * np.arange(N) / N
    y = np.zeros((n_loops, N, 2))
    for m in (1, 2, 3):
        a = rng.normal(size=(n_loops, 2, 2)) / m
        y[:, :, 0] += a[:, 0, 0, None] * np.cos(m * t) + a[:, 0, 1, None] * np.sin(m * t)
        y[:, :, 1] += a[:, 1, 0, None] * np.cos(m * t) + a[:, 1, 1, None] * np.sin(m * t)
    y -= y.mean(1, keepdims=True)
    return radius * y / np.sqrt((y ** 2).sum(2).mean(1))[:, None, None]


def per_loop_close(got, ref, what, compute="f32"):
    """FP32 phase / spin 2e-5, W 2e-3 relative; FP64 1e-12 (W: 1e-11, cosh amplifies the spin)."""
    W, p, s = got
    tp, tw = (2e-5, 2e-3) if compute == "f32" else (1e-12, 1e-11)
    assert np.all(np.isfinite(W)), what
    assert np.max(np.abs(p - ref["phase"]) / np.maximum(1.0, np.abs(ref["phase"]))) < tp, what
    assert np.max(np.abs(s - ref["spin"]) / np.maximum(1.0, np.abs(ref["spin"]))) < tp, what
    assert np.max(np.abs(W - ref["W"]) / np.maximum(1.0, np.abs(ref["W"]))) < tw, what


@pytest.mark.parametrize("compute", ["f32", "f64"])
@pytest.mark.parametrize("n_T,n_rho", [(16, 128), (4, 40)])          # P = 4 x 256 threads and P = 2 x 128 threads (FP32)
@pytest.mark.parametrize("lam", [1.0, 0.2])
def test_every_tier_against_the_oracle(api, o, n_T, n_rho, lam, compute):
    """rho_cm/lambda runs from 0 to 25 (u' = 2 log2(e) rho/lambda up to 72: tier 5 needs u' >= 12), loops of
    radius 0.6 lambda with 1024 smooth points (8 blocks of 128 per loop, each a short arc), sqrt(T) from 0.05 to 3:
    blocks on the axis, blocks that brush it and blocks in every far tier occur in the same launch."""
    n_loops, N = 6, 1024
    y = smooth_loops(n_loops, N, 11 + n_rho, 0.6 * lam)
    T = np.geomspace(0.0025, 9.0, n_T)
    rho = lam * np.concatenate([[0.0, 0.1, 0.35, 0.5], np.geomspace(0.7, 25.0, n_rho - 4)])
    params = (1.7 / lam ** 2, lam)
    f = api.wl_field_create(SECH2, params)
    loops = torch.tensor(y, dtype=torch.float32 if compute == "f32" else torch.float64, device="cuda")
    ref = o.evaluate(SECH2, params, loops.cpu().numpy().astype(np.float64), T, rho, None, per_loop=True)
    W, p, s = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), None, compute=compute)
    torch.cuda.synchronize()
    per_loop_close((W.cpu().numpy(), p.cpu().numpy(), s.cpu().numpy()), ref, "n_T=%d n_rho=%d lambda=%g" % (n_T, n_rho, lam), compute)
    assert np.abs(ref["phase"]).max() > 0.5                          # the field is felt
    # the far tiers matter here: most grid points are many lambda away
    assert np.mean(rho / lam > 4.2) > 0.25


@pytest.mark.parametrize("compute", ["f32", "f64"])
@pytest.mark.parametrize("n_T,n_rho", [(16, 128), (6, 24)])
def test_every_tier_with_phi_cm(api, o, n_T, n_rho, compute):
    """The same with the centres of mass spread round the axis (phi_cm given: the HAS_PHI Terms, whose bound uses both
    components of x_cm); smooth loops are not isotropic, so a wrong sign or a swapped component in the bound would put
    near blocks into a far tier for some angles."""
    n_loops, N, lam = 5, 1024, 0.5
    y = smooth_loops(n_loops, N, 23 + n_rho, 0.6 * lam)
    T = np.geomspace(0.0025, 9.0, n_T)
    rho = lam * np.concatenate([[0.0, 0.2, 0.45], np.geomspace(0.6, 25.0, n_rho - 3)])
    phi = 2.0 * np.pi * ((np.arange(n_rho) * 0.381966) % 1.0)         # golden-angle spread
    params = (1.7 / lam ** 2, lam)
    f = api.wl_field_create(SECH2, params)
    loops = torch.tensor(y, dtype=torch.float32 if compute == "f32" else torch.float64, device="cuda")
    ref = o.evaluate(SECH2, params, loops.cpu().numpy().astype(np.float64), T, rho, phi, per_loop=True)
    W, p, s = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), dev(phi), compute=compute)
    torch.cuda.synchronize()
    per_loop_close((W.cpu().numpy(), p.cpu().numpy(), s.cpu().numpy()), ref, "phi_cm n_T=%d n_rho=%d" % (n_T, n_rho), compute)
    assert np.abs(ref["phase"]).max() > 0.5


@pytest.mark.parametrize("compute", ["f32", "f64"])
def test_a_block_that_crosses_the_axis_inside_a_far_warp(api, o, compute):
    """One grid point sits exactly where the loop passes (its nodes reach w' ~ 0), the other 127 of its warp are far
    away: the warp must take tier 0 for that block, and the far lanes must not notice."""
    N = 512
    t = 2.0 * np.pi * np.arange(N) / N
    y = np.stack([0.5 * np.cos(t), 0.5 * np.sin(t)], axis=1)[None]   # a circle of radius 0.5 round the origin
    y = np.repeat(y, 3, axis=0) * np.array([1.0, 0.7, 1.3])[:, None, None]
    T = np.geomspace(1.0, 1.5, 16)
    rho = np.concatenate([[0.5], np.linspace(6.0, 9.0, 7)])          # sqrt(T) y reaches rho = 0.5 ... 0.61: on the circle
    params = (2.0, 1.0)
    loops = torch.tensor(y, dtype=torch.float32 if compute == "f32" else torch.float64, device="cuda")
    ref = o.evaluate(SECH2, params, loops.cpu().numpy().astype(np.float64), T, rho, None, per_loop=True)
    f = api.wl_field_create(SECH2, params)
    W, p, s = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), None, compute=compute)
    torch.cuda.synchronize()
    per_loop_close((W.cpu().numpy(), p.cpu().numpy(), s.cpu().numpy()), ref, "axis crossing", compute)
    assert np.abs(ref["phase"][:, :, 0]).max() > 0.3


@pytest.mark.parametrize("n_T,n_rho", [(64, 64), (9, 21)])
def test_tier_choice_does_not_change_the_result_beyond_rounding(api, n_T, n_rho):
    """The same (T, rho_cm) points handed over with the rho_cm axis shifted by three entries land in other strips, other
    warps, with other neighbours: other tiers, another shared reciprocal.  Group sums must agree to FP32 rounding
    (the tier polynomials differ by 6e-8) without being the same computation."""
    n_loops, N, G = 64, 512, 4
    loops = api.wl_loops_generate(n_loops, N, 5, torch.float32)
    T = np.geomspace(0.001, 20.0, n_T)
    rho = np.linspace(0.0, 5.0, n_rho)
    rho2 = np.concatenate([rho[3:], [5.5, 6.0, 6.5]])
    f = api.wl_field_create(SECH2, (1.0, 1.0))
    m1, g1 = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=G, compute="f32")
    m2, g2 = api.wl_eval(f, loops, dev(T), dev(rho2), None, n_groups=G, compute="f32")
    torch.cuda.synchronize()
    g1, g2 = g1.cpu().numpy()[:, :, 3:], g2.cpu().numpy()[:, :, :n_rho - 3]
    assert np.max(np.abs(g1 - g2) / np.maximum(1.0, np.abs(g1))) < 2e-6 * (n_loops // G)
    assert not np.array_equal(g1, g2)                                # they are different computations


@pytest.mark.parametrize("compute", ["f32", "f64"])
@pytest.mark.parametrize("n_T,n_rho", [(1, 1), (1, 9), (3, 8), (5, 17), (17, 5), (33, 7), (2, 300), (129, 17), (40, 52)])
def test_strip_walk_touches_every_grid_point_once(api, o, compute, n_T, n_rho):
    """The grid is walked in strips of 8 rho_cm (last strip narrower), in every tile shape (1, 2 or 4 grid points per
    thread).  <W> of the sech^2 tube depends on T and on rho_cm: an entry written to the wrong place, twice or not at
    all disagrees with the oracle."""
    n_loops, N, G = 8, 64, 2
    loops = api.wl_loops_generate(n_loops, N, 9, torch.float64)
    T = np.linspace(0.2, 3.0, n_T) if n_T > 1 else np.array([1.3])
    rho = np.linspace(0.0, 3.0, n_rho) if n_rho > 1 else np.array([0.7])
    params = (2.0, 1.0)
    f = api.wl_field_create(SECH2, params)
    m, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=G, compute=compute)
    torch.cuda.synchronize()
    ref = o.evaluate(SECH2, params, loops.cpu().numpy(), T, rho, None, n_groups=G)
    assert_mean_close(m.cpu().numpy(), ref["W_mean"], compute, what="mean %dx%d" % (n_T, n_rho))
    assert_mean_close(gs.cpu().numpy(), ref["group_sums"], compute, scale=n_loops // G, what="group sums")
    if n_T > 1 and n_rho > 1:                                        # the comparison can tell the entries apart
        assert np.ptp(ref["W_mean"], axis=0).max() > 1e-2 and np.ptp(ref["W_mean"], axis=1).max() > 1e-2
