"""GPU tests added in round 2 for paths the round-1 suite did not reach (VERDICT.md r01 "What's weak"):

  * the FP32 lean kernels at the ends of their lambda window and the generic kernel beyond it, against the oracle
  * the discretisation estimate in the packed FP32 kernels at P = 4 (n_grid >= 2048) and in the 128-thread
    variant (n_grid <= 256), sech^2 and flux tube, against the oracle
  * more jackknife groups than gridDim.y allows (one-loop groups of 70000 loops)
  * wl_eval / wl_eval_discretization on a side stream with their internally allocated scratch
  * option combinations that must be refused before anything is launched; wl_grid_validate
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


@pytest.mark.parametrize("profile", [SECH2, FLUX])
@pytest.mark.parametrize("lam", [5e-5, 1e-4, 2e-4, 5e3, 1e4, 2e4])
def test_fp32_on_both_sides_of_the_lean_kernels_lambda_window(api, o, profile, lam):
    """launch_wilson routes lambda outside [1e-4, 1e4] to the generic (unscaled) kernel; inside, the lean kernels
    carry squared radii scaled by 1/lambda^2.  Loops are sized to the tube (rho/lambda of order one), so the
    profile is resolved on either side of the switch; rho_cm reaches 40 lambda (E = exp(-80): flushed, g -> ln 2/u^2)."""
    n_loops, N = 12, 96
    rng = np.random.default_rng(int(lam * 1e6) % 1000 + profile)
    y = np.cumsum(rng.normal(size=(n_loops, N, 2)) / np.sqrt(N), axis=1)
    y -= y.mean(1, keepdims=True)
    T = np.array([0.1, 1.0, 4.0]) * lam ** 2                       # sqrt(T) y ~ lambda
    rho = np.array([0.0, 0.3, 1.0, 3.0, 40.0]) * lam
    strength = 1.3 / lam ** 2 if profile == SECH2 else 2.0         # phases of order one: eB0 T ~ 1; script-F is dimensionless
    params = (strength, lam)
    ref = o.evaluate(profile, params, y, T, rho, None, per_loop=True)
    f = api.wl_field_create(profile, params)
    loops = torch.tensor(y, dtype=torch.float64, device="cuda")
    W, p, s = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), None, compute="f32")
    torch.cuda.synchronize()
    W, p, s = W.cpu().numpy(), p.cpu().numpy(), s.cpu().numpy()
    assert np.all(np.isfinite(W))
    assert np.max(np.abs(p - ref["phase"]) / np.maximum(1.0, np.abs(ref["phase"]))) < 2e-5
    assert np.max(np.abs(s - ref["spin"]) / np.maximum(1.0, np.abs(ref["spin"]))) < 2e-5
    assert np.max(np.abs(W - ref["W"]) / np.maximum(1.0, np.abs(ref["W"]))) < 2e-3
    assert np.abs(ref["phase"]).max() > 0.05                       # the field is felt: not a vacuous comparison


@pytest.mark.parametrize("profile,params", [(SECH2, (1.0, 1.0)), (FLUX, (3.0, 1.0))])
@pytest.mark.parametrize("n_T,n_rho", [(64, 64), (33, 70), (16, 16), (7, 30)])
def test_discretisation_estimate_fp32_packed_tile_shapes(api, o, profile, params, n_T, n_rho):
    """n_grid >= 2048: 256 threads x P = 4 with three running W sums per grid point (the instantiation most likely
    to spill); n_grid <= 256: the 128-thread x P = 2 variant; against the oracle at the north_star tolerance."""
    n_loops, N, G = 32, 256, 4
    T = np.geomspace(0.02, 3.0, n_T)
    rho = np.linspace(0.0, 3.0, n_rho)
    loops = api.wl_loops_generate(n_loops, N, 77, torch.float32)
    f = api.wl_field_create(profile, params)
    gs3 = api.wl_eval_discretization(f, loops, dev(T), dev(rho), None, n_groups=G, compute="f32")
    per_loop = api.wl_eval_discretization(f, loops, dev(T), dev(rho), None, n_groups=n_loops, compute="f32")
    torch.cuda.synchronize()
    ti = np.unique(np.linspace(0, n_T - 1, 6).astype(int))
    ri = np.unique(np.linspace(0, n_rho - 1, 9).astype(int))
    ref_gs, ref_W = o.evaluate_discretization(profile, params, loops.cpu().numpy(), T[ti], rho[ri], None, n_groups=G,
                                              per_loop=True)
    W = per_loop.cpu().numpy()[:, :, ti][:, :, :, ri]
    assert np.max(np.abs(W - ref_W) / np.maximum(1.0, np.abs(ref_W))) < 2e-3
    for lev in range(3):
        assert_mean_close(gs3.cpu().numpy()[lev][:, ti][:, :, ri], ref_gs[lev], "f32", scale=n_loops // G,
                          what="level %d group sums" % lev)


def test_more_groups_than_a_grid_dimension(api):
    """One-loop groups of 70000 loops: n_groups > 65535 used to fail in k_group_reduce's gridDim.y AFTER k_wilson ran."""
    n_loops, N = 70000, 4
    T, rho = dev([0.5, 2.0]), dev([0.0, 1.0, 2.0])
    loops = api.wl_loops_generate(n_loops, N, 3, torch.float64)
    f = api.wl_field_create(SECH2, (1.0, 1.0))
    mean, gs = api.wl_eval(f, loops, T, rho, None, n_groups=n_loops, compute="f64")
    W, _, _ = api.wl_eval_per_loop(f, loops, T, rho, None, compute="f64", want_phase_spin=False)
    torch.cuda.synchronize()
    assert torch.equal(gs, W)                                      # a group of one loop is that loop's W
    assert torch.allclose(mean, W.mean(0), rtol=1e-13, atol=0)


def test_side_stream_with_internal_scratch(api):
    """the scratch workspace must belong to the stream the kernels run on.  Evaluate on a side stream
    while the default stream allocates and overwrites blocks of the same size; the result must be the reference."""
    c = inputs.config(1)
    T, rho, _ = c.grids()
    Td, rd = dev(T), dev(rho)
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float64)
    f = api.wl_field_create(c.profile, c.params)
    ref_mean, ref_gs = api.wl_eval(f, loops, Td, rd, None, n_groups=c.n_groups, compute="f64")
    ref3 = api.wl_eval_discretization(f, loops, Td, rd, None, n_groups=c.n_groups, compute="f64")
    torch.cuda.synchronize()
    need = api.wl_eval_workspace_bytes(c.n_loops, c.n_ppl, c.n_T, c.n_rho, c.n_groups, "f64")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    for _ in range(10):
        mean, gs = api.wl_eval(f, loops, Td, rd, None, n_groups=c.n_groups, compute="f64", stream=side)
        gs3 = api.wl_eval_discretization(f, loops, Td, rd, None, n_groups=c.n_groups, compute="f64", stream=side)
        for k in range(4):                                         # default stream: same-size blocks, written at once
            junk = torch.empty(need * (1 if k < 2 else 3), dtype=torch.uint8, device="cuda")
            junk.fill_(255)
            del junk
        side.synchronize()
        assert torch.equal(gs, ref_gs) and torch.equal(mean, ref_mean) and torch.equal(gs3, ref3)
    torch.cuda.synchronize()


def test_refused_before_anything_is_launched(api):
    T, rho = dev([0.5, 2.0]), dev([0.0, 1.0])
    loops = api.wl_loops_generate(8, 16, 1, torch.float64)
    f = api.wl_field_create(SECH2, (1.0, 1.0))
    mean = torch.full((2, 2), -7.0, dtype=torch.float64, device="cuda")
    gs = torch.full((2, 2, 2), -7.0, dtype=torch.float64, device="cuda")
    # a shard cannot shuffle across shards
    with pytest.raises(api.WLError) as e:
        api.wl_eval(f, loops, T, rho, None, n_groups=2, compute="f64", W_mean=mean, group_sums=gs,
                    options=api.wl_eval_options(shuffle_seed=1, ensemble_loops=16))
    assert e.value.status == 2
    # ensemble smaller than the shard / not whole groups / unknown staging
    for opt in (api.wl_eval_options(ensemble_loops=4), api.wl_eval_options(ensemble_loops=10), api.wl_eval_options(staging=2)):
        with pytest.raises((api.WLError, ValueError)):
            api.wl_eval(f, loops, T, rho, None, n_groups=2, compute="f64", W_mean=mean, group_sums=gs, options=opt)
    # a struct of another ABI generation
    opt = api.wl_eval_options()
    opt.struct_size = 8
    with pytest.raises((api.WLError, ValueError)):
        api.wl_eval(f, loops, T, rho, None, n_groups=2, compute="f64", W_mean=mean, group_sums=gs, options=opt)
    torch.cuda.synchronize()
    assert float(mean.min()) == -7.0 and float(gs.max()) == -7.0   # nothing was written


def test_grid_validate(api):
    api.wl_grid_validate([0.01, 10.0], [0.0, 4.0])
    for T, rho in (([0.0, 1.0], [0.0]), ([-1.0], [0.0]), ([1.0], [-1e-9]), ([float("nan")], [0.0]), ([1.0], [float("inf")])):
        with pytest.raises(api.WLError) as e:
            api.wl_grid_validate(T, rho)
        assert e.value.status == 1


@pytest.mark.parametrize("n_T,n_rho", [(64, 64), (12, 40), (16, 16)])
def test_scalar_only_sech2_kernel_in_every_tile_shape(api, o, n_T, n_rho):
    """A scalar field in the reducing path runs the packed kernel WITHOUT the spin sum (3 special-function ops per
    point-eval): against the oracle's W = cos(phase), and consistent with the full kernel's per-loop phases."""
    n_loops, N, G = 64, 512, 8
    T, rho = np.geomspace(0.01, 8.0, n_T), np.linspace(0.0, 4.0, n_rho)
    loops = api.wl_loops_generate(n_loops, N, 91, torch.float32)
    fs = api.wl_field_create_particle(SECH2, (1.0, 1.0), api.SCALAR)
    mean, gs = api.wl_eval(fs, loops, dev(T), dev(rho), None, n_groups=G, compute="f32")
    Wl, ph, _ = api.wl_eval_per_loop(fs, loops, dev(T), dev(rho), None, compute="f32")
    torch.cuda.synchronize()
    ref = o.evaluate(SECH2, (1.0, 1.0), loops.cpu().numpy(), T, rho, None, n_groups=G, scalar=True)
    assert_mean_close(mean.cpu().numpy(), ref["W_mean"], "f32")
    assert_mean_close(gs.cpu().numpy(), ref["group_sums"], "f32", scale=n_loops // G, what="group sums")
    # the two kernels round the reciprocal differently: equal to FP32 accuracy, not bit for bit
    regrouped = Wl.reshape(G, n_loops // G, n_T, n_rho).sum(1)
    assert float((regrouped - gs).abs().max()) < 2e-4 * (n_loops // G)
    # a seeded scalar run takes the same kernel: same bits
    m2, g2 = api.wl_eval_seeded(fs, 91, n_loops, N, dev(T), dev(rho), None, n_groups=G, compute="f32", storage=torch.float32)
    torch.cuda.synchronize()
    assert torch.equal(gs, g2)
