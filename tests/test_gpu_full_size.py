"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (wl_eval on
the whole grid and ensemble), checked on sampled outputs the oracle can compute one by one
(SURVEY.md section 8(d) coverage table, readings A12):

  config 3: full grid on the GPU; oracle on a 16 x 16 sub-grid (256 points: both ends of both axes forced in,
            the rest seeded) x ALL loops                                               (<W>, S_g)
  config 4: FP32 kernel AND FP64 kernel on the full 48 x 128 grid (the launches bench.py's `secondary` block and
            profiles/ report: Sech2PackedF32<4> and Sech2LeanF64<2>); oracle on a seeded 8 x 8 sub-grid
  config 5: full grid; oracle on 64 seeded (T, rho) points x 16 seeded WHOLE groups   (S_g)
"""
import numpy as np
import pytest
import torch

from paper_1407_7486_b200 import inputs
from test_gpu_parity import assert_mean_close, dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_1407_7486_b200 import api as _api
    return _api


@pytest.fixture(scope="module")
def o():
    from oracle import wl_oracle
    return wl_oracle


def subgrid(c, n_t, n_r, seed, edges=False):
    """Seeded sub-grid; edges=True forces the first and last index of both axes in (rho_cm = 0 is where the
    near-axis branch of the sech^2 kernels carries most terms; T_min and T_max are the extremes of the scaling)."""
    rng = np.random.default_rng(seed)
    if not edges:
        return np.sort(rng.choice(c.n_T, n_t, replace=False)), np.sort(rng.choice(c.n_rho, n_r, replace=False))
    ti = np.sort(np.concatenate(([0, c.n_T - 1], 1 + rng.choice(c.n_T - 2, n_t - 2, replace=False))))
    ri = np.sort(np.concatenate(([0, c.n_rho - 1], 1 + rng.choice(c.n_rho - 2, n_r - 2, replace=False))))
    return ti, ri


def test_config3_full_fp32_sampled_grid_all_loops(api, o):
    c = inputs.config(3)
    T, rho, _ = c.grids()
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float32)
    f = api.wl_field_create(c.profile, c.params)
    mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=c.n_groups, compute="f32")
    mean2, gs2 = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=c.n_groups, compute="f32")
    # seeded evaluation: no ensemble buffer, same bits as generate + eval
    mean3, gs3 = api.wl_eval_seeded(f, c.seed, c.n_loops, c.n_ppl, dev(T), dev(rho), None, n_groups=c.n_groups,
                                    compute="f32", storage=torch.float32)
    torch.cuda.synchronize()
    assert torch.equal(gs, gs2) and torch.equal(mean, mean2)          # fixed summation order: same bits
    assert torch.equal(gs, gs3) and torch.equal(mean, mean3)
    ti, ri = subgrid(c, 16, 16, 303, edges=True)          # 256 grid points x all loops (~16 s of oracle)
    assert ti[0] == 0 and ti[-1] == c.n_T - 1 and ri[0] == 0 and ri[-1] == c.n_rho - 1
    ref = o.evaluate(c.profile, c.params, loops.cpu().numpy(), T[ti], rho[ri], None, n_groups=c.n_groups)
    assert_mean_close(mean.cpu().numpy()[np.ix_(ti, ri)], ref["W_mean"], "f32")
    assert_mean_close(gs.cpu().numpy()[:, ti][:, :, ri], ref["group_sums"], "f32",
                      scale=c.n_loops // c.n_groups, what="group sums")
    # properties that hold at any size: <W> >= ~1 for the fermion loop at weak field / small T
    # (<W> - 1 -> (eB(rho) T)^2/3), and eq. (61)-(62): mean of group means == mean
    m = mean.cpu().numpy()
    eB = c.params[0] / np.cosh(rho / c.params[1]) ** 2
    lead = (eB[None, :] * T[:, None]) ** 2 / 3.0
    small = T < 0.02
    assert np.max(np.abs(m[small] - 1.0 - lead[small])) < 5e-5
    assert np.max(np.abs(gs.cpu().numpy().sum(0) / c.n_loops - m)) < 1e-12 * np.abs(m).max()


def test_config4_narrow_flux_tube_both_kernels(api, o):
    c = inputs.config(4)
    T, rho, _ = c.grids()
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float32)
    f = api.wl_field_create(c.profile, c.params)
    ti, ri = subgrid(c, 8, 8, 404)
    ti[-1] = c.n_T - 1                       # keep the largest T (largest phases) in the sample
    ri[0] = 0                                # and the axis
    mean32, gs32 = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=c.n_groups, compute="f32")
    # the FP64 kernel on the FULL grid x all loops (~8 s): the launch shape whose throughput is reported
    # (north_star config 4: "FP64-kernel and FP32-kernel variants both reported"), not a 64-point sub-grid launch
    mean64, gs64 = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=c.n_groups, compute="f64")
    torch.cuda.synchronize()
    ref = o.evaluate(c.profile, c.params, loops.cpu().numpy(), T[ti], rho[ri], None, n_groups=c.n_groups)
    assert_mean_close(mean64.cpu().numpy()[np.ix_(ti, ri)], ref["W_mean"], "f64")
    assert_mean_close(gs64.cpu().numpy()[:, ti][:, :, ri], ref["group_sums"], "f64", scale=c.n_loops // c.n_groups,
                      what="group sums")
    # the two kernels against each other on every grid point (the oracle sees 64 of the 6144)
    assert_mean_close(mean32.cpu().numpy(), mean64.cpu().numpy(), "f32")
    assert_mean_close(mean32.cpu().numpy()[np.ix_(ti, ri)], ref["W_mean"], "f32")
    assert_mean_close(gs32.cpu().numpy()[:, ti][:, :, ri], ref["group_sums"], "f32",
                      scale=c.n_loops // c.n_groups, what="group sums")


def test_config5_large_sweep_sampled_points_and_whole_groups(api, o):
    c = inputs.config(5)
    T, rho, _ = c.grids()
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float32)
    f = api.wl_field_create(c.profile, c.params)
    mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=c.n_groups, compute="f32")
    mean_s, gs_s = api.wl_eval_seeded(f, c.seed, c.n_loops, c.n_ppl, dev(T), dev(rho), None, n_groups=c.n_groups,
                                      compute="f32", storage=torch.float32)      # 4.3 GB of coordinates never stored
    torch.cuda.synchronize()
    assert torch.equal(gs, gs_s) and torch.equal(mean, mean_s)
    del gs_s, mean_s
    gs = gs.cpu().numpy()
    rng = np.random.default_rng(505)
    groups = np.sort(rng.choice(c.n_groups, 16, replace=False))
    points = [(int(rng.integers(c.n_T)), int(rng.integers(c.n_rho))) for _ in range(64)]
    per_group = c.n_loops // c.n_groups
    idx = np.concatenate([np.arange(g * per_group, (g + 1) * per_group) for g in groups])
    sub = loops[torch.as_tensor(idx, device="cuda")].cpu().numpy()          # 16 whole groups (reading A12)
    got = np.empty((16, len(points)))
    want = np.empty((16, len(points)))
    for k, (t, r) in enumerate(points):
        ref = o.evaluate(c.profile, c.params, sub, T[t:t + 1], rho[r:r + 1], None, n_groups=16)
        want[:, k] = ref["group_sums"][:, 0, 0]
        got[:, k] = gs[groups, t, r]
    assert_mean_close(got, want, "f32", scale=per_group, what="group sums")
    m = mean.cpu().numpy()
    assert np.all(np.isfinite(m))
    assert np.max(np.abs(gs.sum(0) / c.n_loops - m)) < 1e-12 * np.abs(m).max()
