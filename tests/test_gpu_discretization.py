"""SURVEY.md section 8(f) NEXT-2 on the GPU: the discretisation estimate of Sec. IV.A (eq. (48)-(52),
PAPER.md:269-304) against the oracle, tolerances of tests/test_gpu_parity.py."""
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


CASES = [(inputs.UNIFORM, (1.0,), False), (inputs.SECH2, (1.0, 1.0), False), (inputs.SECH2, (10.0, 0.1), True),
         (inputs.FLUXTUBE, (3.0, 1.0), False), (inputs.FLUXTUBE, (3.0, 1.0), True)]


@pytest.mark.parametrize("compute", ["f64", "f32"])
@pytest.mark.parametrize("profile,params,with_phi", CASES)
@pytest.mark.parametrize("scalar", [False, True])
def test_three_levels_match_the_oracle_per_loop_and_per_group(api, o, compute, profile, params, with_phi, scalar):
    n_loops, N = 96, 1024
    T = np.geomspace(0.02, 2.0 if profile != inputs.SECH2 or params[0] < 5 else 0.3, 7)
    rho = np.linspace(0.0, 2.5, 41) * (params[1] if len(params) > 1 and params[1] < 1 else 1.0)
    phi = np.linspace(0.0, 5.0, len(rho)) if with_phi else None
    loops = api.wl_loops_generate(n_loops, N, 41, torch.float32)
    f = api.wl_field_create_particle(profile, params, api.SCALAR if scalar else api.FERMION)
    per_loop = api.wl_eval_discretization(f, loops, dev(T), dev(rho), dev(phi), n_groups=n_loops, compute=compute)
    grouped = api.wl_eval_discretization(f, loops, dev(T), dev(rho), dev(phi), n_groups=8, compute=compute)
    again = api.wl_eval_discretization(f, loops, dev(T), dev(rho), dev(phi), n_groups=8, compute=compute)
    torch.cuda.synchronize()
    assert torch.equal(grouped, again)
    ref_gs, ref_W = o.evaluate_discretization(profile, params, loops.cpu().numpy(), T, rho, phi, n_groups=8,
                                              per_loop=True, scalar=scalar)
    W = per_loop.cpu().numpy()                                    # one loop per group: the per-loop W
    wtol = 1e-10 if compute == "f64" else 2e-3
    assert np.max(np.abs(W - ref_W) / np.maximum(1.0, np.abs(ref_W))) < wtol
    for lev in range(3):
        assert_mean_close(grouped.cpu().numpy()[lev], ref_gs[lev], compute, scale=n_loops // 8,
                          what="level %d group sums" % lev)
    # the levels differ (the estimate is not trivially zero) unless the field is uniform at small T
    assert float((grouped[2] - grouped[1]).abs().max()) > 1e-6


def test_level_N_over_2_is_the_ordinary_run_on_every_other_point(api):
    """the every-other-point sub-loop is an N/2 loop of its own; eq. (49).  For a profile
    served by the same kernel in both calls the bits agree."""
    loops = api.wl_loops_generate(64, 512, 42, torch.float64)
    T, rho = dev(np.geomspace(0.05, 3.0, 6)), dev(np.linspace(0.0, 3.0, 30))
    f = api.wl_field_create(inputs.FLUXTUBE, (2.0, 0.8))
    gs3 = api.wl_eval_discretization(f, loops, T, rho, None, n_groups=4, compute="f64")
    _, gs = api.wl_eval(f, loops[:, 0::2].contiguous(), T, rho, None, n_groups=4, compute="f64")
    torch.cuda.synchronize()
    assert torch.equal(gs3[1], gs)
    # the lean sech^2 kernels serve both calls too (FP32: 64 x 64 grid so that both run 4 grid points per thread)
    fs = api.wl_field_create(inputs.SECH2, (1.0, 1.0))
    c = inputs.config(3)
    T3, rho3, _ = c.grids()
    for compute in ("f64", "f32"):
        gs3 = api.wl_eval_discretization(fs, loops, dev(T3), dev(rho3), None, n_groups=4, compute=compute)
        _, gs = api.wl_eval(fs, loops[:, 0::2].contiguous(), dev(T3), dev(rho3), None, n_groups=4, compute=compute)
        torch.cuda.synchronize()
        assert torch.equal(gs3[1], gs)


def test_extrapolation_and_error_estimate(api, o):
    c = inputs.config(1)
    T, rho, _ = c.grids()
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float64)
    f = api.wl_field_create(c.profile, c.params)
    gs3 = api.wl_eval_discretization(f, loops, dev(T), dev(rho), None, n_groups=c.n_groups, compute="f64")
    gs_inf, _ = api.wl_extrapolate(gs3, want_delta=False)          # eq. (51) on the group sums (linear)
    means = torch.stack([api.wl_jackknife_finalize(gs3[k], c.n_loops)[0] for k in range(3)])
    W_inf, delta = api.wl_extrapolate(means)
    mean_inf, err_inf = api.wl_jackknife_finalize(gs_inf, c.n_loops)
    torch.cuda.synchronize()
    r_inf, r_delta = o.extrapolate(means.cpu().numpy())
    assert np.max(np.abs(W_inf.cpu().numpy() - r_inf)) < 1e-14 * np.abs(r_inf).max()
    assert np.max(np.abs(delta.cpu().numpy() - r_delta)) < 1e-13
    assert float((mean_inf - W_inf).abs().max()) < 1e-12 * float(W_inf.abs().max())   # eq. (51) commutes with the mean
    ref = o.evaluate_discretization(c.profile, c.params, loops.cpu().numpy(), T, rho, None, n_groups=c.n_groups)
    assert_mean_close(gs3.cpu().numpy().sum(1) / c.n_loops, ref.sum(1) / c.n_loops, "f64")
    # eq. (52) is small where the field is weak on the loop's scale and grows with T
    d = delta.cpu().numpy()
    assert d[0].max() < 1e-6 and d[-1].max() > d[0].max()
    assert torch.all(err_inf > 0)


def test_sizes_and_errors(api):
    f = api.wl_field_create(inputs.SECH2, (1.0, 1.0))
    T, rho = dev([1.0]), dev([0.0, 1.0])
    with pytest.raises(api.WLError) as e:
        api.wl_eval_discretization(f, torch.zeros((8, 6, 2), dtype=torch.float64, device="cuda"), T, rho, None, n_groups=2)
    assert e.value.status == 1                                      # N % 4 != 0
    y = api.wl_loops_generate(8, 4, 1, torch.float64)               # N = 4: sub-worldlines of 2, 1, 1 points
    gs3 = api.wl_eval_discretization(f, y, T, rho, None, n_groups=8, compute="f64")
    torch.cuda.synchronize()
    assert torch.all(torch.isfinite(gs3))
    assert api.wl_eval_workspace_bytes(8, 4, 1, 2, 8, "f64") * 3 >= 0
