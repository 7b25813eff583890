"""SURVEY.md section 8(f) NEXT-1 on the GPU: the paper's flux-tube profile (eq. (68)) and
the scalar-QED output W = cos(phase), against the oracle, same tolerances as
tests/test_gpu_parity.py."""
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


# Fig. 11 / 12 parameters of the paper: script-F = 10, lambda = 1 and 10, plus a narrow tube
@pytest.mark.parametrize("compute", ["f64", "f32"])
@pytest.mark.parametrize("F,lam", [(10.0, 1.0), (10.0, 10.0), (0.5, 0.1)])
@pytest.mark.parametrize("with_phi", [False, True])
def test_fluxtube_parity_per_loop_and_reduced(api, o, compute, F, lam, with_phi):
    n_loops, N, G = 192, 512, 6
    T = np.geomspace(0.01, min(5.0, 3.0 / (2.0 * F / lam ** 2)), 9)     # eB(0) T <= 3
    rho = np.linspace(0.0, 4.0 * lam, 33)
    phi = np.linspace(0.0, 6.0, 33) if with_phi else None
    loops = api.wl_loops_generate(n_loops, N, 31, torch.float32)
    f = api.wl_field_create(inputs.FLUXTUBE, (F, lam))
    W, ph, sp = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), dev(phi), compute=compute)
    mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), dev(phi), n_groups=G, compute=compute)
    torch.cuda.synchronize()
    ref = o.evaluate(o.FLUXTUBE, (F, lam), loops.cpu().numpy(), T, rho, phi, n_groups=G, per_loop=True)
    tol = 1e-12 if compute == "f64" else 2e-5
    assert np.max(np.abs(ph.cpu().numpy() - ref["phase"]) / np.maximum(1, np.abs(ref["phase"]))) < tol
    assert np.max(np.abs(sp.cpu().numpy() - ref["spin"]) / np.maximum(1, np.abs(ref["spin"]))) < tol
    wtol = 1e-10 if compute == "f64" else 2e-3
    assert np.max(np.abs(W.cpu().numpy() - ref["W"]) / np.maximum(1, np.abs(ref["W"]))) < wtol
    assert_mean_close(mean.cpu().numpy(), ref["W_mean"], compute)
    assert_mean_close(gs.cpu().numpy(), ref["group_sums"], compute, scale=n_loops // G, what="group sums")


@pytest.mark.parametrize("compute", ["f64", "f32"])
@pytest.mark.parametrize("profile,params", [(inputs.SECH2, (1.0, 1.0)), (inputs.FLUXTUBE, (10.0, 1.0)),
                                            (inputs.UNIFORM, (1.0,))])
def test_scalar_output_parity(api, o, compute, profile, params):
    n_loops, N, G = 256, 256, 8
    T, rho = np.geomspace(0.01, 6.0, 12), np.linspace(0.0, 3.0, 40)
    loops = api.wl_loops_generate(n_loops, N, 32, torch.float64)
    fs = api.wl_field_create_particle(profile, params, api.SCALAR)
    ff = api.wl_field_create_particle(profile, params, api.FERMION)
    Ws, phs, _ = api.wl_eval_per_loop(fs, loops, dev(T), dev(rho), None, compute=compute)
    Wf, phf, spf = api.wl_eval_per_loop(ff, loops, dev(T), dev(rho), None, compute=compute)
    mean, gs = api.wl_eval(fs, loops, dev(T), dev(rho), None, n_groups=G, compute=compute)
    torch.cuda.synchronize()
    assert torch.equal(phs, phf)                                         # same phase, other combine step
    assert torch.equal(Ws, torch.cos(phs))
    assert float((Wf - Ws * torch.cosh(spf)).abs().max()) < 1e-12 * float(Wf.abs().max())
    assert float(Ws.abs().max()) <= 1.0
    ref = o.evaluate(profile, params, loops.cpu().numpy(), T, rho, None, n_groups=G, scalar=True)
    assert_mean_close(mean.cpu().numpy(), ref["W_mean"], compute)
    assert_mean_close(gs.cpu().numpy(), ref["group_sums"], compute, scale=n_loops // G, what="group sums")


def test_scalar_uniform_field_eq43_at_config2_size(api):
    """eq. (43), at finite N: <cos(eBT A)>_N = prod_k [1 + (x cot(pi k/N)/N)^2]^(-1/2)
    (pinned for the oracle in tests/test_oracle_fluxtube_scalar.py); config-2 ensemble, GPU only."""
    c = inputs.config(2)
    T, rho, phi = c.grids()
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float64)
    f = api.wl_field_create_particle(c.profile, c.params, api.SCALAR)
    _, gs = api.wl_eval(f, loops, dev(T), dev(rho), dev(phi), n_groups=c.n_groups, compute="f64")
    mean, err = api.wl_jackknife_finalize(gs, c.n_loops)
    torch.cuda.synchronize()
    mean, err = mean.cpu().numpy(), err.cpu().numpy()
    k = np.arange(1, c.n_ppl)
    for t in range(0, c.n_T, 3):
        x = c.params[0] * T[t]
        exact = np.prod(1.0 / np.sqrt(1.0 + (x / (c.n_ppl * np.tan(np.pi * k / c.n_ppl))) ** 2))
        assert abs(mean[t, 0] - exact) < 5.0 * err[t, 0] + 1e-9
        assert abs(exact - x / np.sinh(x)) < 0.02 * exact              # and that is eq. (43) up to O(1/N)


def test_fluxtube_field_validation(api):
    with pytest.raises(api.WLError):
        api.wl_field_create(inputs.FLUXTUBE, (1.0,))
    with pytest.raises(api.WLError):
        api.wl_field_create(inputs.FLUXTUBE, (1.0, 0.0))
    with pytest.raises(api.WLError):
        api.wl_field_create_particle(inputs.SECH2, (1.0, 1.0), 7)
