"""SURVEY.md section 8(f) NEXT-3 on the GPU: effective-action integrals on the group sums (eq. (12), (44)-(47),
(70)) against the oracle (pinned in tests/test_oracle_action.py)."""
import numpy as np
import pytest
import torch

from paper_1407_7486_b200 import inputs
from test_gpu_parity import dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_1407_7486_b200 import api as _api
    return _api


@pytest.fixture(scope="module")
def o():
    from oracle import wl_oracle
    return wl_oracle


@pytest.mark.parametrize("profile,params", [(inputs.SECH2, (1.0, 1.0)), (inputs.FLUXTUBE, (10.0, 1.0)),
                                            (inputs.UNIFORM, (1.5,))])
@pytest.mark.parametrize("scalar", [False, True])
def test_whole_chain_nodes_eval_density_radial_matches_the_oracle(api, o, profile, params, scalar):
    n_loops, N, G = 1024, 256, 16
    a, Tmax, n_T, m2 = 0.05, 1.0, 24, 1.0
    T = api.wl_proper_time_nodes(a, Tmax, n_T)
    assert np.max(np.abs(T / o.proper_time_nodes(a, Tmax, n_T) - 1)) < 1e-15 and T[0] == a
    rho = np.linspace(0.0, 4.0, 17)
    loops = api.wl_loops_generate(n_loops, N, 51, torch.float64)
    f = api.wl_field_create_particle(profile, params, api.SCALAR if scalar else api.FERMION)
    _, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=G, compute="f64")
    dens = api.wl_action_density(f, gs, n_loops, dev(T), dev(rho), m2, a, Tmax)
    act = api.wl_action_radial(dens, dev(rho))
    mean, err = api.wl_jackknife_finalize(dens.reshape(G, 1, len(rho)), G)     # one value per group
    amean, aerr = api.wl_jackknife_finalize(act.reshape(G, 1, 1), G)
    torch.cuda.synchronize()
    # same group sums -> same integrals (the kernels' arithmetic, element by element)
    rd = o.action_density(profile, params, gs.cpu().numpy(), n_loops, T, rho, m2, a, Tmax, scalar=scalar)
    ra = o.action_radial(rd, rho)
    d = dens.cpu().numpy()
    assert np.max(np.abs(d - rd)) < 1e-11 * np.abs(rd).max()
    assert np.max(np.abs(act.cpu().numpy() - ra)) < 1e-11 * np.abs(ra).max()
    # and the whole chain against the oracle's own evaluation of the same loops
    ref = o.evaluate(profile, params, loops.cpu().numpy(), T, rho, None, n_groups=G, scalar=scalar)
    rd2 = o.action_density(profile, params, ref["group_sums"], n_loops, T, rho, m2, a, Tmax, scalar=scalar)
    assert np.max(np.abs(d - rd2)) < 1e-8 * np.abs(rd2).max()          # 1e-9 on <W>, divided by T^3 >= a^3... bounded by e^{-T}
    rm, re = o.finalize(rd[:, None, :], G)
    assert np.max(np.abs(mean.cpu().numpy() - rm)) < 1e-12 * np.abs(rm).max()
    assert np.max(np.abs(err.cpu().numpy() - re)) < 1e-10 * np.abs(re).max()
    assert float(aerr) > 0 and np.isfinite(float(amean))
    if profile == inputs.UNIFORM and not scalar:
        # constant field: density -> int_0^inf of the exact integrand (eq. (42), (44)) within a few sigma
        from scipy import integrate
        b = params[0]
        I = lambda t: np.exp(-m2 * t) / t ** 3 * ((b * t) / np.tanh(b * t) - 1 - (b * t) ** 2 / 3) if b * t > 0.2 \
            else np.exp(-m2 * t) / t ** 3 * (-(b * t) ** 4 / 45 + 2 * (b * t) ** 6 / 945 - (b * t) ** 8 / 4725)
        want, _ = integrate.quad(I, 0, np.inf, limit=400)
        m_, e_ = mean.cpu().numpy()[0], err.cpu().numpy()[0]
        assert np.all(np.abs(m_ - want) < 5 * e_ + 0.02 * abs(want))   # + O(1/N) discretisation bias and Simpson (24 nodes)


def test_action_error_statuses(api):
    f = api.wl_field_create(inputs.SECH2, (1.0, 1.0))
    gs = torch.ones((4, 6, 5), dtype=torch.float64, device="cuda")
    T, rho = dev(api.wl_proper_time_nodes(0.05, 1.0, 6)), dev(np.linspace(0, 1, 5))
    with pytest.raises(api.WLError):
        api.wl_proper_time_nodes(0.05, 1.0, 7)
    with pytest.raises(api.WLError):
        api.wl_action_density(f, gs, 10, T, rho, 1.0, 0.05, 1.0)            # 10 % 4
    with pytest.raises(api.WLError):
        api.wl_action_density(f, gs, 8, T, rho, 1.0, -1.0, 1.0)
    with pytest.raises(api.WLError):
        api.wl_action_radial(torch.ones((4, 4), dtype=torch.float64, device="cuda"), dev(np.linspace(0, 1, 4)))
    d = api.wl_action_density(f, gs, 8, T, rho, 1.0, 0.05, 1.0)
    torch.cuda.synchronize()
    assert torch.all(torch.isfinite(d))
