"""Parity of the CUDA path (through the C ABI, paper_1407_7486_b200.api) against the FP64 CPU
oracle, element by element, on identical loop coordinates.

Tolerances (BASELINE.json north_star):
  FP64 kernel : |d<W>| <= 1e-9 * max(1, |<W>|)                         (reading A9)
  FP32 kernel : |d<W>| <= 2e-4 where |<W>| <= 1, <= 1e-3 |<W>| where |<W>| > 1
  group sums  : the same bounds times the loops per group
  jackknife group membership: bit-exact (integer division only, reading A6)
Loops are generated ON THE GPU by wl_loops_generate and copied to the host for the oracle
(reading A11: the CPU twin agrees to ~1e-15, but parity must not depend on that).
"""
import numpy as np
import pytest
import torch

from paper_1407_7486_b200 import inputs

pytestmark = pytest.mark.gpu

F64_RTOL = 1e-9
F32_ATOL = 2e-4
F32_RTOL = 1e-3


@pytest.fixture(scope="module")
def api():
    from paper_1407_7486_b200 import api as _api     # raises if libwl.so is missing: no fallback
    return _api


@pytest.fixture(scope="module")
def o():
    from oracle import wl_oracle
    return wl_oracle


def dev(a):
    return torch.tensor(np.asarray(a), dtype=torch.float64, device="cuda") if a is not None else None


def tdtype(name):
    return torch.float64 if name == "f64" else torch.float32


def assert_mean_close(got, ref, compute, scale=1.0, what="<W>"):
    """north_star tolerance; `scale` = loops per group when comparing group sums."""
    got, ref = np.asarray(got), np.asarray(ref)
    assert got.shape == ref.shape
    assert np.all(np.isfinite(got)), what + " has non-finite entries"
    mag = np.abs(ref) / scale
    if compute == "f64":
        bound = F64_RTOL * np.maximum(1.0, mag) * scale
    else:
        bound = np.where(mag > 1.0, F32_RTOL * mag, F32_ATOL) * scale
    err = np.abs(got - ref)
    k = np.unravel_index(np.argmax(err / bound), err.shape)
    assert np.all(err <= bound), "%s (%s): |err| %.3e > bound %.3e at %s (ref %.6e)" % (
        what, compute, err[k], bound[k], k, ref[k])


def run_gpu(api, cfg, loops, T, rho, phi, G, compute):
    f = api.wl_field_create(cfg.profile, cfg.params)
    mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), dev(phi), n_groups=G, compute=compute)
    fmean, err = api.wl_jackknife_finalize(gs, loops.shape[0]) if G >= 2 else (mean, None)
    torch.cuda.synchronize()
    return mean.cpu().numpy(), gs.cpu().numpy(), fmean.cpu().numpy(), (err.cpu().numpy() if err is not None else None)


# --------------------------------------------------------------------------- generator (a0)

def test_generator_matches_the_oracle_twin(api, o):
    for (n, N, seed) in ((64, 256, 1), (5, 2, 7), (3, 8192, 4), (33, 1024, 2), (3, 16384, 5), (2, 65536, 11), (7, 4, 6)):
        y = api.wl_loops_generate(n, N, seed, torch.float64)
        torch.cuda.synchronize()
        ref = o.generate_loops(seed, n, N)
        assert np.max(np.abs(y.cpu().numpy() - ref)) < 1e-12
        y32 = api.wl_loops_generate(n, N, seed, torch.float32).cpu().numpy()
        assert y32.dtype == np.float32
        assert np.max(np.abs(y32 - ref)) < 2e-7 * max(1.0, np.abs(ref).max())


def test_generator_windows_and_determinism(api):
    a = api.wl_loops_generate(40, 128, 11, torch.float64)
    b = api.wl_loops_generate(40, 128, 11, torch.float64)
    c = api.wl_loops_generate(7, 128, 11, torch.float64, loop_begin=30)
    d = api.wl_loops_generate(40, 128, 12, torch.float64)
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    assert torch.equal(a[30:37], c)                  # loop l is a function of (seed, l) only
    assert not torch.equal(a, d)
    assert float(a.mean(1).abs().max()) < 1e-15      # step (5)
    e = api.wl_loops_generate(0, 128, 11, torch.float64)
    assert e.shape == (0, 128, 2)
    with pytest.raises(api.WLError):
        api.wl_loops_generate(4, 100, 1, torch.float64)


# --------------------------------------------------------------------------- configs 1 and 2: full size, every element

def test_config1_full_fp64_every_element(api, o):
    c = inputs.config(1)
    T, rho, phi = c.grids()
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float64)
    mean, gs, fmean, err = run_gpu(api, c, loops, T, rho, phi, c.n_groups, "f64")
    ref = o.evaluate(c.profile, c.params, loops.cpu().numpy(), T, rho, phi, n_groups=c.n_groups)
    assert_mean_close(mean, ref["W_mean"], "f64")
    assert_mean_close(gs, ref["group_sums"], "f64", scale=c.n_loops // c.n_groups, what="group sums")
    rmean, rerr = o.finalize(ref["group_sums"], c.n_loops)
    assert_mean_close(fmean, rmean, "f64")
    assert np.max(np.abs(err - rerr)) <= 1e-9 * max(1.0, rerr.max())
    # FP32 kernel on the same FP64 loops
    mean32, gs32, _, _ = run_gpu(api, c, loops, T, rho, phi, c.n_groups, "f32")
    assert_mean_close(mean32, ref["W_mean"], "f32")
    assert_mean_close(gs32, ref["group_sums"], "f32", scale=c.n_loops // c.n_groups, what="group sums")


@pytest.mark.parametrize("compute", ["f64", "f32"])
def test_config2_full_uniform_field(api, o, compute):
    c = inputs.config(2)
    T, rho, phi = c.grids()
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, tdtype(c.loop_dtype))
    mean, gs, fmean, err = run_gpu(api, c, loops, T, rho, phi, c.n_groups, compute)
    y = loops.cpu().numpy()
    ref = o.evaluate(c.profile, c.params, y, T, rho, phi, n_groups=c.n_groups)
    assert_mean_close(mean, ref["W_mean"], compute)
    assert_mean_close(gs, ref["group_sums"], compute, scale=c.n_loops // c.n_groups, what="group sums")
    # rotation invariance (reading A13): in a uniform field W does not depend on x_cm
    spread = np.max(np.abs(mean - mean[:, :1]) / np.maximum(1.0, np.abs(mean[:, :1])))
    assert spread < (1e-11 if compute == "f64" else 1e-4)
    # eq. (42), at finite N (pin P3 of tests/test_oracle_ensemble.py): within 5 jackknife sigma
    k = np.arange(1, c.n_ppl)
    for t in range(0, c.n_T, 5):
        x = c.params[0] * T[t]
        exact = np.cosh(x) * np.prod(1.0 / np.sqrt(1.0 + (x / (c.n_ppl * np.tan(np.pi * k / c.n_ppl))) ** 2))
        assert abs(fmean[t, 0] - exact) < 5.0 * err[t, 0] + 1e-6


def test_config2_phase_is_eB_T_times_shoelace_area(api):
    """eq. (19)-(20): the phase is e x flux; for uniform B the discretised phase
    is eB T x the polygon area of the unit loop, for any x_cm (pin P2, here on the GPU output)."""
    c = inputs.config(2)
    T, rho, phi = c.grids()
    loops = api.wl_loops_generate(256, c.n_ppl, c.seed, torch.float64)
    f = api.wl_field_create(c.profile, c.params)
    W, ph, sp = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), dev(phi), compute="f64")
    y = loops.cpu().numpy()
    yn = np.roll(y, -1, axis=1)
    area = 0.5 * np.sum(y[:, :, 0] * yn[:, :, 1] - y[:, :, 1] * yn[:, :, 0], axis=1)
    want = c.params[0] * T[None, :, None] * area[:, None, None]
    got = ph.cpu().numpy()
    assert np.max(np.abs(got - want)) < 1e-11 * max(1.0, np.abs(want).max())
    assert np.max(np.abs(sp.cpu().numpy() - c.params[0] * T[None, :, None])) < 1e-13 * T.max()


# --------------------------------------------------------------------------- reduced-size element-wise parity incl. per-loop values

CASES = [
    # (config, n_loops, grid stride, compute, loop storage)
    (1, 1024, 1, "f64", "f64"),
    (1, 1024, 1, "f32", "f32"),
    (2, 512, 1, "f64", "f64"),
    (2, 512, 1, "f32", "f32"),
    (3, 256, 4, "f32", "f32"),
    (3, 256, 4, "f64", "f32"),
    (4, 128, 8, "f32", "f32"),
    (4, 128, 8, "f64", "f32"),
    (5, 256, 4, "f32", "f32"),
]


@pytest.mark.parametrize("ci,n_loops,stride,compute,storage", CASES)
def test_per_loop_phase_spin_and_W(api, o, ci, n_loops, stride, compute, storage):
    c = inputs.config(ci)
    T, rho, phi = c.grids()
    T, rho = T[::stride], rho[::stride]
    phi = phi[::stride] if phi is not None else None
    G = c.n_groups if n_loops % c.n_groups == 0 else 4
    loops = api.wl_loops_generate(n_loops, c.n_ppl, c.seed, tdtype(storage))
    f = api.wl_field_create(c.profile, c.params)
    W, ph, sp = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), dev(phi), compute=compute)
    mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), dev(phi), n_groups=G, compute=compute)
    torch.cuda.synchronize()
    ref = o.evaluate(c.profile, c.params, loops.cpu().numpy(), T, rho, phi, n_groups=G, per_loop=True)
    W, ph, sp = W.cpu().numpy(), ph.cpu().numpy(), sp.cpu().numpy()
    # per-term arithmetic: FP64 ~ N eps; FP32 ~ sqrt(N) 6e-8 relative to the sum's scale
    tol = 1e-12 if compute == "f64" else 2e-5
    assert np.max(np.abs(ph - ref["phase"]) / np.maximum(1.0, np.abs(ref["phase"]))) < tol
    assert np.max(np.abs(sp - ref["spin"]) / np.maximum(1.0, np.abs(ref["spin"]))) < tol
    wtol = 1e-10 if compute == "f64" else 2e-3
    assert np.max(np.abs(W - ref["W"]) / np.maximum(1.0, np.abs(ref["W"]))) < wtol
    assert_mean_close(mean.cpu().numpy(), ref["W_mean"], compute)
    assert_mean_close(gs.cpu().numpy(), ref["group_sums"], compute, scale=n_loops // G, what="group sums")
