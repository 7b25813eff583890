"""Edge cases, invariants and the boundary's error behaviour on the GPU (through the C ABI)."""
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


@pytest.mark.parametrize("compute", ["f64", "f32"])
@pytest.mark.parametrize("profile,params", [(inputs.UNIFORM, (0.0,)), (inputs.SECH2, (0.0, 0.7))])
def test_zero_field_gives_W_exactly_one(api, compute, profile, params):
    """Pin P1 (north_star): W == 1 exactly, every loop, every grid point, incl. rho_cm = 0 and a
    loop point exactly on the axis (no 0*inf or rsqrt(0) may leak out)."""
    loops = api.wl_loops_generate(48, 64, 3, torch.float64)
    loops[0, 0] = 0.0                                   # a point on the axis when rho_cm = 0
    loops[1] = 0.0                                      # a loop collapsed to the axis
    T = dev([1e-4, 1.0, 50.0])
    rho = dev([0.0, 1e-3, 2.0, 40.0, 1e4])
    f = api.wl_field_create(profile, params)
    W, ph, sp = api.wl_eval_per_loop(f, loops, T, rho, None, compute=compute)
    mean, gs = api.wl_eval(f, loops, T, rho, None, n_groups=4, compute=compute)
    torch.cuda.synchronize()
    assert torch.all(W == 1.0) and torch.all(ph == 0.0) and torch.all(sp == 0.0)
    assert torch.all(mean == 1.0) and torch.all(gs == 12.0)


@pytest.mark.parametrize("compute", ["f64", "f32"])
@pytest.mark.parametrize("n_ppl", [1, 2, 3, 31, 33, 100, 1000, 1025])
def test_ragged_points_per_loop_incl_degenerate(api, o, compute, n_ppl):
    """n_ppl need not be a power of two for wl_eval; N = 1 is a point (phase 0, spin = T b(|x|)),
    N = 2 a segment walked there and back (phase 0)."""
    rng = np.random.default_rng(n_ppl)
    y = rng.normal(size=(12, n_ppl, 2)) * 0.4
    loops = torch.tensor(y, dtype=torch.float64, device="cuda")
    T, rho = np.array([0.05, 1.0, 7.0]), np.array([0.0, 0.3, 1.5, 6.0, 30.0])
    f = api.wl_field_create(inputs.SECH2, (2.0, 0.8))
    W, ph, sp = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), None, compute=compute)
    mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=3, compute=compute)
    torch.cuda.synchronize()
    ref = o.evaluate(o.SECH2, (2.0, 0.8), y, T, rho, None, n_groups=3, per_loop=True)
    tol = 1e-12 if compute == "f64" else 3e-5
    assert np.max(np.abs(ph.cpu().numpy() - ref["phase"]) / np.maximum(1, np.abs(ref["phase"]))) < tol
    assert np.max(np.abs(sp.cpu().numpy() - ref["spin"]) / np.maximum(1, np.abs(ref["spin"]))) < tol
    if n_ppl <= 2:
        assert float(ph.abs().max()) < (1e-15 if compute == "f64" else 1e-6)
    assert_mean_close(mean.cpu().numpy(), ref["W_mean"], compute)


@pytest.mark.parametrize("compute", ["f64", "f32"])
@pytest.mark.parametrize("n_T,n_rho,n_loops,G", [(1, 1, 7, 7), (3, 5, 12, 4), (17, 31, 24, 1), (33, 65, 16, 2),
                                                 (1, 300, 10, 5), (129, 17, 8, 8)])
def test_ragged_grids_and_group_shapes(api, o, compute, n_T, n_rho, n_loops, G):
    """Grids that do not fill a tile of 256 x P grid points, several tiles with a ragged tail,
    G = 1, G = n_loops (one loop per group), with phi_cm given."""
    T = np.geomspace(0.01, 5.0, n_T) if n_T > 1 else np.array([0.7])
    rho = np.linspace(0.0, 3.0, n_rho) if n_rho > 1 else np.array([0.9])
    phi = np.linspace(0.0, 5.0, n_rho)
    loops = api.wl_loops_generate(n_loops, 64, 21, torch.float64)
    f = api.wl_field_create(inputs.SECH2, (1.5, 1.2))
    mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), dev(phi), n_groups=G, compute=compute)
    torch.cuda.synchronize()
    ref = o.evaluate(o.SECH2, (1.5, 1.2), loops.cpu().numpy(), T, rho, phi, n_groups=G)
    assert_mean_close(mean.cpu().numpy(), ref["W_mean"], compute)
    assert_mean_close(gs.cpu().numpy(), ref["group_sums"], compute, scale=n_loops // G, what="group sums")


def test_group_membership_is_bit_exact(api):
    """Reading A6: group g = loops [g N_l/G, (g+1) N_l/G).  Summing the GPU's own per-loop W in
    the documented order (units of consecutive loops, then units in order; the unit size follows
    from wl_eval_workspace_bytes) must reproduce S_g to the last bit; moving one loop across a
    group boundary must not."""
    n_loops, N, G = 96, 128, 6
    T, rho = np.geomspace(0.1, 8.0, 5), np.linspace(0.0, 2.0, 7)
    loops = api.wl_loops_generate(n_loops, N, 5, torch.float64)
    f = api.wl_field_create(inputs.SECH2, (1.0, 1.0))
    for compute in ("f64", "f32"):
        W, _, _ = api.wl_eval_per_loop(f, loops, dev(T), dev(rho), None, compute=compute, want_phase_spin=False)
        mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=G, compute=compute)
        torch.cuda.synchronize()
        W, gs = W.cpu().numpy(), gs.cpu().numpy()
        n_units = api.wl_eval_workspace_bytes(n_loops, N, len(T), len(rho), G, compute) // (8 * len(T) * len(rho))
        lpu = n_loops // n_units
        per_group = n_loops // G
        assert per_group % lpu == 0

        def sums(first_loop_of_group):
            S = np.zeros((G, len(T), len(rho)))
            for g in range(G):
                for u in range(per_group // lpu):
                    part = np.zeros((len(T), len(rho)))
                    for l in range(lpu):
                        part = part + W[first_loop_of_group(g) + u * lpu + l]
                    S[g] = S[g] + part
            return S
        assert np.array_equal(sums(lambda g: g * per_group), gs)
        shifted = sums(lambda g: (g * per_group + 1) % (n_loops - per_group + 1))
        assert not np.array_equal(shifted, gs)
        total = np.zeros_like(gs[0])
        for g in range(G):
            total = total + gs[g]
        assert np.array_equal(total / n_loops, mean.cpu().numpy())           # eq. (61)-(62)


def test_results_do_not_depend_on_loop_window_or_repeat(api):
    """Determinism: the same call twice gives the same bytes; evaluating the two halves of the
    ensemble separately gives the same group sums as the whole (whole groups per call)."""
    c = inputs.config(1)
    T, rho, _ = c.grids()
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float32)
    f = api.wl_field_create(c.profile, c.params)
    for compute in ("f32", "f64"):
        m1, g1 = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=16, compute=compute)
        m2, g2 = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=16, compute=compute)
        _, ga = api.wl_eval(f, loops[:512].contiguous(), dev(T), dev(rho), None, n_groups=8, compute=compute)
        _, gb = api.wl_eval(f, loops[512:].contiguous(), dev(T), dev(rho), None, n_groups=8, compute=compute)
        torch.cuda.synchronize()
        assert torch.equal(m1, m2) and torch.equal(g1, g2)
        assert torch.equal(torch.cat([ga, gb]), g1)


def test_joint_rotation_and_relabelling_invariance(api):
    """Reading A13 / pin P9: rotating x_cm and every loop by the same angle, cyclically relabelling
    the points, or reversing their order leaves every W unchanged (to rounding)."""
    loops = api.wl_loops_generate(32, 256, 8, torch.float64)
    T, rho = dev([0.2, 2.0, 9.0]), dev([0.0, 0.7, 2.5])
    f = api.wl_field_create(inputs.SECH2, (1.3, 0.9))
    W0, _, _ = api.wl_eval_per_loop(f, loops, T, rho, None, compute="f64")
    a = 0.83
    R = torch.tensor([[np.cos(a), np.sin(a)], [-np.sin(a), np.cos(a)]], dtype=torch.float64, device="cuda")
    W1, _, _ = api.wl_eval_per_loop(f, (loops @ R).contiguous(), T, rho, dev([a, a, a]), compute="f64")
    W2, _, _ = api.wl_eval_per_loop(f, torch.roll(loops, 37, dims=1).contiguous(), T, rho, None, compute="f64")
    W3, _, _ = api.wl_eval_per_loop(f, torch.flip(loops, dims=[1]).contiguous(), T, rho, None, compute="f64")
    torch.cuda.synchronize()
    for W in (W1, W2, W3):
        assert float(((W - W0).abs() / W0.abs().clamp(min=1.0)).max()) < 1e-11


def test_sech2_tends_to_uniform_as_lambda_grows(api):
    """Pin P6: lambda -> infinity gives the uniform-field result with eB = eB0, per loop."""
    loops = api.wl_loops_generate(16, 128, 4, torch.float64)
    T, rho = dev([0.5, 3.0]), dev([0.0, 1.0])
    Wu, pu, su = api.wl_eval_per_loop(api.wl_field_create(inputs.UNIFORM, (1.1,)), loops, T, rho, None, compute="f64")
    Ws, ps, ss = api.wl_eval_per_loop(api.wl_field_create(inputs.SECH2, (1.1, 1e4)), loops, T, rho, None, compute="f64")
    torch.cuda.synchronize()
    assert float((pu - ps).abs().max()) < 1e-6 and float((su - ss).abs().max()) < 1e-6


def test_finalize_matches_oracle_and_delete_one_identity(api, o):
    rng = np.random.default_rng(5)
    gs = rng.normal(loc=100.0, scale=3.0, size=(12, 5, 9))
    mean, err, d1 = api.wl_jackknife_finalize(dev(gs), 12 * 50, delete_one=True)
    torch.cuda.synchronize()
    rmean, rerr, rd1 = o.finalize(gs, 12 * 50, delete_one=True)
    assert np.max(np.abs(mean.cpu().numpy() - rmean)) < 1e-13 * 3
    assert np.max(np.abs(err.cpu().numpy() - rerr)) < 1e-13
    assert np.max(np.abs(d1.cpu().numpy() - rd1)) < 1e-13 * 3
    # reading A7: delete-one-group jackknife variance of the mean == eq. (63)^2
    d = d1.cpu().numpy()
    jk = np.sqrt((12 - 1) / 12 * np.sum((d - d.mean(0)) ** 2, axis=0))
    assert np.max(np.abs(jk - err.cpu().numpy())) < 1e-12


def test_host_call_equals_device_call(api):
    c = inputs.config(1)
    T, rho, _ = c.grids()
    loops = api.wl_loops_generate(256, c.n_ppl, c.seed, torch.float32)
    f = api.wl_field_create(c.profile, c.params)
    mean, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=16, compute="f32")
    fm, fe = api.wl_jackknife_finalize(gs, 256)
    torch.cuda.synchronize()
    hm, he, hg = api.wl_eval_host(f, loops.cpu().numpy(), T, rho, None, n_groups=16, compute="f32")
    assert np.array_equal(hm, mean.cpu().numpy()) and np.array_equal(hg, gs.cpu().numpy())
    assert np.array_equal(he, fe.cpu().numpy())
    # a second call reuses the pooled device memory; G = 1 (no error bars, one chunk); FP64 loops with phi
    hm2, _, hg2 = api.wl_eval_host(f, loops.cpu().numpy(), T, rho, None, n_groups=16, compute="f32")
    assert np.array_equal(hm2, hm) and np.array_equal(hg2, hg)
    y64 = loops.double().cpu().numpy()
    phi = np.linspace(0.0, 3.0, len(rho))
    m1, g1 = api.wl_eval(f, loops.double(), dev(T), dev(rho), dev(phi), n_groups=1, compute="f64")
    torch.cuda.synchronize()
    hm3, _, hg3 = api.wl_eval_host(f, y64, T, rho, phi, n_groups=2, compute="f64")
    assert np.array_equal(hg3.sum(0), hg3[0] + hg3[1])
    assert np.max(np.abs(hm3 - m1.cpu().numpy())) < 1e-13 * np.abs(hm3).max()
    api.wl_eval_host_trim()


def test_host_calls_from_two_threads_on_one_device_serialise(api):
    """wl_eval_host shares two streams and a pool per device: concurrent callers on that device take turns
    (one mutex per device) and each gets the result of its own inputs."""
    import threading
    c = inputs.config(1)
    T, rho, _ = c.grids()
    f = api.wl_field_create(c.profile, c.params)
    ys = [api.wl_loops_generate(128, c.n_ppl, seed, torch.float32).cpu().numpy() for seed in (11, 12, 13, 14)]
    want = [api.wl_eval_host(f, y, T, rho, None, n_groups=8, compute="f32") for y in ys]
    got, errors = [None] * len(ys), []

    def work(k):
        try:
            torch.cuda.set_device(0)
            for _ in range(3):
                got[k] = api.wl_eval_host(f, ys[k], T, rho, None, n_groups=8, compute="f32")
        except Exception as exc:                       # surfaced in the main thread below
            errors.append(exc)

    threads = [threading.Thread(target=work, args=(k,)) for k in range(len(ys))]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for (m, e, g), (wm, we, wg) in zip(got, want):
        assert np.array_equal(m, wm) and np.array_equal(e, we) and np.array_equal(g, wg)
    assert not np.array_equal(want[0][0], want[1][0])


def test_error_statuses(api):
    loops = api.wl_loops_generate(8, 16, 1, torch.float64)
    f = api.wl_field_create(inputs.SECH2, (1.0, 1.0))
    T, rho = dev([1.0]), dev([0.0, 1.0])
    with pytest.raises(api.WLError) as e:
        api.wl_eval(f, loops, T, rho, None, n_groups=3, compute="f64")            # 8 % 3
    assert e.value.status == 1
    with pytest.raises(api.WLError) as e:
        api.wl_eval(f, loops, T, rho, None, n_groups=2, compute="f64",
                    workspace=torch.empty(8, dtype=torch.uint8, device="cuda"))
    assert e.value.status == 3
    with pytest.raises(api.WLError):
        api.wl_field_create(inputs.SECH2, (1.0, -1.0))
    with pytest.raises(api.WLError):
        api.wl_jackknife_finalize(torch.zeros((1, 2, 2), dtype=torch.float64, device="cuda"), 8)   # G < 2
    # after the failures the library still works
    mean, _ = api.wl_eval(f, loops, T, rho, None, n_groups=2, compute="f64")
    torch.cuda.synchronize()
    assert torch.all(torch.isfinite(mean))


def test_eval_and_finalize_capture_into_a_cuda_graph(api):
    """include/wl.h: no call except wl_eval_host allocates, copies or synchronises -- so the whole step
    (wl_eval + wl_jackknife_finalize, 4 kernels) can be captured once and replayed as a CUDA graph."""
    c = inputs.config(1)
    T, rho, _ = c.grids()
    loops = api.wl_loops_generate(c.n_loops, c.n_ppl, c.seed, torch.float32)
    f = api.wl_field_create(c.profile, c.params)
    Td, rd = dev(T), dev(rho)
    n_grid = len(T) * len(rho)
    W_mean = torch.empty((len(T), len(rho)), dtype=torch.float64, device="cuda")
    gs = torch.empty((c.n_groups, len(T), len(rho)), dtype=torch.float64, device="cuda")
    ws = torch.empty(api.wl_eval_workspace_bytes(c.n_loops, c.n_ppl, len(T), len(rho), c.n_groups, "f32"),
                     dtype=torch.uint8, device="cuda")
    ref_mean, ref_gs = api.wl_eval(f, loops, Td, rd, None, n_groups=c.n_groups, compute="f32")
    ref_fm, ref_err = api.wl_jackknife_finalize(ref_gs, c.n_loops)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            api.wl_eval(f, loops, Td, rd, None, n_groups=c.n_groups, compute="f32", W_mean=W_mean, group_sums=gs,
                        workspace=ws, stream=side)
            fm, err = api.wl_jackknife_finalize(gs, c.n_loops, stream=side)
    W_mean.zero_()
    gs.zero_()
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(W_mean, ref_mean) and torch.equal(gs, ref_gs)
    assert torch.equal(fm, ref_fm) and torch.equal(err, ref_err)
    assert n_grid == 256
