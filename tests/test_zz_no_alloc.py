"""wl_eval_static: the evaluation for callers that are not allowed to allocate device memory.

Who needs it: a program whose own pool took all of HBM at start-up (a later cudaMalloc fails), or a plug-in /
callback running where its host application forbids cudaMalloc and cudaFree because they stall every stream of
the device.  Such a caller owns input and output buffers and nothing else, so the partial sums that wl_eval keeps
in a caller-allocated workspace sit instead in a fixed 16 MiB array inside libwl.so (include/wl.h).

What is checked: on the same inputs the entry point returns what the existing path (wl_eval with a workspace)
returns -- the same kernels in the same order, so the same bits, which is inside every tolerance the other GPU
tests use -- on two calls in a row that share the array (the second on a different, smaller problem, so stale
contents of the first would show), that the device's free memory does not move across a call, and that sizes
over the limit are refused with their own status before anything runs.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It has no fixtures shared with other files and passes alone in a fresh process as well as after
the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

WL_ERR_STATIC_LIMIT = 5


def _problem(api, inputs, torch, config, n_loops, n_T, n_rho, n_groups, seed):
    c = inputs.config(config)
    T, rho, phi = c.grids()
    T, rho = T[:n_T], rho[:n_rho]
    phi = None if phi is None else phi[:n_rho]
    dev = lambda a: None if a is None else torch.tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")
    field = api.wl_field_create(c.profile, c.params)
    loops = api.wl_loops_generate(n_loops, c.n_ppl, seed, torch.float64)
    return field, loops, dev(T), dev(rho), dev(phi), n_groups


@pytest.mark.gpu
@pytest.mark.parametrize("compute", ["f64", "f32"])
def test_static_scratch_entry_point_matches_wl_eval_on_two_calls_in_a_row(compute):
    import torch
    from paper_1407_7486_b200 import api, inputs

    torch.cuda.set_device(0)
    # call 1: config 1 as BASELINE.json states it (2 MiB of partial sums); call 2: a smaller, ragged problem
    # (uniform field on the circle of config 2: phi_cm given, 5 x 7 grid) that reuses the front of the array
    problems = [_problem(api, inputs, torch, 1, 1024, 16, 16, 16, seed=1),
                _problem(api, inputs, torch, 2, 96, 5, 7, 8, seed=2)]
    expected = []
    for field, loops, T, rho, phi, G in problems:               # the existing path, workspace from the caller
        mean, gs = api.wl_eval(field, loops, T, rho, phi, n_groups=G, compute=compute)
        expected.append((mean.clone(), gs.clone()))
    outs = [(torch.full_like(m, float("nan")), torch.full_like(g, float("nan"))) for m, g in expected]
    torch.cuda.synchronize()

    free_before = None
    for k, ((field, loops, T, rho, phi, G), (mean, gs)) in enumerate(zip(problems, outs)):
        if k == 1:                                              # set-up (address look-up, module load) is behind us
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
        api.wl_eval_static(field, loops, T, rho, phi, G, compute, mean, gs)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before          # the second call took no device memory

    for (mean, gs), (ref_mean, ref_gs) in zip(outs, expected):
        assert torch.isfinite(mean).all() and torch.isfinite(gs).all()
        assert torch.equal(gs, ref_gs)                          # S_g, eq. (60): same order of summation, same bits
        assert torch.equal(mean, ref_mean)                      # <W>, eq. (61)-(62)


def test_limit_is_checked_on_the_host_before_any_cuda_call():
    """No GPU needed: the refusal comes from the sizes alone, so the (never dereferenced) pointers can be dummies."""
    from paper_1407_7486_b200 import build
    lib = C.CDLL(build.build())
    lib.wl_eval_static_max_bytes.restype = C.c_size_t
    lib.wl_eval_workspace_bytes.restype = C.c_size_t
    lib.wl_eval_workspace_bytes.argtypes = [C.c_int64] + [C.c_int] * 5
    lib.wl_field_create.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_void_p)]
    vp = C.c_void_p
    lib.wl_eval_static.argtypes = [vp, vp, C.c_int, C.c_int64, C.c_int, vp, C.c_int, vp, vp, C.c_int, C.c_int, C.c_int,
                                   vp, vp, vp]
    limit = lib.wl_eval_static_max_bytes()
    assert limit == 16 << 20
    field = vp()
    assert lib.wl_field_create(1, (C.c_double * 2)(1.0, 1.0), 2, C.byref(field)) == 0
    dummy = vp(256)
    assert lib.wl_eval_workspace_bytes(4096, 64, 32, 32, 32, 1) > limit
    assert lib.wl_eval_static(field, dummy, 0, 4096, 64, dummy, 32, dummy, None, 32, 32, 1, dummy, dummy, None) \
        == WL_ERR_STATIC_LIMIT
    assert lib.wl_eval_static(field, dummy, 0, 100, 64, dummy, 4, dummy, None, 4, 3, 1, dummy, dummy, None) == 1
    assert lib.wl_eval_static(field, None, 0, 1024, 256, dummy, 16, dummy, None, 16, 16, 1, dummy, dummy, None) == 1
    lib.wl_status_string.restype = C.c_char_p
    assert b"wl_eval_static" in lib.wl_status_string(WL_ERR_STATIC_LIMIT)
    lib.wl_field_destroy.argtypes = [vp]
    lib.wl_field_destroy(field)


@pytest.mark.gpu
def test_static_scratch_entry_point_refuses_what_does_not_fit():
    import torch
    from paper_1407_7486_b200 import api, inputs

    torch.cuda.set_device(0)
    limit = api.wl_eval_static_max_bytes()
    assert limit == 16 << 20
    assert api.wl_eval_workspace_bytes(1024, 256, 16, 16, 16, "f64") <= limit     # config 1 fits
    # 4096 loops on a 32 x 32 grid need 32 MiB of partial sums: refused, and the outputs are left alone
    n_loops, n_T, n_rho, G = 4096, 32, 32, 32
    assert api.wl_eval_workspace_bytes(n_loops, 64, n_T, n_rho, G, "f64") > limit
    c = inputs.config(1)
    field = api.wl_field_create(c.profile, c.params)
    loops = api.wl_loops_generate(n_loops, 64, 7, torch.float32)
    T = torch.linspace(0.1, 1.0, n_T, dtype=torch.float64, device="cuda")
    rho = torch.linspace(0.0, 2.0, n_rho, dtype=torch.float64, device="cuda")
    mean = torch.full((n_T, n_rho), -7.0, dtype=torch.float64, device="cuda")
    gs = torch.full((G, n_T, n_rho), -7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(api.WLError) as err:
        api.wl_eval_static(field, loops, T, rho, None, G, "f64", mean, gs)
    assert err.value.status == WL_ERR_STATIC_LIMIT
    assert "wl_eval_static" in str(err.value)
    torch.cuda.synchronize()
    assert bool((mean == -7.0).all()) and bool((gs == -7.0).all())
    # sizes wl_eval itself refuses keep wl_eval's status (unequal groups)
    with pytest.raises(api.WLError) as err:
        api.wl_eval_static(field, loops[:100], T[:4], rho[:4], None, 3, "f64", mean[:4, :4].contiguous(),
                           gs[:3, :4, :4].contiguous())
    assert err.value.status == 1
