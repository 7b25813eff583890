"""Every shared-memory staging path of k_wilson in one small run, FP32 and FP64.

The three places where a data race would be silent: the two-slot
cp.async.bulk ring with its re-issue after the second barrier (wl_wilson_body.cuh), the seeded path's reuse of
yraw across dloop_begin / dloop_chunk (wl_dloop_device.cuh), and the bounding-box slots written during staging and
read after the barrier (wl_block_bounds.cuh).  The run is sized so that each is exercised more than once per CTA
(N = 2048: two or four chunks per loop; two loops per ring; a 32 x 32 grid, i.e. the 256-thread, P = 4 / P = 2
kernels that the bulk variant is compiled for) and small enough for compute-sanitizer:

    compute-sanitizer --tool memcheck|racecheck|synccheck python -m pytest tests/test_gpu_staging_paths.py -q

(profiles/r03_sanitizer.md: the tool is closed on this GPU pool, so what stands in is this test's own evidence: every
path repeated with bit-identical results, and three differently staged paths agreeing bit for bit).  It checks what
must hold between the paths:
same bits for default / bulk / seeded staging, level N of the discretisation estimate equal to the plain
evaluation, shuffled groups summing to the same total.
"""
import numpy as np
import pytest
import torch

from paper_1407_7486_b200 import inputs

pytestmark = pytest.mark.gpu

N_LOOPS, N_PPL, N_T, N_RHO, G, SEED = 32, 2048, 32, 32, 4, 77


def dev(a):
    return None if a is None else torch.tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")


@pytest.mark.parametrize("compute", ["f32", "f64"])
@pytest.mark.parametrize("profile,params", [(inputs.SECH2, (1.0, 1.0)), (inputs.FLUXTUBE, (10.0, 1.0)),
                                            (inputs.UNIFORM, (1.0,))])
def test_all_staging_paths_agree(profile, params, compute):
    from paper_1407_7486_b200 import api
    T = dev(np.geomspace(0.01, 10.0, N_T))
    rho = dev(np.linspace(0.0, 4.0, N_RHO))
    sdt = torch.float32 if compute == "f32" else torch.float64
    f = api.wl_field_create(profile, params)
    loops = api.wl_loops_generate(N_LOOPS, N_PPL, SEED, sdt)

    m0, g0 = api.wl_eval(f, loops, T, rho, None, n_groups=G, compute=compute)                     # (i) default staging
    m1, g1 = api.wl_eval(f, loops, T, rho, None, n_groups=G, compute=compute,
                         options=api.wl_eval_options(staging=1))                                  # (ii) bulk ring
    m2, g2 = api.wl_eval_seeded(f, SEED, N_LOOPS, N_PPL, T, rho, None, n_groups=G, compute=compute,
                                storage=sdt)                                                      # (iii) seeded
    gs3 = api.wl_eval_discretization(f, loops, T, rho, None, n_groups=G, compute=compute)         # (iv) three levels
    m4, g4 = api.wl_eval(f, loops, T, rho, None, n_groups=G, compute=compute,
                         options=api.wl_eval_options(shuffle_seed=5))                             # (v) shuffled groups
    torch.cuda.synchronize()

    assert torch.isfinite(g0).all()
    # a race in any of the three places would show as bits that change from run to run: every path three more times
    for _ in range(3):
        ra = api.wl_eval(f, loops, T, rho, None, n_groups=G, compute=compute)[1]
        rb = api.wl_eval(f, loops, T, rho, None, n_groups=G, compute=compute, options=api.wl_eval_options(staging=1))[1]
        rc = api.wl_eval_seeded(f, SEED, N_LOOPS, N_PPL, T, rho, None, n_groups=G, compute=compute, storage=sdt)[1]
        rd = api.wl_eval_discretization(f, loops, T, rho, None, n_groups=G, compute=compute)
        torch.cuda.synchronize()
        assert torch.equal(ra, g0) and torch.equal(rb, g0) and torch.equal(rc, g0) and torch.equal(rd, gs3)
    assert torch.equal(g0, g1) and torch.equal(m0, m1)            # same staged values, same walk order: same bits
    assert torch.equal(g0, g2) and torch.equal(m0, m2)
    # the three levels of eq. (48)-(50) are sums over stride-2 / stride-4 sub-worldlines, not the plain N-point sum:
    # their parity is tests/test_gpu_discretization.py's business, here they only have to be finite
    assert torch.isfinite(gs3).all()
    # shuffling moves loops between groups, not out of the ensemble (eq. (61)-(62))
    tot0, tot4 = g0.sum(0), g4.sum(0)
    assert float((tot0 - tot4).abs().max()) <= 1e-12 * float(tot0.abs().max()) * N_LOOPS
    assert float((m0 - m4).abs().max()) <= 1e-12 * float(m0.abs().max())
