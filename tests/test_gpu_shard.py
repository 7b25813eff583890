"""The sharded CUDA path (Sec. V: four GPUs): `shard.wl_eval_sharded` run by TWO
ranks (gloo process group, both on cuda:0 -- their kernels are independent, nothing waits on another rank), each
on its own `loop_begin` window of one ensemble.  The gathered [G][T][rho], mean and error must be BIT-IDENTICAL to
one unsharded wl_eval + wl_jackknife_finalize, and within the north_star tolerance of the oracle.  Also runs
bench.py under torch.distributed.run with one rank so that its NCCL control flow (init, all-gather, barriers,
MAX over ranks, rank-0 print, destroy) executes on the GPU box.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch

from paper_1407_7486_b200 import inputs
from test_gpu_parity import assert_mean_close, dev

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

# (name, profile, params, n_loops, N, seed, storage, compute, G, T, rho)
def _cases():
    c1 = inputs.config(1)
    T1, r1, _ = c1.grids()
    c3 = inputs.config(3)
    T3, r3, _ = c3.grids()
    return [
        ("cfg1_f64", c1.profile, c1.params, c1.n_loops, c1.n_ppl, c1.seed, "f64", "f64", c1.n_groups, T1, r1),
        ("cfg1_f32", c1.profile, c1.params, c1.n_loops, c1.n_ppl, c1.seed, "f64", "f32", c1.n_groups, T1, r1),
        # a 2048-loop slice of config 3 (full grid, N = 2048, FP32 storage and kernel), 8 groups of 256
        ("cfg3_slice", c3.profile, c3.params, 2048, c3.n_ppl, c3.seed, "f32", "f32", 8, T3, r3),
        # sizes at which a shard ALONE would be cut into other units than the whole ensemble (units of 2 loops
        # for 8192 loops on 4 tiles, single loops for 4096): wl_eval_options.ensemble_loops keeps the bits equal
        ("unit_plan", c3.profile, c3.params, 8192, 16, 9, "f32", "f32", 8, T3, r3),
    ]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, outdir):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from paper_1407_7486_b200 import api, shard
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        for (name, profile, params, n_loops, N, seed, storage, compute, G, T, rho) in _cases():
            sh = shard.shard_groups(n_loops, G, world, rank)
            sdt = torch.float64 if storage == "f64" else torch.float32
            loops = api.wl_loops_generate(sh.n_loops, N, seed, sdt, loop_begin=sh.loop_begin)
            f = api.wl_field_create(profile, params)
            mean, err, gs = shard.wl_eval_sharded(f, loops, dev(T), dev(rho), None, sh, compute)
            torch.cuda.synchronize()
            np.savez(os.path.join(outdir, "%s_rank%d.npz" % (name, rank)), mean=mean.cpu().numpy(),
                     err=err.cpu().numpy(), gs=gs.cpu().numpy())
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_are_bit_identical_to_one(tmp_path):
    import torch.multiprocessing as mp
    from oracle import wl_oracle as o
    from paper_1407_7486_b200 import api
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    for (name, profile, params, n_loops, N, seed, storage, compute, G, T, rho) in _cases():
        sdt = torch.float64 if storage == "f64" else torch.float32
        loops = api.wl_loops_generate(n_loops, N, seed, sdt)
        f = api.wl_field_create(profile, params)
        _, gs = api.wl_eval(f, loops, dev(T), dev(rho), None, n_groups=G, compute=compute)
        mean, err = api.wl_jackknife_finalize(gs, n_loops)
        torch.cuda.synchronize()
        r0 = np.load(os.path.join(str(tmp_path), "%s_rank0.npz" % name))
        r1 = np.load(os.path.join(str(tmp_path), "%s_rank1.npz" % name))
        for key, want in (("gs", gs), ("mean", mean), ("err", err)):
            assert np.array_equal(r0[key], r1[key]), (name, key)                    # every rank holds the same result
            assert np.array_equal(r0[key], want.cpu().numpy()), (name, key)         # and it is the unsharded one, bit for bit
        if name != "unit_plan":
            ti = np.array([0, len(T) // 3, len(T) - 1])
            ri = np.array([0, len(rho) // 2, len(rho) - 1])
            ref = o.evaluate(profile, params, loops.cpu().numpy(), T[ti], rho[ri], None, n_groups=G)
            assert_mean_close(r0["mean"][np.ix_(ti, ri)], ref["W_mean"], compute)
            assert_mean_close(r0["gs"][:, ti][:, :, ri], ref["group_sums"], compute, scale=n_loops // G, what="group sums")
            rm, rerr = o.finalize(ref["group_sums"], n_loops)
            assert np.allclose(r0["err"][np.ix_(ti, ri)], rerr, rtol=2e-3, atol=1e-7)


def test_a_shard_alone_would_be_cut_differently(tmp_path):
    """The case above is not vacuous: without ensemble_loops the 4096-loop shard uses other units of loops."""
    from paper_1407_7486_b200 import api
    whole = api.wl_eval_opt_workspace_bytes(8192, 16, 64, 64, 8, "f32")
    alone = api.wl_eval_opt_workspace_bytes(4096, 16, 64, 64, 4, "f32")
    with_ens = api.wl_eval_opt_workspace_bytes(4096, 16, 64, 64, 4, "f32", api.wl_eval_options(ensemble_loops=8192))
    assert alone == 4096 * 4096 * 8 and whole == 4096 * 4096 * 8 and with_ens == 2048 * 4096 * 8


def test_bench_under_torchrun_one_rank():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "1", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", "1", "--steps", "2", "--warmup", "3",
           "--workload", "1", "--no-cpu-baseline"]
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                  # rank 0 prints ONE line
    d = json.loads(lines[0])
    assert d["n_gpus"] == 1 and d["value"] > 0 and d["e2e"]["value"] > 0 and d["gpu_launches"] > 0
    assert d["roofline"]["frac"] > 0 and np.isfinite(d["checksum_sum_W_mean"])
