"""The N>1 path on CPU: world_size-2 `gloo` run of the host-side sharding logic
(paper_1407_7486_b200/shard.py): whole jackknife groups per rank, one all-gather of the group
sums, the same finalise on every rank.  The per-rank evaluation is done here by the ORACLE
(there is no GPU in this container); what is under test is the index arithmetic, the
generator's loop_begin windows, the gather layout and that the result is bit-identical to
the unsharded one (eq. (60)-(63))."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

N_LOOPS, N_PPL, G, SEED = 64, 32, 8, 9
PARAMS = (1.0, 1.0)
T = np.array([0.1, 1.0, 4.0])
RHO = np.array([0.0, 0.5, 2.0, 3.0])


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    from oracle import wl_oracle as o
    # shard.py is host logic; import it without importing api.py (which needs libwl.so + CUDA tensors)
    from paper_1407_7486_b200.shard import all_gather_group_sums, shard_groups
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        sh = shard_groups(N_LOOPS, G, world, rank)
        loops = o.generate_loops(SEED, sh.n_loops, N_PPL, loop_begin=sh.loop_begin)
        res = o.evaluate(o.SECH2, PARAMS, loops, T, RHO, None, n_groups=sh.n_groups)
        gs = all_gather_group_sums(torch.from_numpy(res["group_sums"]), world)
        np.save(os.path.join(out_dir, "gs_rank%d.npy" % rank), gs.numpy())
    finally:
        dist.destroy_process_group()


def test_shard_plan_covers_the_ensemble_by_whole_groups():
    from paper_1407_7486_b200.shard import shard_groups
    for (nl, g, w) in ((16384, 64, 1), (16384, 64, 2), (16384, 64, 8), (65536, 256, 4), (12, 4, 2)):
        shards = [shard_groups(nl, g, w, r) for r in range(w)]
        assert shards[0].loop_begin == 0 and shards[0].group_begin == 0
        for a, b in zip(shards, shards[1:]):
            assert a.loop_begin + a.n_loops == b.loop_begin
            assert a.group_begin + a.n_groups == b.group_begin
        assert shards[-1].loop_begin + shards[-1].n_loops == nl
        assert shards[-1].group_begin + shards[-1].n_groups == g
        for s in shards:
            assert s.n_loops == s.n_groups * (nl // g)            # whole groups only
            assert s.loop_begin == s.group_begin * (nl // g)
    with pytest.raises(ValueError):
        shard_groups(16384, 64, 3, 0)        # 64 groups do not split over 3 ranks
    with pytest.raises(ValueError):
        shard_groups(10, 3, 1, 0)            # unequal groups
    with pytest.raises(ValueError):
        shard_groups(16, 4, 2, 2)            # rank out of range


def test_world_size_2_gloo_matches_the_unsharded_result_bit_for_bit(tmp_path):
    from oracle import wl_oracle as o
    world = 2
    port = _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    gs0 = np.load(tmp_path / "gs_rank0.npy")
    gs1 = np.load(tmp_path / "gs_rank1.npy")
    assert gs0.shape == (G, len(T), len(RHO))
    assert np.array_equal(gs0, gs1)                               # every rank holds the same bits
    loops = o.generate_loops(SEED, N_LOOPS, N_PPL)
    ref = o.evaluate(o.SECH2, PARAMS, loops, T, RHO, None, n_groups=G)
    assert np.array_equal(gs0, ref["group_sums"])                 # and they are the unsharded ones
    mean, err = o.finalize(gs0, N_LOOPS)
    mean_ref, err_ref = o.finalize(ref["group_sums"], N_LOOPS)
    assert np.array_equal(mean, mean_ref) and np.array_equal(err, err_ref)
    assert np.array_equal(mean, ref["W_mean"])


def test_all_gather_world_size_1_is_a_copy():
    from paper_1407_7486_b200.shard import all_gather_group_sums
    x = torch.arange(24, dtype=torch.float64).reshape(2, 3, 4)
    y = all_gather_group_sums(x, 1)
    assert torch.equal(x, y) and y.data_ptr() != x.data_ptr()
    with pytest.raises(ValueError):
        all_gather_group_sums(x.float(), 1)
