"""Multi-GPU sharding of the Wilson-loop path: whole jackknife groups per rank.

Loops are independent and a group sum S_g (eq. (60)) only needs the
loops of group g, so rank r of R owns groups [r G/R, (r+1) G/R) and with them the contiguous loops
[r N_l/R, (r+1) N_l/R) of the ensemble.  Each rank runs the ordinary single-GPU `wl_eval` on its
loops; the only exchange is ONE all-gather of the local group sums [G/R][n_T][n_rho] (FP64, <= 2 MB
per rank at config 3), after which every rank runs the same fixed-order `wl_jackknife_finalize` on
the full [G][n_T][n_rho].  The bits of every S_g, of <W> and of the error are therefore the same for
any number of ranks (an all-reduce of <W> would make them depend on the reduction tree).

This module holds host logic only: index arithmetic and the torch.distributed call.  It works with
any backend (nccl for CUDA tensors; gloo for the CPU tests of tests/test_shard_gloo.py).
"""
from dataclasses import dataclass

import torch
import torch.distributed as dist


@dataclass(frozen=True)
class Shard:
    rank: int
    world_size: int
    loop_begin: int      # first loop of the ensemble this rank owns
    n_loops: int         # loops this rank owns
    group_begin: int     # first jackknife group this rank owns
    n_groups: int        # groups this rank owns


def shard_groups(n_loops: int, n_groups: int, world_size: int, rank: int) -> Shard:
    """Rank `rank`'s share of an ensemble of n_loops loops in n_groups equal groups."""
    if world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("bad rank / world_size")
    if n_groups < 1 or n_loops < 1 or n_loops % n_groups != 0:
        raise ValueError("n_loops must be a positive multiple of n_groups (equal groups, PAPER.md:388)")
    if n_groups % world_size != 0:
        raise ValueError("n_groups (%d) must be a multiple of the number of ranks (%d): ranks own whole groups"
                         % (n_groups, world_size))
    g_local = n_groups // world_size
    per_group = n_loops // n_groups
    return Shard(rank, world_size, rank * g_local * per_group, g_local * per_group, rank * g_local, g_local)


def all_gather_group_sums(local_group_sums: torch.Tensor, world_size: int, group=None) -> torch.Tensor:
    """[G/R][n_T][n_rho] on every rank -> [G][n_T][n_rho] on every rank, rank-major (= group order)."""
    if local_group_sums.dtype != torch.float64 or local_group_sums.dim() != 3:
        raise ValueError("local_group_sums must be float64 [G_local][n_T][n_rho]")
    local = local_group_sums.contiguous()
    g_local = local.shape[0]
    out = torch.empty((world_size * g_local,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    if world_size == 1 and not (dist.is_available() and dist.is_initialized()):
        out.copy_(local)
        return out
    if local.is_cuda and dist.get_backend(group) == "gloo":
        # gloo has no all_gather for CUDA tensors: stage through the host (<= 2 MB per rank); same values, same order
        host = torch.empty(out.shape, dtype=out.dtype)
        dist.all_gather([host[r * g_local:(r + 1) * g_local] for r in range(world_size)], local.cpu(), group=group)
        out.copy_(host)
        return out
    parts = [out[r * g_local:(r + 1) * g_local] for r in range(world_size)]
    dist.all_gather(parts, local, group=group)
    return out


def wl_eval_sharded(field, local_loops, T, rho_cm, phi_cm, shard: Shard, compute, stream=None, group=None,
                    workspace=None, options=None):
    """wl_eval on this rank's loops, all-gather of the group sums, finalise on every rank.

    local_loops: this rank's loops [shard.n_loops][n_ppl][2] (CUDA).  Returns (mean, err, group_sums)
    for the WHOLE ensemble, identical on every rank.  n_groups_total >= 2.
    """
    from . import api
    if local_loops.shape[0] != shard.n_loops:
        raise ValueError("local_loops has %d loops, the shard owns %d" % (local_loops.shape[0], shard.n_loops))
    # the units of loops are those of one call over the whole ensemble: same bits for any number of ranks
    opt = api._own_options(options)                    # a copy: the caller's block keeps ensemble_loops = 0
    opt.ensemble_loops = shard.n_loops * shard.world_size
    _, gs_local = api.wl_eval(field, local_loops, T, rho_cm, phi_cm, n_groups=shard.n_groups, compute=compute,
                              stream=stream, workspace=workspace, options=opt)
    gs = all_gather_group_sums(gs_local, shard.world_size, group=group)
    mean, err = api.wl_jackknife_finalize(gs, shard.n_loops * shard.world_size, stream=stream)
    return mean, err, gs
