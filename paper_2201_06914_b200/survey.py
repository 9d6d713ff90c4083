"""Survey loop over independent shots ("44 ... common receiver gathers", L77, L85 "stack out"):
shot partition across ranks, in-place image stacking on each GPU (rtm_adjoint_image accumulate=1), one
sum-reduce of the stacked image at the end.  Shots are independent, so there is NO data-path collective
inside a shot ("replicas only"); the final all-reduce is bookkeeping over N floats."""
from __future__ import annotations


def partition_shots(nshots: int, world: int, rank: int) -> range:
    """Contiguous, balanced block of shot indices for `rank` (sizes differ by at most one)."""
    if nshots < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("bad partition arguments")
    base, extra = divmod(nshots, world)
    start = rank * base + min(rank, extra)
    return range(start, start + base + (1 if rank < extra else 0))


def stack_across_ranks(image, group=None):
    """Sum the per-rank stacked images (in place).  No-op without an initialised process group."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(image, op=dist.ReduceOp.SUM, group=group)
    return image


def max_over_ranks(value: float, device=None, group=None) -> float:
    """Max over ranks of a scalar (device timings are reported as the slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def migrate_shots(rtm, shots, image, rank: int = 0, world: int = 1):
    """Run this rank's share of `shots` (objects with src_xyz, wav, rec_xyz, data_in) through one Rtm
    context, stacking into `image` (a device tensor shaped like the physical grid)."""
    mine = partition_shots(len(shots), world, rank)
    for i in mine:
        s = shots[i]
        rtm.forward_probe(s.src_xyz, s.wav, s.rec_xyz, data_out=None)
        rtm.adjoint_image(s.rec_xyz, s.data_in, s.src_xyz, image=image, accumulate=True)
    return len(mine)
