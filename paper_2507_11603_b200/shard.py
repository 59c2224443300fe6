"""Photon-id sharding across ranks: the only multi-GPU logic the path needs.

Packets are independent and the RNG is keyed on (seed, photon id), so rank r of R walks the id range
[offset_r, offset_r + count_r) on its own replica of the grid and the integer / fixed-point tallies are summed with
one all-reduce; the result is bit-identical to the one-rank run.  No method arithmetic lives here.
"""


def shard_range(n_photons, rank, world):
    """Contiguous split of [0, n_photons) into `world` ranges whose sizes differ by at most one.
    Returns (offset, count) for `rank`."""
    if not (0 <= rank < world) or n_photons < 0:
        raise ValueError("bad rank / world / n_photons")
    base, rem = divmod(int(n_photons), int(world))
    count = base + (1 if rank < rem else 0)
    offset = rank * base + min(rank, rem)
    return offset, count


def allreduce_tallies(tensors, group=None):
    """Sums integer tally tensors (spectrum, scattering-count histogram, counters, fixed-point cube) over the ranks of
    a torch.distributed process group, in place.  Integer sums are order-independent: every rank ends with the
    tallies of the whole run."""
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return tensors
    for t in tensors:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return tensors
