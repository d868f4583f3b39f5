"""Photon-id sharding across GPUs (one process per GPU) and the one exchange step of the path.

Photons are independent and keyed by their global id, so N GPUs trace disjoint id ranges
of the same field with no data-path collective; the only exchange is the final sum of the int64
tallies, which is exact and order-independent.  Host logic only; works with any torch.distributed
backend (nccl on GPUs, gloo in the CPU tests)."""
import torch
import torch.distributed as dist


def photon_range(rank: int, world: int, n_total: int, first_photon_id: int = 0):
    """Contiguous id range [first, first + count) of `rank` when n_total photons are split over `world`
    ranks (strong scaling); counts differ by at most one and cover the range exactly."""
    if not (0 <= rank < world) or n_total < 0:
        raise ValueError("photon_range: bad rank/world/n_total")
    base, rem = divmod(n_total, world)
    count = base + (1 if rank < rem else 0)
    first = first_photon_id + rank * base + min(rank, rem)
    return first, count


def job_range(rank: int, world: int, job_photons: int):
    """(range_begin, range_count) of `rank` for include/rt.h rt_trace_range: the job's photon INDICES split over
    the ranks.  Every rank passes the same job_photons and first_photon_id, so columns, passes and ids are the
    job's, and the all-reduced integer tallies equal the one-GPU call bit for bit."""
    return photon_range(rank, world, job_photons, 0)


def weak_range(rank: int, world: int, step: int, n_per_gpu: int):
    """Id range of `rank` at `step` when every GPU traces n_per_gpu new photons per step (weak scaling)."""
    return (step * world + rank) * n_per_gpu, n_per_gpu


def allreduce_tallies(tensors, group=None):
    """Sum int64 tally tensors over all ranks in place (exact; a no-op without a process group)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return tensors
    for t in tensors:
        if t is None:
            continue
        if t.dtype != torch.int64:
            raise TypeError("allreduce_tallies: tallies are int64")
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return tensors
