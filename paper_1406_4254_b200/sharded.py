"""Sharded SCF over several GPUs, one process per GPU ("each particle's contribution to
the coefficients is completely independent of all other particles", :221 partial coefficients + MPI_Allreduce).

Every rank holds a contiguous shard of the particles.  One exchange: the ranks' coefficient tables (2T doubles, 4.9-22 KB) are
all-gathered and added in rank order (etics_scf_combine), so every rank ends with bit-identical A, B; each rank then evaluates
its own shard.  torch.distributed is the plumbing (NCCL on GPUs); all arithmetic is in the kernels behind the binding.
MEX does not shard by particle index and stays single-GPU.
"""
from __future__ import annotations


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Particles [first, last) of `rank`: contiguous, sizes differ by at most one, every particle in exactly one shard."""
    if not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(n, world)
    first = rank * base + min(rank, extra)
    return first, first + base + (1 if rank < extra else 0)


def gather_and_combine(local_table, all_gather, combine):
    """local_table: this rank's [A | B]; all_gather(t) -> the ranks' tables stacked in rank order; combine(stack) -> their sum
    in that order.  Split out so that the exchange logic can be exercised on CPU (gloo) with stand-in callables."""
    return combine(all_gather(local_table))


def scf_force_sharded(pos_shard, mass_shard, nmax: int, lmax: int, group=None, workspace=None):
    """SCF full force calculation of a particle set spread over the ranks of `group`.  pos_shard (3, n_r), mass_shard (n_r,)
    CUDA fp64 -> (A, B, acc_shard, pot_shard); A, B are the coefficients of the WHOLE set, identical on every rank."""
    import torch
    import torch.distributed as dist

    from . import binding as E

    T = (nmax + 1) * E.num_lm(lmax)
    local = torch.empty(2 * T, dtype=torch.float64, device=pos_shard.device)
    E.etics_scf_coeffs(pos_shard, mass_shard, nmax, lmax, local[:T], local[T:], workspace)

    def all_gather(t):
        world = dist.get_world_size(group)
        stack = torch.empty((world, t.numel()), dtype=t.dtype, device=t.device)
        dist.all_gather_into_tensor(stack, t, group=group)
        return stack

    table = gather_and_combine(local, all_gather, E.etics_scf_combine)
    A, B = table[:T], table[T:]
    acc, pot = E.etics_scf_force(pos_shard, nmax, lmax, A, B)
    return A, B, acc, pot
