"""Sharded SCF over several GPUs, one process per GPU ("each particle's contribution to
the coefficients is completely independent of all other particles", :221 partial coefficients + MPI_Allreduce).

Every rank holds a contiguous shard of the particles.  One exchange: the ranks' coefficient tables (2T doubles, 4.9-22 KB) are
all-gathered and added in rank order (etics_scf_combine), so every rank ends with bit-identical A, B; each rank then evaluates
its own shard.  torch.distributed is the plumbing (NCCL on GPUs); all arithmetic is in the kernels behind the binding.

MEX does not shard by particle index ("the contribution of each particle depends on its position in a sorted list
(by radius)", :421 "easy for SCF but not so much for MEX"): it is RADIUS-partitioned.  Every rank sorts its
index shard, the ranks agree on world-1 splitter keys from a sample, every particle moves to the rank that owns its key range
(one all-to-all of 32-byte records), each rank runs the MEX sequence on its range — with the cumulative sums of eqs. (11)-(12)
started from the moment totals of the ranks inside / outside (one all-gather of R doubles per rank) — and the results travel
back to the particles' owners.  Only integer key comparisons and data movement happen here; the keys, moments, scans and forces
come from the kernels (etics_mex_sort, etics_mex_shard_moments / _bases / _force).
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


# ---- radius-partitioned MEX ----------------------------------------------------------------------------------------------
SAMPLES_PER_RANK = 64


def _all_gather_rows(t, group=None):
    """The ranks' equally sized 1-D tensors stacked in rank order, (world, len).  (Concatenated output form: the one both the
    NCCL and the gloo backend accept.)"""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    flat = torch.empty(world * t.numel(), dtype=t.dtype, device=t.device)
    dist.all_gather_into_tensor(flat, t.contiguous().reshape(-1), group=group)
    return flat.reshape(world, t.numel())


def sample_positions(n: int, samples: int = SAMPLES_PER_RANK) -> list[int]:
    """`samples` evenly spaced positions of a sorted list of n >= 1 keys (the mid-points of `samples` equal slices)."""
    if n < 1:
        raise ValueError("every rank needs at least one particle")
    return [((2 * j + 1) * n) // (2 * samples) for j in range(samples)]


def choose_splitters(all_samples, world: int):
    """all_samples: the ranks' samples (any shape, world * S int64 keys) -> world-1 splitter keys, the same on every rank:
    the k S-th smallest sample, k = 1 .. world-1.  Rank k owns the keys in [splitter[k-1], splitter[k])."""
    import torch
    flat, _ = torch.sort(all_samples.reshape(-1))
    per = flat.numel() // world
    return flat[per::per][: world - 1].contiguous()


def send_counts(keys_sorted, splitters) -> list[int]:
    """How many of this rank's ascending keys go to each rank: keys < splitter[0] to rank 0, ..., keys >= splitter[-1] to the
    last.  Equal keys always land on ONE rank (the tie-break by particle index is then a local matter)."""
    import torch
    n = keys_sorted.numel()
    cut = torch.searchsorted(keys_sorted, splitters, right=False).tolist() if splitters.numel() else []
    edges = [0] + cut + [n]
    return [edges[k + 1] - edges[k] for k in range(len(edges) - 1)]


class RadiusExchange:
    """The all-to-all plan of one radius partition: forward (records to the owners of the key ranges) and back (results to the
    owners of the particles).  Rows travel in this rank's SORTED order; a receiver sees source 0's rows, then source 1's, ...:
    inside one key the rows are ordered by (source rank, index in the source's shard) = by global particle index when the
    ranks hold contiguous index ranges in rank order (shard_range), which is the tie-break MEX needs (reading G8)."""

    def __init__(self, keys_sorted, perm, group=None, samples: int = SAMPLES_PER_RANK):
        import torch
        import torch.distributed as dist
        self.group, self.perm = group, perm.long()
        world = dist.get_world_size(group)
        mine = keys_sorted[torch.tensor(sample_positions(keys_sorted.numel(), samples), device=keys_sorted.device)]
        self.splitters = choose_splitters(_all_gather_rows(mine, group), world)
        self.send = send_counts(keys_sorted, self.splitters)
        got = torch.empty(world, dtype=torch.int64, device=keys_sorted.device)
        dist.all_to_all_single(got, torch.tensor(self.send, dtype=torch.int64, device=keys_sorted.device), group=group)
        self.recv = got.tolist()

    def forward(self, rows):
        """rows (n_local, k) in ORIGINAL local order -> (n_range, k): the rows of this rank's key range."""
        import torch
        import torch.distributed as dist
        out = torch.empty((sum(self.recv),) + tuple(rows.shape[1:]), dtype=rows.dtype, device=rows.device)
        dist.all_to_all_single(out, rows[self.perm].contiguous(), output_split_sizes=self.recv, input_split_sizes=self.send,
                               group=self.group)
        return out

    def back(self, rows):
        """rows (n_range, k), in the order forward() delivered -> (n_local, k) in ORIGINAL local order."""
        import torch
        import torch.distributed as dist
        got = torch.empty((sum(self.send),) + tuple(rows.shape[1:]), dtype=rows.dtype, device=rows.device)
        dist.all_to_all_single(got, rows.contiguous(), output_split_sizes=self.send, input_split_sizes=self.recv,
                               group=self.group)
        out = torch.empty_like(got)
        out[self.perm] = got
        return out


def mex_force_partitioned(pos_shard, mass_shard, sort, moments, bases, force, group=None):
    """The exchange logic of the radius-partitioned MEX with the four compute steps passed in (the kernels on a GPU; stand-ins
    in the CPU tests):  sort(pos) -> (keys_sorted, perm);  moments(pos_r, mass_r) -> (totals (R,), state);
    bases(parts (world, R), rank) -> base (R,);  force(state, base) -> (acc_r (3, n_r), pot_r (n_r,)).
    pos_shard (3, n), mass_shard (n,) are this rank's contiguous index shard -> (acc (3, n), pot (n,)) in the same order."""
    import torch
    import torch.distributed as dist
    rank = dist.get_rank(group)
    keys_sorted, perm = sort(pos_shard)
    ex = RadiusExchange(keys_sorted, perm, group)
    rec = ex.forward(torch.cat([pos_shard.t(), mass_shard[:, None]], dim=1))      # (n_r, 4): x, y, z, m
    pos_r, mass_r = rec[:, :3].t().contiguous(), rec[:, 3].contiguous()
    n_r = mass_r.numel()
    totals, state = moments(pos_r, mass_r)          # n_r == 0: a zero vector and no state
    parts = _all_gather_rows(totals, group)
    if n_r:
        acc_r, pot_r = force(state, bases(parts, rank))
        res = torch.cat([acc_r.t(), pot_r[:, None]], dim=1)
    else:
        res = torch.empty((0, 4), dtype=pos_shard.dtype, device=pos_shard.device)
    out = ex.back(res)
    return out[:, :3].t().contiguous(), out[:, 3].contiguous()


def mex_force_sharded(pos_shard, mass_shard, lmax: int, group=None):
    """MEX full force calculation of a particle set spread over the ranks of `group` (contiguous index shards in rank order,
    shard_range).  pos_shard (3, n_r), mass_shard (n_r,) CUDA fp64 -> (acc_shard, pot_shard)."""
    import torch

    from . import binding as E

    R = E.etics_mex_shard_rows(lmax)

    def sort(pos):
        return E.etics_mex_sort(pos)

    def moments(pos_r, mass_r):
        n = mass_r.numel()
        if n == 0:
            return torch.zeros(R, dtype=torch.float64, device=pos_r.device), None
        ws = torch.empty(E.etics_workspace_bytes(E.ETICS_WS_MEX_FORCE, n, 0, lmax), dtype=torch.uint8, device=pos_r.device)
        return E.etics_mex_shard_moments(pos_r, mass_r, lmax, ws), (n, ws)

    def bases(parts, rank):
        return E.etics_mex_shard_bases(parts, rank, lmax)

    def force(state, base):
        n, ws = state
        return E.etics_mex_shard_force(n, lmax, E.ETICS_WHAT_BOTH, base, ws)

    return mex_force_partitioned(pos_shard, mass_shard, sort, moments, bases, force, group)
