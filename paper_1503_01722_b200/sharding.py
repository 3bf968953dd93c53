"""Host logic of the multi-GPU path.

Histories are independent and keyed by their index, so the job shards by contiguous history ranges with
no data-path collective: rank r transports histories [r*n, (r+1)*n) of one job of n*world histories into
its own per-batch grids; ONE exchange (sum of the B x nvox grids over ranks) precedes the batch
statistics.  This module holds only the index arithmetic and the call order; the transport, the
reduction and the statistics are passed in (engine + NCCL in bench.py; any stand-in + gloo in the CPU
tests), so the same code is exercised with and without GPUs.
"""
from __future__ import annotations


def history_range(rank: int, world: int, n_per_rank: int):
    """(n_job, h_begin, h_end) of `rank` under weak scaling: every rank owns n_per_rank histories."""
    if not (0 <= rank < world) or n_per_rank <= 0:
        raise ValueError("rank / world / n_per_rank")
    n_job = n_per_rank * world
    if n_job >= 2 ** 32:
        raise ValueError("job too large: n_per_rank * world must be < 2^32 (history index is 32-bit)")
    return n_job, rank * n_per_rank, (rank + 1) * n_per_rank


def split_job(n_job: int, world: int):
    """Strong-scaling split of a fixed job: contiguous, disjoint, covering ranges (sizes differ by <= 1)."""
    if world <= 0 or n_job < 0:
        raise ValueError("world / n_job")
    base, rem = divmod(n_job, world)
    out, h = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((h, h + n))
        h += n
    return out


def run_sharded(rank, world, n_per_rank, run_range, all_reduce_sum, finalize):
    """One step of the sharded job on this rank.

    run_range(n_job, h_begin, h_end) -> this rank's per-batch energy grids (left where they were computed)
    all_reduce_sum(grids)            -> in-place sum over ranks (skipped when world == 1)
    finalize(grids, n_job)           -> (dose, sigma)
    """
    n_job, h0, h1 = history_range(rank, world, n_per_rank)
    grids = run_range(n_job, h0, h1)
    if world > 1:
        all_reduce_sum(grids)
    return finalize(grids, n_job)


def voxel_slice(rank: int, world: int, nvox: int):
    """(chunk, v_begin, v_end): rank r finalizes voxels [r*chunk, min((r+1)*chunk, nvox)), chunk = ceil(nvox / world) — equal
    chunks so that the slices can be all-gathered into one padded buffer of world * chunk entries."""
    if not (0 <= rank < world) or nvox <= 0:
        raise ValueError("rank / world / nvox")
    chunk = -(-nvox // world)
    return chunk, min(rank * chunk, nvox), min((rank + 1) * chunk, nvox)


def agree_on_peer_exchange(ok_here: bool, all_reduce_min) -> bool:
    """The fused (peer-memory) exchange is used only if EVERY rank could map every peer: all_reduce_min(int) -> int is the
    collective minimum over ranks.  One failing rank sends all ranks to the all-reduce fallback together."""
    return bool(all_reduce_min(1 if ok_here else 0))


def run_sharded_peer(rank, world, n_per_rank, nvox, run_range_in_place, barrier, finalize_slice, all_gather):
    """One step of the sharded job with the fused exchange, sliced by voxel.

    run_range_in_place(n_job, h_begin, h_end)   transport into this rank's exported grid buffer
    barrier()                                    all ranks (host barrier: no kernel waits on another rank)
    finalize_slice(n_job, v_begin, v_end)        -> (dose_slice, sigma_slice) of the SUM of all ranks' grids, read in place
    all_gather(slice_padded_to_chunk, chunk)     -> concatenation over ranks (world * chunk entries)
    Returns (dose[nvox], sigma[nvox]) on every rank.
    """
    n_job, h0, h1 = history_range(rank, world, n_per_rank)
    chunk, v0, v1 = voxel_slice(rank, world, nvox)
    run_range_in_place(n_job, h0, h1)
    barrier()                      # every rank's grids are complete
    d, s = finalize_slice(n_job, v0, v1)
    barrier()                      # nobody overwrites its grids while a peer still reads them
    return all_gather(d, chunk)[:nvox], all_gather(s, chunk)[:nvox]
