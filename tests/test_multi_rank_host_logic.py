"""Host logic of the N > 1 path on CPU: two gloo ranks shard one job by history
ranges with paper_1503_01722_b200.sharding (the code bench.py --gpus N runs), one all-reduce of the
per-batch grids, then the batch statistics.  The per-rank transport stand-in is the oracle (there is
no GPU here); the result must equal the single-process run of the whole job."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as tmp

from paper_1503_01722_b200 import sharding
from paper_1503_01722_b200 import workloads as W


def test_history_ranges_are_disjoint_and_cover():
    n = 1000
    seen = []
    for r in range(4):
        nj, a, b = sharding.history_range(r, 4, n)
        assert nj == 4000 and b - a == n
        seen += list(range(a, b, 250))
    assert sorted(seen) == list(range(0, 4000, 250))
    with pytest.raises(ValueError):
        sharding.history_range(0, 8, 2 ** 29)  # 2^32 histories do not fit the 32-bit history index
    with pytest.raises(ValueError):
        sharding.history_range(4, 4, 10)
    for n_job, world in [(10, 3), (7, 8), (0, 2), (2 ** 32 - 1, 8)]:
        parts = sharding.split_job(n_job, world)
        assert parts[0][0] == 0 and parts[-1][1] == n_job
        assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
        sizes = [b - a for a, b in parts]
        assert max(sizes) - min(sizes) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, n_per_rank, B, out_dir):
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = W.config(1)
    orc = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])

    def run_range(n_job, h0, h1):
        e, _ = orc.run_edep(cfg["beam"], n_job, 5, B, h0, h1)
        return torch.from_numpy(e)

    def finalize(g, n_job):
        return orc.finalize(g.numpy(), n_job)

    dose, sig = sharding.run_sharded(rank, world, n_per_rank, run_range, dist.all_reduce, finalize)
    np.save(os.path.join(out_dir, f"dose{rank}.npy"), dose)
    np.save(os.path.join(out_dir, f"sig{rank}.npy"), sig)
    dist.destroy_process_group()


def test_two_gloo_ranks_reproduce_the_single_process_job(tmp_path):
    import oracle
    world, n_per_rank, B = 2, 300, 6
    tmp.spawn(_rank_main, args=(world, _free_port(), n_per_rank, B, str(tmp_path)), nprocs=world, join=True)
    cfg = W.config(1)
    orc = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    d_ref, s_ref, _ = orc.run(cfg["beam"], world * n_per_rank, 5, B)
    for r in range(world):  # every rank holds the full result after the all-reduce
        d = np.load(tmp_path / f"dose{r}.npy")
        s = np.load(tmp_path / f"sig{r}.npy")
        assert np.allclose(d, d_ref, rtol=1e-12, atol=1e-18)
        assert np.allclose(s, s_ref, rtol=1e-9, atol=1e-18)
    assert d_ref.max() > 0


def test_voxel_slices_are_equal_chunks_that_cover():
    for nvox, world in [(10, 3), (8000, 8), (7, 8), (223260, 2), (1, 1)]:
        got = []
        for r in range(world):
            chunk, a, b = sharding.voxel_slice(r, world, nvox)
            assert chunk * world >= nvox and 0 <= a <= b <= nvox and b - a <= chunk
            got += list(range(a, b))
        assert got == list(range(nvox))
    with pytest.raises(ValueError):
        sharding.voxel_slice(2, 2, 10)


def _peer_rank_main(rank, world, port, n_per_rank, B, out_dir, fail_rank):
    """The fused-exchange call order of bench.py --gpus N with stand-ins: the oracle transports, 'peer memory' is an
    all-gather of the grids, the slice statistics are the oracle's.  fail_rank >= 0: that rank cannot map its peers."""
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = W.config(1)
    orc = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    nvox = orc.nvox
    own = {}

    def all_min(v):
        t = torch.tensor([v])
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
        return int(t.item())
    use_peer = sharding.agree_on_peer_exchange(rank != fail_rank, all_min)

    def run_range(n_job, h0, h1):
        own["e"] = torch.from_numpy(orc.run_edep(cfg["beam"], n_job, 5, B, h0, h1)[0])
        return own["e"]

    if use_peer:
        def finalize_slice(n_job, v0, v1):
            grids = [torch.empty_like(own["e"]) for _ in range(world)]
            dist.all_gather(grids, own["e"])  # stand-in for reading the peers' grids in place
            d, s = orc.finalize(sum(grids).numpy(), n_job)
            return torch.from_numpy(d[v0:v1].copy()), torch.from_numpy(s[v0:v1].copy())

        def all_gather(t, chunk):
            pad = torch.zeros(chunk, dtype=t.dtype); pad[:len(t)] = t
            parts = [torch.empty(chunk, dtype=t.dtype) for _ in range(world)]
            dist.all_gather(parts, pad)
            return torch.cat(parts)
        dose, sig = sharding.run_sharded_peer(rank, world, n_per_rank, nvox, run_range, dist.barrier, finalize_slice, all_gather)
        dose, sig = dose.numpy(), sig.numpy()
    else:
        dose, sig = sharding.run_sharded(rank, world, n_per_rank, run_range, dist.all_reduce, lambda g, nj: orc.finalize(g.numpy(), nj))
    np.save(os.path.join(out_dir, f"dose{rank}.npy"), dose)
    np.save(os.path.join(out_dir, f"sig{rank}.npy"), sig)
    with open(os.path.join(out_dir, f"mode{rank}.txt"), "w") as f:
        f.write("peer" if use_peer else "allreduce")
    dist.destroy_process_group()


@pytest.mark.parametrize("fail_rank", [-1, 1])
def test_sliced_peer_exchange_and_joint_fallback_reproduce_the_single_process_job(tmp_path, fail_rank):
    import oracle
    world, n_per_rank, B = 2, 300, 6
    tmp.spawn(_peer_rank_main, args=(world, _free_port(), n_per_rank, B, str(tmp_path), fail_rank), nprocs=world, join=True)
    cfg = W.config(1)
    orc = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    d_ref, s_ref, _ = orc.run(cfg["beam"], world * n_per_rank, 5, B)
    modes = {open(tmp_path / f"mode{r}.txt").read() for r in range(world)}
    assert modes == ({"peer"} if fail_rank < 0 else {"allreduce"})  # all ranks take the same path
    for r in range(world):
        assert np.allclose(np.load(tmp_path / f"dose{r}.npy"), d_ref, rtol=1e-12, atol=1e-18)
        assert np.allclose(np.load(tmp_path / f"sig{r}.npy"), s_ref, rtol=1e-9, atol=1e-18)
