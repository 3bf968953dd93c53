"""Fused exchange + statistics of the sharded job: mc_finalize_multi reads the
ranks' per-batch grids in place (a peer's over NVLink) instead of all-reduce + mc_finalize.  The box has one GPU, so the
two ranks of the second test share it and exchange their grids through CUDA IPC — the same code path as two GPUs,
minus the link.  No kernel waits on another rank: the ranks meet at host barriers only."""
import os
import socket

import numpy as np
import pytest

import paper_1503_01722_b200 as mc
from paper_1503_01722_b200 import sharding
from paper_1503_01722_b200 import workloads as W

pytestmark = pytest.mark.gpu


def test_finalize_multi_equals_finalize_of_the_sum():
    import torch
    assert torch.cuda.is_available()
    cfg = W.config(1)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    n, B = 60000, 6
    parts = sharding.split_job(n, 3)
    grids = []
    for a, b in parts:
        g = torch.zeros(B * eng.nvox, dtype=torch.float32, device="cuda")
        mc.mc_run_range(eng.ctx, cfg["beam"], n, a, b, 3, B, g)
        grids.append(g)
    d1 = torch.zeros(eng.nvox, device="cuda"); s1 = torch.zeros_like(d1)
    mc.mc_finalize_multi(eng.ctx, grids, n, B, d1, s1)
    total = grids[0] + grids[1] + grids[2]
    d0 = torch.zeros_like(d1); s0 = torch.zeros_like(d1)
    mc.mc_finalize(eng.ctx, total, n, B, d0, s0)
    assert torch.allclose(d1, d0, rtol=1e-6, atol=0) and d0.max() > 0
    assert torch.allclose(s1, s0, rtol=1e-4, atol=1e-7 * float(d0.max()))
    # and equals the unsharded run up to fp32 summation order
    dr, sr = eng.run(cfg["beam"], n, 3, B)
    assert np.allclose(d1.cpu().numpy(), dr, rtol=2e-5, atol=1e-7 * dr.max())
    # the context's own buffer can receive a shard without a copy
    p = mc.mc_edep_buffer(eng.ctx, B)
    mc.mc_run_range(eng.ctx, cfg["beam"], n, 0, n, 3, B, p)
    mc.mc_finalize_multi(eng.ctx, [p], n, B, d1, s1)
    assert np.allclose(d1.cpu().numpy(), dr, rtol=2e-5, atol=1e-7 * dr.max())
    with pytest.raises(mc.McError):
        mc.mc_finalize_multi(eng.ctx, [p] * 17, n, B, d1, s1)
    eng.close()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, n_per_rank, B, out_dir):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(rank % torch.cuda.device_count())
    cfg = W.config(4, "e")
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    n_job, h0, h1 = sharding.history_range(rank, world, n_per_rank)
    own = mc.mc_edep_buffer(eng.ctx, B)
    mc.mc_run_range(eng.ctx, cfg["beam"], n_job, h0, h1, 5, B, own)  # shard stays in the context's buffer
    handles = [None] * world
    dist.all_gather_object(handles, mc.mc_ipc_get_handle(own))      # also the barrier: every shard is finished
    peers = [own if r == rank else mc.mc_ipc_open_handle(handles[r]) for r in range(world)]
    dose, sig = np.zeros(eng.nvox, np.float32), np.zeros(eng.nvox, np.float32)
    mc.mc_finalize_multi(eng.ctx, peers, n_job, B, dose, sig)
    # the sliced form bench.py --gpus N uses: this rank's voxel slice of the sum, then an all-gather of the slices
    chunk, v0, v1 = sharding.voxel_slice(rank, world, eng.nvox)
    ds, ss = np.zeros(chunk, np.float32), np.zeros(chunk, np.float32)
    mc.mc_finalize_multi_range(eng.ctx, peers, n_job, B, v0, v1, ds, ss)
    parts = [torch.empty(chunk) for _ in range(world)]
    dist.all_gather(parts, torch.from_numpy(ds))
    assert np.array_equal(torch.cat(parts).numpy()[:eng.nvox], dose)
    dist.all_gather(parts, torch.from_numpy(ss))
    assert np.array_equal(torch.cat(parts).numpy()[:eng.nvox], sig)
    with pytest.raises(mc.McError):
        mc.mc_finalize_multi_range(eng.ctx, peers, n_job, B, 5, eng.nvox + 1, ds, ss)
    dist.barrier()                                                   # nobody frees before everybody has read
    for r in range(world):
        if r != rank:
            mc.mc_ipc_close_handle(peers[r])
    np.save(os.path.join(out_dir, f"dose{rank}.npy"), dose)
    np.save(os.path.join(out_dir, f"sig{rank}.npy"), sig)
    eng.close()
    dist.destroy_process_group()


def test_two_ranks_exchange_their_grids_through_cuda_ipc(tmp_path):
    import torch
    import torch.multiprocessing as tmp
    assert torch.cuda.is_available()
    world, n_per_rank, B = 2, 100000, 10
    tmp.spawn(_rank_main, args=(world, _free_port(), n_per_rank, B, str(tmp_path)), nprocs=world, join=True)
    cfg = W.config(4, "e")
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    d_ref, s_ref = eng.run(cfg["beam"], world * n_per_rank, 5, B)
    eng.close()
    for r in range(world):
        d, s = np.load(tmp_path / f"dose{r}.npy"), np.load(tmp_path / f"sig{r}.npy")
        assert np.allclose(d, d_ref, rtol=2e-5, atol=1e-7 * d_ref.max())
        assert np.allclose(s, s_ref, rtol=5e-3, atol=1e-6 * d_ref.max())
    assert d_ref.max() > 0


@pytest.mark.parametrize("fail_rank", ["", "1"])
def test_bench_two_ranks_on_one_gpu_peer_exchange_and_joint_fallback(fail_rank):
    """bench.py --gpus 2 with both ranks on this box's one GPU (gloo for the plumbing: a functional check, not a measurement):
    the fused, voxel-sliced exchange, and — with a peer-mapping failure injected on rank 1 — the joint fallback of ALL
    ranks to the all-reduce; both give the same statistics as each other."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, MC_BENCH_BACKEND="gloo", MC_BENCH_FAIL_PEER_RANK=fail_rank)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(root, "bench.py"), "--gpus", "2", "--config", "1", "--steps", "2",
           "--warmup", "3", "--no-cpu-baseline", "--no-e2e"]
    out = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["ledger_rel"] < 1e-4
    par = line["config"]["parallelism"]
    assert ("peer mapping failed" in par) == (fail_rank != ""), par
    assert ("one voxel slice per rank" in par) == (fail_rank == ""), par
    # the statistics do not depend on the exchange: same job, same seed
    assert line["mean_rel_sigma_10pct_isodose"] == pytest.approx(0.006, rel=0.25)


def test_bench_gpus_2_without_a_launcher_starts_two_ranks():
    """A plain `python bench.py --gpus 2` (no torchrun around it) must start the two ranks itself and print n_gpus = 2; a
    launcher that started another number of ranks than --gpus says is refused."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    env["MC_BENCH_BACKEND"] = "gloo"
    cmd = [sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--config", "1", "--steps", "2", "--warmup", "3",
           "--no-cpu-baseline", "--no-e2e"]
    out = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["ledger_rel"] < 1e-4 and "x2" in line["config"]["parallelism"]
    out = subprocess.run(cmd[:2] + ["--gpus", "3"] + cmd[4:], env=dict(env, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0"),
                         capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode != 0 and "WORLD_SIZE=1" in (out.stderr + out.stdout)
