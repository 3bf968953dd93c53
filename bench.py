#!/usr/bin/env python
"""bench.py — one JSON line per run (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

A "step" is one pass of the whole hot path (source -> photon / electron transport -> scoring ->
batch statistics) over one job of synthetic histories.  Default workload =
BASELINE.json configs[1]: 15 MeV electron beam, 10x10 cm^2 at SSD 100, 61x61x60 water phantom at
0.5 cm, 1e7 histories, 10 batches, cut-offs 0.2 / 0.01 MeV (the configuration the metric is quoted on).

  value          histories/s with phantom, tables and queues resident in HBM, outputs left on the device
  e2e            the same through the C-ABI call mc_run with HOST buffers: beam description from host memory in,
                 dose and sigma written to host memory, every step, on a resident context; e2e.fresh_context
                 adds mc_create (phantom upload) + mc_build_tables (build + upload) + mc_destroy to every step
  roofline       dominant kernel (electron_kernel): algorithmic thread-instructions per launch (DESIGN.md
                 "Measurement") / its CUDA-event time, against the SM issue peak
  roofline_scoring  dose atomics issued per second against the measured red.global.add.f32 peak
  cpu_baseline   the oracle as it stands on the host cores, bounded sample of the same workload
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1503_01722_b200 import workloads as W  # noqa: E402  (input generators only)

# Algorithmic thread-instructions per unit of work (SURVEY.md 8(d) "Algorithmic work per unit").
# Headline: the figures the survey's own ceiling uses (225 per e- step; mid-range for the rest); beside it the top-of-range
# variant round 1 reported.
INSTR_PER = {"e_step": 225.0, "hard_event": 115.0, "photon_flight": 75.0, "photon_interaction": 150.0}
INSTR_PER_TOP = {"e_step": 240.0, "hard_event": 150.0, "photon_flight": 60.0, "photon_interaction": 150.0}
SM_COUNT, SCHEDULERS_PER_SM, LANES = 148, 4, 32


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="engine", choices=["engine", "reference"])
    ap.add_argument("--config", default="2", help="BASELINE.json config, 1-based (default 2 = configs[1]); p1..p5 = the paper's "
                    "own five cases (128^3 x 0.25 cm, 2x2 cm^2 field: context beside its Tables 2-3)")
    ap.add_argument("--beam", default=None, choices=[None, "e", "g"], help="configs 4, 5: electron or photon beam")
    ap.add_argument("--histories", type=int, default=0, help="override n_histories (the line then says so)")
    ap.add_argument("--ms-model", default="gaussian", choices=["gaussian", "gs"], help="multiple-scattering angle model (north_star: Gaussian or Goudsmit-Saunderson)")
    ap.add_argument("--stepping", default="voxel", choices=["voxel", "multi"], help="electron stepping: one step per voxel (PAPER.md:39) or multi-voxel steps (PAPER.md:167)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extra-configs", action="store_true", help="default run only: leave configs 3 and 5 off the line")
    ap.add_argument("--option", action="append", default=[], help="engine option name=value (mc_set_option)")
    return ap.parse_args()


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the one `ncu --set full` capture of each kernel (the bench does
# not run under ncu, so the figure can only be quoted): valid for the capture's own configuration and nothing else.
# key: (config, beam, ms_model, stepping, histories overridden, kernel) -> (bytes per launch, where it was captured)
NCU_TRAFFIC = {
    ("2", None, "gaussian", "voxel", False, "electron_kernel"):
        (1848283000.0, "profiles/r3_electron_kernel_ncu_full.txt: ncu --set full of this configuration, the 1e7-primary wave"),
}


def ncu_traffic(args, kernel):
    key = (str(args.config), args.beam, args.ms_model, args.stepping, bool(args.histories), kernel)
    if key in NCU_TRAFFIC and not args.option:
        return NCU_TRAFFIC[key]
    return None, "no ncu --set full capture of this kernel on this configuration"


def queue_and_scoring_bytes(acc, steps):
    """Algorithmic DRAM / L2 traffic of one step from the run's own counters: every queued secondary is one 48-byte record
    written and read once, every scoring atomic one 32-byte sector update."""
    rec = (acc["n_secondary_electrons"] + acc["n_secondary_photons"]) / steps
    return {"queue_bytes_per_step": rec * 48 * 2, "scoring_bytes_per_step": acc["n_dose_atomics"] / steps * 32,
            "what": "queued records x 48 B x (write + read); dose atomics x 32 B sector"}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 6 and r[2 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def extras_wanted(args):
    """The default line (BASELINE config 2, nothing overridden) also carries configs 3 and 5; --no-extra-configs drops them."""
    return str(args.config) == "2" and not args.histories and args.ms_model == "gaussian" and args.stepping == "voxel" \
        and not args.option and not args.no_extra_configs


def workload(args):
    cfg = W.config(args.config, args.beam)
    if args.histories:
        cfg["n_histories"] = args.histories
    if args.stepping == "multi":  # steps cross voxel faces (gDPM's scheme; R28); the line says so
        cfg["params"] = dict(cfg["params"], flags=cfg["params"]["flags"] | W.FLAG_MULTI_VOXEL)
    if args.ms_model == "gs":  # Goudsmit-Saunderson angle instead of the Gaussian model (R27); the line says so
        cfg["params"] = dict(cfg["params"], flags=cfg["params"]["flags"] | W.FLAG_MS_GS)
    return cfg


def config_dict(cfg, args, extra=None):
    d = {"workload": (f"paper-shaped case {args.config}: " if str(args.config).startswith("p") else f"BASELINE config {args.config}: ") + cfg["name"], "n_histories_per_step": cfg["n_histories"],
         "n_batches": cfg["n_batches"], "dims": [int(x) for x in cfg["phantom"]["dims"]],
         "voxel_cm": float(cfg["phantom"]["voxel_cm"][0]), "e_cut_MeV": cfg["params"]["e_cut_MeV"],
         "g_cut_MeV": cfg["params"]["g_cut_MeV"], "seed": cfg["seed"],
         "histories_overridden": bool(args.histories), "ms_model": args.ms_model, "stepping": args.stepping}
    d.update(extra or {})
    return d


# ---- the oracle on the host cores (cpu_baseline leg and --impl reference) --------------------------
def oracle_sample_rate(cfg, n_sample, workers):
    import oracle  # test infrastructure: allowed here only (cpu_baseline / reference arm)
    orc = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    _, st, dt = orc.run_sample(cfg["beam"], cfg["n_histories"], n_sample, cfg["seed"], cfg["n_batches"], workers)
    return n_sample / dt, st, dt


def oracle_sample_size(cfg, workers, seconds):
    """Histories for about `seconds` of wall time on `workers` cores, from a 0.5 s single-core probe."""
    import oracle
    orc = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    n_probe, rate = 500, 0.0
    while True:
        _, _, dt = orc.run_sample(cfg["beam"], cfg["n_histories"], n_probe, cfg["seed"], cfg["n_batches"], 1)
        rate = n_probe / dt
        if dt > 0.3 or n_probe >= cfg["n_histories"]:
            break
        n_probe = min(n_probe * 4, cfg["n_histories"])
    return int(max(1000, min(cfg["n_histories"], rate * workers * seconds)))


def cpu_baseline(cfg, seconds=15.0):
    import oracle
    cores = oracle.host_cores()
    n = oracle_sample_size(cfg, cores, seconds)
    rate, st, dt = oracle_sample_rate(cfg, n, cores)
    return {"value": rate, "unit": "histories/s", "cores": cores, "kind": "oracle",
            "sample": f"histories [0, {n}) of the {cfg['n_histories']}-history job, same seed, {cores} processes, {dt:.1f} s",
            "e_steps_per_s": st["n_estep"] / dt, "single_core_equiv": rate / cores}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = workload(args)
    cores = oracle.host_cores()
    # each step = a bounded sample sized so that warmup + steps end within a few minutes
    per_step_s = max(2.0, min(20.0, 150.0 / max(1, args.steps + args.warmup)))
    n = oracle_sample_size(cfg, cores, per_step_s)
    for _ in range(args.warmup):
        oracle_sample_rate(cfg, n, cores)
    t, steps_e = 0.0, 0.0
    for _ in range(args.steps):
        _, st, dt = oracle_sample_rate(cfg, n, cores)
        t += dt
        steps_e += st["n_estep"]
    value = n * args.steps / t
    sample = f"histories [0, {n}) of the {cfg['n_histories']}-history job per step, {cores} processes"
    print(json.dumps({
        "impl": "reference", "metric": "histories/s", "value": value, "unit": "histories/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(cfg, args, {"sample": sample}),
        "e_steps_per_s": steps_e / t,
        "cpu_baseline": {"value": value, "unit": "histories/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "histories/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---- rooflines from the run's own counters and CUDA-event kernel times -----------------------------------
def algorithmic_instr(acc, kernel, per):
    if kernel == "electron_kernel":
        return acc["n_electron_steps"] * per["e_step"] + (acc["n_moller"] + acc["n_brems"]) * per["hard_event"]
    return acc["n_photon_flights"] * per["photon_flight"] + \
        (acc["n_compton"] + acc["n_pair"] + acc["n_photoelectric"]) * per["photon_interaction"]


def kernel_roofline(acc, kernel, K, total_ms, issue_peak, issue_measured, pk_kind, single_gpu=True):
    """Issue-slot roofline of one transport kernel: algorithmic thread-instructions of the timed steps (counters x
    SURVEY 8(d) figures) / the CUDA-event time of that kernel's launches, against the SM issue peak."""
    kms = acc["electron_kernel_ms"] if kernel == "electron_kernel" else acc["photon_kernel_ms"]
    achieved = algorithmic_instr(acc, kernel, INSTR_PER) / (kms * 1e-3) if kms > 0 else 0.0
    achieved_top = algorithmic_instr(acc, kernel, INSTR_PER_TOP) / (kms * 1e-3) if kms > 0 else 0.0
    return {"bound": "alu", "kernel": kernel, "achieved": achieved / 1e12, "peak": issue_peak / 1e12,
            "unit": "Tinstr/s (thread-instructions)", "frac": achieved / issue_peak,
            "instr_per_unit": INSTR_PER, "frac_top_of_range": achieved_top / issue_peak, "instr_per_unit_top_of_range": INSTR_PER_TOP,
            "headline": "frac (SURVEY 8(d) ceiling figures: 225 thread-instructions per e- step, 75 per photon flight)",
            "peak_source": f"148 SM x 4 schedulers x 32 lanes x sm_max_mhz ({pk_kind} MEASURED_PEAKS.json clock)",
            "peak_measured": issue_measured / 1e12, "frac_of_measured": achieved / issue_measured,
            "peak_measured_source": "mc_bench_issue: 2 x 1024-thread CTAs per SM, 8 independent FFMA chains per thread, best of 3",
            "kernel_ms_per_step": kms / K, "kernel_share_of_step": kms / total_ms if single_gpu else None}


def measure_extra_config(mc, torch, stream, flush, name, beam, steps, warmup, issue_peak, issue_measured, pk_kind, red_peak):
    """One more BASELINE config on the same line (north_star quotes the metric for a photon AND an electron beam): the same
    timed region as the headline (L2 flush between steps, CUDA events on the engine's stream), the same rooflines, and e2e
    through mc_run with host buffers.  Single GPU only."""
    a = argparse.Namespace(config=name, beam=beam, histories=0, ms_model="gaussian", stepping="voxel", option=[])
    cfg = workload(a)
    n, B, seed = cfg["n_histories"], cfg["n_batches"], cfg["seed"]
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    mc.mc_set_stream(eng.ctx, stream.cuda_stream)
    dose = torch.empty(eng.nvox, dtype=torch.float32, device="cuda")
    sigma = torch.empty_like(dose)
    acc = {}
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            flush.fill_(1)
            mc.mc_run(eng.ctx, cfg["beam"], n, seed, B, dose, sigma)
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for i in range(steps):
            flush.fill_(1)
            ev[i][0].record(stream)
            mc.mc_run(eng.ctx, cfg["beam"], n, seed, B, dose, sigma)
            ev[i][1].record(stream)
            for k, v in mc.mc_get_stats(eng.ctx).items():
                acc[k] = acc.get(k, 0) + v
        torch.cuda.synchronize()
        total_ms = sum(x.elapsed_time(y) for x, y in ev)
        # e2e: host buffers in and out, wall clock around the calls
        h_dose, h_sigma = np.zeros(eng.nvox, np.float32), np.zeros(eng.nvox, np.float32)
        mc.mc_run(eng.ctx, cfg["beam"], n, seed, B, h_dose, h_sigma)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(steps):
            mc.mc_run(eng.ctx, cfg["beam"], n, seed, B, h_dose, h_sigma)
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
    e_ms, p_ms = acc["electron_kernel_ms"], acc["photon_kernel_ms"]
    dom, other = ("electron_kernel", "photon_kernel") if e_ms >= p_ms else ("photon_kernel", "electron_kernel")
    d, sg = dose.cpu().numpy().astype(np.float64), sigma.cpu().numpy().astype(np.float64)
    m = d >= 0.1 * d.max()
    rel = float(np.mean(sg[m] / d[m]))
    red_rate = acc["n_dose_atomics"] / ((e_ms + p_ms) * 1e-3)
    out = {"config": config_dict(cfg, a), "steps": steps, "warmup": warmup, "ms_per_step": total_ms / steps,
           "value": n * steps / (total_ms * 1e-3), "unit": "histories/s",
           "e_steps_per_s": acc["n_electron_steps"] / (total_ms * 1e-3),
           "photon_flights_per_s": acc["n_photon_flights"] / (total_ms * 1e-3),
           "gpu_launches": int(acc["n_kernel_launches"]),
           "ledger_rel": abs(acc["e_deposited_MeV"] + acc["e_escaped_MeV"] - acc["e_source_MeV"]) / acc["e_source_MeV"],
           "roofline": dict(kernel_roofline(acc, dom, steps, total_ms, issue_peak, issue_measured, pk_kind),
                            traffic=None, traffic_source="no ncu --set full capture of this kernel on this configuration",
                            traffic_algorithmic=queue_and_scoring_bytes(acc, steps)),
           "roofline_scoring": {"bound": "l2_atomic", "achieved": red_rate / 1e9, "peak": red_peak / 1e9, "unit": "Gred/s",
                                "frac": red_rate / red_peak},
           "mean_rel_sigma_10pct_isodose": rel, "time_to_1pct_s": (total_ms / steps * 1e-3) * (rel / 0.01) ** 2,
           "e2e": {"value": n * steps / t_e2e, "unit": "histories/s", "h2d_bytes_per_step": int(3 * 4096 * 4),
                   "d2h_bytes_per_step": int(2 * eng.nvox * 4 + 5 * 4 + 12 * 8 + 3 * 8),
                   "what": "mc_run(beam from host, dose + sigma to host memory) per step on a resident context"}}
    other_ms = p_ms if other == "photon_kernel" else e_ms
    if other_ms > 0.25 * total_ms:
        out["roofline_" + other.split("_")[0]] = kernel_roofline(acc, other, steps, total_ms, issue_peak, issue_measured, pk_kind)
    eng.close()
    return out


# ---- the CUDA engine ---------------------------------------------------------------------------------
def run_engine(args):
    import torch
    import torch.distributed as dist
    import paper_1503_01722_b200 as mc

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:  # the line's n_gpus is the number of ranks that ran: refuse to print anything else
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={world} ranks")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the engine has no CPU path)")
    # one rank per GPU; MC_BENCH_BACKEND=gloo lets the N > 1 code path be exercised on a box with fewer GPUs than
    # ranks (ranks then share devices and the grids are reduced through the host) — a functional check, not a benchmark
    backend = os.environ.get("MC_BENCH_BACKEND", "nccl")
    local = local % torch.cuda.device_count()
    torch.cuda.set_device(local)
    if world > 1:
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
    cfg = workload(args)
    n, B, seed = cfg["n_histories"], cfg["n_batches"], cfg["seed"]
    from paper_1503_01722_b200 import sharding
    n_job, h_lo, h_hi = sharding.history_range(rank, world, n)  # weak scaling: n histories per rank
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    for kv in args.option:
        k, v = kv.split("=")
        mc.mc_set_option(eng.ctx, k, int(v))
    stream = torch.cuda.Stream()
    mc.mc_set_stream(eng.ctx, stream.cuda_stream)
    nvox = eng.nvox
    dose = torch.empty(nvox, dtype=torch.float32, device="cuda")
    sigma = torch.empty_like(dose)
    edep = torch.empty(B * nvox, dtype=torch.float32, device="cuda") if world > 1 else None
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    # N > 1: the one exchange of the sharded job (sum of the ranks' per-batch grids).
    #   peer      (default) every rank leaves its grids in its context's buffer, maps the other ranks' buffers once
    #             through CUDA IPC and reads them in place in mc_finalize_multi (over NVLink): no all-reduce, no copy
    #   allreduce NCCL all-reduce of the grids, then mc_finalize (also the fallback if the peers cannot be mapped)
    exchange, peers = "single GPU", None
    if world > 1:
        exchange = os.environ.get("MC_BENCH_EXCHANGE", "peer")
        if exchange == "peer":
            ok = True
            try:
                own = mc.mc_edep_buffer(eng.ctx, B)
                handles = [None] * world
                dist.all_gather_object(handles, mc.mc_ipc_get_handle(own))
                if os.environ.get("MC_BENCH_FAIL_PEER_RANK") == str(rank):  # fault injection for the fallback test
                    raise RuntimeError("injected peer-mapping failure")
                peers = [None] * world  # filled one by one: what was opened before a failure is closed on fallback
                for r in range(world):
                    peers[r] = own if r == rank else mc.mc_ipc_open_handle(handles[r])
            except Exception as exc:  # noqa: BLE001  (any failure -> every rank falls back together)
                print(f"rank {rank}: peer mapping failed ({exc}); falling back to all-reduce", file=sys.stderr)
                ok = False

            def all_min(v):
                flag = torch.tensor([v], device="cuda" if backend == "nccl" else "cpu")
                dist.all_reduce(flag, op=dist.ReduceOp.MIN)
                return int(flag.item())
            if not sharding.agree_on_peer_exchange(ok, all_min):
                for r in range(world if peers else 0):
                    if r != rank and peers[r] is not None:
                        mc.mc_ipc_close_handle(peers[r])
                exchange, peers = "allreduce (peer mapping failed)", None
            else:
                exchange = "peer, one voxel slice per rank + all-gather of dose and sigma"
    chunk = sharding.voxel_slice(rank, world, nvox)[0]
    d_slice = torch.zeros(chunk, dtype=torch.float32, device="cuda")
    s_slice = torch.zeros_like(d_slice)
    gathered = torch.empty(world * chunk, dtype=torch.float32, device="cuda") if world > 1 else None

    def all_gather(t, _chunk):
        if backend == "nccl":
            dist.all_gather_into_tensor(gathered, t)
            return gathered.clone()  # the buffer is reused for sigma
        parts = [torch.empty(_chunk, dtype=torch.float32) for _ in range(world)]  # gloo: through the host (functional check)
        dist.all_gather(parts, t.cpu())
        return torch.cat(parts).cuda()

    def step(dose_out=None, sigma_out=None, e=None):
        e = e or eng
        d_out, s_out = (dose, sigma) if dose_out is None else (dose_out, sigma_out)
        if world == 1:
            mc.mc_run(e.ctx, cfg["beam"], n, seed, B, d_out, s_out)
        elif peers is not None and e is eng:
            def finalize_slice(nj, v0, v1):
                mc.mc_finalize_multi_range(e.ctx, peers, nj, B, v0, v1, d_slice, s_slice)
                return d_slice, s_slice
            d, sg = sharding.run_sharded_peer(rank, world, n, nvox,
                                              lambda nj, a, b: mc.mc_run_range(e.ctx, cfg["beam"], nj, a, b, seed, B, peers[rank]),
                                              dist.barrier, finalize_slice, all_gather)
            st = mc.mc_get_stats(e.ctx)  # the transport's counters (mc_finalize_multi_range adds one launch)
            if torch.is_tensor(d_out):
                d_out.copy_(d); s_out.copy_(sg)
            else:
                d_out[:] = d.cpu().numpy(); s_out[:] = sg.cpu().numpy()
            return st
        else:
            def run_range(nj, a, b):
                mc.mc_run_range(e.ctx, cfg["beam"], nj, a, b, seed, B, edep)
                return edep
            sharding.run_sharded(rank, world, n, run_range, dist.all_reduce,
                                 lambda g, nj: mc.mc_finalize(e.ctx, g, nj, B, d_out, s_out))
        return mc.mc_get_stats(e.ctx)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            flush.fill_(1)
            step()
        sync_all()
        sampler = ClockSampler(local)
        if rank == 0:
            sampler.start()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        acc = {}
        for i in range(args.steps):
            flush.fill_(1)          # L2 flush between timed iterations (not timed)
            ev[i][0].record(stream)
            st = step()
            ev[i][1].record(stream)
            for k, v in st.items():
                acc[k] = acc.get(k, 0) + v
        sync_all()
        clocks = sampler.stop() if rank == 0 else None
    ms = torch.tensor([sum(a.elapsed_time(b) for a, b in ev)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    total_ms = float(ms.item())
    K = args.steps

    # ---- e2e: the C-ABI call with HOST buffers: beam description (host) in, dose + sigma (host) out, every step ----
    e2e = None
    if not args.no_e2e:
        h_dose, h_sigma = np.zeros(nvox, np.float32), np.zeros(nvox, np.float32)
        ph = cfg["phantom"]

        def host_step(e):
            step(h_dose, h_sigma, e)

        def timed(fn, reps):
            fn()
            sync_all()
            t0 = time.perf_counter()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                fn()
            e1.record(stream)
            sync_all()
            wall = time.perf_counter() - t0
            # host work is part of the call: take the wall clock (>= the device time), max over ranks
            tw = torch.tensor([max(wall, e0.elapsed_time(e1) * 1e-3)], dtype=torch.float64, device="cuda")
            if world > 1:
                dist.all_reduce(tw, op=dist.ReduceOp.MAX)
            return float(tw.item())

        def fresh_step():  # a new context per step: phantom upload + table build + run + teardown
            e = mc.Engine(ph, cfg["materials"], cfg["params"])
            mc.mc_set_stream(e.ctx, stream.cuda_stream)
            host_step(e)
            e.close()

        with torch.cuda.stream(stream):
            t_run = timed(lambda: host_step(eng), K)
            t_fresh = timed(fresh_step, min(K, 3))
        g = mc.mc_export_grid(eng.ctx)
        tab_bytes = (1 + 9 * len(cfg["materials"])) * g["N"] * 8
        e2e = {"value": n_job * K / t_run, "unit": "histories/s",
               "h2d_bytes_per_step": int(3 * 4096 * 4),  # beam energy / pdf / cdf nodes
               "d2h_bytes_per_step": int(2 * nvox * 4 + 5 * 4 + 12 * 8 + 3 * 8),  # dose, sigma, counters, stats, ledger
               "what": "mc_run(beam from host, dose + sigma to host memory) per step on a resident context",
               "fresh_context": {"value": n_job * min(K, 3) / t_fresh, "unit": "histories/s",
                                 "h2d_bytes_per_step": int(nvox * 8 + tab_bytes + 3 * 4096 * 4),
                                 "what": "mc_create + mc_build_tables + mc_run(host outputs) + mc_destroy per step"}}

    # ---- rooflines (rank 0's kernels) ----------------------------------------------------------------------
    pk, pk_kind = peaks()
    issue_peak = SM_COUNT * SCHEDULERS_PER_SM * LANES * pk["sm_max_mhz"] * 1e6  # thread-instructions / s
    issue_measured = max(mc.mc_bench_issue(eng.ctx, 4096) for _ in range(3))  # FFMA micro-benchmark on this GPU
    e_ms, p_ms = acc["electron_kernel_ms"], acc["photon_kernel_ms"]
    dom = "electron_kernel" if e_ms >= p_ms else "photon_kernel"

    traffic, traffic_src = ncu_traffic(args, dom)
    roofline = dict(kernel_roofline(acc, dom, K, total_ms, issue_peak, issue_measured, pk_kind, world == 1),
                    traffic=traffic, traffic_unit="bytes per launch", traffic_source=traffic_src,
                    traffic_algorithmic=queue_and_scoring_bytes(acc, K))
    other = "photon_kernel" if dom == "electron_kernel" else "electron_kernel"
    other_ms = p_ms if dom == "electron_kernel" else e_ms
    roofline_other = kernel_roofline(acc, other, K, total_ms, issue_peak, issue_measured, pk_kind, world == 1) \
        if other_ms > 0.25 * total_ms else None
    # scoring roofline: red.global.add.f32 peak, best over occupancy (1, 2, 4, 8 CTAs of 256 threads per SM) on windows
    # the size of one batch grid of configs 2-4 (0.9 MB) and of config 5 (7.1 MB), random cells (no intra-warp
    # collisions on average), >= 2 ms per launch; mode 1 (one cell per warp) beside it
    red_table, red_peak = [], 0.0
    for cells in (223260, 1786080):
        for per_sm in (1, 2, 4, 8):
            blocks = SM_COUNT * per_sm
            per_thread = int(min(60000, max(64, 4e8 / (blocks * 256))))
            ms = mc.mc_bench_red(eng.ctx, cells, per_thread, 0, blocks)
            rate = blocks * 256 * per_thread / (ms * 1e-3)
            red_table.append({"window_MB": round(cells * 4 / 1e6, 1), "ctas_per_sm": per_sm, "mode": "random cells", "ms": round(ms, 3), "Gred_s": round(rate / 1e9, 1)})
            red_peak = max(red_peak, rate)
    for cells in (223260,):
        blocks = SM_COUNT * 8
        per_thread = 2000
        ms = mc.mc_bench_red(eng.ctx, cells, per_thread, 1, blocks)
        red_table.append({"window_MB": round(cells * 4 / 1e6, 1), "ctas_per_sm": 8, "mode": "one cell per warp", "ms": round(ms, 3),
                          "Gred_s": round(blocks * 256 * per_thread / (ms * 1e-3) / 1e9, 1)})
    red_rate = acc["n_dose_atomics"] / ((e_ms + p_ms) * 1e-3)
    roofline_scoring = {"bound": "l2_atomic", "achieved": red_rate / 1e9, "peak": red_peak / 1e9, "unit": "Gred/s",
                        "frac": red_rate / red_peak, "peak_table": red_table,
                        "peak_source": "mc_bench_red: best of the random-cell rows of peak_table (occupancy x window sweep)"}

    if rank == 0:
        out = {"metric": "histories/s", "value": n_job * K / (total_ms * 1e-3), "unit": "histories/s",
               "n_gpus": world, "steps": K, "warmup": args.warmup, "ms_per_step": total_ms / K,
               "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
               "data": "synthetic",
               "config": config_dict(cfg, args, {"l2": "256 MiB fill between timed steps (L2 flush)",
                                                 "parallelism": f"history ranges x{world}, exchange: {exchange}" if world > 1 else "single GPU"}),
               "e_steps_per_s": acc["n_electron_steps"] * world / (total_ms * 1e-3),
               "photon_flights_per_s": acc["n_photon_flights"] * world / (total_ms * 1e-3),
               "per_history": {"e_steps": acc["n_electron_steps"] / (n * K), "photon_flights": acc["n_photon_flights"] / (n * K),
                               "fictitious_fraction": acc["n_fictitious"] / max(1, acc["n_photon_flights"]),
                               "hard_events": (acc["n_moller"] + acc["n_brems"]) / (n * K),
                               "dose_atomics": acc["n_dose_atomics"] / (n * K),
                               "secondaries": (acc["n_secondary_electrons"] + acc["n_secondary_photons"]) / (n * K)},
               "ledger_rel": abs(acc["e_deposited_MeV"] + acc["e_escaped_MeV"] - acc["e_source_MeV"]) / acc["e_source_MeV"],
               "clocks": clocks, "e2e": e2e, "gpu_launches": int(acc["n_kernel_launches"]),
               "roofline": roofline, "roofline_scoring": roofline_scoring}
        if roofline_other is not None:  # the second kernel where it is more than a quarter of the step
            out["roofline_" + other.split("_")[0]] = roofline_other
        # statistics of the result: mean sigma/D inside the 10 % isodose and time to 1 %
        d, s = dose.cpu().numpy().astype(np.float64), sigma.cpu().numpy().astype(np.float64)
        m = d >= 0.1 * d.max()
        rel = float(np.mean(s[m] / d[m]))
        out["mean_rel_sigma_10pct_isodose"] = rel
        out["time_to_1pct_s"] = (total_ms / K * 1e-3) * (rel / 0.01) ** 2
        if world == 1 and extras_wanted(args):
            # north_star names a 6 MV photon and a 15 MeV electron beam on water, and the heterogeneous phantom: configs 3
            # and 5 (electron beam) ride on the same line, measured like the headline (3 timed steps each)
            eng.close()  # its queues go back to the library's pool and are reused by the next contexts
            out["configs"] = [measure_extra_config(mc, torch, stream, flush, c, b, 3, 3, issue_peak, issue_measured, pk_kind, red_peak)
                              for c, b in (("3", None), ("5", "e"))]
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(cfg)
        print(json.dumps(out))
    if peers is not None:
        dist.barrier()
        for r in range(world):
            if r != rank:
                mc.mc_ipc_close_handle(peers[r])
    eng.close()
    if world > 1:
        dist.destroy_process_group()


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks here (one process per GPU, the same command line the
    driver uses for N > 1) and become that launcher.  NCCL's own environment (NCCL_DEBUG, ...) is passed through untouched."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


if __name__ == "__main__":
    a = parse()
    if a.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if a.impl == "reference":
        run_reference(a)
    else:
        if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
            respawn_under_torchrun(a)
        run_engine(a)
