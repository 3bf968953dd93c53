"""Coupled-mode parity of the CUDA path against the oracle (run on the B200 box with -m gpu); every
call goes through the C ABI.

Bars (BASELINE.json north_star, R19):
  * mean |D_gpu - D_orc| / Dmax over the 10 % isodose <= 1 %
  * >= 99 % of those voxels within 3 combined batch sigma
The oracle runs once per case (seed 1, 40 batches: R19).  The engine runs twice:
  seed 1 — the SAME Philox streams as the oracle: the statistical noise largely cancels, so the 1 % bar is
           applied strictly (a physics difference shows as a bias);
  seed 2 — independent streams: the 3-sigma criterion proper; the mean |difference| bar is then
           1 % + E|noise| = 1 % + 0.8 * mean(sigma_comb)/Dmax (half-normal mean), stated here once.
           Where the oracle is thin (photon configs 3, 4g, 5g: mean combined sigma 2-3 % of Dmax per voxel) that
           allowance makes the seed-2 bar about 3 %: those configs are carried by the seed-1 run (strict 1 %, measured
           2e-5 .. 1e-3) and by the integrated curves of the high-statistics test below (0.3 %), not by seed 2.
Event counters per history (flights, fictitious, Compton, pair, photoelectric, Moller, brems) must agree within 1 %
and the energy ledger of every engine run must close.
"""
import numpy as np
import pytest

import oracle
import paper_1503_01722_b200 as mc
from paper_1503_01722_b200 import workloads as W

pytestmark = pytest.mark.gpu

WORKERS = min(oracle.host_cores(), 32)
B_ORC = 40


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1503_01722_b200 import build
    build.build()


def _metrics(dg, sg, do, so):
    dg, sg = dg.astype(np.float64), sg.astype(np.float64)
    m = do >= 0.1 * do.max()
    diff = np.abs(dg[m] - do[m])
    comb = np.sqrt(sg[m] ** 2 + so[m] ** 2)
    return {"n": int(m.sum()), "mean_diff": float(diff.mean() / do.max()),
            "frac3": float(np.mean(diff <= 3.0 * comb)), "noise": float(0.8 * comb.mean() / do.max())}


EVENTS = ("flights", "fictitious", "compton", "pair", "photoelectric", "moller", "brems")


def _per_history(st, n):
    return {"e_steps": st["n_electron_steps"] / n, "flights": st["n_photon_flights"] / n,
            "fictitious": st["n_fictitious"] / n, "compton": st["n_compton"] / n, "pair": st["n_pair"] / n,
            "photoelectric": st["n_photoelectric"] / n, "moller": st["n_moller"] / n, "brems": st["n_brems"] / n}


def _per_history_orc(st, n):
    return {"e_steps": st["n_estep"] / n, "flights": st["n_flight"] / n, "fictitious": st["n_fict"] / n,
            "compton": st["n_compton"] / n, "pair": st["n_pair"] / n, "photoelectric": st["n_pe"] / n,
            "moller": st["n_moller"] / n, "brems": st["n_brems"] / n}


def _ledger(st):
    return abs(st["e_deposited_MeV"] + st["e_escaped_MeV"] - st["e_source_MeV"]) / st["e_source_MeV"]


def _block_dose(edep, rho, dims, voxel_cm, n_total, f):
    """Dose and batch sigma on f x f x f voxel blocks from per-batch energy grids [B, nvox] (MeV): the R17 / R18
    definitions written out in numpy on block sums — a property that holds at any size, used where the oracle
    cannot afford the statistics of the fine grid."""
    B = edep.shape[0]
    nx, ny, nz = dims
    cx, cy, cz = nx // f, ny // f, nz // f

    def blocks(a):
        a = a.reshape(nz, ny, nx)[:cz * f, :cy * f, :cx * f]
        return a.reshape(cz, f, cy, f, cx, f).sum(axis=(1, 3, 5)).reshape(-1)

    mass = blocks(rho.astype(np.float64)) * float(np.prod(voxel_cm))
    nb = np.array([-(-(b + 1) * n_total // B) - -(-b * n_total // B) for b in range(B)], np.float64)  # ceil edges
    D = np.stack([blocks(edep[b].astype(np.float64)) / (mass * nb[b]) for b in range(B)])
    mean = D.mean(axis=0)
    return mean, np.sqrt(((D - mean) ** 2).sum(axis=0) / (B * (B - 1)))


def _engine_run(eng, cfg, n, seed, coarse):
    ph = cfg["phantom"]
    B = cfg["n_batches"]
    if coarse == 1:
        dg, sg = eng.run(cfg["beam"], n, seed, B)
    else:
        edep = np.zeros((B, eng.nvox), np.float32)
        mc.mc_run_range(eng.ctx, cfg["beam"], n, 0, n, seed, B, edep)
        dg, sg = _block_dose(edep, ph["density"], eng.dims, ph["voxel_cm"], n, coarse)
    st = eng.stats()
    assert st["n_histories"] == n
    assert _ledger(st) < 1e-4, f"engine energy ledger open: {_ledger(st)}"
    return dg, sg, st


ORACLE_SWITCH = {"hinge_overrun_pct": ("hinge_overrun", 0.01), "ms_carry": ("ms_carry", 1.0)}  # engine option -> oracle's


def _run_case(cfg, n_gpu, n_orc, coarse=1, options=None):
    """Oracle: n_orc histories, seed 1.  Engine: seed 1 with n_orc histories (same streams, same batches up to
    the batch count) and seed 2 with n_gpu histories (independent, the size bench.py times).
    options: switches of the readings R8 / R8b set on BOTH sides (engine option name -> value)."""
    ph = cfg["phantom"]
    eng = mc.Engine(ph, cfg["materials"], cfg["params"])
    orc = oracle.Oracle(ph, cfg["materials"], cfg["params"])
    for k, v in (options or {}).items():
        mc.mc_set_option(eng.ctx, k, v)
        orc.set_option(ORACLE_SWITCH[k][0], v * ORACLE_SWITCH[k][1])
    eo, sto = orc.run_edep_parallel(cfg["beam"], n_orc, 1, B_ORC, WORKERS)
    assert sto["max_ledger_rel"] < 1e-5
    if coarse == 1:
        do, so = orc.finalize(eo, n_orc)
    else:
        do, so = _block_dose(eo, ph["density"], eng.dims, ph["voxel_cm"], n_orc, coarse)
    del eo
    out = {}
    for seed, n in ((1, n_orc), (2, n_gpu)):
        dg, sg, st = _engine_run(eng, cfg, n, seed, coarse)
        out[seed] = _metrics(dg, sg, do, so)
        out[seed]["per_history"] = _per_history(st, n)
    eng.close()
    out["orc_per_history"] = _per_history_orc(sto, n_orc)
    out["n_gpu"], out["n_orc"] = n_gpu, n_orc
    return out


def _check(out):
    ref = out["orc_per_history"]
    for seed in (1, 2):
        r = out[seed]
        for k in EVENTS:  # physics events per history: 1 %, or 5 standard errors of the count where that is larger
            tol = max(0.01 * ref[k], 5.0 * np.sqrt(2.0 * max(ref[k], 1e-9) / min(out["n_gpu"], out["n_orc"])), 1e-4)
            assert abs(r["per_history"][k] - ref[k]) <= tol, (seed, k, r["per_history"][k], ref[k], tol)
        # Condensed-history steps per history: with reading R8 (no catch-up steps behind voxel-limited steps) the
        # count no longer depends on fp32-vs-fp64 face decisions: 2 %.
        assert r["per_history"]["e_steps"] == pytest.approx(ref["e_steps"], rel=0.02), (seed, r["per_history"], ref)
        assert r["n"] > 0
    same, indep = out[1], out[2]
    assert same["mean_diff"] <= 0.01, same
    if indep["noise"] < 1e-6:  # no randomness left (pencil beam without MS and hard events): sigma ~ fp32 rounding only
        assert indep["mean_diff"] <= 1e-3, indep
        return
    # >= 99 % within 3 sigma; where the 10 % isodose holds fewer than 100 voxels (the pencil beam of config 1: 20-25)
    # one voxel is already 4-5 %, and with 10 batches a voxel lands beyond 3 sigma ~1 % of the time: allow one there
    assert indep["frac3"] >= 0.99 or (indep["n"] < 100 and round((1.0 - indep["frac3"]) * indep["n"]) <= 1), indep
    assert indep["mean_diff"] <= 0.01 + indep["noise"], indep
    if indep["noise"] <= 0.8 * 0.003:  # mean combined sigma <= 0.3 % of Dmax: north_star's 1 % bar with no allowance
        assert indep["mean_diff"] <= 0.01, indep
    # the independent run's difference must be explained by its noise (no hidden bias)
    assert indep["mean_diff"] <= 1.25 * indep["noise"] + 0.002, indep


# ---- the five BASELINE configs -------------------------------------------------------------------------
def test_config1_electron_pencil_water_full_size():
    cfg = W.config(1)
    _check(_run_case(cfg, cfg["n_histories"], cfg["n_histories"]))


def test_config2_15MeV_electrons_water_full_size():
    cfg = W.config(2)
    _check(_run_case(cfg, cfg["n_histories"], cfg["n_histories"]))


def test_config3_6MV_photons_water_full_size_engine():
    """Engine at the full 1e8 histories (the launch configuration bench.py --config 3 times); the oracle at
    4e7 histories (its sigma enters the combined sigma)."""
    cfg = W.config(3)
    _check(_run_case(cfg, cfg["n_histories"], 4 * 10 ** 7))


def test_config4_slab_electrons_full_size():
    cfg = W.config(4, "e")
    _check(_run_case(cfg, cfg["n_histories"], cfg["n_histories"]))


def test_config4_slab_photons_full_size_engine():
    cfg = W.config(4, "g")
    _check(_run_case(cfg, cfg["n_histories"], 4 * 10 ** 7))


def test_config5_halfslab_electrons_full_size_engine_per_voxel():
    """122x122x120 at 0.25 cm (the half-slab of Fig. 3), 1e8 electron histories on the engine; the oracle
    runs 3e7 (about a minute of the host cores), which brings its per-voxel sigma inside the 10 % isodose to ~1 % of Dmax:
    north_star's criterion voxel by voxel, no block sums."""
    cfg = W.config(5, "e")
    out = _run_case(cfg, cfg["n_histories"], 3 * 10 ** 7)
    print("config 5 e-", out)
    _check(out)


def test_config5_halfslab_photons_full_size_engine_per_voxel():
    cfg = W.config(5, "g")
    out = _run_case(cfg, cfg["n_histories"], 3 * 10 ** 8)
    print("config 5 photons", out)
    _check(out)


# ---- the literal readings of the step rule (PAPER.md:39 d = min[d_vox, ...], :167; R8, R8b) -------------------
@pytest.mark.parametrize("c,beam", [(2, None), (4, "e")])
@pytest.mark.parametrize("options", [{"hinge_overrun_pct": 0}, {"ms_carry": 0}], ids=["no_hinge_overrun", "no_ms_carry"])
def test_literal_step_rule_and_uncarried_ms_match_the_oracle_with_the_same_switch(c, beam, options):
    """The defaults of R8 (a voxel-limited step may run on to the face by 25 % of its second leg) and R8b (scattering power
    travelled but not sampled for is carried) are readings; the plain rule d = min[d_vox, d_maxs, d_maxe, d_event] with no
    overrun, and the planned-path-only MS angle, are run here on both sides with the same switch and must agree to the
    same bars as the defaults."""
    cfg = W.config(c, beam) if beam else W.config(c)
    out = _run_case(cfg, cfg["n_histories"], cfg["n_histories"], options=options)
    print("literal readings", c, beam, options, {k: out[k] for k in (1, 2)})
    _check(out)


# ---- Goudsmit-Saunderson multiple-scattering angle (R27) -------------------
@pytest.mark.parametrize("c,beam", [(1, None), (2, None), (4, "e")])
def test_goudsmit_saunderson_angle_matches_the_oracle_with_the_same_model(c, beam):
    cfg = W.config(c, beam) if beam else W.config(c)
    cfg["params"] = dict(cfg["params"], flags=cfg["params"]["flags"] | W.FLAG_MS_GS)
    out = _run_case(cfg, cfg["n_histories"], cfg["n_histories"])
    print("GS", c, beam, out)
    _check(out)


def test_both_variants_together_on_the_photon_beam_through_the_slab():
    """6 MV photons on the slab phantom with the Goudsmit-Saunderson angle AND multi-voxel steps for the secondary
    electrons (engine at the full 1e8 histories, oracle 4e7): the two options compose."""
    cfg = W.config(4, "g")
    cfg["params"] = dict(cfg["params"], flags=cfg["params"]["flags"] | W.FLAG_MS_GS | W.FLAG_MULTI_VOXEL)
    out = _run_case(cfg, cfg["n_histories"], 4 * 10 ** 7)
    print("GS+MV 4g", out)
    _check(out)


def test_goudsmit_saunderson_angle_changes_the_dose_where_it_should():
    """The model is not a no-op: against the Gaussian model the lateral spread of a 6 MeV pencil beam changes (single-
    scattering tail), while the deposited energy and the energy ledger do not."""
    cfg = W.config(1)
    n, B = 400000, 10
    res = []
    for fl in (0, W.FLAG_MS_GS):
        eng = mc.Engine(cfg["phantom"], cfg["materials"], dict(cfg["params"], flags=fl))
        d, _ = eng.run(cfg["beam"], n, 3, B)
        st = eng.stats()
        assert _ledger(st) < 1e-4
        res.append((d.reshape(20, 20, 20).astype(np.float64), st["e_deposited_MeV"] / st["e_source_MeV"]))
        eng.close()
    (dg, fg), (ds, fs) = res
    assert fg == pytest.approx(fs, abs=5e-3)
    x = (np.arange(20) - 9.5) * 0.5
    r2 = lambda d: float((d.sum(axis=0) * (x[None, :] ** 2 + x[:, None] ** 2)).sum() / d.sum())
    assert abs(r2(ds) / r2(dg) - 1.0) > 0.01, (r2(ds), r2(dg))


# ---- multi-voxel electron stepping (R28) -----------------------------------
@pytest.mark.parametrize("c,beam,extra", [(1, None, 0), (2, None, 0), (4, "e", 0), (4, "e", W.FLAG_MS_GS)])
def test_multi_voxel_stepping_matches_the_oracle_with_the_same_stepping(c, beam, extra):
    cfg = W.config(c, beam) if beam else W.config(c)
    cfg["params"] = dict(cfg["params"], flags=cfg["params"]["flags"] | W.FLAG_MULTI_VOXEL | extra)
    out = _run_case(cfg, cfg["n_histories"], cfg["n_histories"])
    print("MV", c, beam, extra, out)
    _check(out)


def test_multi_voxel_stepping_on_the_half_slab_coarse_blocks():
    """Config 5 (0.25 cm voxels, material interface along x): the case where a step crosses most faces."""
    cfg = W.config(5, "e")
    cfg["params"] = dict(cfg["params"], flags=cfg["params"]["flags"] | W.FLAG_MULTI_VOXEL)
    out = _run_case(cfg, 2 * 10 ** 7, 4 * 10 ** 6, coarse=4)
    print("MV5", out)
    _check(out)


# ---- physics switches, particle types, edge cases ---------------------------------------------------------
def _small_case(flags=0, particle=W.ELECTRON, energy=6.0, n=200000, shape=W.PENCIL, phantom=None):
    ph = phantom or W.homogeneous_phantom((12, 12, 16), 0.5)
    cfg = {"phantom": ph, "materials": W.materials(3), "params": W.params(flags=flags),
           "beam": W.beam(particle, shape, energy=energy, field=(3.0, 3.0)), "n_batches": 10}
    return cfg, n


@pytest.mark.parametrize("flags", [W.FLAG_NO_HARD, W.FLAG_NO_MS, W.FLAG_LOCAL_SECONDARIES,
                                   W.FLAG_NO_HARD | W.FLAG_NO_MS])
def test_physics_switches_match_the_oracle_with_the_same_switches(flags):
    cfg, n = _small_case(flags=flags)
    out = _run_case(cfg, n, n)
    print(flags, out)
    _check(out)
    if flags & W.FLAG_NO_HARD:
        assert out[1]["per_history"]["moller"] == 0 and out[1]["per_history"]["brems"] == 0


def test_no_ms_no_hard_pencil_beam_stays_on_its_column():
    """Without deflection and hard events a pencil beam deposits only along its own voxel column, down to the
    CSDA range: an exact structural property."""
    cfg, n = _small_case(flags=W.FLAG_NO_HARD | W.FLAG_NO_MS, n=5000)
    cfg["beam"] = W.beam(W.ELECTRON, W.PENCIL, energy=6.0, entry=(0.1, 0.1, 0.0))
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    d, s = eng.run(cfg["beam"], n, 3, 10)
    d = d.reshape(16, 12, 12)
    col = d[:, 6, 6]
    assert d.sum() == pytest.approx(col.sum(), rel=1e-6)
    assert np.all(s.reshape(16, 12, 12)[:, 6, 6] < 1e-6 * col.max() + 1e-12)  # every history is identical
    orc = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    do, _, _ = orc.run(cfg["beam"], 10, 3, 2)
    assert np.allclose(col, do.reshape(16, 12, 12)[:, 6, 6], rtol=2e-4, atol=1e-6 * col.max())
    eng.close()


def test_positron_beam_with_annihilation_photons():
    cfg, n = _small_case(particle=W.POSITRON, energy=4.0, n=300000)
    out = _run_case(cfg, n, n)
    print(out)
    _check(out)
    assert out[1]["per_history"]["flights"] > 2.0  # two annihilation photons per history are transported


def test_high_energy_photons_in_bone_pair_production():
    ph = W.homogeneous_phantom((10, 10, 30), 0.5, material=1, density=1.85)
    cfg, n = _small_case(particle=W.PHOTON, energy=18.0, n=1000000, shape=W.POINT_RECT, phantom=ph)
    out = _run_case(cfg, n, n)
    print(out)
    _check(out)


def test_run_range_plus_finalize_equals_run_and_device_outputs():
    import torch
    cfg = W.config(1)
    n, B = 50000, 10
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    d0, s0 = eng.run(cfg["beam"], n, 9, B)
    # two shards into separate grids, summed on the device, finalized
    e1 = torch.zeros(B * eng.nvox, dtype=torch.float32, device="cuda")
    e2 = torch.zeros_like(e1)
    mc.mc_run_range(eng.ctx, cfg["beam"], n, 0, 17001, 9, B, e1)
    mc.mc_run_range(eng.ctx, cfg["beam"], n, 17001, n, 9, B, e2)
    e1 += e2
    torch.cuda.synchronize()
    d1 = torch.zeros(eng.nvox, dtype=torch.float32, device="cuda")
    s1 = torch.zeros_like(d1)
    mc.mc_finalize(eng.ctx, e1, n, B, d1, s1)
    # deterministic per history; grid sums differ only by fp32 summation order
    assert np.allclose(d1.cpu().numpy(), d0, rtol=2e-5, atol=1e-7 * d0.max())
    assert np.allclose(s1.cpu().numpy(), s0, rtol=5e-3, atol=1e-6 * d0.max())
    # ragged batches: n not a multiple of B; n == B (one history per batch)
    d2, s2 = eng.run(cfg["beam"], 1003, 9, 7)
    assert np.isfinite(d2).all() and d2.max() > 0
    d3, s3 = eng.run(cfg["beam"], 5, 9, 5)
    assert np.isfinite(d3).all() and np.isfinite(s3).all()
    eng.close()


def test_finalize_kernel_against_the_oracle_statistics():
    cfg = W.config(1)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    orc = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    rng = np.random.default_rng(0)
    B, n = 7, 1003
    edep = rng.gamma(2.0, 1.0, (B, eng.nvox)).astype(np.float32)
    d, s = np.zeros(eng.nvox, np.float32), np.zeros(eng.nvox, np.float32)
    mc.mc_finalize(eng.ctx, edep, n, B, d, s)
    do, so = orc.finalize(edep.astype(np.float64), n)
    assert np.allclose(d, do, rtol=1e-6) and np.allclose(s, so, rtol=1e-5)
    eng.close()


def test_beam_that_misses_and_energy_ledger_of_escapes():
    cfg = W.config(1)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    miss = W.beam(W.ELECTRON, W.PENCIL, energy=6.0, entry=(40.0, 0.0, 0.0))
    d, s = eng.run(miss, 1000, 1, 4)
    st = eng.stats()
    assert d.max() == 0 and s.max() == 0
    assert st["e_escaped_MeV"] == pytest.approx(6000.0, rel=1e-6) and st["n_electron_steps"] == 0
    eng.close()


def test_queue_overflow_is_reported_never_dropped():
    """R21: with admission control off, a queue too small for the secondaries of one wave -> MC_ERR_QUEUE_OVERFLOW
    and no result; with it on (the default) the scheduler admits fewer primaries per launch and the same tiny
    queue suffices."""
    cfg = W.config(2)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    mc.mc_set_option(eng.ctx, "wave_size", 4096)
    mc.mc_set_option(eng.ctx, "queue_factor", 2)
    mc.mc_set_option(eng.ctx, "adaptive", 0)
    with pytest.raises(mc.McError) as e:
        eng.run(cfg["beam"], 200000, 1, 10)
    assert e.value.status == mc.MC_ERR_QUEUE_OVERFLOW
    mc.mc_set_option(eng.ctx, "adaptive", 1)
    d, _ = eng.run(cfg["beam"], 200000, 1, 10)
    st = eng.stats()
    assert _ledger(st) < 1e-4 and d.max() > 0 and st["n_histories"] == 200000
    eng.close()


def test_scheduling_options_do_not_change_the_result():
    """R14: wave size / refill threshold / blocks per SM are launch-order knobs; every history keeps its own
    stream, so the grids agree to fp32 summation order."""
    cfg = W.config(4, "e")
    n, B = 100000, 10
    ref = None
    for opts in ({}, {"wave_size": 8192, "queue_factor": 16}, {"refill_lanes": 1}, {"refill_lanes": 32, "blocks_per_sm": 1},
                 {"aggregate": 1}, {"aggregate": 0}, {"hard_lanes": 8, "refill_lanes": 48}, {"electron_threads": 512}, {"plan_ahead": 0},
                 {"plan_ahead": 0, "wave_size": 16384}):
        eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
        for k, v in opts.items():
            mc.mc_set_option(eng.ctx, k, v)
        d, _ = eng.run(cfg["beam"], n, 4, B)
        st = eng.stats()
        key = (st["n_electron_steps"], st["n_photon_flights"], st["n_moller"], st["n_brems"])
        if ref is None:
            ref = (d, key)
        else:
            assert key == ref[1], opts
            assert np.allclose(d, ref[0], rtol=1e-4, atol=1e-6 * ref[0].max()), opts
        eng.close()


def test_more_materials_pick_a_smaller_cta_and_give_the_same_histories():
    """8 materials x 256 nodes leave less shared memory for the track pools: the engine falls back to smaller CTAs
    (DESIGN.md "Kernels").  Materials the phantom does not use change nothing: same counters, same dose."""
    cfg = W.config(4, "e")
    n, B = 200000, 10
    mats8 = W.materials(3) + [W.water(), W.bone(), W.lung(), W.water(), W.bone()]
    res = []
    for mats in (cfg["materials"], mats8):
        eng = mc.Engine(cfg["phantom"], mats, cfg["params"])
        d, _ = eng.run(cfg["beam"], n, 6, B)
        st = eng.stats()
        assert _ledger(st) < 1e-4
        res.append((d, (st["n_electron_steps"], st["n_photon_flights"], st["n_moller"], st["n_brems"], st["n_compton"])))
        eng.close()
    assert res[0][1] == res[1][1]
    assert np.allclose(res[0][0], res[1][0], rtol=1e-4, atol=1e-6 * res[0][0].max())
    # 16 materials (the size of the paper's database) on a 128-node grid
    mats16 = mats8 + mats8
    eng = mc.Engine(cfg["phantom"], mats16, W.params(n_grid=128))
    d16, _ = eng.run(cfg["beam"], n, 6, B)
    assert _ledger(eng.stats()) < 1e-4 and abs(d16.sum() / res[0][0].sum() - 1.0) < 0.01
    eng.close()
    # beyond what any CTA size can hold: a clear error, not a crash
    eng = mc.Engine(cfg["phantom"], mats8, W.params(n_grid=1024))
    with pytest.raises(mc.McError) as e:
        eng.run(cfg["beam"], 1000, 1, 2)
    assert e.value.status == mc.MC_ERR_INVALID_ARG and "shared memory" in str(e.value)
    eng.close()


HIGH_STAT = [  # (config, beam, engine histories, oracle histories): the oracle's share is ~30 s of the host cores per case
    pytest.param(2, None, 10 ** 8, 3 * 10 ** 7, id="config2_15MeV_e_water"),
    pytest.param(3, None, 4 * 10 ** 8, 10 ** 8, id="config3_6MV_photons_water"),
    pytest.param(4, "e", 10 ** 8, 3 * 10 ** 7, id="config4_slab_electrons"),
    pytest.param(4, "g", 4 * 10 ** 8, 10 ** 8, id="config4_slab_photons"),
    pytest.param(5, "e", 10 ** 8, 10 ** 7, id="config5_halfslab_electrons"),
    pytest.param(5, "g", 4 * 10 ** 8, 10 ** 8, id="config5_halfslab_photons"),
]


def _curves(edep, rho, dims, voxel_cm, n_total):
    """Per-batch integrated curves from per-batch energy grids [B, nvox] (MeV): the depth curve (energy per history
    and slab) and two lateral profiles (mean dose over y and a 3 cm slab, depths 1-4 cm and 4-7 cm).  Returns
    {name: (mean over batches, standard error of that mean)}."""
    B = edep.shape[0]
    nx, ny, nz = dims
    h = float(voxel_cm[2])
    nb = np.array([-(-(b + 1) * n_total // B) - -(-b * n_total // B) for b in range(B)], np.float64)  # batch sizes (R18)
    inv_mass = 1.0 / (rho.reshape(nz, ny, nx).astype(np.float64) * float(np.prod(voxel_cm)))
    per = {"depth": [], "profile_1_4cm": [], "profile_4_7cm": []}
    for b in range(B):
        e = edep[b].reshape(nz, ny, nx).astype(np.float64) / nb[b]
        per["depth"].append(e.sum(axis=(1, 2)))
        for name, (z0, z1) in (("profile_1_4cm", (1.0, 4.0)), ("profile_4_7cm", (4.0, 7.0))):
            k0, k1 = int(round(z0 / h)), int(round(z1 / h))
            per[name].append((e[k0:k1] * inv_mass[k0:k1]).mean(axis=(0, 1)))
    out = {}
    for k, v in per.items():
        a = np.stack(v)
        out[k] = (a.mean(axis=0), a.std(axis=0, ddof=1) / np.sqrt(B))
    return out


@pytest.mark.parametrize("c,beam,n_gpu,n_orc", HIGH_STAT)
def test_depth_dose_profiles_and_total_energy_agree_at_high_statistics(c, beam, n_gpu, n_orc):
    """Integrated curves at high statistics, independent streams (engine seed 7, oracle seed 1): the laterally
    integrated depth-dose curve, two lateral profiles (PAPER.md:92 compares profiles at fixed depths) and the deposited
    fraction of the source energy.  Integration removes most of the noise, so a systematic difference of a few 0.1 % in
    range, energy loss, scattering or interface handling would show.
    Bars: depth curve within 0.3 % of its maximum, no noise allowance; profiles within 0.3 % of their maximum plus 4
    standard errors of the difference at that point (from the 20 batches of each side; the oracle's statistics are
    what ~30 s of the host cores buy) and within 0.6 % with no allowance; deposited energy fraction within 5e-4."""
    cfg = W.config(c, beam) if beam else W.config(c)
    ph = cfg["phantom"]
    B = 20
    eng = mc.Engine(ph, cfg["materials"], cfg["params"])
    orc = oracle.Oracle(ph, cfg["materials"], cfg["params"])
    eo, sto = orc.run_edep_parallel(cfg["beam"], n_orc, 1, B, WORKERS)
    co = _curves(eo, ph["density"], eng.dims, ph["voxel_cm"], n_orc)
    del eo
    eg = np.zeros((B, eng.nvox), np.float32)
    mc.mc_run_range(eng.ctx, cfg["beam"], n_gpu, 0, n_gpu, 7, B, eg)
    st = eng.stats()
    cg = _curves(eg, ph["density"], eng.dims, ph["voxel_cm"], n_gpu)
    del eg
    eng.close()
    res = {}
    for k in co:
        (mo, so), (mg, sg) = co[k], cg[k]
        diff, sd = np.abs(mg - mo), np.sqrt(so ** 2 + sg ** 2)
        res[k] = {"max_diff": float(diff.max() / mo.max()), "max_sigma": float(sd.max() / mo.max()),
                  "worst_excess": float(np.max(diff - 4.0 * sd) / mo.max())}
    res["energy"] = float(cg["depth"][0].sum() / co["depth"][0].sum())
    res["e_frac"] = (st["e_deposited_MeV"] / st["e_source_MeV"], sto["e_dep"] / sto["e_src"])
    print(c, beam, res)
    assert res["depth"]["max_diff"] < 3e-3, res
    for k in ("profile_1_4cm", "profile_4_7cm"):
        assert res[k]["worst_excess"] < 3e-3, (k, res)
        assert res[k]["max_diff"] < 6e-3, (k, res)  # point by point with no allowance (north_star's bar is 1 %)
    assert res["energy"] == pytest.approx(1.0, abs=5e-4), res
    assert res["e_frac"][0] == pytest.approx(res["e_frac"][1], abs=5e-4), res
    if c == 2:
        # 15 MeV electrons stop: the dose beyond ~the CSDA range (8.7 cm restricted, "fell quickly to
        # zero") is bremsstrahlung tail only
        zg = cg["depth"][0]
        assert zg[int(10.0 / 0.5):].max() < 0.02 * zg.max()


def test_mc_trim_hands_the_queue_pool_back_to_the_driver():
    """Queues of a destroyed context stay in the library's pool (reused by the next context); mc_trim releases them."""
    import torch
    cfg = W.config(1)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    eng.run(cfg["beam"], 400000, 1, 4)  # three queues of 4 x 400000 records x 48 B = 230 MB
    eng.close()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    mc.mc_trim(0)
    free1 = torch.cuda.mem_get_info()[0]
    assert free1 - free0 >= 200e6, (free0, free1)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])  # and a new context simply allocates again
    d, _ = eng.run(cfg["beam"], 20000, 1, 4)
    assert d.max() > 0 and _ledger(eng.stats()) < 1e-4
    eng.close()
