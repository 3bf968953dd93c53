"""Particle-list ("phase-space") source, SURVEY.md 8(f)2 / PAPER.md:84.  CPU part: the oracle's list source against
what its beam source and the invariants fix.  GPU part (-m gpu): mc_run_particles against the oracle."""
import numpy as np
import pytest

import oracle
from paper_1503_01722_b200 import workloads as W


def _orc(ph=None):
    ph = ph or W.homogeneous_phantom((16, 16, 24), 0.5)
    return ph, oracle.Oracle(ph, W.materials(3), W.params())


def test_listed_pencil_particles_reproduce_the_pencil_beam_statistically():
    """A list of identical 6 MeV electrons on the axis is the pencil beam of config 1 up to the stream layout (a listed
    primary starts at Philox block 0, a beam primary at block 1): same mean dose within the batch sigma."""
    cfg = W.config(1)
    orc = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    n, B = 20000, 10
    p = np.zeros(n, W.PARTICLE_DTYPE)
    p["w"], p["E"], p["particle"] = 1.0, 6.0, W.ELECTRON
    d_l, s_l, st_l = orc.run_particles(p, 3, B, workers=4)
    d_b, s_b, st_b = orc.run(cfg["beam"], n, 4, B, workers=4)
    assert st_l["max_ledger_rel"] < 1e-5 and st_l["n_hist"] == n
    m = d_b >= 0.1 * d_b.max()
    zz = (d_l[m] - d_b[m]) / np.sqrt(s_l[m] ** 2 + s_b[m] ** 2)  # studentised differences, ~23 voxels
    assert np.mean(zz ** 2) < 2.0 and np.max(np.abs(zz)) < 5.0
    assert abs(d_l.sum() - d_b.sum()) / d_b.sum() < 0.01
    assert st_l["n_estep"] / n == pytest.approx(st_b["n_estep"] / n, rel=0.02)


def test_list_source_energy_ledger_types_and_misses():
    ph, orc = _orc()
    p = W.phase_space(4000, seed=5, field=(4.0, 4.0))
    p["x"][:100] += 50.0  # 100 particles miss the phantom: escaped, never transported
    dose, sig, st = orc.run_particles(p, 9, 8, workers=2)
    assert st["max_ledger_rel"] < 1e-5
    e_src = float(np.sum(p["E"].astype(np.float64)) + 2 * 0.51099895 * np.sum(p["particle"] == W.POSITRON))
    assert st["e_src"] == pytest.approx(e_src, rel=1e-6)
    e_miss = float(np.sum(p["E"][:100].astype(np.float64)) + 2 * 0.51099895 * np.sum(p["particle"][:100] == W.POSITRON))
    assert st["e_esc"] >= e_miss * (1 - 1e-9)
    mass = ph["density"].astype(np.float64) * 0.125
    assert np.sum(dose * mass) * len(p) == pytest.approx(st["e_dep"], rel=1e-9)
    assert st["n_flight"] > 0 and st["n_estep"] > 0


def test_list_source_sharding_is_exact_and_order_matters_only_through_the_history_index():
    ph, orc = _orc()
    p = W.phase_space(1500, seed=2, field=(4.0, 4.0))
    d1, _, st1 = orc.run_particles(p, 7, 6, workers=1)
    d3, _, st3 = orc.run_particles(p, 7, 6, workers=3)
    assert np.allclose(d1, d3, rtol=1e-12, atol=1e-18) and st1["n_estep"] == st3["n_estep"]
    # a different seed changes the result, the same seed repeats it
    d2, _, _ = orc.run_particles(p, 8, 6)
    assert not np.allclose(d1, d2)
    d1b, _, _ = orc.run_particles(p, 7, 6)
    assert np.array_equal(d1, d1b)


def test_phase_space_generator_is_seeded_and_well_formed():
    a, b = W.phase_space(5000, seed=3), W.phase_space(5000, seed=3)
    assert a.tobytes() == b.tobytes() and a.dtype.itemsize == 32
    nrm = a["u"].astype(np.float64) ** 2 + a["v"].astype(np.float64) ** 2 + a["w"].astype(np.float64) ** 2
    assert np.all(np.abs(nrm - 1) < 1e-6) and np.all(a["E"] > 0) and np.all(a["E"] <= 6.0)
    assert set(np.unique(a["particle"])) == {-1, 0, 1}


# ---- GPU parity ----------------------------------------------------------------------------------------------
@pytest.mark.gpu
def test_mc_run_particles_matches_the_oracle():
    import torch
    import paper_1503_01722_b200 as mc
    assert torch.cuda.is_available()
    ph = W.slab_phantom((31, 31, 40), 0.5)
    mats, prm = W.materials(3), W.params()
    n, B = 1_000_000, 10
    p = W.phase_space(n, seed=11, field=(5.0, 5.0))
    p["x"][:1000] += 40.0  # some misses
    eng = mc.Engine(ph, mats, prm)
    orc = oracle.Oracle(ph, mats, prm)
    do, so, sto = orc.run_particles(p, 1, 40, workers=min(oracle.host_cores(), 32))
    res = {}
    for seed in (1, 2):
        d, s = np.zeros(eng.nvox, np.float32), np.zeros(eng.nvox, np.float32)
        mc.mc_run_particles(eng.ctx, p, seed, B, d, s)
        st = eng.stats()
        assert st["n_histories"] == n
        assert abs(st["e_deposited_MeV"] + st["e_escaped_MeV"] - st["e_source_MeV"]) / st["e_source_MeV"] < 1e-4
        assert st["e_source_MeV"] == pytest.approx(sto["e_src"], rel=1e-6)
        m = do >= 0.1 * do.max()
        diff = np.abs(d[m] - do[m])
        comb = np.sqrt(s[m].astype(np.float64) ** 2 + so[m] ** 2)
        res[seed] = (diff.mean() / do.max(), np.mean(diff <= 3 * comb), 0.8 * comb.mean() / do.max())
        for k_g, k_o in (("n_photon_flights", "n_flight"), ("n_compton", "n_compton"), ("n_moller", "n_moller"),
                         ("n_brems", "n_brems"), ("n_pair", "n_pair")):
            assert st[k_g] / n == pytest.approx(sto[k_o] / n, rel=0.02, abs=2e-3), (k_g, st[k_g], sto[k_o])
    assert res[1][0] <= 0.01, res            # same streams: strict 1 % bar
    assert res[2][1] >= 0.99, res            # independent streams: 3-sigma bar
    assert res[2][0] <= 0.01 + res[2][2], res
    # a device-resident list gives the same result as the host list (same seed)
    t = torch.from_numpy(p.view(np.uint8).reshape(-1)).cuda()
    d2, s2 = torch.zeros(eng.nvox, device="cuda"), torch.zeros(eng.nvox, device="cuda")
    mc.mc_run_particles(eng.ctx, t, 2, B, d2, s2, n=n)
    assert np.allclose(d2.cpu().numpy(), d, rtol=1e-4, atol=1e-6 * d.max())
    # validation of a host list
    bad = p[:10].copy(); bad["E"][3] = 25.0
    with pytest.raises(mc.McError) as e:
        mc.mc_run_particles(eng.ctx, bad, 1, 2, d, s)
    assert e.value.status == mc.MC_ERR_ENERGY_RANGE
    bad = p[:10].copy(); bad["u"][2] = 0.9
    with pytest.raises(mc.McError):
        mc.mc_run_particles(eng.ctx, bad, 1, 2, d, s)
    bad = p[:10].copy(); bad["particle"][4] = 5  # an unknown type is refused, not transported as a positron
    with pytest.raises(mc.McError) as e:
        mc.mc_run_particles(eng.ctx, bad, 1, 2, d, s)
    assert e.value.status == mc.MC_ERR_INVALID_ARG
    for wrong in (0.0, -1.0, float("nan")):  # the header's code for an energy outside (0, e_max]: as for a device list
        bad = p[:10].copy(); bad["E"][1] = wrong
        with pytest.raises(mc.McError) as e:
            mc.mc_run_particles(eng.ctx, bad, 1, 2, d, s)
        assert e.value.status == mc.MC_ERR_ENERGY_RANGE
    # ... and of a device-resident list (checked by one kernel pass, same error codes)
    bad = p[:1000].copy(); bad["E"][777] = 25.0
    tb = torch.from_numpy(bad.view(np.uint8).reshape(-1)).cuda()
    with pytest.raises(mc.McError) as e:
        mc.mc_run_particles(eng.ctx, tb, 1, 2, d2, s2, n=len(bad))
    assert e.value.status == mc.MC_ERR_ENERGY_RANGE
    bad = p[:1000].copy(); bad["u"][5] = 0.9
    tb = torch.from_numpy(bad.view(np.uint8).reshape(-1)).cuda()
    with pytest.raises(mc.McError) as e:
        mc.mc_run_particles(eng.ctx, tb, 1, 2, d2, s2, n=len(bad))
    assert e.value.status == mc.MC_ERR_INVALID_ARG
    bad = p[:1000].copy(); bad["particle"][999] = 5
    tb = torch.from_numpy(bad.view(np.uint8).reshape(-1)).cuda()
    with pytest.raises(mc.McError) as e:
        mc.mc_run_particles(eng.ctx, tb, 1, 2, d2, s2, n=len(bad))
    assert e.value.status == mc.MC_ERR_INVALID_ARG
    mc.mc_run_particles(eng.ctx, t, 2, B, d2, s2, n=n)  # the context still works after a rejected list
    assert np.allclose(d2.cpu().numpy(), d, rtol=1e-4, atol=1e-6 * d.max())
    eng.close()


@pytest.mark.gpu
def test_mc_run_source_user_gpu_and_cpu_functions_reproduce_the_list():
    """"a user can either load source particles from a phase-space file or write a CPU/GPU function".  The
    function is called once per wave; a GPU function enqueues its work on the stream it is given (here: a torch kernel
    plus a device-to-device copy), a CPU function copies from host memory.  Both must reproduce mc_run_particles on the
    same records exactly (same histories, same streams), over several waves."""
    import ctypes as C
    import torch
    import paper_1503_01722_b200 as mc
    assert torch.cuda.is_available()
    cudart = C.CDLL("libcudart.so.12")
    cfg = W.config(4, "g")
    n, B = 60000, 6
    p = W.phase_space(n, seed=5)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    mc.mc_set_option(eng.ctx, "wave_size", 16384)
    d0, s0 = np.zeros(eng.nvox, np.float32), np.zeros(eng.nvox, np.float32)
    mc.mc_run_particles(eng.ctx, p, 3, B, d0, s0)
    st0 = eng.stats()
    t_all = torch.from_numpy(p.view(np.uint8).reshape(-1).copy()).cuda()
    calls = []

    def gpu_fn(h0, cnt, out, stream):
        calls.append((h0, cnt))
        with torch.cuda.stream(torch.cuda.ExternalStream(stream) if stream else torch.cuda.default_stream()):
            chunk = t_all[32 * h0:32 * (h0 + cnt)].clone()  # the user's own kernel, on the library's stream
            rc = cudart.cudaMemcpyAsync(C.c_void_p(out), C.c_void_p(chunk.data_ptr()), C.c_size_t(32 * cnt), 3, C.c_void_p(stream))
            chunk.record_stream(torch.cuda.current_stream())
        return rc

    def cpu_fn(h0, cnt, out, stream):
        q = np.ascontiguousarray(p[h0:h0 + cnt])
        return cudart.cudaMemcpy(C.c_void_p(out), C.c_void_p(q.ctypes.data), C.c_size_t(32 * cnt), 1)

    for fn in (gpu_fn, cpu_fn):
        d, s = np.zeros(eng.nvox, np.float32), np.zeros(eng.nvox, np.float32)
        mc.mc_run_source(eng.ctx, fn, n, 3, B, d, s)
        st = eng.stats()
        assert (st["n_electron_steps"], st["n_photon_flights"], st["n_compton"]) == (st0["n_electron_steps"], st0["n_photon_flights"], st0["n_compton"])
        assert np.allclose(d, d0, rtol=1e-4, atol=1e-6 * d0.max()) and np.allclose(s, s0, rtol=5e-3, atol=1e-6 * d0.max())
    assert calls == [(0, 16384), (16384, 16384), (32768, 16384), (49152, n - 49152)]  # ascending waves of at most wave_size
    # the same on a non-blocking context stream (torch streams are created non-blocking): a plain cudaMemcpy from pageable
    # memory goes through the legacy stream, which such a stream does not wait for by itself — the library orders the two
    side = torch.cuda.Stream()
    mc.mc_set_stream(eng.ctx, side.cuda_stream)
    for fn in (cpu_fn, gpu_fn):
        d, s = np.zeros(eng.nvox, np.float32), np.zeros(eng.nvox, np.float32)
        mc.mc_run_source(eng.ctx, fn, n, 3, B, d, s)
        st = eng.stats()
        assert (st["n_electron_steps"], st["n_photon_flights"], st["n_compton"]) == (st0["n_electron_steps"], st0["n_photon_flights"], st0["n_compton"])
        assert np.allclose(d, d0, rtol=1e-4, atol=1e-6 * d0.max())
    mc.mc_set_stream(eng.ctx, 0)
    calls.clear()
    # a function that fails, and records that break the contract
    with pytest.raises(mc.McError) as e:
        mc.mc_run_source(eng.ctx, lambda *a: 7, n, 3, B, d, s)
    assert e.value.status == mc.MC_ERR_INVALID_ARG
    bad = p.copy(); bad["E"][20000] = 99.0
    with pytest.raises(mc.McError) as e:
        mc.mc_run_source(eng.ctx, lambda h0, cnt, out, stream: cudart.cudaMemcpy(
            C.c_void_p(out), C.c_void_p(np.ascontiguousarray(bad[h0:h0 + cnt]).ctypes.data), C.c_size_t(32 * cnt), 1), n, 3, B, d, s)
    assert e.value.status == mc.MC_ERR_ENERGY_RANGE
    mc.mc_run_source(eng.ctx, cpu_fn, n, 3, B, d, s)  # the context still works
    assert np.allclose(d, d0, rtol=1e-4, atol=1e-6 * d0.max())
    eng.close()
