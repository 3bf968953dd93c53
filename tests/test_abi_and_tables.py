"""CPU-side checks of the C-ABI library (run with -m "not gpu"): it loads, exports every symbol
include/mc.h declares, validates arguments, and its host-side table builder (independent code,
Gauss-Legendre quadratures) agrees with the oracle's tables (Simpson quadratures) node by node.
No compute call is made: without a GPU they must fail loudly with MC_ERR_CUDA."""
import os
import re

import numpy as np
import pytest

import oracle
import paper_1503_01722_b200 as mc
from paper_1503_01722_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_1503_01722_b200 import build
    build.build()


def test_library_exports_every_declared_symbol():
    text = open(os.path.join(ROOT, "include", "mc.h")).read()
    declared = set(re.findall(r"\b(mc_[a-z_0-9]+)\s*\(", text))
    declared -= {"mc_ctx"}
    assert declared == set(mc.SYMBOLS), declared ^ set(mc.SYMBOLS)
    L = mc.lib()
    for s in mc.SYMBOLS:
        assert hasattr(L, s), s
    assert "sm_100a" in mc.mc_version()


def test_python_binding_has_one_function_per_symbol():
    for s in mc.SYMBOLS:
        assert callable(getattr(mc, s)), s


def test_struct_layouts_match_the_header():
    import ctypes as C
    assert C.sizeof(mc._Params) == 28
    assert C.sizeof(mc._Material) == 40
    assert C.sizeof(mc._Beam) == 64
    assert C.sizeof(mc._Stats) == 13 * 8 + 6 * 8 + 8
    assert mc.PARTICLE_DTYPE.itemsize == 32 and W.PARTICLE_DTYPE == mc.PARTICLE_DTYPE  # mc_particle


def test_create_rejects_bad_arguments():
    ph = W.homogeneous_phantom((3, 3, 3), 0.5)
    bad = dict(ph)
    bad["density"] = ph["density"].copy()
    bad["density"][5] = 0.0
    with pytest.raises(mc.McError) as e:
        mc.Engine(bad)
    assert e.value.status == mc.MC_ERR_INVALID_ARG
    bad = dict(ph)
    bad["voxel_cm"] = np.array([0.5, -0.5, 0.5], np.float32)
    with pytest.raises(mc.McError):
        mc.Engine(bad)
    bad = dict(ph)
    bad["dims"] = np.array([3, 0, 3], np.int32)
    bad["material"], bad["density"] = ph["material"][:0], ph["density"][:0]
    with pytest.raises(mc.McError):
        mc.Engine(bad)


def test_build_tables_rejects_bad_arguments_and_run_needs_tables():
    ph = W.homogeneous_phantom((3, 3, 3), 0.5)
    ph["material"][4] = 2
    eng = mc.Engine(ph)
    with pytest.raises(mc.McError) as e:  # material index 2 with one material
        mc.mc_build_tables(eng.ctx, W.materials(1), W.params())
    assert e.value.status == mc.MC_ERR_INVALID_ARG
    with pytest.raises(mc.McError) as e:  # run before tables
        eng.run(W.electron_pencil(6.0), 100, 1, 2)
    assert e.value.status == mc.MC_ERR_STATE
    with pytest.raises(mc.McError):
        mc.mc_export_table(eng.ctx, "mu_tot")
    for k, v in (("n_grid", 4), ("e_cut_MeV", -1.0), ("f_maxe", 0.0), ("d_maxs_cm", 0.0), ("e_max_MeV", 0.3)):
        p = W.params()
        p[k] = v
        with pytest.raises(mc.McError):
            mc.mc_build_tables(eng.ctx, W.materials(3), p)
    mc.mc_build_tables(eng.ctx, W.materials(3), W.params())  # re-callable after failures
    eng.close()


def test_run_argument_validation_happens_before_any_device_work():
    cfg = W.config(1)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    d, s = np.zeros(eng.nvox, np.float32), np.zeros(eng.nvox, np.float32)
    bm = cfg["beam"]
    for n, B in ((100, 1), (5, 10), (0, 2), (2**32, 10)):
        with pytest.raises(mc.McError) as e:
            mc.mc_run(eng.ctx, bm, n, 1, B, d, s)
        assert e.value.status == mc.MC_ERR_INVALID_ARG
    hot = W.electron_pencil(25.0)  # above e_max = 20 MeV
    with pytest.raises(mc.McError) as e:
        mc.mc_run(eng.ctx, hot, 100, 1, 2, d, s)
    assert e.value.status == mc.MC_ERR_ENERGY_RANGE
    tilted = dict(bm)
    tilted["axis"] = np.array([0.0, 0.6, 0.6], np.float32)
    with pytest.raises(mc.McError):
        mc.mc_run(eng.ctx, tilted, 100, 1, 2, d, s)
    with pytest.raises(mc.McError):  # attenuation mode takes photon beams only
        mc.mc_run_atten(eng.ctx, bm, 10, 1, np.zeros(10, np.int32))
    with pytest.raises(mc.McError):
        mc.mc_set_option(eng.ctx, "no_such_option", 1)
    with pytest.raises(mc.McError):
        mc.mc_set_option(eng.ctx, "wave_size", 3)
    eng.close()


def test_no_cpu_fallback_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    cfg = W.config(1)
    eng = mc.Engine(cfg["phantom"], cfg["materials"], cfg["params"])
    with pytest.raises(mc.McError) as e:
        eng.run(cfg["beam"], 1000, 1, 2)
    assert e.value.status == mc.MC_ERR_CUDA
    eng.close()


def test_product_path_never_touches_the_oracle():
    pk = os.path.join(ROOT, "paper_1503_01722_b200")
    for dp, _, fs in os.walk(pk):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "orc_" not in txt, f
                assert "liborc" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r'#include\s+"[^"]*(csrc|mc_|include/)', txt), f
            assert "libmc_b200" not in txt and "import paper_1503" not in txt and "from paper_1503" not in txt, f


# ---- table parity: two independent builders --------------------------------------
TOL = {"mu_tot": 2e-6, "mu_C": 2e-6, "mu_pp": 2e-6, "L": 5e-6, "S_M": 5e-6, "S_hard": 2e-5, "S_max": 2e-5,
       "K1": 5e-6, "R": 2e-5}


@pytest.mark.parametrize("params", [W.params(), W.params(e_cut=0.05, g_cut=0.05, n_grid=128),
                                    W.params(e_cut=0.5, g_cut=0.02, e_max=30.0, n_grid=512)])
def test_engine_tables_match_oracle_tables(params):
    ph = W.slab_phantom((5, 4, 30), 0.5)
    mats = W.materials(3)
    eng = mc.Engine(ph, mats, params)
    orc = oracle.Oracle(ph, mats, params)
    g, og = mc.mc_export_grid(eng.ctx), orc.grid()
    assert g["N"] == og["N"] and g["k_cut"] == og["k_cut"]
    assert g["lnE0"] == pytest.approx(og["lnE0"], abs=1e-13) and g["dln"] == pytest.approx(og["dln"], rel=1e-14)
    kc = g["k_cut"]
    for m in range(3):
        for name, tol in TOL.items():
            a = mc.mc_export_table(eng.ctx, name, m).astype(np.float64)
            b = orc.table(name, m)
            scale = np.maximum(np.abs(b), 1e-3 * np.abs(b).max())
            if name == "R":  # R crosses zero at e_cut: compare against the local node spacing of R
                scale = np.maximum(np.abs(b), np.abs(np.gradient(b)))
                assert a[kc] == 0.0 and b[kc] == 0.0
            err = np.abs(a - b) / scale
            assert err.max() <= tol, (name, m, int(err.argmax()), err.max())
    a, b = mc.mc_export_table(eng.ctx, "mu_maj").astype(np.float64), orc.table("mu_maj")
    assert np.all(np.abs(a - b) <= 3e-7 * b)
    eng.close()


def test_fp32_majorants_dominate_in_the_engine_tables():
    """Woodcock and hard-event thinning need mu_maj >= rho mu and Sigma_max >= Sigma_hard in the fp32
    tables actually used, node by node (lerp preserves dominance)."""
    ph = W.slab_phantom((5, 4, 30), 0.5)
    eng = mc.Engine(ph, W.materials(3), W.params())
    maj = mc.mc_export_table(eng.ctx, "mu_maj")
    rmax = [1.0, 1.85, 0.26]
    for m in range(3):
        mu = mc.mc_export_table(eng.ctx, "mu_tot", m)
        assert np.all(maj.astype(np.float64) >= np.float32(rmax[m]).astype(np.float64) * mu.astype(np.float64))
        sm, sh = mc.mc_export_table(eng.ctx, "S_max", m), mc.mc_export_table(eng.ctx, "S_hard", m)
        assert np.all(sm >= sh) and np.all(np.diff(sm) >= 0)
        R = mc.mc_export_table(eng.ctx, "R", m)
        assert np.all(np.diff(R) > 0)
    eng.close()


def test_set_photon_tables_round_trip():
    ph = W.slab_phantom((5, 4, 30), 0.5)
    eng = mc.Engine(ph, W.materials(3), W.params())
    t = mc.mc_export_photon_tables(eng.ctx, 3)
    t2 = {k: (v * np.float32(1.25) if isinstance(v, np.ndarray) else v) for k, v in t.items()}
    mc.mc_set_photon_tables(eng.ctx, t2)
    got = mc.mc_export_photon_tables(eng.ctx, 3)
    for k in ("mu_maj", "mu_tot", "mu_C", "mu_pp"):
        assert np.array_equal(got[k], t2[k])
    eng.close()


def test_run_particles_argument_validation_before_any_device_work():
    import numpy as np
    ph = W.homogeneous_phantom((4, 4, 4), 0.5)
    eng = mc.Engine(ph)
    p = W.phase_space(16, seed=1, field=(1.0, 1.0))
    d, s = np.zeros(64, np.float32), np.zeros(64, np.float32)
    with pytest.raises(mc.McError) as e:  # tables first
        mc.mc_run_particles(eng.ctx, p, 1, 2, d, s)
    assert e.value.status == mc.MC_ERR_STATE
    mc.mc_build_tables(eng.ctx, W.materials(1), W.params())
    with pytest.raises(mc.McError) as e:  # n_batches > n
        mc.mc_run_particles(eng.ctx, p, 1, 17, d, s)
    assert e.value.status == mc.MC_ERR_INVALID_ARG
    with pytest.raises(mc.McError) as e:  # n_batches < 2
        mc.mc_run_particles(eng.ctx, p, 1, 1, d, s)
    assert e.value.status == mc.MC_ERR_INVALID_ARG
    eng.close()


def test_engine_goudsmit_saunderson_tables_match_the_oracles():
    """Two independent builders of the same definition (R27): the material-independent quantile table
    (ln of the quantiles of 1 - cos theta over scattering power x screening parameter) and the per-material effective
    screening parameter.  Host code only: no device needed."""
    import oracle
    t, y = mc.mc_export_gs_table()
    To = oracle.gs_table()
    tn, An, rn = oracle.gs_nodes()
    assert y.shape == To.shape == oracle.gs_dims()
    assert np.allclose(t, tn, rtol=1e-6)
    assert np.max(np.abs(y - To)) < 3e-3 and np.mean(np.abs(y - To)) < 3e-4  # quantiles of x agree to 0.3 %
    ph = W.homogeneous_phantom((2, 2, 2), 1.0)
    eng = mc.Engine(ph, W.materials(3), W.params())
    orc = oracle.Oracle(ph, W.materials(3), W.params())
    for m in range(3):
        assert np.allclose(mc.mc_export_table(eng.ctx, "lnA", m), orc.table("lnA", m), atol=5e-6)
    eng.close()
