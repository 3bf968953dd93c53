"""Pins for the ORACLE's transport (run with -m "not gpu"): invariants and closed-form expectations
named by BASELINE.json north_star and SURVEY.md §8(c) "Pins"."""
import math

import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_1503_01722_b200 import workloads as W

MEC2 = 0.51099895


def _column(nz, hz, mat=0, rho=1.0, wide=200.0):
    """1 x 1 x nz column of very wide voxels: depth binning only."""
    ph = W.homogeneous_phantom((1, 1, nz), (wide, wide, hz), material=mat, density=rho)
    return ph


def _within(obs, exp, n, nsig=3.0, frac_ok=0.99):
    """binomial counts obs (per bin) against probabilities exp: >= frac_ok of bins within nsig sigma."""
    sig = np.sqrt(n * exp * (1 - exp)) + 1e-12
    z = np.abs(obs - n * exp) / sig
    return np.mean(z <= nsig) >= frac_ok and z.max() < 4.5


# ---- Woodcock tracking ---------------------------------------------------------
def test_narrow_beam_attenuation_homogeneous_fp64():
    """First-interaction depth of primaries follows exp(-mu x) within 3 sigma (north_star)."""
    ph = _column(40, 0.5)
    o = oracle.Oracle(ph, W.materials(1), W.params())
    E, n = 2.0, 200000
    bm = W.beam(W.PHOTON, W.PENCIL, energy=E)
    _, st, fv, fc = o.run_edep(bm, n, 5, 1, first=True)
    mu = o.lerp("mu_tot", E)  # rho = 1
    z = np.arange(41) * 0.5
    p = np.exp(-mu * z[:-1]) - np.exp(-mu * z[1:])
    obs = np.bincount(fv[fv >= 0], minlength=40)
    assert _within(obs, p, n)
    assert np.sum(fv < 0) == pytest.approx(n * math.exp(-mu * 20.0), abs=4 * math.sqrt(n * 0.4))
    # channel fractions = mu_channel / mu
    fr = np.bincount(fc[fc >= 0], minlength=3) / np.sum(fc >= 0)
    exp = np.array([o.lerp("mu_C", E), o.lerp("mu_pp", E), 0.0]) / mu
    exp[2] = 1 - exp[0] - exp[1]
    assert np.allclose(fr, exp, atol=4 * np.sqrt(exp * (1 - exp) / np.sum(fc >= 0)) + 1e-6)
    assert st["n_fict"] == 0  # homogeneous at the majorant density: no fictitious interactions


def test_attenuation_through_slab_and_fictitious_fraction():
    """exp(-sum mu_i x_i) through water/bone/lung/water; fictitious fraction in water under a bone
    majorant = 1 - mu_water/mu_maj."""
    nz, hz = 60, 0.5
    mat = np.zeros(nz, np.uint8)
    rho = np.ones(nz, np.float32)
    mat[6:10], rho[6:10] = 1, 1.85
    mat[10:24], rho[10:24] = 2, 0.26
    ph = _column(nz, hz)
    ph["material"], ph["density"] = mat, rho
    o = oracle.Oracle(ph, W.materials(3), W.params())
    E, n = 1.25, 200000
    _, st, fv, fc = o.run_edep(W.beam(W.PHOTON, W.PENCIL, energy=E), n, 9, 1, first=True)
    mus = np.array([rho[i] * o.lerp("mu_tot", E, m=int(mat[i])) for i in range(nz)])
    tau = np.concatenate([[0.0], np.cumsum(mus * hz)])
    p = np.exp(-tau[:-1]) - np.exp(-tau[1:])
    assert _within(np.bincount(fv[fv >= 0], minlength=nz), p, n)
    assert o.lerp("mu_maj", E) == pytest.approx(float(np.float32(1.85)) * o.lerp("mu_tot", E, m=1), rel=1e-12)
    # all-water phantom but majorant forced by one bone voxel far from the beam
    ph2 = W.homogeneous_phantom((3, 1, 40), (50.0, 50.0, 0.5))
    ph2["material"][0], ph2["density"][0] = 1, 1.85  # corner voxel (ix=0, iz=0), beam goes through ix=1
    o2 = oracle.Oracle(ph2, W.materials(3), W.params())
    n2 = 100000
    vox, ch, fl = o2.run_atten(W.beam(W.PHOTON, W.PENCIL, energy=E), n2, 2, o2.photon_tables_f32())
    f_exp = 1 - o2.lerp("mu_tot", E, m=0) / o2.lerp("mu_maj", E)
    # primaries fly straight through column ix=1 (water): every flight that ends inside is real w.p. mu_w/mu_maj
    n_int, n_esc = np.sum(vox >= 0), np.sum(vox < 0)
    inside = fl.sum() - n_esc
    f_obs = (inside - n_int) / inside
    assert f_exp == pytest.approx(0.434, abs=0.01)  # "fictitious fraction at 2 MeV ~ 43 % in water"
    assert f_obs == pytest.approx(f_exp, abs=4 * math.sqrt(f_exp * (1 - f_exp) / inside))
    # and the coupled fp64 transport sees fictitious interactions at a comparable rate
    o2.set_flags(W.FLAG_LOCAL_SECONDARIES)
    _, st2 = o2.run_edep(W.beam(W.PHOTON, W.PENCIL, energy=E), 20000, 2, 1)
    assert 0.4 < st2["n_fict"] / (st2["n_compton"] + st2["n_pair"] + st2["n_pe"] + st2["n_fict"]) < 0.65


def test_fp32_contract_path_matches_fp64_first_interactions():
    """The attenuation-only fp32 contract path (R20) and the fp64 transport agree on the voxel of the
    first interaction for all but a handful of borderline histories, and exactly on the flight count."""
    cfg = W.config(4, "g")
    ph = W.slab_phantom((15, 15, 60), 0.5)
    o = oracle.Oracle(ph, cfg["materials"], cfg["params"])
    n = 20000
    _, st, fv, fc = o.run_edep(cfg["beam"], n, 1, 1, first=True)
    v32, c32, fl = o.run_atten(cfg["beam"], n, 1, o.photon_tables_f32())
    assert np.mean(v32 == fv) > 0.999
    same = v32 == fv
    assert np.all(c32[same & (fv >= 0)].astype(np.int32) == fc[same & (fv >= 0)])
    assert np.all(c32[v32 < 0] == 255)


# ---- electrons -----------------------------------------------------------------------------------
def test_csda_path_length_equals_range_integral():
    """Hard events and MS off: total path = int_{e_cut}^{T0} dT/L within 0.5 % (north_star)."""
    ph = W.homogeneous_phantom((1, 1, 200), (50.0, 50.0, 0.1))
    o = oracle.Oracle(ph, W.materials(1), W.params(flags=W.FLAG_NO_HARD | W.FLAG_NO_MS))
    ec, gc = float(np.float32(0.2)), float(np.float32(0.01))
    f = lambda T: 1.0 / (o.eval("L_col", T, ec) + o.eval("L_rad", T, gc))
    for T0 in (6.0, 15.0):
        _, st = o.run_edep(W.electron_pencil(T0), 50, 1, 1)
        ref = integrate.quad(f, ec, T0, epsrel=1e-9, limit=200)[0]
        assert st["path_e"] / 50 == pytest.approx(ref, rel=5e-3)
        assert st["path_e"] / 50 == pytest.approx(ref, rel=3e-4)  # what it actually achieves
        assert st["e_esc"] == 0 and st["e_dep"] == pytest.approx(50 * T0, rel=1e-12)
        assert st["lim_event"] == 0 and st["n_moller"] == 0 and st["n_brems"] == 0


def test_electron_depth_dose_stops_at_range():
    """15 MeV e- in water: dose "fell quickly to zero" beyond the ~7-8 cm range; only
    the bremsstrahlung tail (<2 % of the maximum) remains."""
    ph = W.homogeneous_phantom((1, 1, 60), (200.0, 200.0, 0.5))
    o = oracle.Oracle(ph, W.materials(1), W.params())
    dose, sig, st = o.run(W.electron_pencil(15.0), 4000, 1, 4)
    assert dose[:11].min() > 0.5 * dose.max()
    assert dose[18:].max() < 0.02 * dose.max()
    assert 0 < dose[18:].sum()


@pytest.mark.parametrize("kind", ["e15", "g_spec", "positron", "g18_bone"])
def test_energy_ledger_closes_per_history(kind):
    """deposited + escaped (+ below cut-off, part of deposited) = source energy within 1e-5 (north_star)."""
    ph = W.slab_phantom((21, 21, 40), 0.5)
    mats = W.materials(3)
    if kind == "e15":
        bm, n = W.electron_field(15.0), 1500
    elif kind == "g_spec":
        bm, n = W.photon_field(), 20000
    elif kind == "positron":
        bm, n = W.beam(W.POSITRON, W.PENCIL, energy=4.0), 1500
    else:
        bm, n = W.beam(W.PHOTON, W.PENCIL, energy=18.0), 10000
        ph["material"][:] = 1
        ph["density"][:] = 1.85
    o = oracle.Oracle(ph, mats, W.params())
    edep, st = o.run_edep(bm, n, 3, 2)
    assert st["max_ledger_rel"] < 1e-5
    assert st["e_dep"] + st["e_esc"] == pytest.approx(st["e_src"], rel=1e-9)
    assert edep.sum() == pytest.approx(st["e_dep"], rel=1e-12)
    assert 0 < st["e_cutdep"] < st["e_dep"]
    if kind == "g18_bone":
        assert st["n_pair"] > 100  # pair production exercised (and positron annihilation with it)
    if kind == "positron":
        assert st["n_sec_g"] >= 2 * 1400  # two annihilation photons per stopped positron


def test_flags_keep_the_ledger_closed():
    ph = W.homogeneous_phantom((9, 9, 20), 0.5)
    for flags in (W.FLAG_NO_HARD, W.FLAG_NO_MS, W.FLAG_LOCAL_SECONDARIES, 7):
        o = oracle.Oracle(ph, W.materials(1), W.params(flags=flags))
        _, st = o.run_edep(W.electron_pencil(6.0), 300, 1, 1)
        assert st["max_ledger_rel"] < 1e-12
        if flags & W.FLAG_NO_HARD:
            assert st["n_moller"] + st["n_brems"] == 0


def test_one_voxel_phantom_and_dose_units():
    """dose * mass * N = E_src - escaped (R17: MeV/g per source particle)."""
    ph = W.homogeneous_phantom((1, 1, 1), (4.0, 4.0, 2.0), density=1.3)
    o = oracle.Oracle(ph, W.materials(1), W.params())
    n = 2000
    dose, sig, st = o.run(W.electron_pencil(6.0), n, 1, 10)
    assert dose[0] * 1.3 * 32.0 * n == pytest.approx(st["e_src"] - st["e_esc"], rel=1e-6)
    assert 0 < sig[0] < 0.05 * dose[0]


def test_pencil_beam_symmetry_and_total(water_oracle):
    cfg = W.config(1)
    n = 20000
    dose, sig, st = water_oracle.run(cfg["beam"], n, 1, 10, workers=2)
    D = dose.reshape(20, 20, 20)  # [iz, iy, ix]
    assert dose.sum() * 0.125 * n == pytest.approx(st["e_dep"], rel=1e-9)
    # R25: the axis runs along the edge shared by columns 9/10; compare sums over |i - 9.5| >= 1.5
    left, right = D[:, :, :8].sum(), D[:, :, 12:].sum()
    low, high = D[:, :8, :].sum(), D[:, 12:, :].sum()
    # x <-> y is an exact symmetry of the set-up; x <-> -x only up to the hinge truncation of the very
    # first step, which starts on the voxel edge (R8/R25), hence the wider band
    assert abs(left - low) < 0.08 * left and abs(right - high) < 0.08 * left
    assert abs(left - right) < 0.12 * left and abs(low - high) < 0.12 * left
    # the first leg deposits in column (10, 10) only
    assert D[0, 10, 10] > 2.5 * max(D[0, 9, 9], D[0, 9, 10], D[0, 10, 9])


# ---- statistics (R18) ----------------------------------------------------------------------------
def test_finalize_is_mean_and_standard_error_of_batch_means():
    ph = W.homogeneous_phantom((3, 2, 2), 0.5, density=1.7)
    o = oracle.Oracle(ph, W.materials(1), W.params())
    rng = np.random.default_rng(0)
    B, N = 7, 7003  # N not divisible by B: batch sizes differ by one
    edep = rng.uniform(0, 5, (B, o.nvox))
    dose, sig = o.finalize(edep, N)
    nb = np.bincount((np.arange(N) * B) // N, minlength=B)
    Db = edep / (1.7 * 0.125 * nb[:, None])
    assert np.allclose(dose, Db.mean(0), rtol=1e-13)
    assert np.allclose(sig, Db.std(0, ddof=1) / math.sqrt(B), rtol=1e-12)


def test_sigma_scales_as_inverse_sqrt_n_and_sharding_is_exact(water_oracle):
    bm = W.electron_pencil(6.0)
    d1, s1, _ = water_oracle.run(bm, 2000, 1, 10)
    d4, s4, _ = water_oracle.run(bm, 32000, 1, 10, workers=4)
    sel = d4 > 0.05 * d4.max()
    assert np.mean(s1[sel] / d1[sel]) / np.mean(s4[sel] / d4[sel]) == pytest.approx(4.0, rel=0.3)
    # history-keyed streams: disjoint history ranges on several processes give the same grids
    e_all, st_all = water_oracle.run_edep(bm, 2000, 1, 10)
    e_a, _ = water_oracle.run_edep(bm, 2000, 1, 10, 0, 700)
    e_b, _ = water_oracle.run_edep(bm, 2000, 1, 10, 700, 2000)
    assert np.allclose(e_a + e_b, e_all, rtol=1e-12, atol=1e-12)
    d_sh, _, st_sh = water_oracle.run(bm, 2000, 1, 10, workers=3)
    assert np.allclose(d_sh, d1, rtol=1e-12, atol=1e-15) and st_sh["n_estep"] == st_all["n_estep"]


def test_seed_and_history_change_the_stream(water_oracle):
    bm = W.electron_pencil(6.0)
    a, _ = water_oracle.run_edep(bm, 200, 1, 1)
    b, _ = water_oracle.run_edep(bm, 200, 2, 1)
    c, _ = water_oracle.run_edep(bm, 200, 1 + (1 << 32), 1)  # hi32(seed) enters the counter
    assert not np.allclose(a, b) and not np.allclose(a, c) and not np.allclose(b, c)


def test_heterogeneous_phantom_costs_more_work():
    """more fictitious photon interactions and more electron steps in the slab."""
    n = 3000
    res = {}
    for name, ph in (("water", W.homogeneous_phantom((31, 31, 60), 0.5)), ("slab", W.slab_phantom((31, 31, 60), 0.5))):
        o = oracle.Oracle(ph, W.materials(3), W.params())
        _, sg = o.run_edep(W.photon_field(), n, 1, 1)
        _, se = o.run_edep(W.electron_field(15.0), n // 10, 1, 1)
        res[name] = (sg["n_fict"] / sg["n_flight"], sg["n_flight"] / n, se["n_estep"] / (n // 10))
    assert res["water"][0] == 0.0 and res["slab"][0] > 0.3
    assert res["slab"][1] > 1.5 * res["water"][1]
