"""Transport-level pins of the ORACLE's electron code (run with -m "not gpu").

VERDICT round 1 "What's weak" 2: parts of Run::electron that no test would catch if they were wrong —
 (i)   the hard-event rate: d_event from Sigma_max(T) and the thinning Sigma_hard(T')/Sigma_max(T) (R6),
 (ii)  the hinge rule at voxel faces with multiple scattering on (R8) and the MS path bookkeeping (R8b),
 (iii) the MS strength inside transport, a = 1 - exp(-K1(T_mid) rho d) (R7),
 (iv)  the polar-axis branch of the rotation (R25) and the annihilation photons (R9).
Each is pinned to something the mathematics fixes, computed here from the CLOSED FORMS (orc.eval) by independent
quadrature, never from the transport code or its tables: the survival probability exp(-int Sigma/L dT) of an electron
that slows down continuously, and <cos theta> = exp(-int K1/L dT) of Goudsmit-Saunderson theory for any single-scattering law
(Lewis 1950), which every condensed-history MS model must reproduce (PAPER.md:39 random hinge + MS angle).
The per-history observables come from orc_run_probe, which runs the same Run::history as orc_run.
"""
import math

import numpy as np
import pytest
from scipy import integrate, stats

import oracle
from paper_1503_01722_b200 import workloads as W

E_CUT, G_CUT = 0.2, 0.01


def _one_voxel(side=400.0):
    return W.homogeneous_phantom((1, 1, 1), side)


def _L(orc, T, e_cut=E_CUT, g_cut=G_CUT):
    return orc.eval("L_col", T, e_cut) + orc.eval("L_rad", T, g_cut)


# ---- (i) hard-event rate ("distance to the next hard event"; R6) -------------------------------------
def _hard_event_expectations(orc, T0):
    """From the closed forms: an electron that loses energy continuously from T0 to e_cut (rho cancels) meets its first
    hard event at kinetic energy T with density S(T) Sigma_hard(T)/L(T), S(T) = exp(-int_T^T0 Sigma_hard/L)."""
    sm = lambda T: orc.eval("S_M", T, E_CUT)
    sb = lambda T: orc.eval("S_br", T, G_CUT)
    Ts = np.exp(np.linspace(math.log(E_CUT), math.log(T0), 1201))
    rate_m = np.array([sm(t) / _L(orc, t) for t in Ts])
    rate_b = np.array([sb(t) / _L(orc, t) for t in Ts])
    # cumulative integral from T down to ... : I(T) = int_T^T0 (rate_m + rate_b) dT (trapezoid on a fine log grid)
    r = rate_m + rate_b
    seg = 0.5 * (r[1:] + r[:-1]) * np.diff(Ts)
    I = np.concatenate([np.cumsum(seg[::-1])[::-1], [0.0]])  # I[j] = int_{Ts[j]}^{T0}
    S = np.exp(-I)
    p_none = S[0]
    p_m = np.sum(0.5 * (S[1:] * rate_m[1:] + S[:-1] * rate_m[:-1]) * np.diff(Ts))
    p_b = np.sum(0.5 * (S[1:] * rate_b[1:] + S[:-1] * rate_b[:-1]) * np.diff(Ts))
    assert abs(p_none + p_m + p_b - 1.0) < 2e-4  # the three outcomes are exhaustive: checks the quadrature itself
    cdf = lambda T: (np.interp(T, Ts, S) - p_none) / (1.0 - p_none)  # P(T_first <= T | an event happened)
    return p_none, p_m, p_b, cdf


@pytest.mark.parametrize("T0,ms_on", [(2.0, False), (1.0, True), (6.0, False)])
def test_first_hard_event_probability_type_and_spectrum(T0, ms_on):
    """P(no hard event before the cut-off), P(first event is Moller / bremsstrahlung) and the spectrum of the energy at
    the first event against the quadrature of Sigma/L (4 sigma; KS p > 0.003).  Sensitive to the energy the thinning uses
    (T' at the event, not T at the start of the step), to the table it uses and to the d_event sampling: evaluating the
    acceptance at the step's START energy moves P(none) by 2-6 sigma-equivalents at T0 = 1-2 MeV (checked by mutation)."""
    n = 200000
    flags = W.FLAG_LOCAL_SECONDARIES | (0 if ms_on else W.FLAG_NO_MS)
    orc = oracle.Oracle(_one_voxel(), W.materials(1), W.params(flags=flags))
    p_none, p_m, p_b, cdf = _hard_event_expectations(orc, T0)
    pb, st = orc.run_probe(W.beam(W.ELECTRON, W.PENCIL, energy=T0, entry=(0.0, 0.0, 200.0)), n, 11)
    first = pb["first_hard"]
    for k, p in ((0, p_none), (1, p_m), (2, p_b)):
        obs = np.mean(first == k)
        assert abs(obs - p) <= 4.0 * math.sqrt(p * (1 - p) / n) + 2e-4, (T0, k, obs, p)
    Tf = pb["T_first"][first > 0]
    ks = stats.kstest(Tf, cdf)
    assert ks.pvalue > 0.003, (T0, ks)
    # thinning: candidates are rejected with probability 1 - Sigma_hard(T')/Sigma_max(T) > 0 (energy lost inside the step)
    assert pb["fict_before_first"].sum() > 0


def test_event_counts_per_history_match_the_rate_in_a_thin_slab():
    """15 MeV electrons through a 0.2 cm water slab (PAPER.md:39's beam energy): Moller and bremsstrahlung events per history
    = rho Sigma t to first order; second-order terms (energy change after an event) are < 1 % here.  Sigma values:
    SURVEY.md 8(c) pins, Sigma_M/rho(15 MeV) = 0.4218, Sigma_br/rho(15 MeV) = 0.2310 cm^2/g."""
    n, t = 400000, 0.2
    ph = W.homogeneous_phantom((1, 1, 1), (400.0, 400.0, t))
    orc = oracle.Oracle(ph, W.materials(1), W.params(flags=W.FLAG_LOCAL_SECONDARIES | W.FLAG_NO_MS))
    _, st = orc.run_edep(W.beam(W.ELECTRON, W.PENCIL, energy=15.0), n, 3, 1)
    # mean energy in the slab ~ 15 - 0.2 MeV: both cross sections are flat there (d ln Sigma / d ln T < 0.05)
    exp_m, exp_b = 0.4218 * t, 0.2310 * t
    assert st["n_moller"] / n == pytest.approx(exp_m, rel=0.012)
    assert st["n_brems"] / n == pytest.approx(exp_b, rel=0.015)


# ---- (iii) MS strength inside transport, (ii) hinge rule + MS path bookkeeping -------------------------------------
def _G(orc, T0, T1, e_cut):
    """int_{T1}^{T0} K1(T)/L(T) dT from the closed forms (scattering power along the slowing-down)."""
    f = lambda lt: orc.eval("K1", math.exp(lt)) / _L(orc, math.exp(lt), e_cut) * math.exp(lt)
    return integrate.quad(f, math.log(T1), math.log(T0), epsabs=1e-10, epsrel=1e-8)[0]


def _mean_cos(orc, T0, n, angle_deg, seed=5):
    bm = W.beam(W.ELECTRON, W.PENCIL, energy=T0, entry=(0.013, 0.027, 0.0))
    th = math.radians(angle_deg)
    bm["axis"] = np.array((math.sin(th), 0.0, math.cos(th)), np.float32)
    pb, st = orc.run_probe(bm, n, seed)
    ax = bm["axis"].astype(np.float64)
    ax /= np.linalg.norm(ax)
    ok = pb["escaped"] == 0
    assert ok.mean() > 0.99
    c = pb["dir"][ok] @ ax
    return c.mean(), c.std() / math.sqrt(ok.sum()), pb


def test_ms_strength_in_one_voxel_is_the_product_of_the_step_means():
    """Hard events off, one huge voxel: the steps are the same for every history (d = min[d_maxs, d_maxe, d_range]), so
    <Omega . Omega_0> at the cut-off = prod_i <mu_i>, <mu> = 1 - a + 2/(exp(2/a) - 1) exactly for the model of R7 with
    a_i = 1 - exp(-K1(T_mid,i) rho d_i).  The product is rebuilt here from the closed forms and the tabulated range only
    (no transport code).  SURVEY 8(c) pin "MS"."""
    T0, e_cut, n = 15.0, 10.0, 200000
    pr = W.params(e_cut=e_cut, flags=W.FLAG_NO_HARD)
    orc = oracle.Oracle(_one_voxel(), W.materials(1), pr)
    m, se, pb = _mean_cos(orc, T0, n, 0.0)
    # replay the deterministic step sequence
    T, prod = T0, 1.0
    while T > e_cut * (1 + 1e-12):
        R0, L0 = orc.lerp("R", T), orc.lerp("L", T)
        d = min(pr["d_maxs_cm"], pr["f_maxe"] * T / L0, R0)
        Tmid = orc.inv_range(R0 - 0.5 * d)
        a = 1.0 - math.exp(-orc.eval("K1", Tmid) * d)
        prod *= 1.0 - a + 2.0 / math.expm1(2.0 / a)
        T = e_cut if d >= R0 else orc.inv_range(R0 - d)
    assert abs(m - prod) <= 3.5 * se + 2e-5, (m, prod, se)
    # and the product is the Lewis / Goudsmit-Saunderson first moment to the accuracy of the midpoint rule
    assert -math.log(m) == pytest.approx(_G(orc, T0, e_cut, e_cut), rel=0.012)


@pytest.mark.parametrize("vox,T0,e_cut,angle", [(0.25, 15.0, 10.0, 20.0), (0.5, 6.0, 3.0, 10.0), (0.25, 2.0, 1.0, 0.0)])
def test_ms_on_a_voxel_grid_keeps_the_first_moment(vox, T0, e_cut, angle):
    """The same observable on a voxel grid, where most steps end on a face (hinge rule R8): -ln<cos> = int K1/L dT within
    1 % (+ 3 sigma) with the MS path bookkeeping of R8b.  Without it (round-1 reading: the angle is sampled for the planned
    path while the particle travels the actual one) the scattering power comes out 2-7 % too large — asserted too, so that
    the pin is known to see the effect."""
    n = 120000
    nn = int(round(40.0 / vox))
    orc = oracle.Oracle(W.homogeneous_phantom((nn, nn, nn), vox), W.materials(1), W.params(e_cut=e_cut, flags=W.FLAG_NO_HARD))
    G = _G(orc, T0, e_cut, e_cut)
    big = oracle.Oracle(_one_voxel(), W.materials(1), W.params(e_cut=e_cut, flags=W.FLAG_NO_HARD))
    m1, se1, _ = _mean_cos(big, T0, n, angle)   # the model's own value without voxel faces
    m, se, pb = _mean_cos(orc, T0, n, angle)
    ratio, err = -math.log(m) / G, se / m / G
    assert abs(ratio - 1.0) <= 0.01 + 3.0 * err, (ratio, err)
    # finer steps bring the model closer to the exact first moment, never further: between the one-voxel value and G
    assert -math.log(m) >= -math.log(m1) - 3.0 * (se1 / m1 + se / m), (m, m1)
    # bookkeeping identity: what the angles were sampled for = what was travelled (up to the last step's remainder)
    assert pb["q_sampled"].sum() / pb["q_travelled"].sum() == pytest.approx(1.0, abs=2e-3)
    for overrun in (0.0, 0.25):
        orc.set_option("ms_carry", 0)
        orc.set_option("hinge_overrun", overrun)
        mb, seb, pbb = _mean_cos(orc, T0, n, angle)
        assert pbb["q_sampled"].sum() / pbb["q_travelled"].sum() > 1.005  # angles sampled for more path than travelled
        if T0 <= 6.0:
            assert -math.log(mb) / G > 1.02, (overrun, -math.log(mb) / G)
    orc.set_option("ms_carry", 1)
    orc.set_option("hinge_overrun", 0.25)


def test_hinge_overrun_ab_depth_dose():
    """R8 A/B: the second leg may run on to the face by <= 25 % of its planned length (default)
    against the plain rule (0), same seed, config-2 beam on water and on the slab phantom (61 x 61 x 60 at 0.5 cm), 4e5
    histories.  Observables with little noise: energy-weighted mean depth, laterally integrated depth dose, energy-weighted
    <x^2> of the lateral profile at 2.5-3.5 cm and 5-6 cm depth, total energy.  Measured at 1e6 histories with R8b in
    place: mean depth 3.5994 vs 3.6000 cm (water), 3.2392 vs 3.2402 cm (slab), depth dose within 0.2 % of its maximum,
    <x^2> within 0.1 %: the bounds below are those with margin for 4e5 histories.  (Without R8b both rules give a mean
    depth 0.2 % smaller: the over-scattering the grid-MS pin above measures.)"""
    n, B = 400000, 10
    x = (np.arange(61) - 30) * 0.5
    z = (np.arange(60) + 0.5) * 0.5
    for ph in (W.homogeneous_phantom((61, 61, 60), 0.5), W.slab_phantom()):
        res = {}
        for ov in (0.0, 0.25):
            orc = oracle.Oracle(ph, W.materials(3), W.params())
            orc.set_option("hinge_overrun", ov)
            dose, sig, st = orc.run(W.electron_field(15.0), n, 1, B, workers=min(8, oracle.host_cores()))
            e = (dose * ph["density"]).reshape(60, 61, 61)  # energy per voxel (up to the constant voxel volume)
            dd = e.sum(axis=(1, 2))
            x2 = [float((e[lo:hi].sum(axis=(0, 1)) * x * x).sum() / e[lo:hi].sum()) for lo, hi in ((5, 7), (10, 12))]
            res[ov] = (dd, float((dd * z).sum() / dd.sum()), x2, st["n_estep"] / n)
        (dd0, zm0, x20, s0), (dd1, zm1, x21, s1) = res[0.0], res[0.25]
        assert s1 < 0.85 * s0                      # what the rule is for: fewer steps per history
        assert abs(zm1 / zm0 - 1.0) < 1.5e-3, (zm0, zm1)
        assert np.abs(dd1 - dd0).max() / dd0.max() < 0.004
        assert np.allclose(x21, x20, rtol=5e-3), (x20, x21)
        assert dd1.sum() == pytest.approx(dd0.sum(), rel=1e-3)  # total deposited energy


# ---- (iv) rotation at the poles, annihilation photons ----------------------------------------------------------------
def test_rotation_keeps_the_polar_angle_everywhere_including_the_poles():
    """R25: after rotate(d, mu, phi) the new direction is a unit vector at polar cosine mu from d, for generic directions,
    for d = +-z exactly (polar-axis branch) and just off the pole (the general branch at its most ill-conditioned);
    azimuth phi and phi + pi give mirror images about d."""
    rng = np.random.default_rng(3)
    dirs = [np.array([0.0, 0.0, 1.0]), np.array([0.0, 0.0, -1.0])]
    for eps in (1e-6, 2e-5, 1e-3):
        for sgn in (1.0, -1.0):
            dirs.append(np.array([eps, -0.5 * eps, sgn * math.sqrt(1 - 1.25 * eps * eps)]))
    for _ in range(20):
        v = rng.normal(size=3)
        dirs.append(v / np.linalg.norm(v))
    for d in dirs:
        for mu in (1.0, 0.999999, 0.3, -0.7, -1.0):
            for phi in (0.0, 0.4, 2.0, 5.5):
                o = oracle.rotate(d, mu, phi)
                assert abs(np.linalg.norm(o) - 1.0) < 1e-12
                # within 1e-5 rad of the pole the polar-axis branch treats d as +-z exactly (R25: 1 - w^2 < 1e-10)
                # (R25: 1 - w^2 < 1e-10); just outside, the general branch loses digits to the cancellation in 1 - w^2
                s2 = 1.0 - d[2] * d[2]
                tol = 2e-9 if s2 > 1e-4 or abs(d[2]) == 1.0 else (2e-5 if s2 < 1e-10 else 2e-7)
                assert abs(float(o @ d) - mu) < tol, (d, mu, phi, o)
                o2 = oracle.rotate(d, mu, phi + math.pi)
                perp, perp2 = o - mu * d, o2 - mu * d
                assert np.allclose(perp, -perp2, atol=10 * tol)
    # at the pole the azimuth is measured from +x: (sin t cos phi, sin t sin phi, +-cos t)
    o = oracle.rotate([0, 0, 1.0], 0.5, 0.3)
    st = math.sqrt(0.75)
    assert np.allclose(o, [st * math.cos(0.3), st * math.sin(0.3), 0.5], atol=1e-12)


def test_annihilation_photons_are_isotropic_and_back_to_back():
    """R9: the direction sampler the transport code calls is isotropic (<mu> = 0, <mu^2> = 1/3, uniform azimuth, chi-square),
    and a positron that stops emits its two photons exactly back to back (probe of Run::electron)."""
    d = oracle.sample_iso(200000, 9)
    assert np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-12)
    n = len(d)
    assert abs(d[:, 2].mean()) < 4 / math.sqrt(3 * n)
    assert abs((d[:, 2] ** 2).mean() - 1 / 3) < 4 * math.sqrt(4 / 45 / n)
    h, _ = np.histogram(d[:, 2], bins=20, range=(-1, 1))
    assert stats.chisquare(h).pvalue > 0.01
    h, _ = np.histogram(np.arctan2(d[:, 1], d[:, 0]), bins=24, range=(-math.pi, math.pi))
    assert stats.chisquare(h).pvalue > 0.01
    orc = oracle.Oracle(_one_voxel(), W.materials(1), W.params(flags=W.FLAG_LOCAL_SECONDARIES))
    pb, st = orc.run_probe(W.beam(W.POSITRON, W.PENCIL, energy=0.5, entry=(0.0, 0.0, 200.0)), 2000, 2)
    assert np.all(pb["annih_sum"] == 0.0)
    assert st["n_sec_g"] - st["n_brems"] == 2 * 2000  # two annihilation photons per positron (+ a few brems photons)
    assert abs(pb["annih_mu"].mean()) < 4 / math.sqrt(3 * 2000)
    # the rest energy comes back: deposited = kinetic + 2 mc^2 per history with local secondaries
    assert st["e_dep"] == pytest.approx(st["e_src"], rel=1e-12)


@pytest.mark.parametrize("T0", [1.0, 6.0, 15.0])
def test_bremsstrahlung_photon_is_emitted_at_the_most_probable_angle(T0):
    """the bremsstrahlung photon's direction is "the angle with the maximum differential cross section";
    reading R11 takes the textbook position of that maximum, theta = mc^2 / (T + mc^2) (= 1 / gamma) with T the kinetic
    energy AT the emission, about the electron's direction of flight, and leaves the electron's direction unchanged.
    Checked on the primary's first bremsstrahlung event of every history that has one: the angle between the two
    directions is exactly that number (not 1 / gamma of the beam energy, not mc^2 / T, not its cosine taken twice), for
    energies spread between the cut-off and T0; the azimuth is uniform (mean direction along the axis)."""
    mec2 = 0.51099895
    orc = oracle.Oracle(_one_voxel(), W.materials(1), W.params(flags=W.FLAG_LOCAL_SECONDARIES | W.FLAG_NO_MS))
    pb, _ = orc.run_probe(W.beam(W.ELECTRON, W.PENCIL, energy=T0, entry=(0.0, 0.0, 200.0)), 20000, 3)
    has = pb["T_brems"] > 0
    assert has.sum() > 500
    T, c = pb["T_brems"][has], pb["brems_cos"][has]
    assert T.max() <= T0 and T.min() < 0.8 * T0  # emissions along the track, not only at the beam energy
    theta = np.arccos(np.clip(c, -1.0, 1.0))
    assert np.allclose(theta, mec2 / (T + mec2), rtol=0, atol=2e-8)  # arccos near 1 loses half the digits: 1e-16 -> 1e-8
    # plausible mistakes are far outside that: 1/gamma of the beam energy, mc^2 / T, the angle's cosine used as the angle
    for wrong in (mec2 / (T0 + mec2) * np.ones_like(T), mec2 / T, np.cos(mec2 / (T + mec2))):
        assert np.max(np.abs(theta - wrong)) > 1e-3
