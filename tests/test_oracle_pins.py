"""Pins for the ORACLE's closed forms, tables and samplers (run with -m "not gpu").

Each test checks the oracle against something other than itself: published known answers, values
listed in SURVEY.md §8(c) (golden files cite them), textbook limits, numerical integrals of a
*different* formula (a differential cross section integrated to check a total), or analytic pdfs.
"""
import math

import numpy as np
import pytest
from scipy import integrate, stats

import oracle
from conftest import golden
from paper_1503_01722_b200 import workloads as W

MEC2 = 0.51099895
RE = 2.8179403e-13


# ---- RNG (R15) ------------------------------------------------------------------------
def test_philox_known_answers():
    for row in golden("philox4x32_10_kat.txt"):
        v = [int(x, 16) for x in row]
        assert oracle.philox(v[0:4], v[4:6]) == v[6:10]


def test_uniform_is_open_interval_and_fp32_exact():
    # u = ((w >> 9) + 0.5) * 2^-23 : 24 significant bits, never 0 or 1
    for w in (0, 0xFFFFFFFF, 0x000001FF, 0x80000000):
        u = ((w >> 9) + 0.5) * 2.0 ** -23
        assert 0.0 < u < 1.0 and float(np.float32(u)) == u


# ---- photons -------------------------------------------------------------------------------------
def test_water_closed_form_pins(water_oracle):
    for q, E, arg, val, tol in golden("water_closed_form_pins.txt"):
        got = water_oracle.eval(q, float(E), float(arg))
        assert got == pytest.approx(float(val), rel=float(tol) + 6e-4), (q, E)  # +: 4-digit rounding of the pin


def test_sigma_kn_thomson_limit_and_angular_integral(water_oracle):
    ref = {r[0]: r for r in golden("water_reference_data.txt") if r[0] in ("thomson", "compton_xcom")}
    assert water_oracle.eval("sigma_kn", 1e-6 * MEC2) == pytest.approx(float(ref["thomson"][2]), rel=1e-5)
    assert water_oracle.eval("mu_C", 1.0) == pytest.approx(float(ref["compton_xcom"][2]), rel=0.005)

    def dsdo(mu, k):  # Klein-Nishina dsigma/dOmega (textbook form), per electron
        P = 1.0 / (1.0 + k * (1.0 - mu))
        return 0.5 * RE * RE * P * P * (P + 1.0 / P - (1.0 - mu * mu))

    for E in (0.02, 0.3, 1.25, 6.0, 18.0):
        k = E / MEC2
        num = 2 * math.pi * integrate.quad(dsdo, -1, 1, args=(k,), epsabs=0, epsrel=1e-11)[0]
        assert water_oracle.eval("sigma_kn", E) == pytest.approx(num, rel=1e-9)


def test_pair_threshold_continuity_asymptote():
    assert oracle.sigma_pp_reduced(8, 2.0) == 0.0 and oracle.sigma_pp_reduced(8, 1.5) == 0.0
    lo, hi = oracle.sigma_pp_reduced(8, 4.0), oracle.sigma_pp_reduced(8, 4.0 + 1e-9)
    assert lo == pytest.approx(0.3265, rel=1e-3) and hi == pytest.approx(lo, rel=3e-4)
    k = 2.0e4
    assert oracle.sigma_pp_reduced(8, k) == pytest.approx(28.0 / 9.0 * math.log(2 * k) - 218.0 / 27.0, rel=1e-6)
    ks = np.linspace(2.0, 40.0, 400)
    v = np.array([oracle.sigma_pp_reduced(8, x) for x in ks])
    assert np.all(np.diff(v) >= 0)


def test_photoelectric_scaling(water_oracle):
    # Z^5 k^-3.5 per atom: ratio between two energies is exact
    r = water_oracle.eval("mu_pe", 0.02) / water_oracle.eval("mu_pe", 0.08)
    assert r == pytest.approx(4.0 ** 3.5, rel=1e-12)


# ---- electrons -----------------------------------------------------------------------------------
def test_estar_water_sanity(water_oracle):
    o = water_oracle
    for q, E, val, tol in golden("water_reference_data.txt"):
        E, val, tol = float(E), float(val), float(tol)
        if q == "S_col_estar":
            assert o.eval("L_col", E, 1e9) == pytest.approx(val, rel=tol)
        elif q == "S_rad_estar":
            assert o.eval("L_rad", E, 1e9) == pytest.approx(val, rel=tol)
        elif q == "csda_estar":
            r = integrate.quad(lambda T: 1.0 / (o.eval("L_col", T, 1e9) + o.eval("L_rad", T, 1e9)), 0.01, E,
                               epsrel=1e-6, limit=200)[0] + 2.5e-4
            assert r == pytest.approx(val, rel=tol)


def test_restricted_L_identity(water_oracle):
    """L_col(T, Delta) + n_e * int_Delta^{T/2} W dsigma_Moller = unrestricted S_col(T)."""
    o, D = water_oracle, 0.2
    ne = o.material_scalar("ne")
    for T in (0.5, 1.0, 6.0, 15.0):
        hard = integrate.quad(lambda e: e * T * o.eval("moller_dsde", T, e), D / T, 0.5, epsrel=1e-12, epsabs=0)[0]
        assert o.eval("L_col", T, D) + ne * hard == pytest.approx(o.eval("L_col", T, 1e9), rel=1e-12)


def test_moller_total_is_integral_of_differential(water_oracle):
    o = water_oracle
    ne = o.material_scalar("ne")
    assert o.eval("S_M", 0.4, 0.2) == 0.0 and o.eval("S_M", 0.39, 0.2) == 0.0
    for T in (0.41, 0.7, 3.0, 15.0):
        num = integrate.quad(lambda e: o.eval("moller_dsde", T, e), 0.2 / T, 0.5, epsrel=1e-12, epsabs=0)[0]
        assert o.eval("S_M", T, 0.2) == pytest.approx(ne * num, rel=1e-9)


def test_moller_differential_against_textbook_form():
    # dsigma/dW (ICRU 37 eq. 2.14 form): 2 pi r_e^2 mc^2 / (beta^2 T^2) [...] ; here in eps = W/T
    ph = W.homogeneous_phantom((1, 1, 1), 1.0)
    o = oracle.Oracle(ph, W.materials(1), W.params())
    T, eps = 2.0, 0.3
    tau = T / MEC2
    b2 = 1 - 1 / (tau + 1) ** 2
    txt = 2 * math.pi * RE ** 2 / (b2 * tau) * (1 / eps ** 2 + 1 / (1 - eps) ** 2 + (tau / (tau + 1)) ** 2
                                                - (2 * tau + 1) / (tau + 1) ** 2 / (eps * (1 - eps)))
    assert o.eval("moller_dsde", T, eps) == pytest.approx(txt, rel=1e-12)


def test_brems_total_and_radiative_loss_by_independent_quadrature(water_oracle):
    o = water_oracle
    for T in (0.3, 1.0, 15.0):
        # split at the screening kink to help the adaptive integrator
        f = lambda lk: o.eval("brems_kdsdk", T, math.exp(lk))
        num = integrate.quad(f, math.log(0.01), math.log(T), epsrel=1e-9, limit=400)[0]
        assert o.eval("S_br", T, 0.01) == pytest.approx(num, rel=2e-6)
        num2 = integrate.quad(lambda k: o.eval("brems_kdsdk", T, k), 0.0, 0.01, epsrel=1e-10)[0]
        assert o.eval("L_rad", T, 0.01) == pytest.approx(num2, rel=1e-6)


def test_density_effect_limits(water_oracle):
    o = water_oracle
    assert o.eval("delta", 0.05) == 0.0  # below X0
    # high-energy form 2 ln(beta gamma) + C, with C = -(2 ln(I/hnu_p) + 1)
    T = 1.0e4
    bg = math.sqrt((T / MEC2 + 1) ** 2 - 1)
    hnu = 28.816 * math.sqrt(1.0 * o.material_scalar("ZA"))
    C = -(2 * math.log(75.0 / hnu) + 1)
    assert o.eval("delta", T) == pytest.approx(4.606 * math.log10(bg) + C, rel=1e-12)


# ---- tables --------------------------------------------------------------------------------------
def test_grid_puts_cutoffs_on_nodes(water_oracle):
    g = water_oracle.grid()
    E = water_oracle.energies()
    ec = float(np.float32(0.2))  # cut-offs cross the C ABI as fp32
    assert E[g["k_cut"]] == pytest.approx(ec, rel=1e-12)
    n2 = round(math.log(2) / g["dln"])
    assert E[g["k_cut"] + n2] == pytest.approx(2 * ec, rel=1e-12)
    assert E[0] <= 0.01 and E[-1] >= 20.0 and g["N"] == 256


def test_tables_match_closed_forms_at_nodes_and_between(water_oracle):
    o = water_oracle
    E = o.energies()
    ec = float(np.float32(0.2))
    for name, q, arg in (("mu_C", "mu_C", 0), ("S_M", "S_M", ec), ("K1", "K1", 0)):
        t = o.table(name)
        for j in (3, 100, 124, 200, 255):
            assert t[j] == pytest.approx(o.eval(q, E[j], arg), rel=1e-9, abs=1e-300)
    assert o.table("S_M")[123] < 1e-12 and np.all(o.table("S_M")[:123] == 0.0)  # Moller threshold node
    # interpolation error between nodes is small for smooth quantities
    for j in (110, 180, 240):
        Em = math.sqrt(E[j] * E[j + 1])
        assert o.lerp("mu_C", Em) == pytest.approx(o.eval("mu_C", Em), rel=4e-4)
        assert o.lerp("K1", Em) == pytest.approx(o.eval("K1", Em), rel=6e-4)
    L = o.table("L")
    assert L[200] == pytest.approx(o.eval("L_col", E[200], 0.2) + o.eval("L_rad", E[200], 0.01), rel=1e-9)


def test_range_table_against_independent_quadrature(water_oracle):
    o = water_oracle
    ec, gc = float(np.float32(0.2)), float(np.float32(0.01))
    f = lambda T: 1.0 / (o.eval("L_col", T, ec) + o.eval("L_rad", T, gc))
    for T, pin in ((6.0, 3.376), (15.0, 8.705)):  # SURVEY.md §8(c) CSDA pin values (cm in water)
        num = integrate.quad(f, ec, T, epsrel=1e-9, limit=200)[0]
        assert o.lerp("R", T) == pytest.approx(num, rel=1.5e-4)  # lerp of a convex function: <= dln^2/8
        assert num == pytest.approx(pin, rel=5e-4)
    E, R = o.energies(), o.table("R")
    for j in (150, 210, 250):
        assert R[j] == pytest.approx(integrate.quad(f, ec, E[j], epsrel=1e-10, limit=200)[0], rel=1e-7)
    g = o.grid()
    assert o.table("R")[g["k_cut"]] == 0.0
    # inverse of the interpolant
    for T in (0.2001, 0.33, 1.7, 14.9):
        assert o.inv_range(o.lerp("R", T)) == pytest.approx(T, rel=1e-12)
    assert o.inv_range(0.0) == pytest.approx(0.2) and o.inv_range(-1.0) == pytest.approx(0.2)


def test_majorants_dominate():
    cfg = W.config(4, "g")
    o = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    maj = o.table("mu_maj")
    rho_max = {0: 1.0, 1: 1.85, 2: 0.26}
    for m in range(3):
        assert np.all(maj >= rho_max[m] * o.table("mu_tot", m) * (1 - 1e-15))
        smax, sh = o.table("S_max", m), o.table("S_hard", m)
        assert np.all(np.diff(smax) >= 0) and np.all(smax >= sh)
    assert np.allclose(maj, 1.85 * o.table("mu_tot", 1))  # bone is the majorant


# ---- samplers ------------------------------------------------------------------------------------
def _chi2_p(samples, edges, cdf):
    obs, _ = np.histogram(samples, edges)
    exp = np.diff([cdf(e) for e in edges])
    exp = exp / exp.sum() * obs.sum()
    return stats.chisquare(obs, exp).pvalue


@pytest.mark.parametrize("E,mean_pin", [(0.5, 0.6586), (2.0, 0.4692), (6.0, 0.3560)])
def test_klein_nishina_sampler(E, mean_pin):
    """chi-square p > 0.01 for eps and cos(theta) against the analytic KN pdf (north_star), the mean
    energy fraction of SURVEY.md §8(c), and momentum conservation of (gamma', e-)."""
    k = E / MEC2
    s = oracle.sample_kn(E, 200000, seed=7)
    eps, cost = s[:, 0], s[:, 1]
    e0 = 1 / (1 + 2 * k)

    def pdf(e):
        t = (1 - e) / (k * e)
        return (1 / e + e) * (1 - e * t * (2 - t) / (1 + e * e))

    cdf = lambda x: integrate.quad(pdf, e0, x, epsrel=1e-10)[0]
    assert _chi2_p(eps, np.linspace(e0, 1.0, 41), cdf) > 0.01
    # cos(theta) pdf is dsigma/dOmega
    pdo = lambda mu: (lambda P: P * P * (P + 1 / P - (1 - mu * mu)))(1 / (1 + k * (1 - mu)))
    cdf2 = lambda x: integrate.quad(pdo, -1, x, epsrel=1e-10)[0]
    assert _chi2_p(cost, np.linspace(-1, 1, 41), cdf2) > 0.01
    assert eps.mean() == pytest.approx(mean_pin, abs=4 * eps.std() / math.sqrt(len(eps)) + 5e-5)
    assert np.allclose(cost, 1 - (1 - eps) / (k * eps), atol=1e-12)  # Compton relation
    assert s[:, 3].max() < 1e-12  # |p_in - p_gamma' - p_e| / p_in


@pytest.mark.parametrize("T", [0.45, 1.0, 15.0])
def test_moller_sampler(T, water_oracle):
    s = oracle.sample_moller(T, 0.2, 200000, seed=3)
    eps = s[:, 0]
    ec = 0.2 / T
    assert eps.min() >= ec and eps.max() <= 0.5
    cdf = lambda x: integrate.quad(lambda e: water_oracle.eval("moller_dsde", T, e), ec, x, epsrel=1e-11, epsabs=0)[0]
    assert _chi2_p(eps, np.linspace(ec, 0.5, 31), cdf) > 0.01
    # two-body kinematics: transverse momenta cancel, longitudinal momentum and energy conserved
    Wk = eps * T
    p = lambda t: np.sqrt(t * (t + 2 * MEC2))
    c1, c2 = s[:, 1], s[:, 2]
    assert np.allclose(p(T - Wk) * c1 + p(Wk) * c2, p(T), rtol=1e-12)
    assert np.allclose(p(T - Wk) * np.sqrt(1 - c1 ** 2), p(Wk) * np.sqrt(1 - c2 ** 2), rtol=1e-7, atol=1e-9)


@pytest.mark.parametrize("T,m", [(1.0, 0), (15.0, 0), (6.0, 1)])
def test_brems_sampler(T, m):
    cfg = W.config(4, "g")
    o = oracle.Oracle(cfg["phantom"], cfg["materials"], cfg["params"])
    k = o.sample_brems(T, 200000, seed=11, m=m)
    assert k.min() >= 0.01 and k.max() < T
    cdf = lambda x: integrate.quad(lambda lk: o.eval("brems_kdsdk", T, math.exp(lk), m), math.log(0.01), math.log(x),
                                   epsrel=1e-10, limit=300)[0]
    assert _chi2_p(k, np.geomspace(0.01, T, 31), cdf) > 0.01


@pytest.mark.parametrize("a", [0.002, 0.1, 0.7])
def test_ms_polar_sampler(a):
    """p(mu) ~ exp(-(1-mu)/a) on [-1,1]: exact mean 1 - a + 2/(e^(2/a)-1) and chi-square."""
    mu = oracle.sample_ms(a, 200000, seed=5)
    assert mu.min() >= -1.0 and mu.max() <= 1.0
    mean = 1 - a + (2 / math.expm1(2 / a) if a > 0.01 else 0.0)
    assert mu.mean() == pytest.approx(mean, abs=4 * mu.std() / math.sqrt(len(mu)))
    cdf = lambda x: (math.exp(-(1 - x) / a) - math.exp(-2 / a)) / (1 - math.exp(-2 / a))
    edges = 1 - np.geomspace(2.0, 1e-4 * a, 30)
    edges[0] = -1.0
    assert _chi2_p(mu, np.append(edges, 1.0), cdf) > 0.01


def test_source_spectrum_and_field(water_oracle):
    bm = W.photon_field()
    s = water_oracle.sample_source(bm, 200000, seed=1)
    E, x, d = s[:, 0], s[:, 1:4], s[:, 4:7]
    # triangular pdf with vertices 0.25, 1.0, 6.0: mean = (a+b+c)/3, analytic cdf
    assert E.mean() == pytest.approx((0.25 + 1.0 + 6.0) / 3, abs=4 * E.std() / math.sqrt(len(E)))

    def cdf(e):
        a, c, b = 0.25, 1.0, 6.0
        return (e - a) ** 2 / ((b - a) * (c - a)) if e <= c else 1 - (b - e) ** 2 / ((b - a) * (b - c))

    assert _chi2_p(E, np.linspace(0.25, 6.0, 47), cdf) > 0.01
    assert np.all(np.abs(x[:, 0]) <= 5.0) and np.all(np.abs(x[:, 1]) <= 5.0) and np.all(x[:, 2] == 0.0)
    assert _chi2_p(x[:, 0], np.linspace(-5, 5, 21), lambda v: (v + 5) / 10) > 0.01
    assert _chi2_p(x[:, 1], np.linspace(-5, 5, 21), lambda v: (v + 5) / 10) > 0.01
    assert abs(np.corrcoef(x[:, 0], x[:, 1])[0, 1]) < 0.01
    assert np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-14)
    assert np.allclose(d[:, 0] / d[:, 2], x[:, 0] / 100.0, atol=1e-12)  # rays from the point source at SSD
    p = water_oracle.sample_source(W.electron_pencil(6.0), 10, seed=1)
    assert np.all(p[:, 0] == 6.0) and np.all(p[:, 1:4] == 0.0) and np.all(p[:, 4:7] == [0, 0, 1])


def test_contract_ln_accuracy():
    """The self-specified fp32 ln of the attenuation contract (R20) is a faithful ln."""
    rng = np.random.default_rng(0)
    xs = np.concatenate([rng.uniform(0, 1, 2000), 10.0 ** rng.uniform(-7, 2, 2000), [1.0, 0.5, 2.0, 2.0 ** -23]])
    for x in xs.astype(np.float32):
        if x > 0:
            assert oracle.contract_ln(float(x)) == pytest.approx(math.log(float(x)), rel=4e-7, abs=1.5e-7)
