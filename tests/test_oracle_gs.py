"""Pins of the ORACLE's Goudsmit-Saunderson multiple-scattering code (oracle/orc_gs.h; R27; PAPER.md:39:
"the multiple Coulomb scattering angle was determined using the method developed by Kawrakow").  Run with -m "not gpu".

What the mathematics fixes, independently of the code under test:
  * the Legendre moments of the screened-Rutherford law (numerical quadrature of p(mu) P_l(mu));
  * the Goudsmit-Saunderson distribution is the distribution after a Poisson number of single scatterings: brute force
    on small lambda (direct simulation of the collisions with numpy rotations);
  * <P_l> after path s = exp(-lambda G_l) for every l (Goudsmit & Saunderson 1940), checked on the table sampler that
    transport calls, on and between table nodes; l = 1 is Lewis's <cos theta> = exp(-K1 rho s);
  * the effective screening parameter of a pure element is the element's own Moliere parameter (closed form retyped here
    from SURVEY.md 8(c)).
"""
import math

import numpy as np
import pytest
from numpy.polynomial import legendre
from scipy import integrate

import oracle
from paper_1503_01722_b200 import workloads as W

ALPHA, MEC2 = 1.0 / 137.035999, 0.51099895


def _p_single(mu, A):
    return 2.0 * A * (1.0 + A) / (1.0 + 2.0 * A - mu) ** 2


@pytest.mark.parametrize("A", [1e-2, 1e-3, 3e-5])
def test_legendre_moments_of_the_screened_rutherford_law_against_quadrature(A):
    g = oracle.gs_moments(A, 8)
    assert g[0] == 1.0
    for l in range(1, 9):
        c = np.zeros(l + 1); c[l] = 1.0
        # x = 1 - mu on a log scale resolves the forward peak of width ~ A
        f = lambda lx: _p_single(1.0 - math.exp(lx), A) * legendre.legval(1.0 - math.exp(lx), c) * math.exp(lx)
        q = integrate.quad(f, math.log(1e-14), math.log(2.0), limit=400, epsabs=1e-13, epsrel=1e-11)[0]
        assert g[l] == pytest.approx(q, abs=2e-9), (l, g[l], q)
    assert 1.0 - g[1] == pytest.approx(oracle.gs_G1(A), rel=1e-9)
    # moments of a probability law on [-1, 1]: |g_l| <= 1, decreasing for this forward-peaked law — over the range of l
    # the upward Q_l recurrence is used for (l < 5.5 / sqrt(A), the cap gs_cdf applies)
    gl = oracle.gs_moments(A, int(5.5 / math.sqrt(A)))
    assert np.all(np.abs(gl) <= 1.0 + 1e-12) and np.all(np.diff(gl) < 1e-12) and gl[-1] < 1e-3


def _brute_force_mu(lam, A, n, rng):
    """Final direction cosine after a Poisson(lam) number of screened-Rutherford deflections with uniform azimuths."""
    k = rng.poisson(lam, n)
    d = np.zeros((n, 3)); d[:, 2] = 1.0
    for it in range(int(k.max())):
        act = np.nonzero(k > it)[0]
        u = rng.random(act.size)
        mu = 1.0 - 2.0 * A * u / (1.0 + A - u)  # inverse CDF of p(mu): S_1(x) = (1 + A) x / (x + 2A) = u
        phi = 2.0 * math.pi * rng.random(act.size)
        st = np.sqrt(np.maximum(0.0, 1.0 - mu * mu))
        a = d[act]
        # orthonormal frame around a (any): e1 = a x z or a x x
        ref = np.where(np.abs(a[:, 2:3]) < 0.9, np.array([[0.0, 0.0, 1.0]]), np.array([[1.0, 0.0, 0.0]]))
        e1 = np.cross(a, ref); e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
        e2 = np.cross(a, e1)
        d[act] = a * mu[:, None] + st[:, None] * (np.cos(phi)[:, None] * e1 + np.sin(phi)[:, None] * e2)
    return d[:, 2]


@pytest.mark.parametrize("lam,A", [(0.7, 2e-2), (4.0, 5e-3), (12.0, 1e-3)])
def test_cumulative_distribution_against_direct_simulation_of_the_collisions(lam, A):
    n = 400000
    mu = _brute_force_mu(lam, A, n, np.random.default_rng(11))
    x = np.array([1e-9, 0.3 * A, 2 * A, 10 * A, 60 * A, 0.1, 0.5, 1.0, 1.7, 2.0])
    S = oracle.gs_cdf(lam, A, x)
    emp = np.array([(1.0 - mu <= xi).mean() for xi in x])
    se = np.sqrt(np.maximum(S * (1.0 - S), 1e-12) / n)
    assert np.all(np.abs(emp - S) <= 4.5 * se + 1e-6), (emp, S, se)
    assert S[0] == pytest.approx(math.exp(-lam), abs=2e-6)  # the unscattered part
    assert S[-1] == pytest.approx(1.0, abs=1e-9)


@pytest.mark.parametrize("lam,A", [(150.0, 2e-8), (3000.0, 1e-6), (40.0, 1e-4)])
def test_cumulative_distribution_first_moments_at_large_lambda(lam, A):
    """int x dS = 1 - exp(-lam G_1) and int P_2 dS = exp(-lam G_2): moments of the series itself, by quadrature of S."""
    x = np.concatenate(([0.0], np.geomspace(1e-13, 2.0, 6000)))
    S = np.concatenate(([0.0], oracle.gs_cdf(lam, A, x[1:])))
    g = oracle.gs_moments(A, 2)
    m1 = np.sum(0.5 * (x[1:] + x[:-1]) * np.diff(S))
    assert m1 == pytest.approx(1.0 - math.exp(-lam * (1.0 - g[1])), rel=2e-3)
    xm = 0.5 * (x[1:] + x[:-1]); p2 = 0.5 * (3.0 * (1.0 - xm) ** 2 - 1.0)
    assert np.sum(p2 * np.diff(S)) == pytest.approx(math.exp(-lam * (1.0 - g[2])), abs=3e-3 * (1.0 - math.exp(-lam * (1.0 - g[2]))) + 1e-6)
    assert np.all(np.diff(S) >= -1e-9)


def _nodes_and_between():
    t, A, _ = oracle.gs_nodes()
    return [(t[4], A[2]), (t[9], A[1]), (t[12], A[3]),                      # on nodes
            (0.01, 1e-6), (0.02, 3e-6), (0.1, 1e-5), (0.003, 1e-4), (0.3, 5e-5), (0.5, 1e-6), (1.0, 2e-5)]  # between


@pytest.mark.parametrize("t,A", _nodes_and_between())
def test_table_sampler_reproduces_the_goudsmit_saunderson_moments(t, A):
    """The sampler transport calls: 1 - <P_l> against 1 - exp(-lambda G_l).  l = 1 is exact by construction of the table
    (rows scaled to the first moment, t-rows mixed linearly in 1 - exp(-t)): statistical bar only.  l = 2, 3 carry the
    table's interpolation error: 3 %."""
    n = 3000000
    lam = t / oracle.gs_G1(A)
    g = oracle.gs_moments(A, 3)
    mu = oracle.gs_sample(t, A, n, seed=3)
    assert np.all(np.abs(mu) <= 1.0)
    P = [mu, 0.5 * (3 * mu ** 2 - 1), 0.5 * (5 * mu ** 3 - 3 * mu)]
    for l in (1, 2, 3):
        got, se = 1.0 - P[l - 1].mean(), P[l - 1].std() / math.sqrt(n)
        want = 1.0 - math.exp(-lam * (1.0 - g[l]))
        tol = 4.0 * se + (1e-3 if l == 1 else 3e-2) * want
        assert abs(got - want) <= tol, (l, got, want, se)


def test_table_rows_are_quantile_functions_and_the_tail_is_single_scattering():
    T = oracle.gs_table()
    t, A, r = oracle.gs_nodes()
    assert T.shape == oracle.gs_dims() and np.all(np.diff(T, axis=2) >= -1e-12)  # non-decreasing in r
    assert np.all(np.diff(t) > 0) and np.all(np.diff(A) > 0) and r[0] == 0.0 and r[-1] == 1.0
    # far tail: the probability of an angle beyond x0 is that of the exact series (mostly one hard collision)
    for (i, j, x0) in ((3, 2, 0.05), (6, 1, 0.3), (8, 3, 1.0)):
        lam = t[i] / oracle.gs_G1(A[j])
        mu = oracle.gs_sample(t[i], A[j], 4000000, seed=9)
        tail = (1.0 - mu > x0).mean()
        want = 1.0 - oracle.gs_cdf(lam, A[j], np.array([x0]))[0]
        assert tail == pytest.approx(want, rel=0.06, abs=4.0 * math.sqrt(want / 4e6)), (i, j, tail, want)
    # few collisions: the unscattered fraction exp(-lambda) shows as the flat start of the row
    i, j = 0, 4
    lam = t[i] / oracle.gs_G1(A[j])
    mu = oracle.gs_sample(t[i], A[j], 1000000, seed=2)
    assert (1.0 - mu < 1e-9).mean() == pytest.approx(math.exp(-lam), abs=0.04)  # to the 1/32 resolution of the nodes


def test_effective_screening_parameter_of_a_pure_element_is_its_moliere_parameter():
    carbon = W._mat("carbon", {6: 1.0}, 78.0, 1.7)
    orc = oracle.Oracle(W.homogeneous_phantom((1, 1, 1), 10.0), [carbon], W.params())
    g = orc.grid()
    lnA = orc.table("lnA")
    for j in (0, 60, 150, g["N"] - 1):
        T = math.exp(g["lnE0"] + j * g["dln"]) if j != g["k_cut"] else 0.2
        tau = T / MEC2; gam = tau + 1.0; b2 = 1.0 - 1.0 / gam ** 2; bg2 = gam ** 2 - 1.0
        A_mol = ALPHA ** 2 * 6.0 ** (2.0 / 3.0) / (4.0 * 0.885 ** 2 * bg2) * (1.13 + 3.76 * (ALPHA * 6.0) ** 2 / b2)
        assert math.exp(lnA[j]) == pytest.approx(A_mol, rel=1e-6)
        # and for any material K1 = S_el G_1(A) by definition of A
        assert orc.eval("K1", T) == pytest.approx(orc.eval("S_el", T) * oracle.gs_G1(math.exp(lnA[j])), rel=1e-8)
    water = oracle.Oracle(W.homogeneous_phantom((1, 1, 1), 10.0), W.materials(1), W.params())
    lw = water.table("lnA")
    assert np.all(np.diff(lw) < 0)  # screening parameter falls with energy
    assert 2e-8 < math.exp(lw[-1]) and math.exp(lw[0]) < 5e-3


# ---- inside transport (Run::electron with MC_FLAG_MS_GS) --------------------------------------------------------------
def _scattering_power(orc, T0, T1, e_cut, g_cut=0.01):
    """int_{T1}^{T0} K1/L dT from the closed forms."""
    L = lambda T: orc.eval("L_col", T, e_cut) + orc.eval("L_rad", T, g_cut)
    f = lambda lt: orc.eval("K1", math.exp(lt)) / L(math.exp(lt)) * math.exp(lt)
    return integrate.quad(f, math.log(T1), math.log(T0), epsabs=1e-10, epsrel=1e-8)[0]


@pytest.mark.parametrize("vox,T0,e_cut,angle", [(400.0, 15.0, 10.0, 0.0), (0.25, 15.0, 10.0, 20.0), (0.25, 2.0, 1.0, 0.0), (0.5, 1.0, 0.3, 10.0)])
def test_gs_angle_inside_transport_keeps_the_first_moment(vox, T0, e_cut, angle):
    """Hard events off, Goudsmit-Saunderson angle on: <Omega . Omega_0> at the cut-off = exp(-int K1/L dT) (Lewis), in one
    huge voxel and on voxel grids where most steps end on a face and scattering power below the table is carried (R8b,
    R27).  Unlike the Gaussian model's product of step means this holds step by step, so the bar is the midpoint rule's
    (K1 at the mid-step energy) plus statistics: 1 %."""
    n = 100000
    nn = 1 if vox > 100 else int(round(40.0 / vox))
    orc = oracle.Oracle(W.homogeneous_phantom((nn, nn, nn), vox), W.materials(1),
                        W.params(e_cut=e_cut, flags=W.FLAG_NO_HARD | W.FLAG_MS_GS))
    # the track starts well inside the phantom: the single-scattering tail back-scatters a few per cent of the tracks
    bm = W.beam(W.ELECTRON, W.PENCIL, energy=T0, entry=(0.013, 0.027, 0.0 if nn == 1 else 20.0 + 0.031))
    th = math.radians(angle)
    bm["axis"] = np.array((math.sin(th), 0.0, math.cos(th)), np.float32)
    pb, st = orc.run_probe(bm, n, 5)
    ax = bm["axis"].astype(np.float64); ax /= np.linalg.norm(ax)
    ok = pb["escaped"] == 0
    assert ok.mean() > 0.99
    c = pb["dir"][ok] @ ax
    m, se = c.mean(), c.std() / math.sqrt(ok.sum())
    G = _scattering_power(orc, T0, e_cut, e_cut)
    assert -math.log(m) / G == pytest.approx(1.0, abs=0.01 + 3.0 * se / m / G), (m, G)
    assert pb["q_sampled"].sum() / pb["q_travelled"].sum() == pytest.approx(1.0, abs=3e-3)
