// Physics-table builder (host, fp64).  Models: BASELINE.json north_star list, formulas as recorded
// in DESIGN.md "Closed forms": Klein-Nishina, parametric photoelectric, Maximon
// pair, Bethe restricted stopping power + Sternheimer-Peierls density effect, Moller,
// Bethe-Heitler-style bremsstrahlung, screened-Rutherford first transport cross section.
// Quadratures are Gauss-Legendre panels split at the bremsstrahlung screening kink.
#include "mc_tables.h"
#include "mc_gs.h"

#include <algorithm>
#include <cmath>
#include <thread>

namespace mcb {
namespace {

const double kMe = 0.51099895;         // MeV
const double kRe = 2.8179403e-13;      // cm
const double kNa = 6.02214076e23;
const double kAlpha = 1.0 / 137.035999;
const double kPi = 3.14159265358979323846;
const double kZeta3 = 1.2020569031595942;

// 16-point Gauss-Legendre rule on [-1, 1] by Newton iteration on P_16.
struct GL16 {
    double x[16], w[16];
    GL16() {
        const int n = 16;
        for (int i = 0; i < n; ++i) {
            double z = std::cos(kPi * (i + 0.75) / (n + 0.5)), pp = 0;
            for (int it = 0; it < 100; ++it) {
                double p1 = 1, p2 = 0;
                for (int j = 0; j < n; ++j) { double p3 = p2; p2 = p1; p1 = ((2 * j + 1) * z * p2 - j * p3) / (j + 1); }
                pp = n * (z * p1 - p2) / (z * z - 1);
                double dz = p1 / pp;
                z -= dz;
                if (std::fabs(dz) < 1e-15) break;
            }
            x[i] = z; w[i] = 2 / ((1 - z * z) * pp * pp);
        }
    }
};
const GL16& gl() { static GL16 g; return g; }

template <class F> double integrate(F f, double a, double b, int panels) {
    if (!(b > a)) return 0;
    const GL16& g = gl();
    double sum = 0, hp = (b - a) / panels;
    for (int p = 0; p < panels; ++p) {
        double c = a + (p + 0.5) * hp, r = 0.5 * hp, s = 0;
        for (int i = 0; i < 16; ++i) s += g.w[i] * f(c + r * g.x[i]);
        sum += s * r;
    }
    return sum;
}

struct Mat {
    std::vector<Element> el;
    double I, rho0;
    double n_el;     // electrons per gram
    double z_over_a; // <Z/A>
    double c_br;     // N_A sum (w/A) Z (Z+1)
    double l_scr;    // screening cap of the bremsstrahlung logarithm
};

Mat prepare(const MaterialSpec& s) {
    Mat m; m.el = s.el; m.I = s.I_eV; m.rho0 = s.rho_nominal;
    double wsum = 0;
    for (auto& e : m.el) wsum += e.w;
    m.z_over_a = 0; m.c_br = 0;
    double num = 0, den = 0;
    for (auto& e : m.el) {
        e.w /= wsum;
        m.z_over_a += e.w * e.Z / e.A;
        double c = e.w / e.A * e.Z * (e.Z + 1.0);
        m.c_br += c;
        num += c * std::log(183.0 / std::cbrt((double)e.Z));
        den += c;
    }
    m.c_br *= kNa;
    m.n_el = kNa * m.z_over_a;
    m.l_scr = num / den + 0.5;
    return m;
}

// --- photons -----------------------------------------------------------------------------------
double kn_total(double k) {  // per electron
    double q = 1 + 2 * k, lg = std::log(q);
    double t1 = (1 + k) / (k * k) * (2 * (1 + k) / q - lg / k);
    double t2 = lg / (2 * k);
    double t3 = (1 + 3 * k) / (q * q);
    return 2 * kPi * kRe * kRe * (t1 + t2 - t3);
}
double pe_atom(int Z, double k) {
    double thomson = 8 * kPi * kRe * kRe / 3;
    double a4 = kAlpha * kAlpha * kAlpha * kAlpha;
    double z5 = (double)Z * Z * Z * Z * Z;
    return 1.25 * 4 * std::sqrt(2.0) * a4 * thomson * z5 / (k * k * k * std::sqrt(k));
}
double pair_atom(int Z, double k) {
    if (k <= 2) return 0;
    double pref = kAlpha * kRe * kRe * Z * Z;
    if (k <= 4) {
        double e = (2 * k - 4) / (2 + k + 2 * std::sqrt(2 * k));
        double c3 = (k - 2) / k;
        double series = 1 + e * (0.5 + e * (23.0 / 40 + e * (11.0 / 60 + e * 29.0 / 960)));
        return pref * (2 * kPi / 3) * c3 * c3 * c3 * series;
    }
    double L = std::log(2 * k), r2 = 4 / (k * k);
    double a0 = 28 * L / 9 - 218.0 / 27;
    double a2 = 6 * L - 3.5 + 2 * L * L * L / 3 - L * L - kPi * kPi * L / 3 + 2 * kZeta3 + kPi * kPi / 6;
    double a4 = 3 * L / 16 + 0.125;
    double a6 = 29 * L / 2304 - 77.0 / 13824;
    return pref * (a0 + r2 * (a2 - r2 * (a4 + r2 * a6)));
}

// --- electrons ---------------------------------------------------------------------------------
double delta_sp(const Mat& m, double T) {  // Sternheimer-Peierls
    double gam = 1 + T / kMe;
    double X = 0.5 * std::log10(gam * gam - 1);
    double plasma = 28.816 * std::sqrt(m.rho0 * m.z_over_a);
    double C = -(2 * std::log(m.I / plasma) + 1), X0, X1;
    if (m.I < 100) { X1 = 2; X0 = (-C < 3.681) ? 0.2 : -0.326 * C - 1.0; }
    else { X1 = 3; X0 = (-C < 5.215) ? 0.2 : -0.326 * C - 1.5; }
    if (X < X0) return 0;
    double lin = 4.606 * X + C;
    if (X >= X1) return lin;
    double a = (-C - 4.606 * X0) / ((X1 - X0) * (X1 - X0) * (X1 - X0));
    double d = X1 - X;
    return lin + a * d * d * d;
}
double l_col(const Mat& m, double T, double cut) {
    double tau = T / kMe, gam = tau + 1, beta2 = tau * (tau + 2) / (gam * gam);
    double tc = std::min(cut / kMe, 0.5 * tau);
    double ired = m.I * 1e-6 / kMe;
    double f = -1 - beta2 + std::log((tau - tc) * tc) + tau / (tau - tc) +
               (0.5 * tc * tc + (2 * tau + 1) * std::log1p(-tc / tau)) / (gam * gam);
    double bracket = std::log(2 * (tau + 2)) - 2 * std::log(ired) + f - delta_sp(m, T);
    return 2 * kPi * kRe * kRe * kMe * m.n_el * bracket / beta2;
}
double moller_total(double T, double cut) {  // per electron
    if (T <= 2 * cut) return 0;
    double tau = T / kMe, gam = tau + 1, beta2 = tau * (tau + 2) / (gam * gam), ec = cut / T;
    double a = (tau / gam) * (tau / gam), b = (2 * tau + 1) / (gam * gam);
    double s = 1 / ec - 1 / (1 - ec) + a * (0.5 - ec) - b * (std::log1p(-ec) - std::log(ec));
    return 2 * kPi * kRe * kRe * s / (beta2 * tau);
}
double brems_k_dsdk(const Mat& m, double T, double k) {
    double E = T + kMe, Ef = E - k, r = Ef / E;
    double lu = std::log(2 * E * Ef / (kMe * k));
    return m.c_br * 4 * kAlpha * kRe * kRe * (1 + r * r - 2 * r / 3) * (std::min(lu, m.l_scr) - 0.5);
}
double brems_kink(const Mat& m, double T) {  // k where the unscreened logarithm meets the cap
    double E = T + kMe;
    return 2 * E * E / (kMe * std::exp(m.l_scr) + 2 * E);
}
double brems_total(const Mat& m, double T, double kc) {
    if (T <= kc) return 0;
    double ks = std::min(std::max(brems_kink(m, T), kc), T);
    auto f = [&](double lk) { return brems_k_dsdk(m, T, std::exp(lk)); };
    return integrate(f, std::log(kc), std::log(ks), 4) + integrate(f, std::log(ks), std::log(T), 4);
}
double l_rad(const Mat& m, double T, double kc) {
    double top = std::min(kc, T), ks = std::min(brems_kink(m, T), top);
    auto f = [&](double k) { return brems_k_dsdk(m, T, k); };
    return integrate(f, 0, ks, 2) + integrate(f, ks, top, 2);
}
// ln of the effective screening parameter A of the mixture (R27): G_1(A) = K1 / Sigma_el with both sums over the elements
// of the same screened-Rutherford law (total cross section of an element ~ Z(Z+1) / (A_i (1 + A_i)))
double ln_screening(const Mat& m, double T) {
    double tau = T / kMe, gam = tau + 1, bg2 = tau * (tau + 2), beta2 = bg2 / (gam * gam), first = 0, total = 0;
    for (const auto& e : m.el) {
        double az = kAlpha * e.Z / std::sqrt(beta2);
        double scr = kAlpha * kAlpha * std::cbrt((double)e.Z * e.Z) / (4 * 0.885 * 0.885 * bg2) * (1.13 + 3.76 * az * az);
        double c = e.w / e.A * e.Z * (e.Z + 1.0);
        first += 2 * c * (std::log1p(1 / scr) - 1 / (1 + scr));
        total += c / (scr * (1 + scr));
    }
    return std::log(gs_screening_from_ratio(first / total));
}
double k1_transport(const Mat& m, double T) {
    double tau = T / kMe, gam = tau + 1, bg2 = tau * (tau + 2), beta2 = bg2 / (gam * gam), s = 0;
    for (const auto& e : m.el) {
        double az = kAlpha * e.Z / std::sqrt(beta2);
        double scr = kAlpha * kAlpha * std::cbrt((double)e.Z * e.Z) / (4 * 0.885 * 0.885 * bg2) * (1.13 + 3.76 * az * az);
        double g1 = std::log1p(1 / scr) - 1 / (1 + scr);
        s += e.w / e.A * e.Z * (e.Z + 1.0) * g1;
    }
    return kNa * 2 * kPi * kRe * kRe * s / (gam * gam * beta2 * beta2);
}

// fn(i) for i in [0, n) on a few host threads (the nodes of a table are independent; the build is part of the
// end-to-end time of a fresh context)
template <class F> void parallel_for(int n, F fn) {
    int nt = (int)std::min<unsigned>(std::max(1u, std::thread::hardware_concurrency()), 16u);
    nt = std::min(nt, std::max(1, n / 8));
    if (nt <= 1) { for (int i = 0; i < n; ++i) fn(i); return; }
    std::vector<std::thread> th;
    for (int t = 0; t < nt; ++t)
        th.emplace_back([=]() { for (int i = t; i < n; i += nt) fn(i); });
    for (auto& x : th) x.join();
}

}  // namespace

std::string build_tables(const std::vector<MaterialSpec>& specs, const TableParams& p,
                         const std::vector<double>& rho_max, Tables& out) {
    if (specs.empty()) return "no materials";
    if (!(p.e_cut > 0) || !(p.g_cut > 0) || !(p.e_max > 2 * p.e_cut) || !(p.e_max > p.g_cut)) return "bad cut-offs";
    if (p.n_grid < 8 || p.n_grid > 1024) return "n_grid out of range (8..1024)";
    for (const auto& s : specs) {
        if (s.el.empty() || !(s.I_eV > 0) || !(s.rho_nominal > 0)) return "bad material";
        for (const auto& e : s.el) if (e.Z < 1 || e.Z > 100 || !(e.A > 0) || !(e.w >= 0)) return "bad element";
    }
    // grid: spacing ln2/n2 so that e_cut and 2 e_cut (Moller threshold) are nodes; origin <= min cut-off
    const int N = p.n_grid;
    const double e_low = std::min(p.e_cut, p.g_cut), ln2 = std::log(2.0);
    int n2 = (int)std::floor(ln2 / (std::log(p.e_max / e_low) / (N - 1)));
    bool ok = false;
    for (; n2 >= 1 && !ok; --n2) {
        out.dln = ln2 / n2;
        out.k_cut = (int)std::ceil(std::log(p.e_cut / e_low) / out.dln - 1e-12);
        out.lnE0 = std::log(p.e_cut) - out.k_cut * out.dln;
        ok = out.lnE0 + (N - 1) * out.dln >= std::log(p.e_max);
    }
    if (!ok) return "cannot place the energy grid (n_grid too small)";
    out.N = N; out.n_mat = (int)specs.size();
    std::vector<double> E(N);
    for (int j = 0; j < N; ++j) E[j] = std::exp(out.lnE0 + j * out.dln);
    E[out.k_cut] = p.e_cut;
    for (int id = 0; id < T_COUNT; ++id) out.t[id].assign(specs.size(), std::vector<float>(N, 0.f));
    out.lscr.clear();
    std::vector<std::vector<double>> mu_tot(specs.size(), std::vector<double>(N));
    for (size_t mi = 0; mi < specs.size(); ++mi) {
        Mat m = prepare(specs[mi]);
        out.lscr.push_back((float)m.l_scr);
        auto L = [&](double T) { return l_col(m, T, p.e_cut) + l_rad(m, T, p.g_cut); };
        std::vector<double> range(N, 0.0), s_hard(N, 0.0), segv(N, 0.0);
        parallel_for(N, [&](int j) {
            double k = E[j] / kMe, pe = 0, pp = 0;
            for (const auto& e : m.el) { pe += e.w / e.A * pe_atom(e.Z, k); pp += e.w / e.A * pair_atom(e.Z, k); }
            double muC = m.n_el * kn_total(k), muP = kNa * pp;
            mu_tot[mi][j] = muC + muP + kNa * pe;
            double sM = m.n_el * moller_total(E[j], p.e_cut);
            s_hard[j] = sM + brems_total(m, E[j], p.g_cut);
            out.t[T_MU_TOT][mi][j] = (float)mu_tot[mi][j];
            out.t[T_MU_C][mi][j] = (float)muC;
            out.t[T_MU_PP][mi][j] = (float)muP;
            out.t[T_L][mi][j] = (float)L(E[j]);
            out.t[T_S_MOLLER][mi][j] = (float)sM;
            out.t[T_S_HARD][mi][j] = (float)s_hard[j];
            out.t[T_K1][mi][j] = (float)k1_transport(m, E[j]);
            out.t[T_LNA][mi][j] = (float)ln_screening(m, E[j]);
            // range integral over the segment [node j, node j + 1]
            if (j + 1 < N) segv[j] = integrate([&](double lt) { double T = std::exp(lt); return T / L(T); }, std::log(E[j]), std::log(E[j + 1]), 1);
        });
        double run_max = 0;
        for (int j = 0; j < N; ++j) { run_max = std::max(run_max, s_hard[j]); out.t[T_S_MAX][mi][j] = (float)run_max; }
        for (int j = out.k_cut; j + 1 < N; ++j) range[j + 1] = range[j] + segv[j];
        for (int j = out.k_cut - 1; j >= 0; --j) range[j] = range[j + 1] - segv[j];
        for (int j = 0; j < N; ++j) out.t[T_RANGE][mi][j] = (float)range[j];
        // fp32 rounding must not break the dominance Sigma_max >= Sigma_hard nor monotonicity of R
        for (int j = 0; j < N; ++j) {
            float& sm = out.t[T_S_MAX][mi][j];
            sm = std::max(sm, out.t[T_S_HARD][mi][j]);
            if (j) sm = std::max(sm, out.t[T_S_MAX][mi][j - 1]);
        }
    }
    out.mu_maj.assign(N, 0.f);
    for (int j = 0; j < N; ++j) {
        double mx = 0;
        for (size_t mi = 0; mi < specs.size(); ++mi) mx = std::max(mx, rho_max[mi] * mu_tot[mi][j]);
        // round up so that the fp32 majorant dominates rho * fp32(mu_tot) for every voxel
        float f = (float)mx;
        for (size_t mi = 0; mi < specs.size(); ++mi)
            while ((double)f < (double)(float)rho_max[mi] * (double)out.t[T_MU_TOT][mi][j]) f = std::nextafterf(f, INFINITY);
        out.mu_maj[j] = f;
    }
    return "";
}

}  // namespace mcb
