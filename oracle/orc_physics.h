// ORACLE — test infrastructure only (parity reference + timed CPU baseline).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// use anything under oracle/.  It shares no code with the CUDA path (paper_1503_01722_b200/csrc).
//
// Closed-form physics models in fp64, units MeV / cm / g.  The paper says only that
// electron data come from "analytical formula" and photon data from NIST XCOM; XCOM is not
// available, so every model below is the closed form BASELINE.json north_star lists, in the
// reading DESIGN.md §"Closed forms" records.
#pragma once
#include <cmath>
#include <vector>
#include <algorithm>

namespace orc {

constexpr double MEC2 = 0.51099895;        // electron rest energy, MeV
constexpr double RE = 2.8179403e-13;       // classical electron radius, cm
constexpr double NA = 6.02214076e23;       // Avogadro
constexpr double ALPHA = 1.0 / 137.035999; // fine structure constant
constexpr double PI = 3.14159265358979323846;
constexpr double ZETA3 = 1.2020569031595942;

struct Material {
    std::vector<int> Z;
    std::vector<double> A, w;  // atomic mass, mass fraction
    double I_eV = 75.0, rho_nominal = 1.0;
    // derived
    double ne = 0;    // electrons per gram  N_A sum w Z/A
    double ZA = 0;    // <Z/A>
    double Cbr = 0;   // N_A sum (w/A) Z(Z+1)
    double Lscr = 0;  // brems screening cap
    void derive() {
        ZA = 0; Cbr = 0; double num = 0, den = 0;
        for (size_t i = 0; i < Z.size(); ++i) {
            ZA += w[i] * Z[i] / A[i];
            double c = w[i] / A[i] * Z[i] * (Z[i] + 1.0);
            Cbr += NA * c;
            num += c * std::log(183.0 * std::pow((double)Z[i], -1.0 / 3.0));
            den += c;
        }
        ne = NA * ZA;
        Lscr = num / den + 0.5;
    }
};

// ---- photons (Compton, pair production, photoelectric absorption) -----------------
// Klein-Nishina total cross section per free electron, cm^2; k = E/mc^2.
inline double sigma_kn(double k) {
    double a = 1.0 + 2.0 * k, l = std::log(a);
    return 2.0 * PI * RE * RE * ((1.0 + k) / (k * k) * (2.0 * (1.0 + k) / a - l / k) + l / (2.0 * k)
                                 - (1.0 + 3.0 * k) / (a * a));
}
// Parametric photoelectric cross section per atom (Born K-shell x 5/4), cm^2.
inline double sigma_pe(int Z, double k) {
    double sT = 8.0 * PI * RE * RE / 3.0;
    return 1.25 * 4.0 * std::sqrt(2.0) * std::pow(ALPHA, 4) * sT * std::pow((double)Z, 5) * std::pow(k, -3.5);
}
// Pair production in the nuclear field, unscreened (Maximon's two expansions), per atom, cm^2.
inline double sigma_pp(int Z, double k) {
    if (k <= 2.0) return 0.0;
    double c = ALPHA * RE * RE * Z * Z;
    if (k <= 4.0) {
        double e = (2.0 * k - 4.0) / (2.0 + k + 2.0 * std::sqrt(2.0 * k));
        double t = (k - 2.0) / k;
        return c * (2.0 * PI / 3.0) * t * t * t *
               (1.0 + e / 2.0 + 23.0 * e * e / 40.0 + 11.0 * e * e * e / 60.0 + 29.0 * e * e * e * e / 960.0);
    }
    double L = std::log(2.0 * k), r = 2.0 / k, r2 = r * r;
    return c * (28.0 * L / 9.0 - 218.0 / 27.0
                + r2 * (6.0 * L - 3.5 + (2.0 / 3.0) * L * L * L - L * L - (PI * PI / 3.0) * L + 2.0 * ZETA3 + PI * PI / 6.0)
                - r2 * r2 * (3.0 * L / 16.0 + 0.125)
                - r2 * r2 * r2 * (29.0 * L / 2304.0 - 77.0 / 13824.0));
}
inline double mu_compton(const Material& m, double E) { return m.ne * sigma_kn(E / MEC2); }  // cm^2/g
inline double mu_pe(const Material& m, double E) {
    double s = 0;
    for (size_t i = 0; i < m.Z.size(); ++i) s += m.w[i] / m.A[i] * sigma_pe(m.Z[i], E / MEC2);
    return NA * s;
}
inline double mu_pp(const Material& m, double E) {
    double s = 0;
    for (size_t i = 0; i < m.Z.size(); ++i) s += m.w[i] / m.A[i] * sigma_pp(m.Z[i], E / MEC2);
    return NA * s;
}

// ---- electrons (restricted stopping power, Moller, bremsstrahlung, MS) ----------
// Sternheimer-Peierls density-effect correction from (I, rho_nominal, <Z/A>).
inline double density_effect(const Material& m, double T) {
    double g = T / MEC2 + 1.0, bg = std::sqrt(g * g - 1.0);
    double X = std::log10(bg);
    double hnu = 28.816 * std::sqrt(m.rho_nominal * m.ZA);  // eV
    double C = -(2.0 * std::log(m.I_eV / hnu) + 1.0);
    double X0, X1;
    if (m.I_eV < 100.0) { X1 = 2.0; X0 = (-C < 3.681) ? 0.2 : -0.326 * C - 1.0; }
    else { X1 = 3.0; X0 = (-C < 5.215) ? 0.2 : -0.326 * C - 1.5; }
    double a = (-C - 4.606 * X0) / std::pow(X1 - X0, 3);
    if (X < X0) return 0.0;
    if (X < X1) return 4.606 * X + C + a * std::pow(X1 - X, 3);
    return 4.606 * X + C;
}
// Collision stopping power restricted to losses below delta (Bethe with Moller restriction),
// MeV cm^2/g.  delta >= T/2 gives the unrestricted Bethe value.
inline double L_col(const Material& m, double T, double delta) {
    double tau = T / MEC2, g = tau + 1.0, b2 = 1.0 - 1.0 / (g * g);
    double tup = std::min(delta / MEC2, tau / 2.0);
    double Imc = m.I_eV * 1e-6 / MEC2;
    double F = -1.0 - b2 + std::log((tau - tup) * tup) + tau / (tau - tup)
               + (tup * tup / 2.0 + (2.0 * tau + 1.0) * std::log(1.0 - tup / tau)) / (g * g);
    return 2.0 * PI * RE * RE * MEC2 * m.ne / b2 * (std::log(2.0 * (g + 1.0) / (Imc * Imc)) + F - density_effect(m, T));
}
// Moller differential cross section per electron in eps = W/T, cm^2.
inline double moller_dsde(double T, double eps) {
    double tau = T / MEC2, g = tau + 1.0, b2 = 1.0 - 1.0 / (g * g);
    double q1 = (g - 1.0) / g; q1 *= q1;
    double q2 = (2.0 * g - 1.0) / (g * g);
    return 2.0 * PI * RE * RE / (b2 * tau) * (1.0 / (eps * eps) + 1.0 / ((1.0 - eps) * (1.0 - eps)) + q1 - q2 / (eps * (1.0 - eps)));
}
// Moller total cross section per electron for W >= e_cut, cm^2.
inline double moller_sigma(double T, double e_cut) {
    if (T <= 2.0 * e_cut) return 0.0;
    double tau = T / MEC2, g = tau + 1.0, b2 = 1.0 - 1.0 / (g * g), ec = e_cut / T;
    double q1 = (g - 1.0) / g; q1 *= q1;
    double q2 = (2.0 * g - 1.0) / (g * g);
    return 2.0 * PI * RE * RE / (b2 * tau) * (1.0 / ec - 1.0 / (1.0 - ec) + q1 * (0.5 - ec) - q2 * std::log((1.0 - ec) / ec));
}
// Bremsstrahlung: k dSigma/dk per unit density, cm^2/g (dimensionless k weighting), k < T.
inline double brems_kdsdk(const Material& m, double T, double k) {
    if (k > T) return 0.0;
    double E = T + MEC2, Ep = E - k, r = Ep / E;
    double Lu = std::log(2.0 * E * Ep / (MEC2 * k));
    return m.Cbr * 4.0 * ALPHA * RE * RE * (1.0 + r * r - 2.0 * r / 3.0) * (std::min(Lu, m.Lscr) - 0.5);
}
// composite Simpson
template <class F> inline double simpson(F f, double a, double b, int n) {
    if (b <= a) return 0.0;
    double h = (b - a) / n, s = f(a) + f(b);
    for (int i = 1; i < n; ++i) s += f(a + i * h) * ((i & 1) ? 4.0 : 2.0);
    return s * h / 3.0;
}
// Macroscopic brems cross section for k >= g_cut, cm^2/g: integral of (k dS/dk) d ln k.
inline double brems_sigma(const Material& m, double T, double g_cut) {
    if (T <= g_cut) return 0.0;
    return simpson([&](double x) { return brems_kdsdk(m, T, std::min(std::exp(x), T)); }, std::log(g_cut), std::log(T), 2000);
}
// Radiative stopping power restricted to k < kmax, MeV cm^2/g: integral_0^min(kmax,T) k dS/dk dk.
inline double L_rad(const Material& m, double T, double kmax) {
    double top = std::min(kmax, T);
    return simpson([&](double k) { return k <= 0 ? m.Cbr * 4.0 * ALPHA * RE * RE * (4.0 / 3.0) * (m.Lscr - 0.5) : brems_kdsdk(m, T, k); },
                   0.0, top, 4000);
}
inline double L_total(const Material& m, double T, double e_cut, double g_cut) { return L_col(m, T, e_cut) + L_rad(m, T, g_cut); }
// First transport cross section (screened Rutherford, Moliere screening), cm^2/g.
inline double K1(const Material& m, double T) {
    double tau = T / MEC2, g = tau + 1.0, b2 = 1.0 - 1.0 / (g * g), bg2 = g * g - 1.0;
    double s = 0;
    for (size_t i = 0; i < m.Z.size(); ++i) {
        double Z = m.Z[i];
        double az = ALPHA * Z;
        double Ai = ALPHA * ALPHA * std::pow(Z, 2.0 / 3.0) / (4.0 * 0.885 * 0.885 * bg2) * (1.13 + 3.76 * az * az / b2);
        s += m.w[i] / m.A[i] * 2.0 * PI * RE * RE * Z * (Z + 1.0) * (1.0 - b2) / (b2 * b2) * (std::log((1.0 + Ai) / Ai) - 1.0 / (1.0 + Ai));
    }
    return NA * s;
}

// Total elastic cross section of the same screened-Rutherford law (cm^2/g): per element
// sigma_el = pi r_e^2 Z(Z+1) (1 - beta^2)/beta^4 / (A_i (1 + A_i))  (integral of the law K1 is the first moment of).
inline double S_el(const Material& m, double T) {
    double tau = T / MEC2, g = tau + 1.0, b2 = 1.0 - 1.0 / (g * g), bg2 = g * g - 1.0;
    double s = 0;
    for (size_t i = 0; i < m.Z.size(); ++i) {
        double Z = m.Z[i];
        double az = ALPHA * Z;
        double Ai = ALPHA * ALPHA * std::pow(Z, 2.0 / 3.0) / (4.0 * 0.885 * 0.885 * bg2) * (1.13 + 3.76 * az * az / b2);
        s += m.w[i] / m.A[i] * PI * RE * RE * Z * (Z + 1.0) * (1.0 - b2) / (b2 * b2) / (Ai * (1.0 + Ai));
    }
    return NA * s;
}

}  // namespace orc
