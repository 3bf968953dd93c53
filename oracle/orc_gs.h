// ORACLE (test infrastructure, never on the product path): Goudsmit-Saunderson multiple-scattering angle.
//
// The paper's electrons use "the random hinge method, where the multiple Coulomb scattering angle was determined
// using the method developed by Kawrakow (Kawrakow, 2000)" (section 2.1): the exact angular
// distribution after a path s for a given single-scattering law (Goudsmit & Saunderson),
//     F(mu; s) = sum_l (l + 1/2) exp(-lambda G_l) P_l(mu),   lambda = s / lambda_el,  G_l = 1 - <P_l>_single,
// sampled from pre-computed tables.  The single-scattering law here is the screened-Rutherford law the K_1 table is
// already built from (SURVEY.md 8(c) "Multiple scattering"): p(mu) = 2A(1+A) / (1 + 2A - mu)^2.  Reading R27 of
// DESIGN.md fixes everything the paper leaves to its reference:
//   * per material and energy ONE effective screening parameter A with  K_1 = Sigma_el G_1(A)  (total elastic cross
//     section Sigma_el = sum over elements, first transport cross section K_1 as tabulated): the distribution after a
//     step then depends on two numbers only, the scattering power t = K_1 rho s and A  (lambda = t / G_1(A));
//   * one material-independent table of quantiles of x = 1 - mu on a grid of NT values of t (uniform in
//     ln t + 4 sqrt t) x NA values of A (uniform in ln A); every row scaled so that its sampled <x> = 1 - exp(-t);
//     quantile nodes r_k = k/32 (k = 0..31), then 1 - r = 2^-6 .. 2^-16, then r = 1: 44 nodes; stored as y = ln x;
//   * sampling: the row is chosen by stochastic interpolation (upper t-node with the probability that reproduces
//     1 - exp(-t) exactly, i.e. <cos theta> = exp(-t); upper A-node with probability linear in ln A) from the 9 low
//     bits of the two Philox words whose 23 high bits give the uniforms (R15), then the inverse CDF is interpolated
//     linearly in y inside a quantile interval (linearly in x inside the first);
//   * t below the table (t < GS_T_MIN) is not sampled: it is carried to the next step (R8b).
// Functions: gs_G1, gs_effective_A (closed forms), gs_moments (Legendre moments by the Q_l recurrence), gs_cdf (the
// Legendre series of the cumulative distribution with the unscattered and single-scattered parts split off), GsTable.
// Pins: tests/test_oracle_gs.py (moments against quadrature, sampled <P_l> against exp(-lambda G_l), the no-scatter and
// single-scattering limits, <cos theta> = exp(-t) between nodes).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

namespace orc {

constexpr int GS_NT = 16, GS_NA = 5, GS_NQ = 44;
constexpr double GS_T_MIN = 1e-4, GS_T_MAX = 1.6, GS_A_MIN = 2e-8, GS_A_MAX = 5e-4, GS_X_MIN = 1e-12;

// first transport coefficient of the screened-Rutherford law: G_1 = 1 - <mu> = 2A(1+A) [ln((1+A)/A) - 1/(1+A)]
inline double gs_G1(double A) { return 2.0 * A * (1.0 + A) * (std::log((1.0 + A) / A) - 1.0 / (1.0 + A)); }

// A with K1 = S_el G_1(A), by bisection on ln A (G_1 is increasing in A)
inline double gs_effective_A(double K1, double S_el) {
    double target = K1 / S_el, lo = std::log(1e-12), hi = std::log(10.0);
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (gs_G1(std::exp(mid)) < target) lo = mid; else hi = mid;
    }
    return std::exp(0.5 * (lo + hi));
}

// Legendre moments g_l = <P_l> of p(mu), l = 0..lmax:  g_0 = 1,  g_l = l [Q_{l-1}(z) - z Q_l(z)],  z = 1 + 2A,
// Q_l = Legendre functions of the second kind by their upward recurrence (long double: the recurrence loses
// exp(4 l sqrt(A)) of relative accuracy, callers keep l below ~ 5.5 / sqrt(A)).
inline std::vector<double> gs_moments(double A, int lmax) {
    std::vector<double> g(lmax + 1);
    long double z = 1.0L + 2.0L * (long double)A;
    long double q0 = 0.5L * std::log((1.0L + (long double)A) / (long double)A), q1 = z * q0 - 1.0L;
    g[0] = 1.0;
    if (lmax >= 1) g[1] = (double)(q0 - z * q1);
    for (int l = 1; l < lmax; ++l) {
        long double q2 = ((2 * l + 1) * z * q1 - l * q0) / (l + 1);
        g[l + 1] = (double)((l + 1) * (q1 - z * q2));
        q0 = q1; q1 = q2;
    }
    return g;
}

// Cumulative distribution S(x) = P(1 - mu <= x) of the Goudsmit-Saunderson law at the points x (0 < x <= 2):
//   S = e^-lambda + lambda e^-lambda S_1(x) + 1/2 sum_l c_l [P_{l-1}(mu) - P_{l+1}(mu)],   mu = 1 - x,  P_{-1} = 1,
//   c_l = exp(-lambda G_l) - e^-lambda - lambda e^-lambda g_l   (two or more collisions),  S_1 = (1+A) x / (x + 2A)
// (integral of (l + 1/2) P_l from mu to 1 = [P_{l-1} - P_{l+1}] / 2).
inline std::vector<double> gs_cdf(double lambda, double A, const std::vector<double>& x) {
    int lcap = (int)std::min(60000.0, 5.5 / std::sqrt(A));
    std::vector<double> g = gs_moments(A, lcap);
    double e0 = std::exp(-lambda), e1 = lambda * e0;
    std::vector<double> c;
    int quiet = 0;
    for (int l = 0; l <= lcap; ++l) {
        double cl = std::exp(-lambda * (1.0 - g[l])) - e0 - e1 * g[l];
        c.push_back(cl);
        quiet = std::fabs(cl) < 1e-13 ? quiet + 1 : 0;
        if (quiet >= 30) break;
    }
    int L = (int)c.size();
    std::vector<double> S(x.size());
    for (size_t i = 0; i < x.size(); ++i) {
        const double mu = 1.0 - x[i];
        double sum = c[0] * (1.0 - mu);  // l = 0: P_{-1} - P_1
        double plm1 = 1.0, pl = mu;      // P_{l-1}, P_l at l = 1
        for (int l = 1; l < L; ++l) {
            const double plp1 = ((2 * l + 1) * mu * pl - l * plm1) / (l + 1);
            sum += c[l] * (plm1 - plp1);
            plm1 = pl; pl = plp1;
        }
        S[i] = e0 + e1 * (1.0 + A) * x[i] / (x[i] + 2.0 * A) + 0.5 * sum;
    }
    return S;
}

// ---- the sampling table (reading R27) ------------------------------------------------------------------------------
// t-grid: uniform in c(t) = ln t + 4 sqrt(t) — logarithmic where the shape of the distribution in x / t changes slowly
// (small t), denser where the sphere saturates it (t ~ 1)
inline double gs_c(double t) { return std::log(t) + 4.0 * std::sqrt(t); }
inline double gs_t_node(int i) {
    const double c = gs_c(GS_T_MIN) + (gs_c(GS_T_MAX) - gs_c(GS_T_MIN)) * i / (GS_NT - 1);
    double lo = std::log(GS_T_MIN), hi = std::log(GS_T_MAX);
    for (int it = 0; it < 100; ++it) { const double mid = 0.5 * (lo + hi); if (gs_c(std::exp(mid)) < c) lo = mid; else hi = mid; }
    return i == 0 ? GS_T_MIN : (i == GS_NT - 1 ? GS_T_MAX : std::exp(0.5 * (lo + hi)));
}
inline double gs_A_node(int j) { return GS_A_MIN * std::pow(GS_A_MAX / GS_A_MIN, (double)j / (GS_NA - 1)); }
// cumulative probability of quantile node k
inline double gs_r_node(int k) { return k < 32 ? k / 32.0 : (k < GS_NQ - 1 ? 1.0 - std::ldexp(1.0, -(5 + (k - 31))) : 1.0); }

// mean of x = 1 - mu that the sampling rule below produces from one row (y = ln of the quantile nodes): the first
// interval is uniform in x on [0, x_1], the others are exponentials of a linear function; values above 2 count as 2
inline double gs_row_mean(const double* y) {
    double m = 0.0;
    for (int k = 0; k < GS_NQ - 1; ++k) {
        const double p = gs_r_node(k + 1) - gs_r_node(k);
        if (k == 0) { m += p * 0.5 * std::min(std::exp(y[1]), 2.0); continue; }
        const int n = 64;  // midpoint rule inside the interval (the clamp at 2 makes a closed form awkward)
        double a = 0.0;
        for (int q = 0; q < n; ++q) a += std::min(std::exp(y[k] + (q + 0.5) / n * (y[k + 1] - y[k])), 2.0);
        m += p * a / n;
    }
    return m;
}

struct GsTable {
    std::vector<double> y;  // [GS_NT][GS_NA][GS_NQ]: ln of the quantiles of x = 1 - mu (clamped below at ln GS_X_MIN)
    double tn[GS_NT], an[GS_NT];  // the t-nodes and 1 - exp(-t) at them
    bool built = false;
    const double* row(int i, int j) const { return y.data() + ((size_t)i * GS_NA + j) * GS_NQ; }
    void build() {
        if (built) return;
        y.assign((size_t)GS_NT * GS_NA * GS_NQ, 0.0);
        for (int i = 0; i < GS_NT; ++i) { tn[i] = gs_t_node(i); an[i] = 1.0 - std::exp(-tn[i]); }
        // abscissae: log-spaced from GS_X_MIN to 2
        const int nx = 560;
        std::vector<double> x(nx);
        for (int i = 0; i < nx; ++i) x[i] = GS_X_MIN * std::pow(2.0 / GS_X_MIN, (double)i / (nx - 1));
        x[nx - 1] = 2.0;
        for (int i = 0; i < GS_NT; ++i)
            for (int j = 0; j < GS_NA; ++j) {
                const double t = tn[i], A = gs_A_node(j), lambda = t / gs_G1(A);
                std::vector<double> S = gs_cdf(lambda, A, x);
                for (int k = 1; k < nx; ++k) S[k] = std::max(S[k], S[k - 1]);  // monotone to rounding
                double* q = y.data() + ((size_t)i * GS_NA + j) * GS_NQ;
                for (int k = 0; k < GS_NQ; ++k) {
                    const double r = gs_r_node(k);
                    double v;
                    if (k == GS_NQ - 1) v = std::log(2.0);
                    else if (r <= S[0]) v = std::log(GS_X_MIN);  // inside the unscattered part: x = 0
                    else {
                        int hi = (int)(std::upper_bound(S.begin(), S.end(), r) - S.begin());
                        if (hi >= nx) hi = nx - 1;
                        const int lo = hi - 1;
                        const double f = S[hi] > S[lo] ? (r - S[lo]) / (S[hi] - S[lo]) : 0.0;
                        v = std::log(x[lo]) + f * (std::log(x[hi]) - std::log(x[lo]));  // S linear in ln x between abscissae
                    }
                    q[k] = v;
                }
                // the row is scaled (x -> s x, a shift of y) until the sampling rule reproduces the exact first moment
                // <1 - mu> = 1 - exp(-t): quantile interpolation alone is off by 1 - 3 %
                for (int it = 0; it < 8; ++it) {
                    const double shift = std::log((1.0 - std::exp(-t)) / gs_row_mean(q));
                    for (int k = 0; k < GS_NQ; ++k) if (q[k] > std::log(GS_X_MIN)) q[k] += shift;
                }
            }
        built = true;
    }
};

// 1 - mu for scattering power t >= GS_T_MIN and screening A, from the two Philox words of the step (R15: the 23 high bits
// of w_mu are the uniform r, its 9 low bits choose the t-row, the 9 low bits of w_phi choose the A-row).
inline double gs_sample_omu(const GsTable& T, double t, double A, uint32_t w_mu, uint32_t w_phi) {
    const double dc = (gs_c(GS_T_MAX) - gs_c(GS_T_MIN)) / (GS_NT - 1), dA = std::log(GS_A_MAX / GS_A_MIN) / (GS_NA - 1);
    // t-row: weights linear in 1 - exp(-t), so that the mixture has <cos theta> = exp(-t)
    double tc = std::min(std::max(t, GS_T_MIN), GS_T_MAX);
    int i = std::min(std::max((int)std::floor((gs_c(tc) - gs_c(GS_T_MIN)) / dc), 0), GS_NT - 2);
    while (i > 0 && tc < T.tn[i]) --i;  // the nodes come from a bisection: keep t inside [t_i, t_i+1]
    while (i < GS_NT - 2 && tc >= T.tn[i + 1]) ++i;
    const double a = 1.0 - std::exp(-tc), a0 = T.an[i], a1 = T.an[i + 1];
    const double ft = std::min(std::max((a - a0) / (a1 - a0), 0.0), 1.0);
    if ((double)(w_mu & 511u) + 0.5 < ft * 512.0) ++i;
    // A-row: weights linear in ln A
    const double al = std::log(std::min(std::max(A, GS_A_MIN), GS_A_MAX) / GS_A_MIN) / dA;
    int j = std::min(std::max((int)std::floor(al), 0), GS_NA - 2);
    if ((double)(w_phi & 511u) + 0.5 < (al - j) * 512.0) ++j;
    const double* q = T.row(i, j);
    // inverse CDF
    const double r = ((double)(w_mu >> 9) + 0.5) * (1.0 / 8388608.0), s = (1.0 - r) * 32.0;
    int k;
    double f;
    if (s > 1.0) { k = (int)std::floor(32.0 * r); f = 32.0 * r - k; }
    else {
        const int jj = std::min((int)std::floor(-std::log2(s)), GS_NQ - 33);  // 0..11
        k = 31 + jj;
        f = jj < GS_NQ - 33 ? 2.0 * (1.0 - std::ldexp(s, jj)) : 1.0 - std::ldexp(s, jj);
    }
    const double x = k == 0 ? std::exp(q[1]) * f : std::exp(q[k] + f * (q[k + 1] - q[k]));
    return std::min(x, 2.0);
}

}  // namespace orc
