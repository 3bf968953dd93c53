// Builder of the engine's Goudsmit-Saunderson table (mc_gs.h; R27).
//
// Single scattering: screened Rutherford, p(mu) = 2A(1+A) / (1 + 2A - mu)^2.  After a path with lambda = t / G_1(A)
// mean collisions the direction cosine has the Goudsmit-Saunderson law sum_l (l + 1/2) exp(-lambda (1 - g_l)) P_l(mu).
// Its cumulative distribution in x = 1 - mu is evaluated here as
//     C(x) = e^-lambda + lambda e^-lambda (1+A) x / (x + 2A) + sum_l w_l [P_{l-1}(1-x) - P_{l+1}(1-x)] / 2,
//     w_l = exp(-lambda (1 - g_l)) - e^-lambda (1 + lambda g_l)
// (no collision + one collision in closed form, the rest as a Legendre series that converges once g_l is small), then
// inverted at the quantile nodes.
#include "mc_gs.h"

#include <algorithm>
#include <cmath>
#include <mutex>
#include <thread>

namespace mcb {

namespace {

double g1_of(double A) { return 2 * A * (1 + A) * (std::log1p(1 / A) - 1 / (1 + A)); }

// moments g_0 .. g_n of the single-scattering law.  With z = 1 + 2A and the Legendre functions of the second kind,
// int P_l(mu) / (z - mu)^2 dmu = -2 Q_l'(z) and (z^2 - 1) Q_l' = l (z Q_l - Q_{l-1}) give g_l = l (Q_{l-1} - z Q_l).
void single_moments(double A, int n, std::vector<double>& g) {
    g.assign(n + 1, 0.0);
    g[0] = 1.0;
    const long double z = 1 + 2 * (long double)A;
    long double prev = std::log1p(1 / (long double)A) / 2;  // Q_0
    long double cur = z * prev - 1;                          // Q_1
    for (int l = 1; l <= n; ++l) {
        g[l] = (double)(l * (prev - z * cur));
        const long double nxt = ((2 * l + 1) * z * cur - l * prev) / (l + 1);
        prev = cur; cur = nxt;
    }
}

double node_r(int k) { return k < 32 ? k / 32.0 : (k == kGsNQ - 1 ? 1.0 : 1.0 - std::exp2(-(double)(k - 26))); }

// <x> produced by the sampling rule from one row: uniform in x on the first interval, exp(linear) on the others, x
// capped at 2
double sampled_mean(const double* y) {
    const double top = std::log(2.0);
    double m = (node_r(1) - node_r(0)) * 0.5 * std::min(std::exp(y[1]), 2.0);
    for (int k = 1; k + 1 < kGsNQ; ++k) {
        const double p = node_r(k + 1) - node_r(k), a = y[k], b = y[k + 1], d = b - a;
        auto piece = [](double a0, double d0) { return std::fabs(d0) < 1e-9 ? std::exp(a0) : std::exp(a0) * std::expm1(d0) / d0; };
        if (b <= top || d <= 0) m += p * std::min(piece(a, d), 2.0);
        else if (a >= top) m += p * 2.0;
        else {  // crosses the cap inside the interval
            const double f = (top - a) / d;
            m += p * (f * piece(a, top - a) + (1 - f) * 2.0);
        }
    }
    return m;
}

void build_row(double t, double A, const std::vector<double>& xs, double* y) {
    const double lambda = t / g1_of(A), e0 = std::exp(-lambda);
    const int cap = (int)std::min(60000.0, 5.5 / std::sqrt(A));
    std::vector<double> g;
    single_moments(A, cap, g);
    std::vector<double> w;
    w.reserve(cap + 1);
    for (int l = 0, calm = 0; l <= cap && calm < 30; ++l) {
        w.push_back(std::exp(-lambda * (1 - g[l])) - e0 * (1 + lambda * g[l]));
        calm = std::fabs(w.back()) < 1e-13 ? calm + 1 : 0;
    }
    const size_t nx = xs.size();
    std::vector<double> C(nx), pa(nx, 1.0), pb(nx);  // pa = P_{l-1}, pb = P_l at every abscissa
    for (size_t i = 0; i < nx; ++i) { pb[i] = 1 - xs[i]; C[i] = w[0] * xs[i]; }  // l = 0: P_{-1} - P_1 = x
    for (size_t l = 1; l < w.size(); ++l)
        for (size_t i = 0; i < nx; ++i) {
            const double mu = 1 - xs[i], pn = ((2 * l + 1) * mu * pb[i] - l * pa[i]) / (l + 1);
            C[i] += w[l] * (pa[i] - pn);
            pa[i] = pb[i]; pb[i] = pn;
        }
    for (size_t i = 0; i < nx; ++i) {
        C[i] = e0 + lambda * e0 * (1 + A) * xs[i] / (xs[i] + 2 * A) + 0.5 * C[i];
        if (i) C[i] = std::max(C[i], C[i - 1]);
    }
    const double floor_y = std::log(kGsXMin);
    for (int k = 0; k < kGsNQ; ++k) {
        const double r = node_r(k);
        if (k == kGsNQ - 1) { y[k] = std::log(2.0); continue; }
        if (r <= C[0]) { y[k] = floor_y; continue; }
        size_t hi = std::upper_bound(C.begin(), C.end(), r) - C.begin();
        hi = std::min(hi, nx - 1);
        const size_t lo = hi - 1;
        const double f = C[hi] > C[lo] ? (r - C[lo]) / (C[hi] - C[lo]) : 0.0;
        y[k] = std::log(xs[lo]) + f * std::log(xs[hi] / xs[lo]);
    }
    // scale the row until the sampling rule gives <x> = 1 - exp(-t) (R27)
    for (int it = 0; it < 8; ++it) {
        const double s = std::log(-std::expm1(-t) / sampled_mean(y));
        for (int k = 0; k < kGsNQ; ++k) if (y[k] > floor_y) y[k] += s;
    }
}

}  // namespace

double gs_grid_coordinate(double t) { return std::log(t) + 4 * std::sqrt(t); }

double gs_screening_from_ratio(double g1) {
    // Newton on u = ln A for ln G_1(e^u) = ln g1; G_1 ~ 2A (ln(1/A) - 1) for small A
    double u = std::log(std::max(g1, 1e-300) / 20.0);
    for (int it = 0; it < 60; ++it) {
        const double A = std::exp(u), f = std::log(g1_of(A)) - std::log(g1);
        const double h = 1e-6, fp = (std::log(g1_of(std::exp(u + h))) - std::log(g1_of(std::exp(u - h)))) / (2 * h);
        const double du = f / fp;
        u -= du;
        if (std::fabs(du) < 1e-13) break;
    }
    return std::exp(u);
}

const GsTable& gs_table() {
    static GsTable T;
    static std::once_flag once;
    std::call_once(once, [] {
        const double c0 = gs_grid_coordinate(kGsTMin), c1 = gs_grid_coordinate(kGsTMax);
        double tn[kGsNT];
        for (int i = 0; i < kGsNT; ++i) {
            const double c = c0 + (c1 - c0) * i / (kGsNT - 1);
            double t = std::sqrt(kGsTMin * kGsTMax);  // Newton on c(t) = c in ln t
            for (int it = 0; it < 80; ++it) {
                const double step = (gs_grid_coordinate(t) - c) / (1 + 2 * std::sqrt(t));  // dc/dln t = 1 + 2 sqrt t
                t *= std::exp(-step);
                if (std::fabs(step) < 1e-15) break;
            }
            tn[i] = i == 0 ? kGsTMin : (i == kGsNT - 1 ? kGsTMax : t);
            T.t[i] = (float)tn[i];
            T.an[i] = (float)(-std::expm1(-tn[i]));
        }
        const int nx = 640;
        std::vector<double> xs(nx);
        for (int i = 0; i < nx; ++i) xs[i] = kGsXMin * std::pow(2.0 / kGsXMin, (double)i / (nx - 1));
        xs[nx - 1] = 2.0;
        std::vector<double> y((size_t)kGsNT * kGsNA * kGsNQ);
        auto rows = [&](int begin, int end) {
            for (int q = begin; q < end; ++q) {
                const int i = q / kGsNA, j = q % kGsNA;
                const double A = kGsAMin * std::pow(kGsAMax / kGsAMin, (double)j / (kGsNA - 1));
                build_row(tn[i], A, xs, y.data() + (size_t)q * kGsNQ);
            }
        };
        const int total = kGsNT * kGsNA, nth = 8;
        std::vector<std::thread> th;
        for (int k = 0; k < nth; ++k) th.emplace_back(rows, total * k / nth, total * (k + 1) / nth);
        for (auto& x : th) x.join();
        T.y.resize(y.size());
        for (size_t k = 0; k < y.size(); ++k) T.y[k] = (float)y[k];
    });
    return T;
}

}  // namespace mcb
