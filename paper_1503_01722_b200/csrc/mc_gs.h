// Goudsmit-Saunderson multiple-scattering table of the engine ("the multiple Coulomb scattering angle was
// determined using the method developed by Kawrakow"; reading R27).  Host-side builder, fp64 -> fp32.
// Independent of oracle/ (no shared code): only the DEFINITION of the table is common — nodes, variable, row
// normalisation and sampling rule as stated in DESIGN.md R27.
#pragma once
#include <vector>

namespace mcb {

constexpr int kGsNT = 16, kGsNA = 5, kGsNQ = 44;     // scattering-power nodes, screening nodes, quantile nodes
constexpr double kGsTMin = 1e-4, kGsTMax = 1.6;      // t = K1 rho s covered by the table (below: carried; above: last row)
constexpr double kGsAMin = 2e-8, kGsAMax = 5e-4;     // effective screening parameter covered by the table
constexpr double kGsXMin = 1e-12;                    // quantiles of x = 1 - cos(theta) are stored as ln x >= ln kGsXMin

struct GsTable {
    std::vector<float> y;   // [kGsNT][kGsNA][kGsNQ] ln of the quantiles of 1 - cos(theta)
    float an[kGsNT];        // 1 - exp(-t_i) at the t-nodes (row mixing weights)
    float t[kGsNT];         // the t-nodes
};

// c(t) = ln t + 4 sqrt(t): the t-grid is uniform in c
double gs_grid_coordinate(double t);
// The table (built once per process, thread-safe).
const GsTable& gs_table();
// Effective screening parameter A of a mixture from the ratio K1 / Sigma_el = G_1(A).
double gs_screening_from_ratio(double g1);

}  // namespace mcb
