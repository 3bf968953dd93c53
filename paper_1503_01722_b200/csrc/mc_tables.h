// Host-side physics-table builder of the CUDA engine ("A computer program was also
// developed to create physics data needed by oclMC based on a user-defined material composition").
// fp64 closed forms -> fp32 tables on a uniform ln E grid.  Independent of oracle/ (no shared code).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace mcb {

struct Element { int Z; double A, w; };
struct MaterialSpec {
    std::vector<Element> el;
    double I_eV, rho_nominal;
};
struct TableParams {
    double e_cut, g_cut, e_max;
    int n_grid;
};

enum TableId { T_MU_TOT = 0, T_MU_C, T_MU_PP, T_RANGE, T_L, T_S_HARD, T_S_MOLLER, T_S_MAX, T_K1,
               T_LNA,  // ln of the effective screening parameter of the Goudsmit-Saunderson model (R27)
               T_COUNT };

struct Tables {
    int N = 0, k_cut = 0, n_mat = 0;
    double lnE0 = 0, dln = 0;
    std::vector<std::vector<float>> t[T_COUNT];  // t[id][material][node]
    std::vector<float> lscr;                     // per material: bremsstrahlung screening cap
    std::vector<float> mu_maj;                   // 1/cm, needs the phantom's max density per material
};

// Returns empty string on success, else an error message.
std::string build_tables(const std::vector<MaterialSpec>& mats, const TableParams& p,
                         const std::vector<double>& rho_max_per_material, Tables& out);

}  // namespace mcb
