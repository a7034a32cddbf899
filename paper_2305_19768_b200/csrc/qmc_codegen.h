// qmc_codegen.h -- lowering of a sector's polynomial description to straight-line CUDA.
// Host-only C++; no CUDA types.  See qmc_codegen.cpp.
#ifndef QMC_CODEGEN_H_
#define QMC_CODEGEN_H_

#include <cstdint>
#include <string>
#include <vector>

namespace qmc {

// Deep copy of a qmc_sector_desc (include/qmc.h).
struct SectorSpec {
    int kind = 0, dim = 1, transform = 0, deformed = 0, first_order = 0, n_orders = 1;
    int a[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    double p = 0.0, q = 0.0, lambda = 0.0, f_im = 0.0;
    std::vector<double> U_coef, F_coef, logc;
    std::vector<uint8_t> U_exp, F_exp;  // n x dim row-major
};

struct SectorCode {
    std::string text;     // "struct Sector_<id> { ... };"
    bool cplx = false;    // deformed class: complex values, 3 accumulators per order
    int J = 1, D = 1, TR = 0;
    double ops = 0.0;     // FP64 instructions per evaluation of the emitted code, incl. lattice,
                          // transform, elementary functions and accumulation (fma = 1)
    int n_const = 0;      // doubles in the sector's __constant__ pool (64 KB per module in all)
    double flops = 0.0;   // flops per evaluation by SURVEY.md 8(d)'s model (monomial by monomial)
    double eflops = 0.0;  // flops per evaluation of the emitted code (fma = 2): what the kernel executes
};

// Generates the device struct `Sector_<case_id>` with
//   static constexpr int D, TR, J; static constexpr bool CPLX;
//   static double wscale();                       // 140^D for Korobov-3, else 1
//   static int eval(const double (&x)[D], double (&g)[CPLX ? 2*J : J]);   // returns Im F >= 0
SectorCode generate_sector(const SectorSpec& s, int case_id);

// __constant__ arrays qmc_tab_log / qmc_tab_exp (/ qmc_tab_trig) of qmc_math.cuh as CUDA source, and their values.
std::string math_tables_source(bool with_trig);
void math_tables(std::vector<double>& log_tab, std::vector<double>& exp_tab);
void math_trig_table(std::vector<double>& trig_tab);   // 256 x (cos, sin)(2 pi j / 256)

}  // namespace qmc
#endif
