// host_tables.hpp -- step S0 of the hot path: everything the kernels need that is derived once on
// the host in fp64 and rounded to fp32 (readings P2, P3, P5, P6).  Pure host C++, no CUDA.
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/bvfdtd.h"

namespace bvfdtd {

// Physical per-material constants of the one-mechanism standard linear solid (reading P3).
struct Derived {
    double rho, piR, muR, tauP, tauS, piU, muU, cU;
};

// Row of the kernels' private coefficient table (8 floats = 32 B, one LDS.128 pair).
// With beta = dt/(2 tau_sigma), A = (1-beta)/(1+beta), B = 2 beta/(1+beta):
//   normal stresses:  r' = A r - (bP th - bS (th - v_ii));  s += (eP th - eS (th - v_ii)) + dt/2 (r' + r)
//   shear nodes:      mu_h = 4 / sum(invMu) (0 if any cell is fluid), ts_h = mean(tauS)
struct KRow {
    float rho;    // density
    float eP;     // dt * pi_U
    float eS;     // 2 dt * mu_U
    float bP;     // B * pi_R * tau_p
    float bS;     // 2 B * mu_R * tau_s
    float invMu;  // 1 / mu_R, or 0 for a fluid (mu_R = 0)
    float tauS;   // tau_s
    float solid;  // 1 if mu_R > 0 else 0
};

struct PmlAxis {
    std::vector<float> a_int, b_int, a_half, b_half;
};

// returns BVFDTD_OK or BVFDTD_EINVAL
int derive_materials(const bvfdtd_material *table, int n, double f0, std::vector<Derived> &out);
void kernel_rows(const std::vector<Derived> &d, double dt, double f0, std::vector<KRow> &rows);
void pml_axis(int n, int pml, double dx, double dt, double f0, double R, double c_ref, PmlAxis &p, bool open_lo = false,
              bool open_hi = false);
double max_courant(const std::vector<Derived> &d, double dt, double dx);

}  // namespace bvfdtd
