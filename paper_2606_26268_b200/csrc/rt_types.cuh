// rt_types.cuh — plain structs passed by value to the kernels (device pointers + sizes).
#pragma once
#include <stdint.h>

namespace rtm1 {

// Separable metric factors (R-G9).  For every cell (i,j,k) and direction d
//   V            = vf[0][i] vf[1][j] vf[2][k]
//   A_d(face f)  = wf[d][f] * prod_{e != d} af[d][e][idx_e]
//   A_d / V      = wf[d][f] * cg[d][0][i] cg[d][1][j] cg[d][2][k]      (cg[d][d] = 1/vf[d], cg[d][e] = af[d][e]/vf[e])
//   dl_d         = len[d][0][i] len[d][1][j] len[d][2][k],  1/dl_d = product of ilen[d][e]
struct GridDev {
    int n[3];    // interior cells
    int gh[3];   // ghosts per side (2 if active else 0)
    int nt[3];   // n + 2 gh
    int bc[6];
    int geometry;
    long long stride[3];  // element strides of x1, x2, x3 in the ghosted arrays
    long long ntot;       // nt1 nt2 nt3
    const double* xf[3];  // edges, n_d + 1
    const double* wf[3];  // n_d + 1
    const double* vf[3];  // n_d
    const double* af[3][3];
    const double* cg[3][3];
    const double* len[3][3];
    const double* ilen[3][3];
    const double* invr;   // <1/r> (spherical) or <1/R> (cylindrical), n1
    const double* cot;    // <cot theta> (spherical), n2
};

struct OpacDev {
    int set;   // 0: never set -> kappa = 0
    int kind;  // 0 power law, 1 table
    int n2a, n2b;  // 2a, 2b when both are integers with |.| <= 64 (half-integer fast path), else INT_MIN
    int fast;      // both exponents are half-integers with |2a|, |2b| <= 15: straight-line evaluation (power_law_fast)
    double kappa0, irho0, iT0, a, b, kmin, kmax;
    int n_lrho, n_lT;
    double lrho_min, lrho_max, lT_min, lT_max;
    double su, sv;  // (n_lrho - 1)/(lrho_max - lrho_min), (n_lT - 1)/(lT_max - lT_min)
    double rho_unit, T_unit;
    const double* tab;  // device, n_lT x n_lrho
};

struct ParamsDev {
    double chat, c, a_R, c_v, E_floor;
    int solver, thick_limit, feedback_momentum;
};

struct Fields4 {
    double* q[4];
};
struct Fields3 {
    double* q[3];
};

}  // namespace rtm1
