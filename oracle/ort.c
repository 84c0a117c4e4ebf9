/* oracle/ort.c — plain, slow, double-precision CPU ORACLE of one gray-M1 radiation sub-step.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.  It shares no code with the CUDA path.
 *
 * What it follows: PAPER.md (arxiv 2606.26268, Scepi & Lesur), Sect. 2.4-2.8.  The method is a
 * discretisation, so the oracle is the algorithm step by step in the paper's order (L109-120):
 *   1 ghost fill (L111) -> 3 reconstruct (Eq. 17-18) -> 4 f-preserving fix (Eq. 19-21) ->
 *   5 wave speeds (Eq. 22-26) -> 6 Riemann flux (L150) -> 7 flux divergence (L117) ->
 *   8 implicit sources (Eq. 29-33, 30, 28) -> 10 time step (L120).
 * No tiling, no fusion, no algebraic shortcuts: every face flux is stored in a full array and the
 * divergence is taken with full 3-D face areas and volumes.  "R-Gn" = reading Gn of DESIGN.md.
 *
 * Parity pins live in tests/test_oracle_*.py.  Readings that nothing outside this repo fixes (R-G7 tau_face = min
 * of the two cells and dx = the cell's largest extent, R-G9 source form, R-G11 floor placement, R-G15 CFL formula)
 * stay conventions; what IS pinned is that the code implements them as stated: tau_cell and the Eq. 25-26 wiring by
 * the hand-worked interface fluxes and the clamp-active diffusion rates of tests/test_oracle_thick_limit.py (each
 * mutation of that block turns one of them red: DESIGN.md Sect. 7), the sources by the curvilinear residual tests,
 * the CFL form by its two closed forms.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC oracle/ort.c -o oracle/libort.so -lm
 */
#include "ort.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

struct ort_grid {
    int geometry;
    int n[3];    /* interior cells */
    int gh[3];   /* ghosts per side: 2 if active else 0 */
    int nt[3];   /* n + 2 gh */
    int bc[6];
    double* xf[3]; /* n[d]+1 edges */
    ort_params par;
    int have_par;
    ort_opacity opac[3];
    double* table[3];
    int have_opac[3];
    long long n_floor, n_clip;
    const double* div_firr; /* caller-owned, ghosted layout, or NULL (Sect. 2.9) */
    int face_fix;           /* ORT_FIX_* (zero-initialised: the f-preserving scheme of Eq. 19-21) */
    int recon;              /* ORT_RECON_* (zero-initialised: PLM + van Leer) */
    double limo3_r;         /* LimO3: radius of the asymptotic region in units of the cell length (<= 0: no switch) */
};

/* ------------------------------------------------------------------------------------------ */
/* point-wise physics                                                                          */
/* ------------------------------------------------------------------------------------------ */

/* Eq. 13 (L75): xi = (3 + 4 f^2) / (5 + 2 sqrt(4 - 3 f^2)) */
double ort_eddington_factor(double f) {
    return (3.0 + 4.0 * f * f) / (5.0 + 2.0 * sqrt(4.0 - 3.0 * f * f));
}

/* reduced flux f = ||F||/E capped at 1 (Eq. 14; the cap is a round-off guard, DESIGN R-G4) */
static double reduced_flux(double E, const double F[3]) {
    double normF = sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
    double f = normF / E;
    if (f > 1.0) f = 1.0;
    return f;
}

/* Eq. 11-12 (L71-73): P^{ij} = D^{ij} E, D^{ij} = (1-xi)/2 delta^{ij} + (3 xi - 1)/2 n^i n^j,
 * n = F/||F|| (L77); the n n term is dropped when ||F|| = 0 (then 3 xi - 1 = 0 anyway). */
void ort_pressure_tensor(double E, const double F[3], double P[9]) {
    double normF = sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
    double f = reduced_flux(E, F);
    double xi = ort_eddington_factor(f);
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) {
            double D = (i == j) ? 0.5 * (1.0 - xi) : 0.0;
            if (normF > 0.0) {
                double ni = F[i] / normF, nj = F[j] / normF;
                D += 0.5 * (3.0 * xi - 1.0) * ni * nj;
            }
            P[3 * i + j] = D * E;
        }
    }
}

/* Eq. 22-24 (L156-162).  theta = angle between F and direction d (L165).
 * lam[0] = lambda_1 (minus sign), lam[1] = lambda_2, lam[2] = lambda_3 (plus sign).
 * zeta^2 is clamped at 0 against round-off at f -> 1 (DESIGN R-G6). */
void ort_wave_speeds(double E, const double F[3], int32_t d, double lam[3]) {
    double normF = sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
    double f = reduced_flux(E, F);
    double cth = (normF > 0.0) ? F[d] / normF : 0.0;
    double s = sqrt(4.0 - 3.0 * f * f);
    double z2 = (2.0 / 3.0) * (4.0 - 3.0 * f * f - s) + 2.0 * cth * cth * (2.0 - f * f - s);
    if (z2 < 0.0) z2 = 0.0;
    double zeta = sqrt(z2);
    lam[0] = (f * cth - zeta) / s;
    lam[2] = (f * cth + zeta) / s;
    /* Eq. 23: (3 xi - 1)/(2 f) cos(theta); its f -> 0 limit is 0 (L167) */
    lam[1] = (f > 0.0) ? (3.0 * ort_eddington_factor(f) - 1.0) / (2.0 * f) * cth : 0.0;
}

/* PLM with the van Leer (harmonic mean) limiter, L132 (DESIGN R-G3): index-space slope */
double ort_vanleer_slope(double qm, double q0, double qp) {
    double dm = q0 - qm, dp = qp - q0;
    if (dm * dp > 0.0) return 2.0 * dm * dp / (dm + dp);
    return 0.0;
}

/* Compact third-order reconstruction LimO3 (L132: Cada & Torrilhon 2009, J. Comput. Phys. 228, 4118; the formula is not
 * printed in PAPER.md: DESIGN R-G22 restates it).  With d- = u_i - u_{i-1}, d+ = u_{i+1} - u_i, theta = d-/d+:
 *   u at the upper face = u_i + 1/2 phi(theta)   d+,      u at the lower face = u_i - 1/2 phi(1/theta) d-,
 *   phi_3(theta)  = (2 + theta)/3                              (unlimited: the quadratic through the three cell averages)
 *   phi_L(theta)  = max(0, min(phi_3, max(-theta/2, min(2 theta, phi_3, 1.6))))
 *   eta = (d-^2 + d+^2)/(r dx)^2;  phi = phi_3 if eta <= 1 - eps, phi_L if eta >= 1 + eps, their linear blend in between,
 *   eps = 1e-12; r <= 0 switches the smooth-extremum detector off (phi = phi_L).
 * A vanishing denominator: phi(theta) d+ -> 0 as d+ -> 0 (phi_L is bounded by 1.6 and by 0 for theta -> -inf). */
static double limo3_phi_times(double dnum, double dden, double eta_or_neg) {
    /* returns phi(dnum/dden) * dden.  phi_3(theta) d+ = (2 d+ + d-)/3 needs no quotient; phi_L(theta) d+ -> 0 for d+ -> 0 */
    double p3 = (2.0 * dden + dnum) / 3.0;
    double pL = 0.0;
    if (dden != 0.0) {
        double theta = dnum / dden;
        double phi3 = (2.0 + theta) / 3.0;
        pL = fmax(0.0, fmin(phi3, fmax(-0.5 * theta, fmin(fmin(2.0 * theta, phi3), 1.6)))) * dden;
    }
    if (eta_or_neg < 0.0) return pL; /* no smoothness switch */
    const double eps = 1.0e-12;
    double eta = eta_or_neg;
    if (eta <= 1.0 - eps) return p3;
    if (eta >= 1.0 + eps) return pL;
    return 0.5 * ((1.0 - (eta - 1.0) / eps) * p3 + (1.0 + (eta - 1.0) / eps) * pL);
}

void ort_limo3_faces(double um, double u0, double up, double dx, double r, double* lo, double* hi) {
    double dm = u0 - um, dp = up - u0;
    double eta = -1.0;
    if (r > 0.0) eta = (dm * dm + dp * dp) / ((r * dx) * (r * dx));
    *hi = u0 + 0.5 * limo3_phi_times(dm, dp, eta);   /* theta = d-/d+ */
    *lo = u0 - 0.5 * limo3_phi_times(dp, dm, eta);   /* 1/theta = d+/d- */
}

/* Eq. 19-21 (L140-146), DESIGN R-G4.  E_f = R(E).  Keep F_f = R(F) iff ||R(F)||/R(E) <= 1 and
 * ||R(F)||/R(E) > ||F_c||/E_c, else F_f = F_c R(E)/E_c.  The two ratio tests are evaluated with
 * the squares cross-multiplied (no division); all three flux components are replaced together. */
void ort_fpreserving_face(const double Uc[4], const double RU[4], double Uf[4]) {
    double Ec = Uc[0], Ef = RU[0];
    double F2c = Uc[1] * Uc[1] + Uc[2] * Uc[2] + Uc[3] * Uc[3];
    double F2f = RU[1] * RU[1] + RU[2] * RU[2] + RU[3] * RU[3];
    Uf[0] = Ef;
    if (F2f <= Ef * Ef && F2f * (Ec * Ec) > F2c * (Ef * Ef)) {
        Uf[1] = RU[1]; Uf[2] = RU[2]; Uf[3] = RU[3];
    } else {
        double r = Ef / Ec;
        Uf[1] = Uc[1] * r; Uf[2] = Uc[2] * r; Uf[3] = Uc[3] * r;
    }
}

/* The "PLUTO reconstruction scheme" as the paper states it (L136): flat reconstruction, E_f = E_c and
 * F_f = F_c, whenever ||R(F)|| > R(E); the reconstructed values otherwise.  Squares compared, no division. */
void ort_pluto_face(const double Uc[4], const double RU[4], double Uf[4]) {
    double Ef = RU[0];
    double F2f = RU[1] * RU[1] + RU[2] * RU[2] + RU[3] * RU[3];
    if (F2f > Ef * Ef) {
        for (int q = 0; q < 4; ++q) Uf[q] = Uc[q];
    } else {
        for (int q = 0; q < 4; ++q) Uf[q] = RU[q];
    }
}

/* Eq. 36-38 (L272-279), the scheme of Fig. 5's first panel: E_f = R(E); F_f = R(F) while
 * ||R(F)||/R(E) <= 1, otherwise R(F) rescaled to ||F_f|| = R(E) (direction kept). */
void ort_clip_face(const double RU[4], double Uf[4]) {
    double Ef = RU[0];
    double F2f = RU[1] * RU[1] + RU[2] * RU[2] + RU[3] * RU[3];
    Uf[0] = Ef;
    if (F2f <= Ef * Ef) {
        Uf[1] = RU[1]; Uf[2] = RU[2]; Uf[3] = RU[3];
    } else {
        double r = Ef / sqrt(F2f);
        Uf[1] = RU[1] * r; Uf[2] = RU[2] * r; Uf[3] = RU[3] * r;
    }
}

/* physical flux of Eq. 5-6 (L49-51) through a face normal to d: chat (F^d, P^{1d}, P^{2d}, P^{3d}) */
static void physical_flux(const double U[4], int d, double chat, double flux[4]) {
    double P[9];
    ort_pressure_tensor(U[0], &U[1], P);
    flux[0] = chat * U[1 + d];
    flux[1] = chat * P[3 * 0 + d];
    flux[2] = chat * P[3 * 1 + d];
    flux[3] = chat * P[3 * 2 + d];
}

/* L150 + Sect. 2.6.  HLL (two-wave, textbook form; DESIGN R-G5) with
 * S_L = chat min(lam1(U_L), lam1(U_R), 0), S_R = chat max(lam3(U_L), lam3(U_R), 0) (R-G6),
 * then Eq. 25-26: S_L = max(S_L, -lim), S_R = min(S_R, lim), lim = 4 chat/(3 tau) (R-G7).
 * den = S_R - S_L; den > 0 ? HLL formula : plain average (R-G8).
 * GLF: 1/2 (F_L + F_R) - 1/2 alpha (U_R - U_L), alpha = min(chat, lim).
 * Rusanov ("Lax-Friedrichs-Rusanov", L150; DESIGN R-G5): the same form with the LOCAL bound
 * alpha = min(chat max(|lam1(U_L)|, |lam3(U_L)|, |lam1(U_R)|, |lam3(U_R)|), lim). */
void ort_riemann_flux(const double UL[4], const double UR[4], int32_t d, double chat, int32_t solver,
                      double lim, double flux[4]) {
    double FL[4], FR[4];
    physical_flux(UL, d, chat, FL);
    physical_flux(UR, d, chat, FR);
    if (solver == ORT_SOLVER_GLF) {
        double alpha = (chat < lim) ? chat : lim;
        for (int q = 0; q < 4; ++q) flux[q] = 0.5 * (FL[q] + FR[q]) - 0.5 * alpha * (UR[q] - UL[q]);
        return;
    }
    double lamL[3], lamR[3];
    ort_wave_speeds(UL[0], &UL[1], d, lamL);
    ort_wave_speeds(UR[0], &UR[1], d, lamR);
    if (solver == ORT_SOLVER_RUSANOV) {
        double alpha = fmax(fmax(fabs(lamL[0]), fabs(lamL[2])), fmax(fabs(lamR[0]), fabs(lamR[2]))) * chat;
        if (alpha > lim) alpha = lim;
        for (int q = 0; q < 4; ++q) flux[q] = 0.5 * (FL[q] + FR[q]) - 0.5 * alpha * (UR[q] - UL[q]);
        return;
    }
    double SL = fmin(fmin(lamL[0], lamR[0]), 0.0) * chat;
    double SR = fmax(fmax(lamL[2], lamR[2]), 0.0) * chat;
    if (SL < -lim) SL = -lim;
    if (SR > lim) SR = lim;
    double den = SR - SL;
    for (int q = 0; q < 4; ++q) {
        if (den > 0.0)
            flux[q] = (SR * FL[q] - SL * FR[q] + SR * SL * (UR[q] - UL[q])) / den;
        else
            flux[q] = 0.5 * (FL[q] + FR[q]);
    }
}

/* L299 (power law, clipped) and L375 (table, here 2-D bilinear in log10; DESIGN R-G14) */
double ort_opacity_eval(const ort_opacity* o, double rho, double T) {
    if (o->kind == 0) {
        double k = o->kappa0 * pow(rho / o->rho0, o->a) * pow(T / o->T0, o->b);
        if (k < o->kmin) k = o->kmin;
        if (k > o->kmax) k = o->kmax;
        return k;
    }
    const double* tab = o->log10_kappa;
    double y = log10(T * o->T_unit);
    if (y < o->lT_min) y = o->lT_min;
    if (y > o->lT_max) y = o->lT_max;
    double v = (y - o->lT_min) / (o->lT_max - o->lT_min) * (double)(o->n_lT - 1);
    int j0 = (int)floor(v);
    if (j0 < 0) j0 = 0;
    if (j0 > o->n_lT - 2) j0 = o->n_lT - 2;
    double tv = v - (double)j0;
    double val;
    if (o->n_lrho == 1) {
        val = (1.0 - tv) * tab[j0] + tv * tab[j0 + 1];
    } else {
        double x = log10(rho * o->rho_unit);
        if (x < o->lrho_min) x = o->lrho_min;
        if (x > o->lrho_max) x = o->lrho_max;
        double u = (x - o->lrho_min) / (o->lrho_max - o->lrho_min) * (double)(o->n_lrho - 1);
        int i0 = (int)floor(u);
        if (i0 < 0) i0 = 0;
        if (i0 > o->n_lrho - 2) i0 = o->n_lrho - 2;
        double tu = u - (double)i0;
        int nr = o->n_lrho;
        double v00 = tab[j0 * nr + i0], v01 = tab[j0 * nr + i0 + 1];
        double v10 = tab[(j0 + 1) * nr + i0], v11 = tab[(j0 + 1) * nr + i0 + 1];
        val = (1.0 - tv) * ((1.0 - tu) * v00 + tu * v01) + tv * ((1.0 - tu) * v10 + tu * v11);
    }
    return pow(10.0, val);
}

/* Eq. 29-33 (L195-216) solved per cell; DESIGN R-G12: the analytic inverse of the 2x2 of Eq. 33,
 *   det = C_v (1 + g_r) + 4 g a_R T^3,
 *   E'  = [E (C_v + 4 g a_R T^3) + g_r C_v a_R T^4] / det,
 *   T'  = [(1 + g_r) C_v T + 3 g a_R T^4 + g E] / det,
 * with g_r = dt chat kappa_P rho (gamma_abs,red), g = dt c kappa_P rho (gamma_abs), C_v = rho c_v.
 * Eq. 30 (L198): F' = F / (1 + dt chat chi rho).  Eq. 28 (L183): m' = m - (F' - F)/chat.
 * Irradiation (Sect. 2.9, Eq. 34-35): Q = -div F_irr dt is added to S_1 = C_v T + 3 g a_R T^4 of Eq. 33;
 * with S_0 = E - 3 g_r a_R T^4 the analytic inverse reads
 *   E' = [S_0 (C_v + 4 g a_R T^3) + 4 g_r a_R T^3 S_1] / det,   T' = [g S_0 + (1 + g_r) S_1] / det,
 * which is the form above for Q = 0; it is evaluated as that form plus the two Q terms. */
void ort_implicit_cell(const ort_params* p, double dt, double rho, double kappaP, double chi,
                       double* E, double F[3], double* T, double* mom, double Q) {
    double T0 = *T, E0 = *E;
    double gr = dt * p->chat * kappaP * rho;
    double g = dt * p->c * kappaP * rho;
    double Cv = rho * p->c_v;
    double aT3 = p->a_R * T0 * T0 * T0;
    double aT4 = aT3 * T0;
    double det = Cv * (1.0 + gr) + 4.0 * g * aT3;
    *E = (E0 * (Cv + 4.0 * g * aT3) + gr * Cv * aT4) / det;
    *T = ((1.0 + gr) * Cv * T0 + 3.0 * g * aT4 + g * E0) / det;
    if (Q != 0.0) {
        *E += 4.0 * gr * aT3 * Q / det;
        *T += (1.0 + gr) * Q / det;
    }
    double damp = 1.0 + dt * p->chat * chi * rho;
    for (int q = 0; q < 3; ++q) {
        double Fn = F[q] / damp;
        if (mom) mom[q] = mom[q] - (Fn - F[q]) / p->chat;
        F[q] = Fn;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* grid, metrics                                                                               */
/* ------------------------------------------------------------------------------------------ */

static inline long IDX(const ort_grid* g, int i, int j, int k) {
    return ((long)(k + g->gh[2]) * g->nt[1] + (j + g->gh[1])) * g->nt[0] + (i + g->gh[0]);
}
static inline long total_cells(const ort_grid* g) { return (long)g->nt[0] * g->nt[1] * g->nt[2]; }

int32_t ort_grid_create(int32_t geometry, const int32_t n[3], int32_t nghost,
                        const double* x1f, const double* x2f, const double* x3f,
                        const int32_t bc[6], ort_grid** out) {
    if (!n || !x1f || !x2f || !x3f || !bc || !out) return ORT_ERR_INVALID_ARG;
    if (geometry < 0 || geometry > 2 || nghost != 2) return ORT_ERR_INVALID_ARG;
    const double* xf[3] = {x1f, x2f, x3f};
    for (int d = 0; d < 3; ++d) {
        if (n[d] < 1) return ORT_ERR_INVALID_ARG;
        for (int i = 0; i <= n[d]; ++i)
            if (!isfinite(xf[d][i])) return ORT_ERR_INVALID_ARG;
        for (int i = 0; i < n[d]; ++i)
            if (!(xf[d][i + 1] > xf[d][i])) return ORT_ERR_INVALID_ARG;
        if (bc[2 * d] < 0 || bc[2 * d] > 3 || bc[2 * d + 1] < 0 || bc[2 * d + 1] > 3) return ORT_ERR_INVALID_ARG;
        if ((bc[2 * d] == ORT_BC_PERIODIC) != (bc[2 * d + 1] == ORT_BC_PERIODIC)) return ORT_ERR_INVALID_ARG;
    }
    if (geometry != ORT_CARTESIAN && x1f[0] < 0.0) return ORT_ERR_INVALID_ARG;
    if (geometry == ORT_SPHERICAL && (x2f[0] < 0.0 || x2f[n[1]] > M_PI)) return ORT_ERR_INVALID_ARG;
    ort_grid* g = (ort_grid*)calloc(1, sizeof(ort_grid));
    g->geometry = geometry;
    for (int d = 0; d < 3; ++d) {
        g->n[d] = n[d];
        g->gh[d] = (n[d] > 1) ? nghost : 0;
        g->nt[d] = n[d] + 2 * g->gh[d];
        g->bc[2 * d] = bc[2 * d];
        g->bc[2 * d + 1] = bc[2 * d + 1];
        g->xf[d] = (double*)malloc(sizeof(double) * (size_t)(n[d] + 1));
        memcpy(g->xf[d], xf[d], sizeof(double) * (size_t)(n[d] + 1));
    }
    *out = g;
    return ORT_OK;
}

int32_t ort_grid_destroy(ort_grid* g) {
    if (!g) return ORT_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d) free(g->xf[d]);
    for (int w = 0; w < 3; ++w) free(g->table[w]);
    free(g);
    return ORT_OK;
}

/* DESIGN R-G9 (the paper gives no metric formulas, L15/L409): exact finite-volume integrals.
 *  Cartesian   V = dx1 dx2 dx3
 *  Cylindrical V = 1/2 D(R^2) Dphi Dz                    (R, phi, z)
 *  Spherical   V = 1/3 D(r^3) D(-cos th) Dphi            (r, theta, phi) */
static double cell_volume(const ort_grid* g, int i, int j, int k) {
    double a0 = g->xf[0][i], a1 = g->xf[0][i + 1];
    double b0 = g->xf[1][j], b1 = g->xf[1][j + 1];
    double c0 = g->xf[2][k], c1 = g->xf[2][k + 1];
    if (g->geometry == ORT_CARTESIAN) return (a1 - a0) * (b1 - b0) * (c1 - c0);
    if (g->geometry == ORT_CYLINDRICAL) return 0.5 * (a1 * a1 - a0 * a0) * (b1 - b0) * (c1 - c0);
    return (a1 * a1 * a1 - a0 * a0 * a0) / 3.0 * (cos(b0) - cos(b1)) * (c1 - c0);
}

/* area of the LOWER face in direction d of cell (i,j,k); the index along d may equal n[d]
 * (the last upper face).  R-G9:
 *  Cartesian   A1 = dx2 dx3, A2 = dx1 dx3, A3 = dx1 dx2
 *  Cylindrical A_R = R_f Dphi Dz, A_phi = DR Dz, A_z = 1/2 D(R^2) Dphi
 *  Spherical   A_r = r_f^2 D(-cos th) Dphi, A_th = 1/2 D(r^2) sin(th_f) Dphi, A_phi = 1/2 D(r^2) Dth */
static double face_area(const ort_grid* g, int d, int i, int j, int k) {
    const double* x1 = g->xf[0];
    const double* x2 = g->xf[1];
    const double* x3 = g->xf[2];
    if (g->geometry == ORT_CARTESIAN) {
        if (d == 0) return (x2[j + 1] - x2[j]) * (x3[k + 1] - x3[k]);
        if (d == 1) return (x1[i + 1] - x1[i]) * (x3[k + 1] - x3[k]);
        return (x1[i + 1] - x1[i]) * (x2[j + 1] - x2[j]);
    }
    if (g->geometry == ORT_CYLINDRICAL) {
        if (d == 0) return x1[i] * (x2[j + 1] - x2[j]) * (x3[k + 1] - x3[k]);
        if (d == 1) return (x1[i + 1] - x1[i]) * (x3[k + 1] - x3[k]);
        return 0.5 * (x1[i + 1] * x1[i + 1] - x1[i] * x1[i]) * (x2[j + 1] - x2[j]);
    }
    if (d == 0) return x1[i] * x1[i] * (cos(x2[j]) - cos(x2[j + 1])) * (x3[k + 1] - x3[k]);
    if (d == 1) return 0.5 * (x1[i + 1] * x1[i + 1] - x1[i] * x1[i]) * sin(x2[j]) * (x3[k + 1] - x3[k]);
    return 0.5 * (x1[i + 1] * x1[i + 1] - x1[i] * x1[i]) * (x2[j + 1] - x2[j]);
}

/* physical length of cell (i,j,k) along d, used by tau_cell (L175) and the CFL (L120). R-G9:
 * Cartesian dx_d; cylindrical DR, R_c Dphi, Dz; spherical Dr, r_c Dth, r_c sin(th_c) Dphi, with
 * arithmetic-mean centres. */
static double cell_length(const ort_grid* g, int d, int i, int j, int k) {
    const double* x1 = g->xf[0];
    const double* x2 = g->xf[1];
    const double* x3 = g->xf[2];
    double d1 = x1[i + 1] - x1[i], d2 = x2[j + 1] - x2[j], d3 = x3[k + 1] - x3[k];
    if (g->geometry == ORT_CARTESIAN) return d == 0 ? d1 : (d == 1 ? d2 : d3);
    double rc = 0.5 * (x1[i] + x1[i + 1]);
    if (g->geometry == ORT_CYLINDRICAL) return d == 0 ? d1 : (d == 1 ? rc * d2 : d3);
    double thc = 0.5 * (x2[j] + x2[j + 1]);
    return d == 0 ? d1 : (d == 1 ? rc * d2 : rc * sin(thc) * d3);
}

int32_t ort_grid_get_metrics(const ort_grid* g, double* vol, double* area1, double* area2, double* area3) {
    if (!g) return ORT_ERR_INVALID_ARG;
    const int n1 = g->n[0], n2 = g->n[1], n3 = g->n[2];
    if (vol)
        for (int k = 0; k < n3; ++k)
            for (int j = 0; j < n2; ++j)
                for (int i = 0; i < n1; ++i) vol[((long)k * n2 + j) * n1 + i] = cell_volume(g, i, j, k);
    if (area1)
        for (int k = 0; k < n3; ++k)
            for (int j = 0; j < n2; ++j)
                for (int i = 0; i <= n1; ++i) area1[((long)k * n2 + j) * (n1 + 1) + i] = face_area(g, 0, i, j, k);
    if (area2)
        for (int k = 0; k < n3; ++k)
            for (int j = 0; j <= n2; ++j)
                for (int i = 0; i < n1; ++i) area2[((long)k * (n2 + 1) + j) * n1 + i] = face_area(g, 1, i, j, k);
    if (area3)
        for (int k = 0; k <= n3; ++k)
            for (int j = 0; j < n2; ++j)
                for (int i = 0; i < n1; ++i) area3[((long)k * n2 + j) * n1 + i] = face_area(g, 2, i, j, k);
    return ORT_OK;
}

int32_t ort_set_params(ort_grid* g, const ort_params* p) {
    if (!g || !p) return ORT_ERR_INVALID_ARG;
    if (!(p->chat > 0.0) || !(p->c > 0.0) || !(p->a_R >= 0.0) || !(p->c_v > 0.0) || !(p->E_floor >= 0.0))
        return ORT_ERR_INVALID_ARG;
    if (p->solver != ORT_SOLVER_HLL && p->solver != ORT_SOLVER_GLF && p->solver != ORT_SOLVER_RUSANOV) return ORT_ERR_INVALID_ARG;
    g->par = *p;
    g->have_par = 1;
    return ORT_OK;
}

int32_t ort_set_opacity(ort_grid* g, int32_t which, const ort_opacity* o) {
    if (!g || !o || which < 0 || which > 2) return ORT_ERR_INVALID_ARG;
    if (o->kind == 0) {
        if (!(o->rho0 > 0.0) || !(o->T0 > 0.0) || !(o->kmax >= o->kmin) || !(o->kmin >= 0.0)) return ORT_ERR_INVALID_ARG;
    } else if (o->kind == 1) {
        if (!o->log10_kappa || o->n_lT < 2 || (o->n_lrho < 2 && o->n_lrho != 1)) return ORT_ERR_INVALID_ARG;
        if (!(o->lT_max > o->lT_min) || !(o->T_unit > 0.0)) return ORT_ERR_INVALID_ARG;
        if (o->n_lrho > 1 && (!(o->lrho_max > o->lrho_min) || !(o->rho_unit > 0.0))) return ORT_ERR_INVALID_ARG;
    } else {
        return ORT_ERR_INVALID_ARG;
    }
    free(g->table[which]);
    g->table[which] = NULL;
    g->opac[which] = *o;
    if (o->kind == 1) {
        size_t sz = sizeof(double) * (size_t)o->n_lT * (size_t)o->n_lrho;
        g->table[which] = (double*)malloc(sz);
        memcpy(g->table[which], o->log10_kappa, sz);
        g->opac[which].log10_kappa = g->table[which];
    }
    g->have_opac[which] = 1;
    return ORT_OK;
}

/* an opacity that was never set is zero */
static double opacity_of(const ort_grid* g, int which, double rho, double T) {
    if (!g->have_opac[which]) return 0.0;
    return ort_opacity_eval(&g->opac[which], rho, T);
}

/* ------------------------------------------------------------------------------------------ */
/* step 1: boundary conditions (L111)                                                          */
/* ------------------------------------------------------------------------------------------ */
/* periodic: copy from the opposite interior; outflow: copy the nearest interior cell into both
 * ghosts (L260); reflect: mirror, normal flux component negated (L291); fixed: left as the
 * caller wrote them (injection boundary, L289).  Axis by axis: x1, then x2 over the x1-extended
 * range, then x3 over the x1,x2-extended range. */
int32_t ort_fill_ghosts(ort_grid* g, double* const U[4]) {
    if (!g || !U) return ORT_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d) {
        if (g->gh[d] == 0) continue;
        int lo[3], hi[3]; /* loop bounds of the other axes */
        for (int a = 0; a < 3; ++a) {
            if (a < d) { lo[a] = -g->gh[a]; hi[a] = g->n[a] + g->gh[a]; }
            else       { lo[a] = 0;         hi[a] = g->n[a]; }
        }
        for (int side = 0; side < 2; ++side) {
            int kind = g->bc[2 * d + side];
            if (kind == ORT_BC_FIXED) continue;
            for (int gl = 0; gl < g->gh[d]; ++gl) {
                int dst = side == 0 ? -1 - gl : g->n[d] + gl;
                int src;
                if (kind == ORT_BC_PERIODIC) src = side == 0 ? g->n[d] - 1 - gl : gl;
                else if (kind == ORT_BC_OUTFLOW) src = side == 0 ? 0 : g->n[d] - 1;
                else src = side == 0 ? gl : g->n[d] - 1 - gl; /* reflect */
                int c[3];
                lo[d] = 0; hi[d] = 1;
                for (c[2] = lo[2]; c[2] < hi[2]; ++c[2])
                    for (c[1] = lo[1]; c[1] < hi[1]; ++c[1])
                        for (c[0] = lo[0]; c[0] < hi[0]; ++c[0]) {
                            int cd[3] = {c[0], c[1], c[2]}, cs[3] = {c[0], c[1], c[2]};
                            cd[d] = dst; cs[d] = src;
                            long id = IDX(g, cd[0], cd[1], cd[2]), is = IDX(g, cs[0], cs[1], cs[2]);
                            for (int q = 0; q < 4; ++q) U[q][id] = U[q][is];
                            if (kind == ORT_BC_REFLECT) U[1 + d][id] = -U[1 + d][is];
                        }
            }
        }
    }
    return ORT_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* steps 3-7: explicit transport                                                               */
/* ------------------------------------------------------------------------------------------ */

/* steps 3+4 for one cell and one direction: PLM (Eq. 17-18) then the f-preserving fix (Eq. 19-21;
 * or, on request, the flat fallback of L136 / the clip of Eq. 36-38: ort_set_face_fix)
 * for the cell's lower-face state (the RIGHT state of face i-1/2) and upper-face state (the LEFT
 * state of face i+1/2). */
static void cell_face_states(const ort_grid* g, double* const U[4], long idx, long stride, double dx,
                             double Ulo[4], double Uhi[4]) {
    double Uc[4], Rlo[4], Rhi[4];
    for (int q = 0; q < 4; ++q) {
        double qm = U[q][idx - stride], q0 = U[q][idx], qp = U[q][idx + stride];
        Uc[q] = q0;
        if (g->recon == ORT_RECON_LIMO3) {
            ort_limo3_faces(qm, q0, qp, dx, g->limo3_r, &Rlo[q], &Rhi[q]);
        } else {
            double slope = ort_vanleer_slope(qm, q0, qp);
            Rlo[q] = q0 - 0.5 * slope;
            Rhi[q] = q0 + 0.5 * slope;
        }
    }
    if (g->face_fix == ORT_FIX_PLUTO) {
        ort_pluto_face(Uc, Rlo, Ulo);
        ort_pluto_face(Uc, Rhi, Uhi);
    } else if (g->face_fix == ORT_FIX_CLIP) {
        ort_clip_face(Rlo, Ulo);
        ort_clip_face(Rhi, Uhi);
    } else {
        ort_fpreserving_face(Uc, Rlo, Ulo);
        ort_fpreserving_face(Uc, Rhi, Uhi);
    }
}

/* tau_cell = rho chi dx, dx = the cell's largest physical extent over active dimensions
 * (L175 "cell of maximum size dx"; DESIGN R-G7), chi = kappa_R + sigma (L89). */
static double tau_cell(const ort_grid* g, const double* rho, const double* T, int i, int j, int k) {
    long id = IDX(g, i, j, k);
    double chi = opacity_of(g, ORT_OPAC_ROSSELAND, rho[id], T[id]) + opacity_of(g, ORT_OPAC_SCATTER, rho[id], T[id]);
    double dx = 0.0;
    for (int d = 0; d < 3; ++d)
        if (g->gh[d] > 0) dx = fmax(dx, cell_length(g, d, i, j, k));
    return rho[id] * chi * dx;
}

static inline int wrap_or_clamp(const ort_grid* g, int d, int i) {
    if (i >= 0 && i < g->n[d]) return i;
    if (g->bc[2 * d] == ORT_BC_PERIODIC) return (i + g->n[d]) % g->n[d];
    return i < 0 ? 0 : g->n[d] - 1;
}

int32_t ort_explicit_step(ort_grid* g, double dt, const double* rho, const double* T,
                          double* const U_in[4], double* const U_out[4]) {
    if (!g || !U_in || !U_out || !g->have_par) return g && !g->have_par ? ORT_ERR_BAD_STATE : ORT_ERR_INVALID_ARG;
    if (!(dt > 0.0) || !isfinite(dt)) return ORT_ERR_INVALID_ARG;
    for (int q = 0; q < 4; ++q)
        if (!U_in[q] || !U_out[q] || U_in[q] == U_out[q]) return ORT_ERR_INVALID_ARG;
    const ort_params* p = &g->par;
    if (p->thick_limit && (!rho || !T)) return ORT_ERR_INVALID_ARG;
    const int n1 = g->n[0], n2 = g->n[1], n3 = g->n[2];
    const long stride[3] = {1, g->nt[0], (long)g->nt[0] * g->nt[1]};

    /* step 1 */
    ort_fill_ghosts(g, U_in);

    /* per-cell optical depth for Eq. 25-26; ghosts of tau: periodic wrap, else nearest interior (R-G7) */
    double* tau = NULL;
    if (p->thick_limit) {
        tau = (double*)malloc(sizeof(double) * (size_t)total_cells(g));
#pragma omp parallel for collapse(2)
        for (int k = -g->gh[2]; k < n3 + g->gh[2]; ++k)
            for (int j = -g->gh[1]; j < n2 + g->gh[1]; ++j)
                for (int i = -g->gh[0]; i < n1 + g->gh[0]; ++i)
                    tau[IDX(g, i, j, k)] = tau_cell(g, rho, T, wrap_or_clamp(g, 0, i), wrap_or_clamp(g, 1, j),
                                                    wrap_or_clamp(g, 2, k));
    }

    /* steps 3-6: one full array of face fluxes per active direction */
    double* flux[3][4] = {{0}};
    for (int d = 0; d < 3; ++d) {
        if (g->gh[d] == 0) continue;
        int nf[3] = {n1, n2, n3};
        nf[d] += 1;
        size_t sz = (size_t)nf[0] * nf[1] * nf[2];
        for (int q = 0; q < 4; ++q) flux[d][q] = (double*)malloc(sizeof(double) * sz);
#pragma omp parallel for collapse(2)
        for (int k = 0; k < nf[2]; ++k)
            for (int j = 0; j < nf[1]; ++j)
                for (int i = 0; i < nf[0]; ++i) {
                    /* face between cell a = (i,j,k) - e_d and cell b = (i,j,k) */
                    long ib = IDX(g, i, j, k), ia = ib - stride[d];
                    double aLo[4], aHi[4], bLo[4], bHi[4];
                    /* LimO3's smoothness switch wants the cell's length along d (ghost cells: that of the nearest
                     * interior cell) */
                    int ca[3] = {i, j, k}, cb[3] = {i, j, k};
                    ca[d] -= 1;
                    for (int e = 0; e < 3; ++e) {
                        ca[e] = ca[e] < 0 ? 0 : (ca[e] > g->n[e] - 1 ? g->n[e] - 1 : ca[e]);
                        cb[e] = cb[e] > g->n[e] - 1 ? g->n[e] - 1 : cb[e];
                    }
                    cell_face_states(g, U_in, ia, stride[d], cell_length(g, d, ca[0], ca[1], ca[2]), aLo, aHi);
                    cell_face_states(g, U_in, ib, stride[d], cell_length(g, d, cb[0], cb[1], cb[2]), bLo, bHi);
                    double lim = INFINITY;
                    if (p->thick_limit) {
                        double tf = fmin(tau[ia], tau[ib]);
                        lim = 4.0 * p->chat / (3.0 * tf);
                    }
                    double f4[4];
                    ort_riemann_flux(aHi, bLo, d, p->chat, p->solver, lim, f4);
                    size_t fi = ((size_t)k * nf[1] + j) * nf[0] + i;
                    for (int q = 0; q < 4; ++q) flux[d][q][fi] = f4[q];
                }
    }

    /* step 7: U* = U^n - dt sum_d [A+ F+ - A- F-]/V + dt S_geo(U^n)   (L117; R-G9) */
#pragma omp parallel for collapse(2)
    for (int k = 0; k < n3; ++k)
        for (int j = 0; j < n2; ++j)
            for (int i = 0; i < n1; ++i) {
                long id = IDX(g, i, j, k);
                double V = cell_volume(g, i, j, k);
                double div[4] = {0, 0, 0, 0};
                for (int d = 0; d < 3; ++d) {
                    if (g->gh[d] == 0) continue;
                    int nf[3] = {n1, n2, n3};
                    nf[d] += 1;
                    int c[3] = {i, j, k};
                    size_t lo = ((size_t)c[2] * nf[1] + c[1]) * nf[0] + c[0];
                    c[d] += 1;
                    size_t hi = ((size_t)c[2] * nf[1] + c[1]) * nf[0] + c[0];
                    double Am = face_area(g, d, i, j, k);
                    double Ap = face_area(g, d, c[0], c[1], c[2]);
                    for (int q = 0; q < 4; ++q) div[q] += (Ap * flux[d][q][hi] - Am * flux[d][q][lo]) / V;
                }
                /* geometric sources from the cell-centred closure P(U^n) with volume-averaged
                 * metric factors (R-G9).  E has none.
                 *  cyl: S(F^R) = +chat P^{phiphi} <1/R>,  S(F^phi) = -chat P^{Rphi} <1/R>
                 *  sph: S(F^r)  = chat (P^{thth} + P^{phph}) <1/r>
                 *       S(F^th) = chat (-P^{rth} + <cot th> P^{phph}) <1/r>
                 *       S(F^ph) = chat (-P^{rph} - <cot th> P^{thph}) <1/r> */
                double S[4] = {0, 0, 0, 0};
                if (g->geometry != ORT_CARTESIAN) {
                    double Uc[4] = {U_in[0][id], U_in[1][id], U_in[2][id], U_in[3][id]};
                    double P[9];
                    ort_pressure_tensor(Uc[0], &Uc[1], P);
                    double r0 = g->xf[0][i], r1 = g->xf[0][i + 1];
                    if (g->geometry == ORT_CYLINDRICAL) {
                        double invR = (r1 - r0) / (0.5 * (r1 * r1 - r0 * r0));
                        S[1] = p->chat * P[3 * 1 + 1] * invR;
                        S[2] = -p->chat * P[3 * 0 + 1] * invR;
                    } else {
                        double invr = 0.5 * (r1 * r1 - r0 * r0) / ((r1 * r1 * r1 - r0 * r0 * r0) / 3.0);
                        double t0 = g->xf[1][j], t1 = g->xf[1][j + 1];
                        double cot = (sin(t1) - sin(t0)) / (cos(t0) - cos(t1));
                        S[1] = p->chat * (P[3 * 1 + 1] + P[3 * 2 + 2]) * invr;
                        S[2] = p->chat * (-P[3 * 0 + 1] + cot * P[3 * 2 + 2]) * invr;
                        S[3] = p->chat * (-P[3 * 0 + 2] - cot * P[3 * 1 + 2]) * invr;
                    }
                }
                for (int q = 0; q < 4; ++q) U_out[q][id] = U_in[q][id] - dt * div[q] + dt * S[q];
            }

    for (int d = 0; d < 3; ++d)
        for (int q = 0; q < 4; ++q) free(flux[d][q]);
    free(tau);
    return ORT_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* step 8: floor / clip, opacities, implicit coupling                                          */
/* ------------------------------------------------------------------------------------------ */
/* Sect. 2.5 / 3.2: which face fix the explicit step applies */
int32_t ort_set_face_fix(ort_grid* g, int32_t mode) {
    if (!g || mode < ORT_FIX_FPRESERVING || mode > ORT_FIX_CLIP) return ORT_ERR_INVALID_ARG;
    g->face_fix = mode;
    return ORT_OK;
}

/* L132: which standard reconstruction R() the explicit step applies */
int32_t ort_set_reconstruction(ort_grid* g, int32_t kind, double r) {
    if (!g || (kind != ORT_RECON_PLM && kind != ORT_RECON_LIMO3) || !isfinite(r)) return ORT_ERR_INVALID_ARG;
    g->recon = kind;
    g->limo3_r = r;
    return ORT_OK;
}

/* Sect. 2.9: div F_irr per cell (host, ghosted layout, caller-owned; NULL switches irradiation off) */
int32_t ort_set_irradiation(ort_grid* g, const double* div_firr) {
    if (!g) return ORT_ERR_INVALID_ARG;
    g->div_firr = div_firr;
    return ORT_OK;
}

/* Sect. 3.7 (L379-383), gray (DESIGN R-G21).  Eq. 48: tau_irr(r) = int_{r_in}^{r} kappa rho dr' with rho constant in a
 * cell: tau at the upper face of cell i = tau at its lower face + kappa rho_i (r_{i+1/2} - r_{i-1/2}).  Eq. 47 with the
 * frequency integral collapsed to one gray band: F_irr(r) = L0 e^{-tau}/r^2 r_hat, L0 = F_s R_s^2.  Finite-volume
 * divergence of a purely radial flux in a spherical cell: [A_+ F_+ - A_- F_-]/V = 3 (r_+^2 F_+ - r_-^2 F_-)/(r_+^3 - r_-^3)
 * = 3 L0 (e^{-tau_+} - e^{-tau_-})/(r_+^3 - r_-^3); the difference of exponentials is written e^{-tau_-} expm1(-dtau)
 * (the same number, without the cancellation of optically thin cells).  Cartesian: plane-parallel rays along x1,
 * F_irr = L0 e^{-tau}, div = (F_+ - F_-)/dx. */
int32_t ort_irradiation_radial(ort_grid* g, double L0, double kappa_irr, double tau_in, const double* rho,
                               double* tau_hi, double* div_firr) {
    if (!g || !rho || !div_firr) return ORT_ERR_INVALID_ARG;
    if (g->geometry == ORT_CYLINDRICAL) return ORT_ERR_INVALID_ARG;
    if (!(kappa_irr >= 0.0) || !(tau_in >= 0.0) || !isfinite(L0) || !isfinite(kappa_irr) || !isfinite(tau_in)) return ORT_ERR_INVALID_ARG;
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j) {
            double tau_lo = tau_in;
            for (int i = 0; i < g->n[0]; ++i) {
                long id = IDX(g, i, j, k);
                double rm = g->xf[0][i], rp = g->xf[0][i + 1];
                double dtau = kappa_irr * rho[id] * (rp - rm);
                double geo = g->geometry == ORT_SPHERICAL ? 3.0 / (rp * rp * rp - rm * rm * rm) : 1.0 / (rp - rm);
                div_firr[id] = L0 * exp(-tau_lo) * expm1(-dtau) * geo;
                tau_lo = tau_lo + dtau;
                if (tau_hi) tau_hi[id] = tau_lo;
            }
        }
    return ORT_OK;
}

int32_t ort_implicit_step(ort_grid* g, double dt, const double* rho, double* T,
                          double* const mom[3], double* const U[4]) {
    if (!g || !U || !rho || !T) return ORT_ERR_INVALID_ARG;
    if (!g->have_par) return ORT_ERR_BAD_STATE;
    if (!(dt > 0.0) || !isfinite(dt)) return ORT_ERR_INVALID_ARG;
    const ort_params* p = &g->par;
    int feedback = p->feedback_momentum && mom != NULL;
    long long nfl = 0, ncl = 0;
#pragma omp parallel for collapse(2) reduction(+ : nfl, ncl)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i) {
                long id = IDX(g, i, j, k);
                double E = U[0][id];
                double F[3] = {U[1][id], U[2][id], U[3][id]};
                /* positivity of E (L250) and f <= 1 at the cell centre (L81); DESIGN R-G11 */
                if (E < p->E_floor) { E = p->E_floor; ++nfl; }
                double normF = sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
                if (normF > E) {
                    for (int q = 0; q < 3; ++q) F[q] = F[q] * E / normF;
                    ++ncl;
                }
                double kP = opacity_of(g, ORT_OPAC_PLANCK, rho[id], T[id]);
                double chi = opacity_of(g, ORT_OPAC_ROSSELAND, rho[id], T[id]) +
                             opacity_of(g, ORT_OPAC_SCATTER, rho[id], T[id]);
                double Tc = T[id];
                double m[3] = {0, 0, 0};
                if (feedback)
                    for (int q = 0; q < 3; ++q) m[q] = mom[q][id];
                double Q = g->div_firr ? -g->div_firr[id] * dt : 0.0; /* Eq. 34-35 */
                ort_implicit_cell(p, dt, rho[id], kP, chi, &E, F, &Tc, feedback ? m : NULL, Q);
                U[0][id] = E; U[1][id] = F[0]; U[2][id] = F[1]; U[3][id] = F[2];
                T[id] = Tc;
                if (feedback)
                    for (int q = 0; q < 3; ++q) mom[q][id] = m[q];
            }
    g->n_floor += nfl;
    g->n_clip += ncl;
    return ORT_OK;
}

/* ------------------------------------------------------------------------------------------ */
/* step 10: time step (L120; DESIGN R-G15)                                                     */
/* dt = C_a / max_cells sum_{d active} chat max(|lam1|,|lam3|)(U_i; d) / dl_d(i)               */
/* ------------------------------------------------------------------------------------------ */
int32_t ort_cfl_dt(ort_grid* g, const double* const U[4], double cfl, double* dt) {
    if (!g || !U || !dt || !(cfl > 0.0)) return ORT_ERR_INVALID_ARG;
    if (!g->have_par) return ORT_ERR_BAD_STATE;
    double rate = 0.0;
#pragma omp parallel for collapse(2) reduction(max : rate)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i) {
                long id = IDX(g, i, j, k);
                double F[3] = {U[1][id], U[2][id], U[3][id]};
                double sum = 0.0;
                for (int d = 0; d < 3; ++d) {
                    if (g->gh[d] == 0) continue;
                    double lam[3];
                    ort_wave_speeds(U[0][id], F, d, lam);
                    sum += g->par.chat * fmax(fabs(lam[0]), fabs(lam[2])) / cell_length(g, d, i, j, k);
                }
                if (sum > rate) rate = sum;
            }
    *dt = cfl / rate;
    return ORT_OK;
}

int32_t ort_get_floor_counts(ort_grid* g, int64_t* n_floor, int64_t* n_clip) {
    if (!g) return ORT_ERR_INVALID_ARG;
    if (n_floor) *n_floor = g->n_floor;
    if (n_clip) *n_clip = g->n_clip;
    g->n_floor = 0;
    g->n_clip = 0;
    return ORT_OK;
}

void ort_set_num_threads(int32_t n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int32_t ort_get_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
