/* oracle/ort.h — C interface of the CPU ORACLE for the gray-M1 radiation sub-step.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this library.  It shares
 * no code, header, table or constant with the CUDA path (paper_2606_26268_b200/).
 *
 * Everything is host memory, double precision, SoA, one contiguous array per field,
 * index ((k+g3)*nt2 + (j+g2))*nt1 + (i+g1), x1 fastest, g_d = 2 ghosts per side on
 * every ACTIVE dimension (n_d > 1) and 0 on inactive ones (n_d == 1).
 *
 * Citations are PAPER.md:L<line> (section / equation); "R-Gn" = reading Gn listed in
 * DESIGN.md (points where the paper is silent, ambiguous or garbled).
 */
#ifndef ORT_H
#define ORT_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORT_OK = 0, ORT_ERR_INVALID_ARG = 1, ORT_ERR_BAD_STATE = 2 };
enum { ORT_CARTESIAN = 0, ORT_CYLINDRICAL = 1 /* (R,phi,z) */, ORT_SPHERICAL = 2 /* (r,theta,phi) */ };
enum { ORT_BC_PERIODIC = 0, ORT_BC_OUTFLOW = 1, ORT_BC_REFLECT = 2, ORT_BC_FIXED = 3 };
enum { ORT_SOLVER_HLL = 0, ORT_SOLVER_GLF = 1, ORT_SOLVER_RUSANOV = 2 };
enum { ORT_OPAC_PLANCK = 0, ORT_OPAC_ROSSELAND = 1, ORT_OPAC_SCATTER = 2 };
/* how f <= 1 is enforced on the reconstructed face states (Sect. 2.5, Sect. 3.2 Eq. 36-38) */
enum { ORT_FIX_FPRESERVING = 0 /* Eq. 19-21 */, ORT_FIX_PLUTO = 1 /* flat fallback, L136 */, ORT_FIX_CLIP = 2 /* Eq. 36-38 */ };

/* the "standard reconstruction method" R() of Sect. 2.5 (L132): PLM with the van Leer limiter, or the compact third-order
 * LimO3 of Cada & Torrilhon 2009 (the scheme of the paper's Fig. 1-5); DESIGN.md R-G22 */
enum { ORT_RECON_PLM = 0, ORT_RECON_LIMO3 = 1 };

typedef struct {
    double chat;    /* reduced speed of light, PAPER.md:L179 (Sect. 2.7) */
    double c;       /* speed of light in code units */
    double a_R;     /* radiation constant, Eq. 15 */
    double c_v;     /* specific heat: C_v = rho*c_v, Eq. 31 L204 (R-G12) */
    double E_floor; /* positivity floor on E_r, L250 (R-G11) */
    int32_t solver;            /* ORT_SOLVER_* (L150) */
    int32_t thick_limit;       /* 0/1: Eq. 25-26 */
    int32_t feedback_momentum; /* 0/1: Eq. 28 */
} ort_params;

typedef struct {
    int32_t kind;   /* 0: power law kappa = clip(kappa0 (rho/rho0)^a (T/T0)^b, kmin, kmax)  (L299)
                       1: table of log10(kappa) on a uniform (log10 rho, log10 T) grid, bilinear (L375, R-G14) */
    double kappa0, rho0, T0, a, b, kmin, kmax;
    int32_t n_lrho, n_lT;
    double lrho_min, lrho_max, lT_min, lT_max;
    double rho_unit, T_unit;       /* table inputs are rho*rho_unit, T*T_unit (L97) */
    const double* log10_kappa;     /* n_lT x n_lrho, lrho fastest; copied */
} ort_opacity;

typedef struct ort_grid ort_grid;

int32_t ort_grid_create(int32_t geometry, const int32_t n[3], int32_t nghost,
                        const double* x1f, const double* x2f, const double* x3f,
                        const int32_t bc[6], ort_grid** out);
int32_t ort_grid_destroy(ort_grid* g);
/* full 3-D arrays: vol[n3][n2][n1]; area_d has n_d+1 entries along d (lower faces + last upper face) */
int32_t ort_grid_get_metrics(const ort_grid* g, double* vol, double* area1, double* area2, double* area3);
int32_t ort_set_params(ort_grid* g, const ort_params* p);
int32_t ort_set_opacity(ort_grid* g, int32_t which, const ort_opacity* o);

/* steps 1,3-7 of L111-117: ghost fill of U_in (in place), then U_out(interior) = transported U_in */
int32_t ort_explicit_step(ort_grid* g, double dt, const double* rho, const double* T,
                          double* const U_in[4], double* const U_out[4]);
/* step 8 of L118 (+ floor/clip R-G11): in place on U, T and (optionally) mom */
int32_t ort_implicit_step(ort_grid* g, double dt, const double* rho, double* T,
                          double* const mom[3], double* const U[4]);
/* step 10 of L120 (R-G15) */
int32_t ort_cfl_dt(ort_grid* g, const double* const U[4], double cfl, double* dt);
/* ghost fill alone (step 1 L111), exposed for tests */
int32_t ort_fill_ghosts(ort_grid* g, double* const U[4]);
/* activations of the E floor and of the cell f<=1 clip since the last call (then reset) */
int32_t ort_get_floor_counts(ort_grid* g, int64_t* n_floor, int64_t* n_clip);
void ort_set_num_threads(int32_t n);
int32_t ort_get_max_threads(void);

/* ---- point-wise pieces, exposed so the tests can pin each formula on its own ---- */
double ort_eddington_factor(double f);                                     /* Eq. 13 */
void ort_pressure_tensor(double E, const double F[3], double P[9]);        /* Eq. 11-14 */
void ort_wave_speeds(double E, const double F[3], int32_t d, double lam[3]); /* Eq. 22-24: lam1<=lam2<=lam3 */
double ort_vanleer_slope(double qm, double q0, double qp);                 /* L132 (R-G3) */
/* Eq. 19-21: cell value Uc[4], reconstructed RU[4] -> face state Uf[4] */
void ort_fpreserving_face(const double Uc[4], const double RU[4], double Uf[4]);
/* "PLUTO reconstruction" L136: U_f = U_c (E and F) whenever ||R(F)|| > R(E), else U_f = R(U) */
void ort_pluto_face(const double Uc[4], const double RU[4], double Uf[4]);
/* Eq. 36-38: E_f = R(E); F_f = R(F) if ||R(F)|| <= R(E), else R(F) R(E)/||R(F)|| */
void ort_clip_face(const double RU[4], double Uf[4]);
/* LimO3 (L132; Cada & Torrilhon 2009; DESIGN R-G22) for one field of one cell: values um, u0, up of the cells i-1, i, i+1,
 * the cell's length dx along the direction and the radius r of the asymptotic region (r <= 0: the limiter alone, no
 * smoothness switch) -> the values at the cell's lower and upper face */
void ort_limo3_faces(double um, double u0, double up, double dx, double r, double* lo, double* hi);
/* which reconstruction the explicit step applies (default ORT_RECON_PLM) and LimO3's r */
int32_t ort_set_reconstruction(ort_grid* g, int32_t kind, double r);
/* which of the three the explicit step applies (default ORT_FIX_FPRESERVING) */
int32_t ort_set_face_fix(ort_grid* g, int32_t mode);
/* L150 (R-G5,G6,G8): face flux from the two face states; lim = 4 chat/(3 tau_face) or +inf */
void ort_riemann_flux(const double UL[4], const double UR[4], int32_t d, double chat, int32_t solver,
                      double lim, double flux[4]);
double ort_opacity_eval(const ort_opacity* o, double rho, double T);       /* L299, L375 */
/* Eq. 29-33 L195-216 + Eq. 30: in/out E, F[3], T; optional mom[3] (may be NULL) */
int32_t ort_set_irradiation(ort_grid* g, const double* div_firr);
/* Sect. 3.7, Eq. 47-48 L379-383 in gray form (DESIGN R-G21): along every x1 ray tau_irr at the radial faces
 * (tau_in at the inner edge, + kappa_irr rho_i dr_i per cell), F_irr = L0 e^{-tau}/r^2 (spherical; L0 e^{-tau}
 * along x1 on a Cartesian grid) and its finite-volume divergence.  rho, tau_hi (optional: tau at each cell's
 * UPPER face), div_firr: host, ghosted field layout; only interior cells are written. */
int32_t ort_irradiation_radial(ort_grid* g, double L0, double kappa_irr, double tau_in, const double* rho,
                               double* tau_hi, double* div_firr);
void ort_implicit_cell(const ort_params* p, double dt, double rho, double kappaP, double chi,
                       double* E, double F[3], double* T, double* mom, double Q);

#ifdef __cplusplus
}
#endif
#endif
