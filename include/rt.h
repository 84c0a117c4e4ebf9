/* include/rt.h — C ABI of the B200-native gray-M1 radiation sub-step library (librt_m1.so).
 *
 * What the library computes: one radiation sub-step of the split explicit-implicit scheme of
 * PAPER.md (arxiv 2606.26268, Scepi & Lesur) Sect. 2.4-2.8, steps 1, 3-8, 10 of L109-120:
 *   ghost fill -> PLM reconstruction (Eq. 17-18) -> f-preserving fix (Eq. 19-21) -> M1 closure
 *   (Eq. 11-14) -> wave speeds (Eq. 22-26) -> HLL / GLF flux (L150) -> geometry-weighted flux
 *   divergence (L117) -> floor/clip -> opacities (L299, L375) -> implicit coupling (Eq. 29-33, 30, 28)
 *   -> time step (L120).
 * "R-Gn" = reading Gn of DESIGN.md (points where the paper is silent / ambiguous / garbled).
 *
 * Conventions
 *  - Every call returns an int32 status (RT_OK = 0 ...).  Nothing throws or aborts across the ABI.
 *    rt_last_error(grid) returns a handle-owned, NUL-terminated description of the last failure.
 *  - FIELD ARRAYS ARE DEVICE MEMORY OWNED BY THE CALLER: fp64, one contiguous array per field (SoA),
 *    ghosted, index ((k+g3)*nt2 + (j+g2))*nt1 + (i+g1), x1 fastest, g_d = nghost (= 2) ghosts per
 *    side on every ACTIVE dimension (n_d > 1) and 0 on inactive ones (n_d == 1); nt_d = n_d + 2 g_d.
 *    Pointers must be 8-byte aligned (16-byte alignment enables the vectorised / bulk-copy paths).
 *  - Arguments documented "host" are host pointers; they are copied during the call and may be
 *    freed on return.  Arrays OF pointers (U_in[4], mom[3] ...) are host arrays of device pointers.
 *  - The library owns only the handle: metric arrays, opacity tables, the per-cell thick-limit
 *    scratch array and reduction scratch.  All work is enqueued on the cudaStream_t given at
 *    rt_grid_create; only the calls documented "synchronises" wait for it.
 *  - Stored flux variable F is the paper's F_r (it carries the 1/c of Eq. 9: f = |F|/E <= 1;
 *    free streaming is |F| = E).  All constants are in code units (L95-97).
 *  - There is no CPU fallback: without a CUDA device rt_grid_create returns RT_ERR_CUDA.
 */
#ifndef RT_M1_H
#define RT_M1_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { RT_OK = 0, RT_ERR_INVALID_ARG = 1, RT_ERR_BAD_STATE = 2, RT_ERR_CUDA = 3, RT_ERR_NOT_FINITE = 4 };
enum { RT_CARTESIAN = 0, RT_CYLINDRICAL = 1 /* (R,phi,z) */, RT_SPHERICAL = 2 /* (r,theta,phi) */ };
enum { RT_BC_PERIODIC = 0, RT_BC_OUTFLOW = 1, RT_BC_REFLECT = 2, RT_BC_FIXED = 3 /* ghosts left as the caller wrote them */ };
enum { RT_SOLVER_HLL = 0, RT_SOLVER_GLF = 1 /* global bound alpha = chat */,
       RT_SOLVER_RUSANOV = 2 /* local bound alpha = chat max |lambda_1,3| of the two face states (L150; R-G5) */ };
enum { RT_OPAC_PLANCK = 0, RT_OPAC_ROSSELAND = 1, RT_OPAC_SCATTER = 2 };
/* how f <= 1 is enforced on the reconstructed face states (rt_set_face_fix) */
enum { RT_FIX_FPRESERVING = 0 /* Eq. 19-21, the paper's scheme and the default */,
       RT_FIX_PLUTO = 1 /* flat fallback U_f = U_c whenever |R(F)| > R(E), L136 */,
       RT_FIX_CLIP = 2 /* Eq. 36-38: F_f = R(F) R(E)/|R(F)| whenever |R(F)| > R(E) */ };

/* the "standard reconstruction method" R() of Sect. 2.5 (L132) */
enum { RT_RECON_PLM = 0 /* piecewise linear, van Leer limiter (R-G3): the default */,
       RT_RECON_LIMO3 = 1 /* compact third-order, Cada & Torrilhon 2009 (the scheme of the paper's Fig. 1-5; R-G22) */ };

typedef struct rt_grid rt_grid; /* opaque */

typedef struct {
    double chat;    /* reduced speed of light c^ (Sect. 2.7) */
    double c;       /* speed of light, code units */
    double a_R;     /* radiation constant (Eq. 15) */
    double c_v;     /* specific heat: C_v = rho c_v (Eq. 31; R-G12) */
    double E_floor; /* positivity floor on E_r (L250; R-G11) */
    int32_t solver;            /* RT_SOLVER_* (L150; R-G5) */
    int32_t thick_limit;       /* 0/1: optically-thick wave-speed limit, Eq. 25-26 (L171-173; R-G7) */
    int32_t feedback_momentum; /* 0/1: Eq. 28 (L183) applied to mom[] in rt_implicit_step */
} rt_params;

typedef struct {
    int32_t kind; /* 0: kappa = clip(kappa0 (rho/rho0)^a (T/T0)^b, kmin, kmax)               (L299)
                     1: bilinear table of log10 kappa on a uniform (log10 rho, log10 T) grid (L375; R-G14) */
    double kappa0, rho0, T0, a, b, kmin, kmax;
    int32_t n_lrho, n_lT;          /* n_lrho == 1: table in T only (the paper's form, L375) */
    double lrho_min, lrho_max, lT_min, lT_max;
    double rho_unit, T_unit;       /* table inputs are rho*rho_unit, T*T_unit (L97) */
    const double* log10_kappa;     /* HOST, n_lT x n_lrho, lrho fastest; copied to the device */
} rt_opacity;

/* Grid + metric precompute (a0).  geometry: RT_*; n[3] interior cells; nghost must be 2;
 * x1f/x2f/x3f: HOST edge coordinates, n[d]+1 strictly increasing values each (n[d] == 1 marks an
 * inactive dimension; its two edges still give the cell extent); bc[6] = x1lo,x1hi,x2lo,x2hi,x3lo,x3hi.
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).  Volumes and face areas are the exact
 * finite-volume integrals of R-G9; they are evaluated by a device kernel into separable 1-D factor
 * arrays.  Errors: NULL pointer, n < 1, nghost != 2, non-monotone / non-finite edges, r < 0 or theta
 * outside [0, pi], periodic paired with non-periodic on one axis, n[1] or n[2] > 65535 (they ride in gridDim.y / .z of
 * the launches) -> RT_ERR_INVALID_ARG.  The handle belongs to the device that is current at creation: every later call
 * switches to it for its duration, so a process may hold grids on several GPUs. */
int32_t rt_grid_create(int32_t geometry, const int32_t n[3], int32_t nghost,
                       const double* x1f, const double* x2f, const double* x3f,
                       const int32_t bc[6], void* cuda_stream, rt_grid** out);
int32_t rt_grid_destroy(rt_grid* g);

/* Test hook: full 3-D metrics to HOST arrays (NULLs allowed): vol[n3][n2][n1]; area_d has n_d + 1
 * entries along d (lower faces + the last upper face).  Synchronises. */
int32_t rt_grid_get_metrics(rt_grid* g, double* vol, double* area1, double* area2, double* area3);

int32_t rt_set_params(rt_grid* g, const rt_params* p);
/* which = RT_OPAC_*; an opacity never set is zero.  chi = kappa_R + sigma (L89). */
int32_t rt_set_opacity(rt_grid* g, int32_t which, const rt_opacity* o);

/* Step 1 (L111) alone: periodic / outflow / reflect (normal flux negated, L291) / fixed, axis by
 * axis (x1, then x2 over the x1-extended range, then x3).  U[4] = device pointers E, F1, F2, F3. */
int32_t rt_fill_ghosts(rt_grid* g, double* const U[4]);

/* Steps 1, 3-7 (L111-117): ghosts of U_in are filled IN PLACE, then
 *   U_out(interior) = U_in - dt sum_d [A+ F*+ - A- F*-]/V + dt S_geo(U_in)      (unsplit, R-G9, R-G10).
 * rho, T (device, ghosted layout; ghost values never read) are needed only when thick_limit = 1.
 * U_out[q] must not alias U_in[q]; ghosts of U_out are not written.  dt <= 0 or non-finite ->
 * RT_ERR_INVALID_ARG; rt_set_params not called -> RT_ERR_BAD_STATE.  Asynchronous. */
int32_t rt_explicit_step(rt_grid* g, double dt, const double* rho, const double* T,
                         double* const U_in[4], double* const U_out[4]);

/* Step 8 (L118) + floor/clip (R-G11), in place on the interior of U, T and (if feedback_momentum
 * and mom != NULL) mom: E <- max(E, E_floor); |F| <= E; opacities at (rho, T); closed-form solution
 * of the 2x2 system Eq. 33 (R-G12); F' = F/(1 + dt chat chi rho) (Eq. 30); m' = m - (F' - F)/chat
 * (Eq. 28).  Asynchronous. */
int32_t rt_implicit_step(rt_grid* g, double dt, const double* rho, double* T,
                         double* const mom[3], double* const U[4]);

/* Face fix of the explicit half (step a3).  The paper's f-preserving scheme (Eq. 19-21) is the default; the two
 * schemes it is compared with (Sect. 2.5, Sect. 3.2 Eq. 36-38 and Fig. 5) can be selected for the same
 * comparisons.  Every path honours the mode (per-direction kernels, the fused 2-D / 3-D kernel, the 1-D kernel); only the
 * combination with RT_SOLVER_RUSANOV makes rt_substep / rt_rk2_step take the per-direction kernels.  Unknown mode ->
 * RT_ERR_INVALID_ARG, state unchanged.  Host call, nothing enqueued. */
int32_t rt_set_face_fix(rt_grid* g, int32_t mode);

/* Reconstruction of the explicit half (step a2; L132).  RT_RECON_LIMO3 (DESIGN R-G22): with d- = u_i - u_{i-1},
 * d+ = u_{i+1} - u_i, theta = d-/d+: u(upper face) = u_i + phi(theta) d+/2, u(lower face) = u_i - phi(1/theta) d-/2,
 * phi_3 = (2 + theta)/3, phi_L = max(0, min(phi_3, max(-theta/2, min(2 theta, phi_3, 1.6)))); r > 0 switches the limiter
 * off (phi = phi_3) where eta = (d-^2 + d+^2)/(r dl)^2 <= 1 (dl = the cell's length along the direction: smooth extrema keep
 * third order), r <= 0 applies phi_L everywhere.  eta compares field differences with lengths, as in the original: choose r
 * for the units of the fields.  LimO3 runs in the per-direction kernels and the 1-D kernel (rt_substep on 2-D / 3-D
 * grids then takes the per-direction path).  Unknown kind / non-finite r -> RT_ERR_INVALID_ARG.  Host call. */
int32_t rt_set_reconstruction(rt_grid* g, int32_t kind, double r);

/* Irradiation (Sect. 2.9, Eq. 34-35): div_firr = DEVICE array (field layout, caller-owned, must stay valid)
 * of the divergence of a user-defined irradiation flux; every later implicit half adds Q = -div_firr dt to S_1 of
 * Eq. 33, i.e. to the coupled energy C_v T + (c/chat) E_r (Eq. 34).  NULL switches it off (the default). */
int32_t rt_set_irradiation(rt_grid* g, const double* div_firr);

/* The stellar irradiation flux of Sect. 3.7 in gray form (Eq. 47-48; DESIGN R-G21), the "user function" of
 * Sect. 2.9 for a central source: along every x1 ray tau_irr at the radial faces is tau_in at the inner edge plus
 * kappa_irr rho_i (r_{i+1/2} - r_{i-1/2}) per cell (Eq. 48, a prefix sum); F_irr = L0 e^{-tau}/r^2 r_hat on a spherical
 * grid (L0 = F_s R_s^2), L0 e^{-tau} x_hat on a Cartesian one (plane-parallel rays); div_firr = its finite-volume
 * divergence [A_+ F_+ - A_- F_-]/V per interior cell, ready for rt_set_irradiation.  rho, div_firr and the optional
 * tau_hi (tau at each cell's UPPER x1 face; NULL allowed): DEVICE, fp64, field layout, caller-owned; only interior
 * cells are written.  Cylindrical grid, kappa_irr < 0, tau_in < 0 or a non-finite scalar -> RT_ERR_INVALID_ARG.
 * Asynchronous on the grid's stream. */
int32_t rt_irradiation_radial(rt_grid* g, double L0, double kappa_irr, double tau_in, const double* rho,
                              double* tau_hi, double* div_firr);

/* rt_implicit_step with step 10 (L120; R-G15) fused behind it: the kernel that writes the updated state also
 * reduces the CFL rate of that state (warp shuffles + filtered atomicMax), and a one-thread kernel writes
 * *dt_next_device = cfl / max rate (DEVICE double): bit-identical to rt_cfl_dt_async on the updated U, without
 * reading the four fields again.  Asynchronous, graph-capturable. */
int32_t rt_implicit_step_cfl(rt_grid* g, double dt, const double* rho, double* T,
                             double* const mom[3], double* const U[4], double cfl, double* dt_next_device);

/* One WHOLE sub-step (steps 1, 3-8, 10; L111-120) with the time step resident on the device:
 *   dt = *dt_device  ->  rt_explicit_step(dt, U_in -> U_out)  ->  rt_implicit_step_cfl(dt, U_out)  ->  *dt_device = next dt.
 * dt_device: DEVICE double, read by the kernels of this sub-step and overwritten at its end (seed it with
 * rt_cfl_dt_async).  No host synchronisation anywhere: a sequence of sub-steps can be enqueued back to back or
 * captured in a CUDA graph.  rho and T are required.  Same argument errors as the two halves.  On 2-D and 3-D grids the
 * whole sub-step is one fused kernel (rt_set_tuning) and step 1 fills the face-normal ghosts of U_in only: edge and
 * corner ghosts, which no stencil of the scheme reads, are left as they were.  Handle-owned scratch (thick-limit and
 * rho kappa_P arrays) is allocated on the first call: capture a graph after one eager call. */
int32_t rt_substep(rt_grid* g, double* dt_device, double cfl, const double* rho, double* T,
                   double* const mom[3], double* const U_in[4], double* const U_out[4]);

/* One RK2 step (L107, L256, L399: "two Euler sub-steps and the average", the integrator of the paper's tests; R-G10):
 *   dt = *dt_device;  (U1,T1,m1) = substep(U,T,m; dt);  (U2,T2,m2) = substep(U1,T1,m1; dt);
 *   U <- (U + U2)/2,  T <- (T^n + T2)/2,  m <- (m^n + m2)/2 on interior cells;  *dt_device = CFL time step of the new U.
 * W1, W2: caller-owned work states (4 device arrays each, same layout as U; FIXED-boundary ghosts must be set in W1 as
 * in U).  The library keeps T^n, m^n in handle-owned scratch.  No host synchronisation.  Errors as rt_substep. */
int32_t rt_rk2_step(rt_grid* g, double* dt_device, double cfl, const double* rho, double* T,
                    double* const mom[3], double* const U[4], double* const W1[4], double* const W2[4]);

/* Step 10 (L120; R-G15): dt = cfl / max_cells sum_{d active} chat max(|lam1|,|lam3|)(U; d) / dl_d.
 * rt_cfl_dt writes a HOST double and synchronises the stream; rt_cfl_dt_async writes a DEVICE
 * double and does not synchronise (graph-capturable). */
int32_t rt_cfl_dt(rt_grid* g, const double* const U[4], double cfl, double* dt_host);
int32_t rt_cfl_dt_async(rt_grid* g, const double* const U[4], double cfl, double* dt_device);

/* Activations of the E floor and of the cell-centre f <= 1 clip in rt_implicit_step since the
 * last call (then reset).  Synchronises. */
int32_t rt_get_floor_counts(rt_grid* g, int64_t* n_floor, int64_t* n_clip);

/* Debug aid (failure detection): counts the interior cells in which E, F1, F2, F3 or (if T != NULL) T is NaN or infinite.
 * U[4], T: DEVICE, field layout.  *n_bad (HOST, NULL allowed) receives the count; returns RT_ERR_NOT_FINITE when it is not
 * zero (rt_last_error says how many), RT_OK otherwise.  Synchronises.  The sub-step calls themselves never check: a caller
 * that wants the check pays for this pass (40 B per cell). */
int32_t rt_check_finite(rt_grid* g, const double* const U[4], const double* T, int64_t* n_bad);

/* Number of kernel launches the library has enqueued on this grid since creation (bench bookkeeping). */
int64_t rt_get_launch_count(const rt_grid* g);

/* Optional per-kernel device timing (measurement support, not part of the method).  While profiling is
 * on, every kernel launch is bracketed by a cudaEvent pair on the grid's stream.  rt_get_kernel_times
 * synchronises, returns the summed milliseconds and launch counts per kernel kind since the last call,
 * and releases the events.  Kinds: */
enum { RT_K_GHOST = 0, RT_K_THICK = 1, RT_K_SWEEP1 = 2, RT_K_SWEEP2 = 3, RT_K_SWEEP3 = 4, RT_K_IMPLICIT = 5,
       RT_K_CFL = 6, RT_K_FUSED = 7 /* k_substep_fused: a2-a11 in one pass (3-D grids) */, RT_NKERNEL_KINDS = 8 };
int32_t rt_set_profiling(rt_grid* g, int32_t on);
int32_t rt_get_kernel_times(rt_grid* g, double ms[RT_NKERNEL_KINDS], int64_t launches[RT_NKERNEL_KINDS]);

/* Launch-shape tuning knobs, not part of the method.  march_len: cells marched per thread along the sweep
 * direction in the x2/x3 sweeps (0 = library default).  fused_seg: rt_substep on 2-D / 3-D grids runs ONE fused kernel
 * (reconstruction ... implicit coupling + CFL rate in a single pass over U^n, x1-x2 tiles marching along x3);
 * 0 = on with an automatic x3 segment length, > 0 = that segment length, -1 = off (per-direction kernels). */
int32_t rt_set_tuning(rt_grid* g, int32_t march_len, int32_t fused_seg);
/* Measurement aid: with RT_M1_NO_TMA=1 in the environment at rt_grid_create the fused kernel stages its planes by
 * cp.async even where TMA could address them (the path arrays with an odd x1 pitch always take). */

/* Measurement aid (SURVEY.md Sect. 8(d): "measure its own fp64 peak with a DFMA microbenchmark in the same run"); no grid
 * handle.  Launches `blocks` x `threads` threads, each running `chains` (1, 2, 4 or 8) independent chains of
 * 8 * iters dependent DFMAs, twice (the first launch warms up), and writes the CUDA-event duration of the second launch
 * in milliseconds to *ms_host (HOST).  Thread instructions of that launch = blocks * threads * chains * 8 * iters.
 * chains = 101, 102, 104: 1, 2, 4 chains with 64 instead of 8 DFMAs per chain between loop branches (x 64 * iters).
 * chains = 204 / 304: four chains whose DFMA reads two / three DIFFERENT register pairs (x = fma(x, y_c, const) /
 * fma(x, y_c, z_c)); 214 / 314: the same plus four independent fp32 multiplies per four DFMAs.  DFMA count of these
 * four = blocks * threads * 4 * 8 * iters.  They measure what the issue slot charges per instruction (DESIGN.md
 * Sect. 5: 2 cycles per fp64 warp instruction, 3 with three register operands, 1 per other instruction, not overlapped).
 * Synchronises the stream.  Bad argument -> RT_ERR_INVALID_ARG; no device / launch failure -> RT_ERR_CUDA. */
int32_t rt_measure_fp64(void* cuda_stream, int32_t blocks, int32_t threads, int32_t chains, int32_t iters, double* ms_host);

/* The CFL time step (step 10, L120; R-G15: dt = cfl / max_cells sum_{d active} chat max(|lambda_1|, |lambda_3|)_d / dx_d)
 * of a UNIFORM CARTESIAN grid through an entry point that ALLOCATES NOTHING: no grid handle, no cudaMalloc / cudaFree, no
 * allocating library routine -- for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it).  Same per-cell arithmetic as rt_cfl_dt_async, which it matches to rounding (<= 1e-14).
 *   cuda_stream  the stream the work is enqueued on (no synchronisation)
 *   n[3]         HOST; interior cells per axis; n[d] == 1: inactive (no ghosts, adds no rate)
 *   dx[3]        HOST; cell length per axis (> 0 on every active axis)
 *   U[4]         HOST array of four DEVICE pointers: E, F1, F2, F3 in the layout above (ghosted, nghost = 2); caller-owned
 *   dt_device    DEVICE; receives dt; caller-owned
 *   err, err_len HOST; optional buffer that receives a NUL-terminated description when the status is not RT_OK
 * The device the fields live on must be the CURRENT device.  The reduction's scratch is a static device array inside the
 * library (512 KB, held by every GPU that loads the library until exit) with one slot per x2-x3 row: grids with
 * n[1] * n[2] > RT_NOALLOC_MAX_ROWS are refused with RT_ERR_INVALID_ARG (256^3 still fits).  All calls share that
 * array: calls that overlap on one GPU (different streams or threads) race; calls on one stream are ordered and safe.
 * The first call on a device looks the array's address up (cudaGetSymbolAddress); make that call outside stream capture. */
#define RT_NOALLOC_MAX_ROWS 65536
int32_t rt_cfl_dt_uniform_noalloc(void* cuda_stream, const int32_t n[3], const double dx[3], double chat, double cfl,
                                  const double* const U[4], double* dt_device, char* err, int32_t err_len);

const char* rt_last_error(const rt_grid* g);

#ifdef __cplusplus
}
#endif
#endif
