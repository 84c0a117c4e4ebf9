// rt_kernels_aux.cuh — metric precompute (a0), ghost fill (a1), opacity evaluation (a9),
// thick-limit pre-pass (part of a5) and the CFL reduction (a11).  SURVEY.md Sect. 8(a) row names.
#pragma once
#include <limits.h>

#include "rt_math.cuh"
#include "rt_types.cuh"

namespace rtm1 {

constexpr int RT_OPAC_SCATTER_IDX = 2;

// ------------------------------------------------------------------------------------------------
// a0: metric precompute.  The paper gives no metric formulas (L15, L409); DESIGN.md R-G9: exact
// finite-volume integrals, written as separable 1-D factors.
//   Cartesian   V = dx1 dx2 dx3;                     A_d = prod_{e != d} dx_e
//   Cylindrical V = 1/2 D(R^2) Dphi Dz;              A_R = R_f Dphi Dz, A_phi = DR Dz, A_z = 1/2 D(R^2) Dphi
//   Spherical   V = 1/3 D(r^3) D(-cos th) Dphi;      A_r = r_f^2 D(-cos th) Dphi,
//               A_th = 1/2 D(r^2) sin(th_f) Dphi,    A_phi = 1/2 D(r^2) Dth
// Lengths (CFL, tau_cell): Cartesian dx_d; cyl DR, R_c Dphi, Dz; sph Dr, r_c Dth, r_c sin(th_c) Dphi.
// Sources: <1/R> = DR / (1/2 D(R^2)); <1/r> = 1/2 D(r^2) / (1/3 D(r^3)); <cot th> = D(sin th)/D(-cos th).
// Output pointers are the (writable) aliases of the arrays in GridDev.
// ------------------------------------------------------------------------------------------------
struct MetricOut {
    double* wf[3];
    double* vf[3];
    double* af[3][3];
    double* cg[3][3];
    double* len[3][3];
    double* ilen[3][3];
    double* invr;
    double* cot;
};

static __global__ void k_metric_precompute(GridDev g, MetricOut m) {
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    const int nth = gridDim.x * blockDim.x;
    const int geo = g.geometry;
    for (int e = 0; e < 3; ++e) {
        const double* x = g.xf[e];
        // faces
        for (int f = tid; f <= g.n[e]; f += nth) {
            double w = 1.0;
            if (geo == 1 && e == 0) w = x[f];
            if (geo == 2 && e == 0) w = x[f] * x[f];
            if (geo == 2 && e == 1) w = sin(x[f]);
            m.wf[e][f] = w;
        }
        // cells
        for (int c = tid; c < g.n[e]; c += nth) {
            const double a0 = x[c], a1 = x[c + 1];
            const double dx = a1 - a0;
            double vf = dx;                 // volume factor along e
            double afe[3] = {dx, dx, dx};   // area factor along e of the face normal to d (d != e)
            double len_e[3] = {1.0, 1.0, 1.0};  // factor along e of the length along d
            len_e[e] = dx;
            if (geo == 1) {  // (R, phi, z)
                if (e == 0) {
                    const double hR2 = 0.5 * (a1 * a1 - a0 * a0);
                    vf = hR2;
                    afe[1] = dx;   // A_phi = DR Dz
                    afe[2] = hR2;  // A_z = 1/2 D(R^2) Dphi
                    len_e[1] = 0.5 * (a0 + a1);  // R_c Dphi
                    m.invr[c] = dx / hR2;
                }
            } else if (geo == 2) {  // (r, theta, phi)
                if (e == 0) {
                    const double tr3 = (a1 * a1 * a1 - a0 * a0 * a0) / 3.0;
                    const double hr2 = 0.5 * (a1 * a1 - a0 * a0);
                    vf = tr3;
                    afe[1] = hr2;
                    afe[2] = hr2;
                    const double rc = 0.5 * (a0 + a1);
                    len_e[1] = rc;
                    len_e[2] = rc;
                    m.invr[c] = hr2 / tr3;
                } else if (e == 1) {
                    const double dmc = cos(a0) - cos(a1);
                    vf = dmc;
                    afe[0] = dmc;  // A_r = r_f^2 D(-cos th) Dphi
                    afe[2] = dx;   // A_phi = 1/2 D(r^2) Dth
                    len_e[2] = sin(0.5 * (a0 + a1));
                    m.cot[c] = (sin(a1) - sin(a0)) / dmc;
                }
            }
            m.vf[e][c] = vf;
            for (int d = 0; d < 3; ++d) {
                const double a = (d == e) ? 1.0 : afe[d];
                m.af[d][e][c] = a;
                m.cg[d][e][c] = (d == e) ? 1.0 / vf : a / vf;
                m.len[d][e][c] = len_e[d];
                m.ilen[d][e][c] = 1.0 / len_e[d];
            }
        }
    }
}

// Test hook behind rt_grid_get_metrics: full 3-D volume and face areas from the separable factors.
static __global__ void k_metric_expand(GridDev g, double* vol, double* a1, double* a2, double* a3) {
    const int n1 = g.n[0], n2 = g.n[1], n3 = g.n[2];
    const long long tot = (long long)(n1 + 1) * (n2 + 1) * (n3 + 1);
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < tot; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % (n1 + 1));
        const int j = (int)((t / (n1 + 1)) % (n2 + 1));
        const int k = (int)(t / ((long long)(n1 + 1) * (n2 + 1)));
        if (vol && i < n1 && j < n2 && k < n3) vol[((long long)k * n2 + j) * n1 + i] = g.vf[0][i] * g.vf[1][j] * g.vf[2][k];
        if (a1 && j < n2 && k < n3) a1[((long long)k * n2 + j) * (n1 + 1) + i] = g.wf[0][i] * g.af[0][1][j] * g.af[0][2][k];
        if (a2 && i < n1 && k < n3) a2[((long long)k * (n2 + 1) + j) * n1 + i] = g.wf[1][j] * g.af[1][0][i] * g.af[1][2][k];
        if (a3 && i < n1 && j < n2) a3[((long long)k * n2 + j) * n1 + i] = g.wf[2][k] * g.af[2][0][i] * g.af[2][1][j];
    }
}

// ------------------------------------------------------------------------------------------------
// a1: ghost fill along one axis d (step 1, L111).  periodic: copy from the opposite interior;
// outflow: nearest interior cell into both ghosts (L260); reflect: mirror, normal flux negated
// (L291); fixed: untouched (L289).  Axes e < d run over their ghost-extended range.
// One thread per (ghost layer, side, other-axis position).
// ------------------------------------------------------------------------------------------------
static __global__ void k_fill_ghosts(GridDev g, Fields4 U, int d) {
    int lo[3], ext[3];
    for (int e = 0; e < 3; ++e) {
        lo[e] = (e < d) ? -g.gh[e] : 0;
        ext[e] = (e < d) ? g.nt[e] : g.n[e];
    }
    const int ea = (d == 0) ? 1 : 0, eb = (d == 2) ? 1 : 2;  // the two other axes, ea < eb
    const long long na = ext[ea], nb = ext[eb];
    const long long tot = 4 * na * nb;
    const int nd = g.n[d];
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < tot; t += (long long)gridDim.x * blockDim.x) {
        const int a = (int)(t % na);
        const int b = (int)((t / na) % nb);
        const int ls = (int)(t / (na * nb));  // 0..3
        const int gl = ls & 1, side = ls >> 1;
        const int kind = g.bc[2 * d + side];
        if (kind == 3) continue;
        const int dst = side == 0 ? -1 - gl : nd + gl;
        int src;
        if (kind == 0) src = side == 0 ? nd - 1 - gl : gl;
        else if (kind == 1) src = side == 0 ? 0 : nd - 1;
        else src = side == 0 ? gl : nd - 1 - gl;
        int c[3];
        c[ea] = lo[ea] + a;
        c[eb] = lo[eb] + b;
        c[d] = 0;
        const long long base = (c[0] + g.gh[0]) * g.stride[0] + (c[1] + g.gh[1]) * g.stride[1] + (c[2] + g.gh[2]) * g.stride[2];
        const long long id = base + dst * g.stride[d], is = base + src * g.stride[d];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            double v = U.q[q][is];
            if (kind == 2 && q == 1 + d) v = -v;
            U.q[q][id] = v;
        }
    }
}

// a1 for the sub-step kernels, ONE launch: the face-normal ghosts of every active axis (other axes over their
// interior range only).  The scheme never reads edge / corner ghosts — each direction's stencil leaves the
// interior along its own axis only — so rt_substep does not need the axis-by-axis ordering of k_fill_ghosts.
// block `block` of `nblocks` blocks of blockDim.x threads
__device__ __forceinline__ void fill_faces_body(const GridDev& g, const Fields4& U, int block, int nblocks) {
    // one work item = both ghost layers of one (transverse cell, side) of one axis; along x1 the two layers are one
    // 16-byte store (they share a 32-byte sector: item-per-layer traffic was twice the sectors)
    long long cnt[3], tot = 0;
    for (int d = 0; d < 3; ++d) {
        const int ea = (d == 0) ? 1 : 0, eb = (d == 2) ? 1 : 2;
        const bool skip = g.gh[d] == 0 || (g.bc[2 * d] == 3 && g.bc[2 * d + 1] == 3);
        cnt[d] = skip ? 0 : 2LL * g.n[ea] * g.n[eb];
        tot += cnt[d];
    }
    for (long long t = block * (long long)blockDim.x + threadIdx.x; t < tot; t += (long long)nblocks * blockDim.x) {
        long long r = t;
        int d = 0;
        while (r >= cnt[d]) {
            r -= cnt[d];
            ++d;
        }
        const int ea = (d == 0) ? 1 : 0, eb = (d == 2) ? 1 : 2;
        const long long na = g.n[ea], nb = g.n[eb];
        const int a = (int)(r % na);
        const int b = (int)((r / na) % nb);
        const int side = (int)(r / (na * nb));  // 0..1
        const int kind = g.bc[2 * d + side];
        if (kind == 3) continue;
        const int nd = g.n[d];
        // the two ghost cells in address order: index dlo and dlo + 1 along d, filled from slo and shi
        const int dlo = side == 0 ? -2 : nd;
        int slo, shi;
        if (kind == 0) {
            slo = side == 0 ? nd - 2 : 0;
            shi = slo + 1;
        } else if (kind == 1) {
            slo = shi = side == 0 ? 0 : nd - 1;
        } else {
            slo = side == 0 ? 1 : nd - 1;
            shi = side == 0 ? 0 : nd - 2;
        }
        int c[3];
        c[ea] = a;
        c[eb] = b;
        c[d] = 0;
        const long long base = (c[0] + g.gh[0]) * g.stride[0] + (c[1] + g.gh[1]) * g.stride[1] + (c[2] + g.gh[2]) * g.stride[2];
        const long long id = base + dlo * g.stride[d];
        const long long is0 = base + slo * g.stride[d], is1 = base + shi * g.stride[d];
        double v0[4], v1[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            v0[q] = U.q[q][is0];
            v1[q] = U.q[q][is1];
            if (kind == 2 && q == 1 + d) {
                v0[q] = -v0[q];
                v1[q] = -v1[q];
            }
        }
        const bool pair = d == 0 && (id & 1) == 0;  // the fields are 16-byte aligned (include/rt.h)
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (pair) {
                *reinterpret_cast<double2*>(U.q[q] + id) = make_double2(v0[q], v1[q]);
            } else {
                U.q[q][id] = v0[q];
                U.q[q][id + g.stride[d]] = v1[q];
            }
        }
    }
}

static __global__ void k_fill_faces(const __grid_constant__ GridDev g, const __grid_constant__ Fields4 U) {
    fill_faces_body(g, U, (int)blockIdx.x, (int)gridDim.x);
}

// Debug aid (SURVEY.md Sect. 5 "failure detection"): count the interior cells in which any of up to five fields is not finite.
struct FiniteArgs {
    const double* f[5];
    int n;
};
static __global__ void __launch_bounds__(128) k_check_finite(const __grid_constant__ GridDev g, const __grid_constant__ FiniteArgs v,
                                                      unsigned long long* __restrict__ bad) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool b = false;
    if (i < g.n[0]) {
        const long long id = (i + g.gh[0]) + (blockIdx.y + g.gh[1]) * g.stride[1] + (blockIdx.z + g.gh[2]) * g.stride[2];
        for (int q = 0; q < v.n; ++q) b = b || !isfinite(v.f[q][id]);
    }
    const unsigned m = __ballot_sync(0xffffffffu, b);
    if (m && (threadIdx.x & 31) == 0) atomicAdd(bad, (unsigned long long)__popc(m));
}

// RK2 (L107, L256: two Euler sub-steps and the average of every evolved variable): q <- (q0 + q2)/2 on interior cells.
// a[] = the fields holding q0 on entry and the average on exit; b[] = q2.  n = 4 (U), 1 (T) or 3 (m) pairs per launch.
struct AvgArgs {
    double* a[8];
    const double* b[8];
    int n;
};
static __global__ void __launch_bounds__(128) k_rk2_average(const __grid_constant__ GridDev g, const __grid_constant__ AvgArgs v) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n[0]) return;
    const long long id = (i + g.gh[0]) + (blockIdx.y + g.gh[1]) * g.stride[1] + (blockIdx.z + g.gh[2]) * g.stride[2];
    for (int q = 0; q < v.n; ++q) v.a[q][id] = 0.5 * (v.a[q][id] + v.b[q][id]);
}

// ------------------------------------------------------------------------------------------------
// Radial irradiation (Sect. 3.7, Eq. 47-48, gray: R-G21).  One warp per x1 ray, 32 consecutive cells per
// pass (coalesced 256-B rows): dtau = kappa rho dr per lane, inclusive scan over the warp by shuffles, the ray's
// running tau carried from pass to pass in a register.  div F_irr = L0 e^{-tau_-} expm1(-dtau) x 3/(r_+^3 - r_-^3)
// (spherical: [A_+ F_+ - A_- F_-]/V of F = L0 e^{-tau}/r^2) or x 1/dx (Cartesian, plane-parallel rays along x1).
// HBM: 8 B read + 8 B written per cell (+ 8 B with tau_hi).
// ------------------------------------------------------------------------------------------------
static __global__ void __launch_bounds__(128) k_irradiation_radial(const __grid_constant__ GridDev g, double L0, double kappa,
                                                            double tau_in, const double* __restrict__ rho,
                                                            double* __restrict__ tau_hi, double* __restrict__ div) {
    const int lane = threadIdx.x & 31;
    const long long ray = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (ray >= (long long)g.n[1] * g.n[2]) return;  // whole warps leave together
    const int j = (int)(ray % g.n[1]), k = (int)(ray / g.n[1]);
    const long long row = g.gh[0] + (j + g.gh[1]) * g.stride[1] + (k + g.gh[2]) * g.stride[2];
    const int n1 = g.n[0];
    const bool sph = g.geometry == 2;
    double carry = tau_in;
#pragma unroll 2
    for (int i0 = 0; i0 < n1; i0 += 32) {
        const int i = i0 + lane;
        const bool on = i < n1;
        double dtau = 0.0, geo = 0.0;
        if (on) {
            const double rm = g.xf[0][i], rp = g.xf[0][i + 1];
            dtau = kappa * rho[row + i] * (rp - rm);
            geo = sph ? 3.0 / (rp * rp * rp - rm * rm * rm) : 1.0 / (rp - rm);
        }
        double incl = dtau;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const double up = __shfl_up_sync(0xffffffffu, incl, s);
            if (lane >= s) incl += up;
        }
        double excl = __shfl_up_sync(0xffffffffu, incl, 1);
        if (lane == 0) excl = 0.0;
        const double tlo = carry + excl, thi = carry + incl;
        if (on) {
            div[row + i] = L0 * exp(-tlo) * expm1(-dtau) * geo;
            if (tau_hi) tau_hi[row + i] = thi;
        }
        carry = __shfl_sync(0xffffffffu, thi, 31);
    }
}

// ------------------------------------------------------------------------------------------------
// a9: opacities.  Power law kappa0 (rho/rho0)^a (T/T0)^b clipped (L299) or bilinear table of
// log10 kappa on a uniform (log10 rho, log10 T) grid (L375; R-G14).
// ------------------------------------------------------------------------------------------------
// x^(n2/2) for integer n2: sqrt for the odd part, binary powering for the rest (warp-uniform control
// flow); Newton sqrt / reciprocal of rt_math.cuh (x > 0 normal), so ~1-2 ulp against libm pow().
__device__ __forceinline__ double pow_half_int(double x, int n2) {
    int m = n2 < 0 ? -n2 : n2;
    double r = (m & 1) ? fsqrt(x) : 1.0;
    int k = m >> 1;
    double base = x;
    while (k) {
        if (k & 1) r *= base;
        base *= base;
        k >>= 1;
    }
    return n2 < 0 ? frcp(r) : r;
}

// log10 of the table inputs, shared by every table opacity of a cell when their units agree
struct LogRT {
    double lrho, lT;
};

// x^(m2/2) for 0 <= m2 <= 15, m2 uniform over the launch: binary powering with uniform predicates (no jump table,
// no loop), one optional square root
__device__ __forceinline__ double pow_half_small(double x, int m2) {
    // the empty asm statements keep these launch-uniform tests real (uniform) branches: if-converted, each costs a
    // multiplication plus two FSEL per cell whether taken or not
    double r = 1.0;
    if (m2 & 2) { r = x; asm volatile(""); }
    if (m2 & 12) {
        const double x2 = x * x;
        if (m2 & 4) { r *= x2; asm volatile(""); }
        if (m2 & 8) { r *= x2 * x2; asm volatile(""); }
    }
    if (m2 & 1) { r *= fsqrt(x); asm volatile(""); }
    return r;
}

// kappa0 (rho/rho0)^a (T/T0)^b with half-integer a, b (|2a|, |2b| <= 15): positive powers multiply, negative powers
// share ONE reciprocal.  ~1-2 ulp against libm pow().  The scalars are passed in so that a caller looping over
// cells keeps them in registers.
__device__ __forceinline__ double power_law_fast_v(double kappa0, double irho0, double iT0, int na, int nb, double kmin,
                                                   double kmax, double rho, double T) {
    const double pr = pow_half_small(rho * irho0, na < 0 ? -na : na);
    const double pt = pow_half_small(T * iT0, nb < 0 ? -nb : nb);
    double num = kappa0, den = 1.0;   // launch-uniform tests kept as uniform branches (see pow_half_small)
    if (na < 0) { den = pr; asm volatile(""); } else { num *= pr; asm volatile(""); }
    if (nb < 0) { den *= pt; asm volatile(""); } else { num *= pt; asm volatile(""); }
    if ((na | nb) < 0) { num *= frcp(den); asm volatile(""); }
    return dmin(dmax(num, kmin), kmax);
}
__device__ __forceinline__ double power_law_fast(const OpacDev& o, double rho, double T) {
    return power_law_fast_v(o.kappa0, o.irho0, o.iT0, o.n2a, o.n2b, o.kmin, o.kmax, rho, T);
}

__device__ __forceinline__ double power_law_eval(const OpacDev& o, double rho, double T) {
    if (o.fast) return power_law_fast(o, rho, T);
    const double xr = rho * o.irho0, xt = T * o.iT0;
    double pr, pt;
    if (o.n2a != INT_MIN) pr = pow_half_int(xr, o.n2a); else pr = pow(xr, o.a);
    if (o.n2b != INT_MIN) pt = pow_half_int(xt, o.n2b); else pt = pow(xt, o.b);
    double k = o.kappa0 * pr * pt;
    k = dmax(k, o.kmin);
    k = dmin(k, o.kmax);
    return k;
}

__device__ __forceinline__ double table_eval(const OpacDev& o, const LogRT& l) {
    const double y = dmin(dmax(l.lT, o.lT_min), o.lT_max);
    const double v = (y - o.lT_min) * o.sv;
    int j0 = (int)v;  // v >= 0: truncation = floor
    j0 = max(0, min(j0, o.n_lT - 2));
    const double tv = v - (double)j0;
    double val;
    if (o.n_lrho == 1) {
        val = (1.0 - tv) * __ldg(o.tab + j0) + tv * __ldg(o.tab + j0 + 1);
    } else {
        const double x = dmin(dmax(l.lrho, o.lrho_min), o.lrho_max);
        const double u = (x - o.lrho_min) * o.su;
        int i0 = (int)u;
        i0 = max(0, min(i0, o.n_lrho - 2));
        const double tu = u - (double)i0;
        const double* p = o.tab + (long long)j0 * o.n_lrho + i0;
        const double v00 = __ldg(p), v01 = __ldg(p + 1), v10 = __ldg(p + o.n_lrho), v11 = __ldg(p + o.n_lrho + 1);
        val = (1.0 - tv) * ((1.0 - tu) * v00 + tu * v01) + tv * ((1.0 - tu) * v10 + tu * v11);
    }
    return fexp10(val);
}

__device__ __forceinline__ LogRT log_inputs(const OpacDev& o, double rho, double T) {
    LogRT l;
    l.lT = flog10(T * o.T_unit);
    l.lrho = o.n_lrho > 1 ? flog10(rho * o.rho_unit) : 0.0;
    return l;
}

__device__ __forceinline__ double opacity_eval(const OpacDev& o, double rho, double T) {
    if (!o.set) return 0.0;
    if (o.kind == 0) return power_law_eval(o, rho, T);
    return table_eval(o, log_inputs(o, rho, T));
}

// Several opacities of one cell.  share = the host found that every TABLE among them has the same
// rho_unit, T_unit (and n_lrho > 1 or == 1 alike): log10 rho, log10 T are then evaluated once.
struct OpacSet {
    int share;  // 1: >= 2 tables in the set and all of them share their log inputs
    int src;    // RT_OPAC_* index of the table whose units define the shared inputs
};

__device__ __forceinline__ double opacity_eval_shared(const OpacDev& o, double rho, double T, bool share, const LogRT& l) {
    if (!o.set) return 0.0;
    if (o.kind == 0) return power_law_eval(o, rho, T);
    return share ? table_eval(o, l) : table_eval(o, log_inputs(o, rho, T));
}

// ------------------------------------------------------------------------------------------------
// Thick-limit pre-pass (Eq. 25-26; R-G7): per interior cell
//   limd = 4 / (3 tau_cell),  tau_cell = rho chi dx,  chi = kappa_R + sigma (L89),
//   dx = the cell's largest physical extent over the active dimensions.
// The sweeps use lim_face = max(limd_a, limd_b) = 4/(3 min(tau_a, tau_b)) of the two cells next to a face, so of the
// ghost layers only the first, face-normal one is ever used: the thread of a boundary cell also writes that ghost
// (the periodic image, or the copy of the nearest interior cell: rho and T ghosts are never read).  The remaining
// ghosts of the array keep the zeros of its allocation.
// ------------------------------------------------------------------------------------------------
constexpr int kThickRows = 4;  // x2 rows per block: one-row blocks cost more to schedule than to run

// x^(N/2) for a compile-time N: straight-line code, one reciprocal for N < 0, one square root for odd N
template <int N>
__device__ __forceinline__ double pow_half_ct(double x) {
    if (N == 0) return 1.0;
    constexpr int M = N < 0 ? -N : N;
    const double b = N < 0 ? frcp(x) : x;
    double r = 1.0;
    if (M >> 1) {
        r = b;                      // b^(M >> 1) by repeated squaring, unrolled at compile time
        constexpr int K = M >> 1;
        double acc = 1.0, base = b;
        bool first = true;
#pragma unroll
        for (int bit = 0; bit < 3; ++bit) {
            if (K & (1 << bit)) {
                acc = first ? base : acc * base;
                first = false;
            }
            if ((K >> (bit + 1)) != 0) base = base * base;
        }
        r = acc;
    }
    if (M & 1) {
        const double root = N < 0 ? fsqrt(x) * b : fsqrt(x);
        r = (M >> 1) ? r * root : root;
    }
    return r;
}

// x^(n/2) for a LAUNCH-UNIFORM -15 <= n <= 15: one uniform multi-way branch into the straight-line code of that
// exponent.  (Binary powering behind run-time tests of n cost the pre-pass ~280 instructions per cell, most of them
// selects and moves; this form costs the branch.)  ~1-2 ulp against libm pow().
__device__ __forceinline__ double pow_half_uniform(double x, int n) {
    switch (n) {
#define RT_PH(N) case N: return pow_half_ct<N>(x);
        RT_PH(-15) RT_PH(-14) RT_PH(-13) RT_PH(-12) RT_PH(-11) RT_PH(-10) RT_PH(-9) RT_PH(-8) RT_PH(-7) RT_PH(-6) RT_PH(-5)
        RT_PH(-4) RT_PH(-3) RT_PH(-2) RT_PH(-1) RT_PH(1) RT_PH(2) RT_PH(3) RT_PH(4) RT_PH(5) RT_PH(6) RT_PH(7) RT_PH(8)
        RT_PH(9) RT_PH(10) RT_PH(11) RT_PH(12) RT_PH(13) RT_PH(14) RT_PH(15)
#undef RT_PH
        default: return 1.0;
    }
}

// One or two half-integer power laws kappa0 (rho/rho0)^(na/2) (T/T0)^(nb/2) clipped to [kmin, kmax] (L299) that share
// rho0 and T0; exponents launch-uniform, prepared on the host.
struct LeanLaws {
    double irho0, iT0;
    double k0[2], kmin[2], kmax[2];
    int na[2], nb[2];  // 2a, 2b (|.| <= 15)
    int two;           // evaluate the second law (kappa_P) as well
    int same_ab;       // the second law has the exponents of the first (only kappa0 / the clip differ)
};
__device__ __forceinline__ void lean_eval(const LeanLaws& L, double rho, double T, double& k_first, double& k_second) {
    const double xr = rho * L.irho0, xt = T * L.iT0;
    const double m0 = pow_half_uniform(xr, L.na[0]) * pow_half_uniform(xt, L.nb[0]);
    k_first = dmin(dmax(L.k0[0] * m0, L.kmin[0]), L.kmax[0]);
    k_second = k_first;
    if (L.two) {
        const double m1 = L.same_ab ? m0 : pow_half_uniform(xr, L.na[1]) * pow_half_uniform(xt, L.nb[1]);
        k_second = dmin(dmax(L.k0[1] * m1, L.kmin[1]), L.kmax[1]);
    }
}

// The same for R cells of one thread at a time: the launch-uniform multi-way branches are taken once per batch instead
// of once per cell (per cell they were a quarter of the pre-pass's instructions).
template <int R>
__device__ __forceinline__ void pow_half_batch(const double (&x)[R], int n, double (&out)[R]) {
    switch (n) {
#define RT_PH(N)                                                                       \
    case N:                                                                            \
        _Pragma("unroll") for (int r = 0; r < R; ++r) out[r] = pow_half_ct<N>(x[r]);   \
        break;
        RT_PH(-15) RT_PH(-14) RT_PH(-13) RT_PH(-12) RT_PH(-11) RT_PH(-10) RT_PH(-9) RT_PH(-8) RT_PH(-7) RT_PH(-6) RT_PH(-5)
        RT_PH(-4) RT_PH(-3) RT_PH(-2) RT_PH(-1) RT_PH(1) RT_PH(2) RT_PH(3) RT_PH(4) RT_PH(5) RT_PH(6) RT_PH(7) RT_PH(8)
        RT_PH(9) RT_PH(10) RT_PH(11) RT_PH(12) RT_PH(13) RT_PH(14) RT_PH(15)
#undef RT_PH
        default:
#pragma unroll
            for (int r = 0; r < R; ++r) out[r] = 1.0;
    }
}
template <int R>
__device__ __forceinline__ void lean_eval_batch(const LeanLaws& L, const double (&rho)[R], const double (&T)[R],
                                                double (&k_first)[R], double (&k_second)[R]) {
    double xr[R], xt[R], pr[R], pt[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        xr[r] = rho[r] * L.irho0;
        xt[r] = T[r] * L.iT0;
    }
    pow_half_batch<R>(xr, L.na[0], pr);
    pow_half_batch<R>(xt, L.nb[0], pt);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        pr[r] *= pt[r];
        k_first[r] = dmin(dmax(L.k0[0] * pr[r], L.kmin[0]), L.kmax[0]);
        k_second[r] = k_first[r];
    }
    if (L.two) {
        if (!L.same_ab) {
            pow_half_batch<R>(xr, L.na[1], pr);
            pow_half_batch<R>(xt, L.nb[1], pt);
#pragma unroll
            for (int r = 0; r < R; ++r) pr[r] *= pt[r];
        }
#pragma unroll
        for (int r = 0; r < R; ++r) k_second[r] = dmin(dmax(L.k0[1] * pr[r], L.kmin[1]), L.kmax[1]);
    }
}
__device__ __forceinline__ void prefetch_global_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// LEAN: chi is ONE half-integer power law (kappa_R fast, no scattering) and kappa_P, when asked for (kpr != nullptr:
// the fused sub-step, whose implicit half then evaluates no opacity at all), is the same law or another fast law with
// the same rho0, T0.  Otherwise the general evaluation (tables share their log10 inputs: OpacSet).
// One thread per x1 column of a block of kThickRows x2 rows; the loads of the next row are issued before the
// arithmetic of the current one.
// MODE 2: kappa_R (and kappa_P, when asked for and not the same law) are 2-D tables on the SAME axes and units, no
// scattering: the two log10, the cell of the table and the interpolation weights are found once, then one 2 x 2 gather
// and one 10^x per table (C5).  Same arithmetic as table_eval, without the per-opacity tests of the general path.
struct TablePair {
    const double* tabR;
    const double* tabP;  // nullptr: kappa_P is not wanted or is the same table
    int n_lrho, n_lT;
    double lrho_min, lrho_max, lT_min, lT_max, su, sv, rho_unit, T_unit;
};
__device__ __forceinline__ void table_pair_eval(const TablePair& tp, double rho, double T, double& kR, double& kP) {
    const double x = dmin(dmax(flog10(rho * tp.rho_unit), tp.lrho_min), tp.lrho_max);
    const double y = dmin(dmax(flog10(T * tp.T_unit), tp.lT_min), tp.lT_max);
    const double u = (x - tp.lrho_min) * tp.su, v = (y - tp.lT_min) * tp.sv;
    const int i0 = max(0, min((int)u, tp.n_lrho - 2)), j0 = max(0, min((int)v, tp.n_lT - 2));
    const double tu = u - (double)i0, tv = v - (double)j0;
    const int off = j0 * tp.n_lrho + i0;
    {
        const double* p = tp.tabR + off;
        const double v00 = __ldg(p), v01 = __ldg(p + 1), v10 = __ldg(p + tp.n_lrho), v11 = __ldg(p + tp.n_lrho + 1);
        kR = fexp10((1.0 - tv) * ((1.0 - tu) * v00 + tu * v01) + tv * ((1.0 - tu) * v10 + tu * v11));
    }
    kP = kR;
    if (tp.tabP) {
        const double* p = tp.tabP + off;
        const double v00 = __ldg(p), v01 = __ldg(p + 1), v10 = __ldg(p + tp.n_lrho), v11 = __ldg(p + tp.n_lrho + 1);
        kP = fexp10((1.0 - tv) * ((1.0 - tu) * v00 + tu * v01) + tv * ((1.0 - tu) * v10 + tu * v11));
    }
}

// block (bxi, byi, bzi) of the pre-pass: x1 columns bxi * blockDim.x ..., x2 rows byi * rows_per_block ..., x3 plane bzi
template <int MODE>
__device__ __forceinline__ void thick_limit_body(const GridDev& g, const OpacDev& oR, const OpacDev& oS, const OpacSet& os,
                                                 const double* __restrict__ rho, const double* __restrict__ T,
                                                 double* __restrict__ lim, const OpacDev& oP, int same_PR,
                                                 double* __restrict__ kpr, const LeanLaws& laws, const TablePair& tp, int bxi,
                                                 int byi, int bzi, int rows_per_block) {
    constexpr bool LEAN = MODE == 1 || MODE == 3;  // 3: the register-batch form (large grids)
    const int i = bxi * blockDim.x + threadIdx.x;
    const int k = bzi;
    if (i >= g.n[0]) return;
    const bool share = MODE == 0 && os.share != 0;
    const int s1 = (int)g.stride[1], s2 = (int)g.stride[2];
    const int n0 = g.n[0], n1 = g.n[1], n2 = g.n[2];
    const bool act1 = g.gh[1] > 0, act2 = g.gh[2] > 0;
    // x1 and x3 factors of the three cell lengths (0 for an inactive direction)
    double l02[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) l02[d] = g.gh[d] > 0 ? __ldg(g.len[d][0] + i) * __ldg(g.len[d][2] + k) : 0.0;
    // face-normal ghost this cell also fills along x1 / x3 (offset 0: none): the periodic image or the clamped copy
    int goff0 = 0, goff2 = 0;
    if (g.gh[0] > 0) {
        const bool per = g.bc[0] == 0;
        if (i == 0) goff0 = per ? n0 : -1;
        if (i == n0 - 1) goff0 = per ? -n0 : 1;
    }
    if (act2) {
        const bool per = g.bc[4] == 0;
        if (k == 0) goff2 = (per ? n2 : -1) * s2;
        if (k == n2 - 1) goff2 = (per ? -n2 : 1) * s2;
    }
    const bool per1 = g.bc[2] == 0;
    const int j0 = byi * rows_per_block;  // rows_per_block: a multiple of kThickRows
    const int j1 = min(j0 + rows_per_block, n1);
    const double* __restrict__ len01 = g.len[0][1];
    const double* __restrict__ len11 = g.len[1][1];
    const double* __restrict__ len21 = g.len[2][1];
    int id = (i + g.gh[0]) + (j0 + g.gh[1]) * s1 + (k + g.gh[2]) * s2;
    // what follows the opacities of one cell: rho kappa_P, tau, lim and the ghost copies of lim
    auto finish = [&](int j, int idc, double rc, double chi, double kP) {
        if (kpr) kpr[idc] = kP * rc;
        double dx = l02[0] * __ldg(len01 + j);
        if (act1) dx = dmax(dx, l02[1] * __ldg(len11 + j));
        if (act2) dx = dmax(dx, l02[2] * __ldg(len21 + j));
        const double tau = rc * chi * dx;
        // any value >= 1 means "no limit" (|lambda| <= 1, L167): tau -> 0 maps to +inf without a division by zero
        const double v = tau > 1.0e-100 ? 4.0 * frcp(3.0 * tau) : __builtin_huge_val();
        lim[idc] = v;
        if (goff0 | goff2) {
            if (goff0) lim[idc + goff0] = v;
            if (goff2) lim[idc + goff2] = v;
        }
        if (act1 && (j == 0 || j == n1 - 1)) {
            if (j == 0) lim[idc + (per1 ? n1 : -1) * s1] = v;
            if (j == n1 - 1) lim[idc + (per1 ? -n1 : 1) * s1] = v;
        }
    };
    if (MODE == 3) {
        // kThickRows cells at a time as one register batch (the plan's launch-uniform branches once per batch); the next
        // batch's rho, T are on their way into L2 while this one is computed (a prefetch holds no registers)
        constexpr int R = kThickRows;
#pragma unroll 1
        for (int jb = j0; jb < j1; jb += R, id += R * s1) {
            double rb[R], tb[R], chi[R], kP[R];
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const int idq = id + min(q, j1 - 1 - jb) * s1;  // rows past the end repeat the last one (not stored)
                rb[q] = __ldg(rho + idq);
                tb[q] = __ldg(T + idq);
            }
            if (jb + R < j1) {
#pragma unroll
                for (int q = 0; q < R; ++q) {
                    const int idq = id + min(R + q, j1 - 1 - jb) * s1;
                    prefetch_global_l2(rho + idq);
                    prefetch_global_l2(T + idq);
                }
            }
            lean_eval_batch<R>(laws, rb, tb, chi, kP);
#pragma unroll
            for (int q = 0; q < R; ++q)
                if (jb + q < j1) finish(jb + q, id + q * s1, rb[q], chi[q], kP[q]);
        }
        return;
    }
    double r = __ldg(rho + id), t = __ldg(T + id);
#pragma unroll 1
    for (int j = j0; j < j1; ++j, id += s1) {
        const double rc = r, tc = t;
        if (j + 1 < j1) {
            r = __ldg(rho + id + s1);
            t = __ldg(T + id + s1);
        }
        double chi, kP;
        if (LEAN) {
            lean_eval(laws, rc, tc, chi, kP);
        } else if (MODE == 2) {
            table_pair_eval(tp, rc, tc, chi, kP);
        } else {
            LogRT l = {0.0, 0.0};
            if (share) l = log_inputs(os.src == RT_OPAC_SCATTER_IDX ? oS : (os.src == 1 ? oR : oP), rc, tc);
            const double kR = opacity_eval_shared(oR, rc, tc, share, l);
            chi = kR + opacity_eval_shared(oS, rc, tc, share, l);
            kP = !kpr ? 0.0 : (same_PR ? kR : opacity_eval_shared(oP, rc, tc, share, l));
        }
        finish(j, id, rc, chi, kP);
    }
}

template <int MODE>
__global__ void __launch_bounds__(256) k_thick_limit(const __grid_constant__ GridDev g, const __grid_constant__ OpacDev oR,
                                                     const __grid_constant__ OpacDev oS, const __grid_constant__ OpacSet os,
                                                     const double* __restrict__ rho, const double* __restrict__ T,
                                                     double* __restrict__ lim, const __grid_constant__ OpacDev oP,
                                                     int same_PR, double* __restrict__ kpr, const __grid_constant__ LeanLaws laws,
                                                     const __grid_constant__ TablePair tp, int rows_per_block) {
    thick_limit_body<MODE>(g, oR, oS, os, rho, T, lim, oP, same_PR, kpr, laws, tp, (int)blockIdx.x, (int)blockIdx.y, (int)blockIdx.z,
                           rows_per_block);
}

// The pre-pass and the ghost fill of a sub-step in ONE launch (rt_substep on 2-D / 3-D grids): they touch different
// arrays (lim, rho kappa_P from rho, T | the ghosts of U), so nbg blocks of the 1-D grid, spread evenly over it, do the
// ghost fill -- short, bound by the sector traffic of the x1 ghosts -- beside the issue-bound pre-pass blocks (the l-th
// of which is block bxi + gx (byi + gy bzi) of the pre-pass); one launch gap less per sub-step.
template <int MODE>
__global__ void __launch_bounds__(256) k_thick_limit_faces(const __grid_constant__ GridDev g, const __grid_constant__ OpacDev oR,
                                                           const __grid_constant__ OpacDev oS, const __grid_constant__ OpacSet os,
                                                           const double* __restrict__ rho, const double* __restrict__ T,
                                                           double* __restrict__ lim, const __grid_constant__ OpacDev oP,
                                                           int same_PR, double* __restrict__ kpr,
                                                           const __grid_constant__ LeanLaws laws, const __grid_constant__ TablePair tp,
                                                           const __grid_constant__ Fields4 U, int nbg, int gx, int gy, int rows_per_block) {
    // ghost-fill blocks are every stride-th block of the grid, so that they are resident beside pre-pass blocks
    const int tot = (int)gridDim.x, stride = tot / nbg, b = (int)blockIdx.x;
    if (b % stride == 0 && b / stride < nbg) {
        fill_faces_body(g, U, b / stride, nbg);
        return;
    }
    const int l = b - min(nbg, (b + stride - 1) / stride);
    const int bxi = l % gx, t = l / gx;
    thick_limit_body<MODE>(g, oR, oS, os, rho, T, lim, oP, same_PR, kpr, laws, tp, bxi, t % gy, t / gy, rows_per_block);
}

// ------------------------------------------------------------------------------------------------
// a11: CFL (step 10, L120; R-G15).  rate_i = sum_{d active} chat max(|lam1|,|lam3|)/dl_d;
// max over cells by warp shuffles -> one atomicMax per block on the bit pattern (rates are >= 0,
// so the unsigned order equals the numeric order); the last block to finish writes
// dt = cfl / rate and re-arms the scratch words.
// ------------------------------------------------------------------------------------------------
struct CflScratch {
    unsigned long long rate_bits;
    unsigned int blocks_done;
    unsigned int pad;
};

// il[d] = 1/dl_d of the cell (0 for an inactive direction: it then adds nothing)
__device__ __forceinline__ double cell_rate_il(double chat, double E, double F1, double F2, double F3, const double il[3]) {
    const double E2 = E * E;
    const double Fq = fma(F3, F3, fma(F2, F2, F1 * F1));
    const Closure c = closure_of(E, E2, Fq);
    const double F[3] = {F1, F2, F3};
    double sum = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double b = c.gE * F[d];
        const double z2 = (2.0 * c.dE) * fma(-b, F[d], c.sE);
        const double z = fsqrt(fabs(z2) + kTiny);  // see flux_and_speeds
        sum = fma((fabs(F[d]) + z) * c.rsE, il[d], sum);
    }
    return sum * chat;
}

__device__ __forceinline__ void cell_inv_lengths(const GridDev& g, int i, int j, int k, double il[3]) {
#pragma unroll
    for (int d = 0; d < 3; ++d) il[d] = g.gh[d] == 0 ? 0.0 : g.ilen[d][0][i] * g.ilen[d][1][j] * g.ilen[d][2][k];
}

__device__ __forceinline__ double cell_rate(const GridDev& g, double chat, double E, double F1, double F2, double F3, int i,
                                            int j, int k) {
    double il[3];
    cell_inv_lengths(g, i, j, k, il);
    return cell_rate_il(chat, E, F1, F2, F3, il);
}

__device__ __forceinline__ void block_max_to_global(double v, CflScratch* scr, double cfl, double* dt_out, unsigned nblocks) {
    __shared__ double sred[32];
    __shared__ bool last;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = dmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) sred[w] = v;
    __syncthreads();
    if (w == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        v = l < nw ? sred[l] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = dmax(v, __shfl_xor_sync(0xffffffffu, v, o));
        if (l == 0) {
            atomicMax(&scr->rate_bits, (unsigned long long)__double_as_longlong(v));
            __threadfence();
            const unsigned done = atomicAdd(&scr->blocks_done, 1u);
            last = (done == nblocks - 1);
        }
    }
    __syncthreads();
    if (last && threadIdx.x == 0) {
        __threadfence();
        const unsigned long long bits = atomicExch(&scr->rate_bits, 0ull);
        scr->blocks_done = 0;
        *dt_out = cfl / __longlong_as_double((long long)bits);
    }
}

// dt = cfl / (running max of the rate), then re-arm the running max (fused-CFL path of k_implicit)
static __global__ void k_cfl_finalize(CflScratch* scr, double cfl, double* dt_out) {
    const unsigned long long bits = scr->rate_bits;
    scr->rate_bits = 0ull;
    *dt_out = cfl / __longlong_as_double((long long)bits);
}

static __global__ void __launch_bounds__(256) k_cfl(GridDev g, double chat, const double* __restrict__ E, const double* __restrict__ F1,
                                             const double* __restrict__ F2, const double* __restrict__ F3, CflScratch* scr,
                                             double cfl, double* dt_out) {
    // a persistent-style grid (a few blocks per SM) walks the rows, so that only O(1000) atomics are issued
    const long long nrows = (long long)g.n[1] * g.n[2];
    double rate = 0.0;
    for (long long row = blockIdx.x; row < nrows; row += gridDim.x) {
        const int j = (int)(row % g.n[1]), k = (int)(row / g.n[1]);
        const long long rb = g.gh[0] * g.stride[0] + (j + g.gh[1]) * g.stride[1] + (k + g.gh[2]) * g.stride[2];
        for (int i = threadIdx.x; i < g.n[0]; i += blockDim.x) {
            const long long id = rb + i;
            rate = dmax(rate, cell_rate(g, chat, E[id], F1[id], F2[id], F3[id], i, j, k));
        }
    }
    block_max_to_global(rate, scr, cfl, dt_out, gridDim.x);
}

}  // namespace rtm1
