// rt_kernels_step.cuh — the fused reconstruct -> f-fix -> closure -> Riemann -> divergence sweeps
// (a2-a7) and the floor + opacity + implicit coupling kernel (a8-a10).  SURVEY.md Sect. 8(a).
// These per-direction kernels serve rt_explicit_step / rt_implicit_step and 1-D grids; on 2-D / 3-D grids rt_substep
// runs k_substep_fused (rt_kernels_fused.cuh), which shares implicit_cell() and the arithmetic of rt_math.cuh.
//
// Sweep design: face states, face fluxes and wave speeds never touch HBM.
//  * x1 sweep: one warp owns 32 consecutive cells of one row; every lane builds both face states of
//    its cell, the upper-face state moves one lane up and the area-weighted face flux one lane down
//    by warp shuffles, so each closure and each Riemann flux is evaluated once; lanes 1..30 write.
//  * x2 / x3 sweeps: lanes along x1 (coalesced), each thread marches along the sweep direction and
//    carries the previous cell's upper-face state and the previous face flux in registers: every
//    field value is loaded once per sweep, every face quantity is computed once.
// All directions start from U^n (unsplit, step 7 L117): the x1 sweep writes U_out = U_in - ..., the
// later sweeps accumulate into U_out while reading the stencil from U_in.
#pragma once
#include "rt_kernels_aux.cuh"

namespace rtm1 {

struct SweepArgs {
    const double* uin[4];
    double* uout[4];
    const double* lim;  // thick-limit pre-pass array (ghosted) or nullptr
    double dtc;         // dt * chat (host-supplied dt)
    const double* dt_dev;  // device-resident dt (rt_substep) or nullptr; then dt * chat = *dt_dev * chat
    double chat;
    int rusanov;  // RT_SOLVER_RUSANOV (the HLL instantiation computes the wave speeds it needs)
    int fix;      // RT_FIX_* (rt_set_face_fix): 0 = f-preserving (Eq. 19-21), 1 = flat fallback (L136), 2 = clip (Eq. 36-38)
    int recon;    // RT_RECON_* (rt_set_reconstruction): 0 = PLM + van Leer, 1 = LimO3 (L132)
    double limo3_r;  // LimO3: radius of the asymptotic region in cell lengths (<= 0: no smoothness switch)
};

// both face states of one cell with the reconstruction the launch selected (a uniform branch: two code copies)
template <int D, bool HLL>
__device__ __forceinline__ void cell_faces_sel(const SweepArgs& a, const double q0[4], const double dm[4], const double dp[4],
                                               bool want_lo, bool want_hi, State& lo, State& hi, double dx) {
    if (a.recon) cell_faces<D, HLL, false, true>(q0, dm, dp, want_lo, want_hi, lo, hi, 0.0, 0.0, 0.0, a.fix, a.limo3_r * dx);
    else cell_faces<D, HLL>(q0, dm, dp, want_lo, want_hi, lo, hi, 0.0, 0.0, 0.0, a.fix);
}
// the cell's length along D (LimO3's smoothness switch); ghost cells take the nearest interior cell's
__device__ __forceinline__ double cell_len(const GridDev& g, int D, int i, int j, int k) {
    i = min(max(i, 0), g.n[0] - 1);
    j = min(max(j, 0), g.n[1] - 1);
    k = min(max(k, 0), g.n[2] - 1);
    return g.len[D][0][i] * g.len[D][1][j] * g.len[D][2][k];
}

__device__ __forceinline__ double sweep_dtc(const SweepArgs& a) { return a.dt_dev ? __ldg(a.dt_dev) * a.chat : a.dtc; }

constexpr double kInf = __builtin_huge_val();

// ------------------------------------------------------------------------------------------------
// x1 sweep.  Warp task = (chunk of 30 output cells, row).  FIRST: always (x1 is the first active
// direction whenever n1 > 1).  CURVI: area weights + geometric sources (R-G9) from the
// cell-centred closure:  cyl: S(F^R) = +chat P^{phiphi}<1/R>, S(F^phi) = -chat P^{Rphi}<1/R>
//   sph: S(F^r) = chat (P^{thth}+P^{phph})<1/r>, S(F^th) = chat(-P^{rth} + <cot>P^{phph})<1/r>,
//        S(F^ph) = chat(-P^{rph} - <cot>P^{thph})<1/r>.
// ------------------------------------------------------------------------------------------------
constexpr int kXOut = 30;  // output cells per warp

template <bool HLL, bool THICK, bool CURVI>
__global__ void __launch_bounds__(128) k_sweep_x(const __grid_constant__ GridDev g, const __grid_constant__ SweepArgs a,
                                                 int nchunk, long long ntask) {
    const int lane = threadIdx.x & 31;
    const long long task = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (task >= ntask) return;
    const int ch = (int)(task % nchunk);
    const long long row = task / nchunk;
    const int j = (int)(row % g.n[1]), k = (int)(row / g.n[1]);
    const int n1 = g.n[0];
    const int i = ch * kXOut - 1 + lane;      // this lane's cell, -1 .. n1
    const int ic = i > n1 ? n1 : i;           // clamp idle lanes onto a valid cell
    const long long id = (ic + g.gh[0]) + (j + g.gh[1]) * g.stride[1] + (k + g.gh[2]) * g.stride[2];

    double q0[4], dm[4], dp[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const double* __restrict__ u = a.uin[q];
        const double um = u[id - 1], uc = u[id], up = u[id + 1];
        q0[q] = uc;
        dm[q] = uc - um;
        dp[q] = up - uc;
    }
    double limd = kInf;
    if (THICK) limd = dmax(a.lim[id - 1], a.lim[id]);

    State lo, hi;
    cell_faces_sel<0, HLL>(a, q0, dm, dp, true, true, lo, hi, a.recon ? cell_len(g, 0, i, j, k) : 0.0);

    // left state of this lane's lower face = upper-face state of the lane below
    State L;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        L.U[q] = __shfl_up_sync(0xffffffffu, hi.U[q], 1);
        L.G[q] = __shfl_up_sync(0xffffffffu, hi.G[q], 1);
    }
    if (HLL) {
        L.lm = __shfl_up_sync(0xffffffffu, hi.lm, 1);
        L.lp = __shfl_up_sync(0xffffffffu, hi.lp, 1);
    }
    double fl[4];
    riemann<HLL>(L, lo, limd, fl, a.rusanov != 0);
    if (CURVI) {
        const double w = g.wf[0][ic < 0 ? 0 : ic];
#pragma unroll
        for (int q = 0; q < 4; ++q) fl[q] *= w;
    }
    double fu[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) fu[q] = __shfl_down_sync(0xffffffffu, fl[q], 1);

    if (lane >= 1 && lane <= kXOut && i < n1) {
        const double dtc = sweep_dtc(a);
        const double coef = dtc * g.cg[0][0][i] * g.cg[0][1][j] * g.cg[0][2][k];
        double out[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) out[q] = fma(-coef, fu[q] - fl[q], q0[q]);
        if (CURVI) {
            const double E2 = q0[0] * q0[0];
            const double F2 = fma(q0[3], q0[3], fma(q0[2], q0[2], q0[1] * q0[1]));
            const Closure c = closure_of(q0[0], E2, F2);
            const double s = dtc * g.invr[i];
            if (g.geometry == 1) {
                out[1] = fma(s, fma(c.gE * q0[2], q0[2], c.dE), out[1]);
                out[2] = fma(-s, c.gE * q0[1] * q0[2], out[2]);
            } else {
                const double ct = g.cot[j];
                const double Ptt = fma(c.gE * q0[2], q0[2], c.dE);
                const double Ppp = fma(c.gE * q0[3], q0[3], c.dE);
                const double Prt = c.gE * q0[1] * q0[2];
                const double Prp = c.gE * q0[1] * q0[3];
                const double Ptp = c.gE * q0[2] * q0[3];
                out[1] = fma(s, Ptt + Ppp, out[1]);
                out[2] = fma(s, fma(ct, Ppp, -Prt), out[2]);
                out[3] = fma(-s, fma(ct, Ptp, Prp), out[3]);
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) a.uout[q][id] = out[q];
    }
}

// ------------------------------------------------------------------------------------------------
// x2 / x3 sweeps: marching.  Thread = (i, o, segment); o = the other transverse index (k for D = 1,
// j for D = 2); the segment covers cells [ca, cb) along D.  Step c in [ca-1, cb] builds the face
// states of cell c (only the upper one at c = ca-1, only the lower one at c = cb), the flux at the
// lower face of cell c, and then finishes cell c-1.  Accumulates into U_out (never the first sweep).
// ------------------------------------------------------------------------------------------------
template <int D, bool HLL, bool THICK, bool CURVI>
__global__ void __launch_bounds__(128) k_sweep_march(const __grid_constant__ GridDev g, const __grid_constant__ SweepArgs a,
                                                     int seglen) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n[0]) return;
    constexpr int EO = (D == 1) ? 2 : 1;
    const int o = blockIdx.y;
    const int nd = g.n[D];
    const int ca = blockIdx.z * seglen;
    const int cb = min(ca + seglen, nd);
    const long long S = g.stride[D];
    // index of the cell with sweep coordinate 0
    const long long id0 = (i + g.gh[0]) + (long long)g.gh[D] * S + (long long)(o + g.gh[EO]) * g.stride[EO];
    const double K = sweep_dtc(a) * g.cg[D][0][i] * g.cg[D][EO][o];
    const double* __restrict__ cgd = g.cg[D][D];
    const double* __restrict__ wfd = g.wf[D];

    long long p = id0 + (long long)(ca - 1) * S;
    double qc[4], dm[4], qn[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const double* __restrict__ u = a.uin[q];
        qc[q] = u[p];
        dm[q] = qc[q] - u[p - S];
        qn[q] = u[p + S];
    }
    double limp = kInf, limc = kInf;
    if (THICK) limc = a.lim[p];

    State hiPrev;
    double Fprev[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll 1
    for (int c = ca - 1; c <= cb; ++c, p += S) {
        // loads issued first: next stencil value, next limiter, accumulation base of cell c-1
        double qnn[4], base[4], limn = kInf;
        if (c < cb) {
#pragma unroll
            for (int q = 0; q < 4; ++q) qnn[q] = a.uin[q][p + 2 * S];
            if (THICK) limn = a.lim[p + S];
        }
        if (c > ca) {
#pragma unroll
            for (int q = 0; q < 4; ++q) base[q] = a.uout[q][p - S];
        }
        double dp[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) dp[q] = qn[q] - qc[q];
        State lo, hi;
        {
            double dxc = 0.0;
            if (a.recon) dxc = D == 1 ? cell_len(g, 1, i, c, o) : cell_len(g, 2, i, o, c);
            cell_faces_sel<D, HLL>(a, qc, dm, dp, c >= ca, c < cb, lo, hi, dxc);
        }
        if (c >= ca) {
            double fl[4];
            riemann<HLL>(hiPrev, lo, THICK ? dmax(limp, limc) : kInf, fl, a.rusanov != 0);
            if (CURVI) {
                const double w = wfd[c];
#pragma unroll
                for (int q = 0; q < 4; ++q) fl[q] *= w;
            }
            if (c > ca) {
                const double coef = K * cgd[c - 1];
#pragma unroll
                for (int q = 0; q < 4; ++q) a.uout[q][p - S] = fma(-coef, fl[q] - Fprev[q], base[q]);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) Fprev[q] = fl[q];
        }
        hiPrev = hi;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            dm[q] = dp[q];
            qc[q] = qn[q];
            qn[q] = qnn[q];
        }
        limp = limc;
        limc = limn;
    }
}

// ------------------------------------------------------------------------------------------------
// a8-a10: floor / clip (L81, L250; R-G11), opacities, implicit coupling (Eq. 29-33; R-G12):
//   g_r = dt chat kappa_P rho, g = dt c kappa_P rho, C_v = rho c_v, det = C_v (1 + g_r) + 4 g a_R T^3
//   E' = [E (C_v + 4 g a_R T^3) + g_r C_v a_R T^4] / det
//   T' = [(1 + g_r) C_v T + 3 g a_R T^4 + g E] / det
//   F' = F / (1 + dt chat chi rho) (Eq. 30);   m' = m - (F' - F)/chat (Eq. 28).
// ------------------------------------------------------------------------------------------------
struct ImplicitArgs {
    double* U[4];
    const double* rho;
    double* T;
    double* mom[3];
    double dt;
    const double* dt_dev;  // device-resident dt (rt_substep) or nullptr
    CflScratch* scr;       // CFL: running max of the rate, as the bit pattern of a non-negative double
    int feedback;
    int same_PR;  // kappa_P and kappa_R are the same law: evaluate once
    OpacSet os;   // shared log10 inputs of the table opacities
    double ichat; // 1 / chat
    unsigned long long* counters;  // [0] floor activations, [1] clip activations
    const double* divfirr;         // div F_irr per cell (Sect. 2.9, Eq. 34-35) or nullptr
    // RK2 (L107, L256): the second stage stores the average of its result with the state the step started from (AVG
    // instantiations only; nullptr: off).  avgU may be the output arrays themselves (each cell is read, then written, by
    // its own thread); the CFL rate is then that of the averaged state
    const double* avgU[4];
    const double* avgT;
    const double* avgm[3];
    // where the updated T and m go: the arrays they were read from (in place), or, for the first RK2 stage, scratch
    // arrays, so that T^n and m^n survive for the average without being copied first
    double* Tout;
    double* mout[3];
};

// CFL = true additionally evaluates the step-10 rate (R-G15) of the UPDATED state of each cell and folds it
// into scr->rate_bits: warp-shuffle max, then one atomicMax per warp that beats the running maximum (a plain
// load filters the rest, so a few hundred atomics reach L2 instead of one per warp); k_cfl_finalize turns the
// maximum into dt.  The result equals rt_cfl_dt of the updated state bit for bit (same cell_rate, max is exact).
// One cell of a8-a10 (+ the CFL rate of the updated state when CFL): shared by k_implicit and the fused
// sub-step kernel.  E, F: the state after the explicit half; writes through the pointers of `a` at index id.
// CHIGIVEN: rho chi and rho kappa_P of the cell are passed in (the fused kernel recovers the first from the
// thick-limit array of the SAME sub-step, lim = 4/(3 rho chi dx), and gets the second from the same pre-pass): no
// opacity is evaluated here.
template <bool FEEDBACK, bool CFL, bool CHIGIVEN = false, bool AVG = false>
__device__ __forceinline__ double implicit_cell(const GridDev& g, const ParamsDev& par, const OpacDev& oP, const OpacDev& oR,
                                                const OpacDev& oS, const ImplicitArgs& a, double dt, long long id,
                                                const double il[3] /* 1/dl_d of the cell (CFL only) */, double E, double F[3],
                                                double rho, double T0, const double m[3], bool& floored, bool& clipped,
                                                double rhochi_given = 0.0, double rhokp_given = 0.0) {
    // second RK2 stage (launch-uniform): the values to average with, loaded first so that the arithmetic below covers
    // their latency
    const bool avg = AVG && a.avgU[0] != nullptr;
    double avE = 0.0, avT = 0.0, avF[3] = {0.0, 0.0, 0.0}, avm[3] = {0.0, 0.0, 0.0};
    if (avg) {
        avE = a.avgU[0][id];
        avT = a.avgT[id];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            avF[q] = a.avgU[1 + q][id];
            if (FEEDBACK) avm[q] = a.avgm[q][id];
        }
    }
    // irradiation (Eq. 34-35): Q = -div F_irr dt joins S_1 of Eq. 33; a launch-uniform branch
    const bool irr = a.divfirr != nullptr;
    double Q = 0.0;
    if (irr) {
        Q = -__ldg(a.divfirr + id) * dt;
        asm volatile("");
    }
    if (E < par.E_floor) {
        E = par.E_floor;
        floored = true;
    }
    const double F2 = fma(F[2], F[2], fma(F[1], F[1], F[0] * F[0]));
    if (F2 > E * E) {
        const double sc = E * rsqrt(F2);
#pragma unroll
        for (int q = 0; q < 3; ++q) F[q] *= sc;
        clipped = true;
    }
    double rhokp, rhochi;
    if (CHIGIVEN) {
        rhokp = rhokp_given;
        rhochi = rhochi_given;
    } else {
        LogRT lg = {0.0, 0.0};
        const bool share = a.os.share != 0;
        if (share) lg = log_inputs(a.os.src == 0 ? oP : (a.os.src == 1 ? oR : oS), rho, T0);
        const double kP = opacity_eval_shared(oP, rho, T0, share, lg);
        const double kR = a.same_PR ? kP : opacity_eval_shared(oR, rho, T0, share, lg);
        rhokp = kP * rho;
        rhochi = (kR + opacity_eval_shared(oS, rho, T0, share, lg)) * rho;
    }
    const double gr = dt * par.chat * rhokp;
    const double gg = dt * par.c * rhokp;
    const double Cv = rho * par.c_v;
    const double aT3 = par.a_R * T0 * T0 * T0;
    const double aT4 = aT3 * T0;
    const double det = fma(Cv, 1.0 + gr, 4.0 * gg * aT3);
    const double idet = frcp(det);
    double En_ = fma(E, fma(4.0 * gg, aT3, Cv), gr * Cv * aT4) * idet;
    double Tn_ = fma((1.0 + gr) * Cv, T0, fma(3.0 * gg, aT4, gg * E)) * idet;
    if (irr) {  // E' += 4 g_r a_R T^3 Q / det,  T' += (1 + g_r) Q / det
        const double qd = Q * idet;
        En_ = fma(4.0 * gr * aT3, qd, En_);
        Tn_ = fma(1.0 + gr, qd, Tn_);
        asm volatile("");
    }
    double En = En_, Tn = Tn_;
    const double idamp = frcp(fma(dt * par.chat, rhochi, 1.0));
    if (avg) {
        En = 0.5 * (En + avE);
        Tn = 0.5 * (Tn + avT);
    }
    a.U[0][id] = En;
    a.Tout[id] = Tn;
    const double ichat = a.ichat;
    double Fn[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        Fn[q] = F[q] * idamp;
        if (FEEDBACK) {
            double mn = fma(-(Fn[q] - F[q]), ichat, m[q]);
            if (avg) mn = 0.5 * (mn + avm[q]);
            a.mout[q][id] = mn;
        }
        if (avg) Fn[q] = 0.5 * (Fn[q] + avF[q]);
        a.U[1 + q][id] = Fn[q];
    }
    return CFL ? cell_rate_il(par.chat, En, Fn[0], Fn[1], Fn[2], il) : 0.0;
}

// fold a warp's CFL rates into the running maximum (see k_implicit) and count floor / clip activations
template <bool CFL>
__device__ __forceinline__ void implicit_warp_epilogue(const ImplicitArgs& a, double rate, int nfloor, int nclip) {
    if (CFL) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) rate = dmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
        if ((threadIdx.x & 31) == 0) {
            const unsigned long long bits = (unsigned long long)__double_as_longlong(rate);
            if (bits > *(volatile unsigned long long*)&a.scr->rate_bits) atomicMax(&a.scr->rate_bits, bits);
        }
    }
    // rare: count floor / clip activations (debug counters, SURVEY.md Sect. 8(d) "Parity")
    if (__any_sync(0xffffffffu, (nfloor | nclip) != 0)) {
        nfloor = __reduce_add_sync(0xffffffffu, nfloor);
        nclip = __reduce_add_sync(0xffffffffu, nclip);
        if ((threadIdx.x & 31) == 0) {
            if (nfloor) atomicAdd(&a.counters[0], (unsigned long long)nfloor);
            if (nclip) atomicAdd(&a.counters[1], (unsigned long long)nclip);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Small 1-D grids (BASELINE config 1: 256 cells): the WHOLE sub-step in one CTA and one launch — ghost fill (step 1),
// thick-limit values, face states + Riemann fluxes, divergence (+ geometric sources), floor / clip, opacities, implicit
// coupling and the new time step (step 10).  Such grids are bound by launch latency, not by any pipe: the five to six
// launches of the per-direction path cost ~28 us per sub-step, this one a single launch.  One thread per FACE builds
// both states of its face from the staged row (each cell's slopes are evaluated by its two faces: twice the
// reconstruction work, which is irrelevant here, and no state exchange), then one thread per CELL finishes it.
// ------------------------------------------------------------------------------------------------
constexpr int K1D_MAXN = 512;   // cells: 10.5 doubles of shared memory per cell, 43 KB in all
constexpr int K1D_NT = 256;

template <bool HLL, bool THICK, bool CURVI, bool FEEDBACK>
__global__ void __launch_bounds__(K1D_NT) k_substep_1d(const __grid_constant__ GridDev g, const __grid_constant__ ParamsDev par,
                                                       const __grid_constant__ OpacDev oP, const __grid_constant__ OpacDev oR,
                                                       const __grid_constant__ OpacDev oS, const __grid_constant__ SweepArgs sw,
                                                       const __grid_constant__ ImplicitArgs im, double cfl, double* dt_out) {
    __shared__ double sU[4][K1D_MAXN + 4];
    __shared__ double sLim[K1D_MAXN + 2];
    __shared__ double sFl[4][K1D_MAXN + 1];
    __shared__ double sred[K1D_NT / 32];
    const int tid = threadIdx.x;
    const int n = g.n[0], gh = g.gh[0];
    const double dt = __ldg(im.dt_dev);
    const double dtc = dt * sw.chat;
    // step 1 (L111): stage the row with its ghosts; ghosts other than FIXED ones are also written back to U_in
    for (int e = tid; e < 4 * (n + 4); e += K1D_NT) {
        const int q = e / (n + 4), c = e - q * (n + 4) - 2;
        int src = c;
        bool flip = false;
        int kind = 3;
        if (c < 0 || c >= n) {
            kind = g.bc[c < 0 ? 0 : 1];
            if (kind == 0) src = c < 0 ? c + n : c - n;
            else if (kind == 1) src = c < 0 ? 0 : n - 1;
            else if (kind == 2) {
                src = c < 0 ? -1 - c : 2 * n - 1 - c;
                flip = q == 1;
            }
        }
        double v = sw.uin[q][src + gh];
        if (flip) v = -v;
        sU[q][c + 2] = v;
        if (kind != 3) const_cast<double*>(sw.uin[q])[c + gh] = v;
    }
    // Eq. 25-26 (R-G7): lim = 4 / (3 rho chi dx) of the cells -1 .. n (ghosts: periodic image or nearest interior cell)
    if (THICK) {
        for (int j = tid - 1; j <= n; j += K1D_NT) {
            int c = j;
            if (c < 0) c = g.bc[0] == 0 ? c + n : 0;
            else if (c >= n) c = g.bc[0] == 0 ? c - n : n - 1;
            const double r = __ldg(im.rho + c + gh), t = im.T[c + gh];
            const double chi = opacity_eval(oR, r, t) + opacity_eval(oS, r, t);
            const double tau = r * chi * (g.len[0][0][c] * g.len[0][1][0] * g.len[0][2][0]);
            sLim[j + 1] = tau > 1.0e-100 ? 4.0 * frcp(3.0 * tau) : kInf;
        }
    }
    __syncthreads();
    // steps 3-6: the flux through face i (between cells i-1 and i), i = 0 .. n
    for (int i = tid; i <= n; i += K1D_NT) {
        double qa[4], qb[4], dma[4], dpa[4], dpb[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            qa[q] = sU[q][i + 1];
            qb[q] = sU[q][i + 2];
            dma[q] = qa[q] - sU[q][i];
            dpa[q] = qb[q] - qa[q];
            dpb[q] = sU[q][i + 3] - qb[q];
        }
        State loa, hia, lob, hib;
        cell_faces_sel<0, HLL>(sw, qa, dma, dpa, false, true, loa, hia, sw.recon ? cell_len(g, 0, i - 1, 0, 0) : 0.0);
        cell_faces_sel<0, HLL>(sw, qb, dpa, dpb, true, false, lob, hib, sw.recon ? cell_len(g, 0, i, 0, 0) : 0.0);
        const double limd = THICK ? dmax(sLim[i], sLim[i + 1]) : kInf;
        double fe[4];
        riemann<HLL>(hia, lob, limd, fe, sw.rusanov != 0);
        const double w = CURVI ? g.wf[0][i] : 1.0;
#pragma unroll
        for (int q = 0; q < 4; ++q) sFl[q][i] = fe[q] * w;
    }
    __syncthreads();
    // step 7 (+ geometric sources, R-G9), then a8-a11 per cell
    double rate = 0.0;
    int nfloor = 0, nclip = 0;
    const double cyz = g.cg[0][1][0] * g.cg[0][2][0];
    const double il12 = g.ilen[0][1][0] * g.ilen[0][2][0];
    for (int i = tid; i < n; i += K1D_NT) {
        const double coef = dtc * g.cg[0][0][i] * cyz;
        double q0[4], out[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            q0[q] = sU[q][i + 2];
            out[q] = fma(-coef, sFl[q][i + 1] - sFl[q][i], q0[q]);
        }
        if (CURVI) {
            const double E2 = q0[0] * q0[0];
            const double F2 = fma(q0[3], q0[3], fma(q0[2], q0[2], q0[1] * q0[1]));
            const Closure c = closure_of(q0[0], E2, F2);
            const double s = dtc * g.invr[i];
            if (g.geometry == 1) {
                out[1] = fma(s, fma(c.gE * q0[2], q0[2], c.dE), out[1]);
                out[2] = fma(-s, c.gE * q0[1] * q0[2], out[2]);
            } else {
                const double ct = g.cot[0];
                const double Ptt = fma(c.gE * q0[2], q0[2], c.dE);
                const double Ppp = fma(c.gE * q0[3], q0[3], c.dE);
                const double Prt = c.gE * q0[1] * q0[2];
                const double Prp = c.gE * q0[1] * q0[3];
                const double Ptp = c.gE * q0[2] * q0[3];
                out[1] = fma(s, Ptt + Ppp, out[1]);
                out[2] = fma(s, fma(ct, Ppp, -Prt), out[2]);
                out[3] = fma(-s, fma(ct, Ptp, Prp), out[3]);
            }
        }
        const long long id = i + gh;
        double F[3] = {out[1], out[2], out[3]};
        double m[3] = {0.0, 0.0, 0.0};
        if (FEEDBACK) {
#pragma unroll
            for (int q = 0; q < 3; ++q) m[q] = im.mom[q][id];
        }
        const double il[3] = {g.ilen[0][0][i] * il12, 0.0, 0.0};
        bool floored = false, clipped = false;
        const double r = implicit_cell<FEEDBACK, true>(g, par, oP, oR, oS, im, dt, id, il, out[0], F, __ldg(im.rho + id), im.T[id], m,
                                                        floored, clipped);
        rate = dmax(rate, r);
        nfloor += floored ? 1 : 0;
        nclip += clipped ? 1 : 0;
    }
    // step 10 (L120; R-G15): dt = cfl / max rate; floor / clip counters
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) rate = dmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
    if ((tid & 31) == 0) sred[tid >> 5] = rate;
    if (__any_sync(0xffffffffu, (nfloor | nclip) != 0)) {
        nfloor = __reduce_add_sync(0xffffffffu, nfloor);
        nclip = __reduce_add_sync(0xffffffffu, nclip);
        if ((tid & 31) == 0) {
            if (nfloor) atomicAdd(&im.counters[0], (unsigned long long)nfloor);
            if (nclip) atomicAdd(&im.counters[1], (unsigned long long)nclip);
        }
    }
    __syncthreads();
    if (tid == 0) {
        double r = sred[0];
#pragma unroll
        for (int k = 1; k < K1D_NT / 32; ++k) r = dmax(r, sred[k]);
        *dt_out = cfl / r;
    }
}

template <bool FEEDBACK, bool CFL>
__global__ void __launch_bounds__(128) k_implicit(const __grid_constant__ GridDev g, const __grid_constant__ ParamsDev par,
                                                  const __grid_constant__ OpacDev oP, const __grid_constant__ OpacDev oR,
                                                  const __grid_constant__ OpacDev oS, const __grid_constant__ ImplicitArgs a) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y, k = blockIdx.z;
    bool floored = false, clipped = false;
    double rate = 0.0;
    const double dt = a.dt_dev ? __ldg(a.dt_dev) : a.dt;
    if (i < g.n[0]) {
        const long long id = (i + g.gh[0]) + (j + g.gh[1]) * g.stride[1] + (k + g.gh[2]) * g.stride[2];
        const double E = a.U[0][id];
        double F[3] = {a.U[1][id], a.U[2][id], a.U[3][id]};
        const double rho = a.rho[id];
        const double T0 = a.T[id];
        double m[3] = {0.0, 0.0, 0.0};
        if (FEEDBACK) {
#pragma unroll
            for (int q = 0; q < 3; ++q) m[q] = a.mom[q][id];
        }
        double il[3] = {0.0, 0.0, 0.0};
        if (CFL) cell_inv_lengths(g, i, j, k, il);
        rate = implicit_cell<FEEDBACK, CFL>(g, par, oP, oR, oS, a, dt, id, il, E, F, rho, T0, m, floored, clipped);
    }
    implicit_warp_epilogue<CFL>(a, rate, floored ? 1 : 0, clipped ? 1 : 0);
}

}  // namespace rtm1
