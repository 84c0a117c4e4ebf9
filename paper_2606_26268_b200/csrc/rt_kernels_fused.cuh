// rt_kernels_fused.cuh — ONE kernel for the whole sub-step on 3-D grids (SURVEY.md Sect. 8(f) NEXT-1):
// steps 3-8 and the rate of step 10 in a single pass over U^n.
//
// Design.  A CTA owns an x1-x2 tile of 30 x FTY cells and marches
// along x3 through a segment [ka, kb).  The x1-x2 planes of U^n (and of the thick-limit array) it
// needs — tile + 2 ghost cells on each side — are staged in shared memory by cp.async into a ring of
// four planes (c-1, c, c+1 in use, c+2 in flight), so every stencil value is read from HBM/L2 once per
// CTA and the loads never occupy registers.  Thread (lx, ly) owns cell (i0-1+lx, j0-1+ly): lanes 0 and
// 31 and rows 0 and FTY+1 are the halo whose face states the tile's outer faces need.  Per plane c:
//   Z  : both x3 face states of cell c (Eq. 17-21 + closure + speeds), Riemann flux at face c-1/2 against
//        the upper-face state of cell c-1 kept in this thread's shared-memory slot;
//   FIN: cell c-1 is complete: U* = acc - dt/V [A F]_z, then floor/clip, opacities, implicit coupling
//        (Eq. 29-33, 30, 28), stores, CFL rate of the updated state (a8-a11);
//   Y  : x2 face states; upper-face states and face fluxes are exchanged through shared memory;
//   X  : x1 face states; exchanged by warp shuffles; + geometric sources;   acc = U^n - dt/V([AF]_x + [AF]_y).
// Every closure, wave speed and Riemann flux is evaluated once per face inside the tile; the halo costs
// 32/30 in x1 and (3 FTY + 1)/(3 FTY) in x2.  Face states, fluxes and U* never touch HBM.
#pragma once
#include "rt_kernels_step.cuh"

namespace rtm1 {

constexpr int FTX = 30;           // output cells per CTA along x1 (32 lanes, 1 halo lane each side)
constexpr int FTY = 6;            // output cells per CTA along x2
constexpr int FNY = FTY + 2;      // thread rows
constexpr int FNT = 32 * FNY;     // threads per CTA
constexpr int FPW = 34;           // staged plane width  (cells i0-2 .. i0+31)
constexpr int FPH = FTY + 4;      // staged plane height (cells j0-2 .. j0+FTY+1)
constexpr int FPHW = FPW * FPH;
constexpr int FNARR = 5;          // E, F1, F2, F3, lim
constexpr int FNSLOT = 4;
constexpr int FNST = 10;          // doubles of an exchanged face state: U[4], G[4], lm, lp
constexpr size_t kFusedSmemBytes = sizeof(double) * (size_t)(FNSLOT * FNARR * FPHW + 2 * FNST * FNT + 4 * FNT);

struct FusedArgs {
    const double* src[FNARR];  // U_in[4], lim (or nullptr)
    ImplicitArgs im;           // U = U_out, rho, T, mom, dt / dt_dev, scratch, counters
    double chat;
};

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <bool HLL>
__device__ __forceinline__ void state_store(double* buf, int t, const State& s) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        buf[q * FNT + t] = s.U[q];
        buf[(4 + q) * FNT + t] = s.G[q];
    }
    if (HLL) {
        buf[8 * FNT + t] = s.lm;
        buf[9 * FNT + t] = s.lp;
    }
}
template <bool HLL>
__device__ __forceinline__ void state_load(const double* buf, int t, State& s) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        s.U[q] = buf[q * FNT + t];
        s.G[q] = buf[(4 + q) * FNT + t];
    }
    if (HLL) {
        s.lm = buf[8 * FNT + t];
        s.lp = buf[9 * FNT + t];
    } else {
        s.lm = 0.0;
        s.lp = 0.0;
    }
}

template <bool HLL, bool THICK, bool CURVI, bool FEEDBACK>
__global__ void __launch_bounds__(FNT, 2)
    k_substep_fused(const __grid_constant__ GridDev g, const __grid_constant__ ParamsDev par, const __grid_constant__ OpacDev oP,
                    const __grid_constant__ OpacDev oR, const __grid_constant__ OpacDev oS, const __grid_constant__ FusedArgs a,
                    int seglen) {
    extern __shared__ double sm[];
    double* const planes = sm;
    double* const zhi = planes + FNSLOT * FNARR * FPHW;
    double* const yhi = zhi + FNST * FNT;
    double* const yfl = yhi + FNST * FNT;

    const int lx = threadIdx.x, ly = threadIdx.y;
    const int tid = ly * 32 + lx;
    const int i0 = blockIdx.x * FTX, j0 = blockIdx.y * FTY;
    const int ka = blockIdx.z * seglen;
    const int kb = min(ka + seglen, g.n[2]);
    const int i = i0 - 1 + lx, j = j0 - 1 + ly;
    const bool row_in = (ly >= 1) && (ly <= FTY);
    const bool writer = row_in && lx >= 1 && lx <= FTX && i < g.n[0] && j < g.n[1];
    const int ic = min(max(i, 0), g.n[0] - 1), jc = min(max(j, 0), g.n[1] - 1);
    const int o = (ly + 1) * FPW + lx + 1;  // this thread's cell inside a staged plane

    const double dt = a.im.dt_dev ? __ldg(a.im.dt_dev) : a.im.dt;
    const double dtc = dt * a.chat;
    const double kx = dtc * g.cg[0][0][ic] * g.cg[0][1][jc];
    const double ky = dtc * g.cg[1][0][ic] * g.cg[1][1][jc];
    const double kz = dtc * g.cg[2][0][ic] * g.cg[2][1][jc];
    double wx = 1.0, wy = 1.0;
    if (CURVI) {
        wx = g.wf[0][min(max(i, 0), g.n[0])];
        wy = g.wf[1][min(max(j, 0), g.n[1])];
    }
    // element index of cell (i, j, 0) in the ghosted arrays
    const long long id0 = (ic + g.gh[0]) + (long long)(jc + g.gh[1]) * g.stride[1] + (long long)g.gh[2] * g.stride[2];

    constexpr int NA = THICK ? 5 : 4;
    auto load_plane = [&](int c) {
        double* dst = planes + ((c + 4) & 3) * (FNARR * FPHW);
        const long long zoff = (long long)(c + g.gh[2]) * g.stride[2];
        for (int e = tid; e < NA * FPHW; e += FNT) {
            const int arr = e / FPHW, r = e - arr * FPHW;
            const int row = r / FPW, col = r - row * FPW;
            const int gi = min(i0 + col, g.nt[0] - 1), gj = min(j0 + row, g.nt[1] - 1);
            cp_async8(dst + e, a.src[arr] + zoff + (long long)gj * g.stride[1] + gi);
        }
        cp_async_commit();
    };
    load_plane(ka - 2);
    load_plane(ka - 1);
    load_plane(ka);

    double acc[4] = {0.0, 0.0, 0.0, 0.0};  // U^n - dt/V ([AF]_x + [AF]_y) + dt S_geo of the previous plane's cell
    double Fz[4] = {0.0, 0.0, 0.0, 0.0};   // area-weighted flux through the lower x3 face of that cell
    int nfloor = 0, nclip = 0;  // cells of this thread whose floor / clip fired
    double rate = 0.0;

#pragma unroll 1
    for (int c = ka - 1; c <= kb; ++c) {
        cp_async_wait_all();
        __syncthreads();
        if (c + 2 <= kb + 1) load_plane(c + 2);
        const double* pc = planes + ((c + 4) & 3) * (FNARR * FPHW);

        if (row_in) {
            // ---------------------------------------------------------------- Z
            const double* pm = planes + ((c + 3) & 3) * (FNARR * FPHW);
            const double* pp = planes + ((c + 5) & 3) * (FNARR * FPHW);
            double flz[4];
            {
                double q0[4], dm[4], dp[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    q0[q] = pc[q * FPHW + o];
                    dm[q] = q0[q] - pm[q * FPHW + o];
                    dp[q] = pp[q * FPHW + o] - q0[q];
                }
                State lo, hi;
                cell_faces<2, HLL>(q0, dm, dp, c >= ka, c < kb, lo, hi);
                if (c >= ka) {
                    State L;
                    state_load<HLL>(zhi, tid, L);
                    const double limd = THICK ? dmax(pm[4 * FPHW + o], pc[4 * FPHW + o]) : kInf;
                    riemann<HLL>(L, lo, limd, flz);
                    if (CURVI) {
                        const double w = g.wf[2][c];
#pragma unroll
                        for (int q = 0; q < 4; ++q) flz[q] *= w;
                    }
                }
                if (c < kb) state_store<HLL>(zhi, tid, hi);
            }
            // ---------------------------------------------------------------- FIN (cell c-1)
            if (c > ka) {
                const double coef = kz * g.cg[2][2][c - 1];
                double E = fma(-coef, flz[0] - Fz[0], acc[0]);
                double F[3];
#pragma unroll
                for (int q = 0; q < 3; ++q) F[q] = fma(-coef, flz[1 + q] - Fz[1 + q], acc[1 + q]);
                if (writer) {
                    const long long id = id0 + (long long)(c - 1) * g.stride[2];
                    const double rho = a.im.rho[id];
                    const double T0 = a.im.T[id];
                    double m[3] = {0.0, 0.0, 0.0};
                    if (FEEDBACK) {
#pragma unroll
                        for (int q = 0; q < 3; ++q) m[q] = a.im.mom[q][id];
                    }
                    bool floored = false, clipped = false;
                    const double r = implicit_cell<FEEDBACK, true>(g, par, oP, oR, oS, a.im, dt, id, i, j, c - 1, E, F, rho, T0, m,
                                                                   floored, clipped);
                    rate = dmax(rate, r);
                    nfloor += floored ? 1 : 0;
                    nclip += clipped ? 1 : 0;
                }
            }
            if (c >= ka) {
#pragma unroll
                for (int q = 0; q < 4; ++q) Fz[q] = flz[q];
            }
        }

        if (c >= ka && c < kb) {  // block-uniform
            // ---------------------------------------------------------------- Y
            double fly[4], qy[4];
            {
                double dm[4], dp[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    qy[q] = pc[q * FPHW + o];
                    dm[q] = qy[q] - pc[q * FPHW + o - FPW];
                    dp[q] = pc[q * FPHW + o + FPW] - qy[q];
                }
                State lo, hi;
                cell_faces<1, HLL>(qy, dm, dp, ly >= 1, ly <= FTY, lo, hi);
                if (ly <= FTY) state_store<HLL>(yhi, tid, hi);
                __syncthreads();
                if (ly >= 1) {
                    State L;
                    state_load<HLL>(yhi, tid - 32, L);
                    const double limd = THICK ? dmax(pc[4 * FPHW + o - FPW], pc[4 * FPHW + o]) : kInf;
                    riemann<HLL>(L, lo, limd, fly);
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        if (CURVI) fly[q] *= wy;
                        yfl[q * FNT + tid] = fly[q];
                    }
                }
                __syncthreads();
            }
            if (row_in) {
                const double cy = ky * g.cg[1][2][c];
#pragma unroll
                for (int q = 0; q < 4; ++q) acc[q] = fma(-cy, yfl[q * FNT + tid + 32] - fly[q], qy[q]);
                // ------------------------------------------------------------ X
                double dm[4], dp[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    dm[q] = qy[q] - pc[q * FPHW + o - 1];
                    dp[q] = pc[q * FPHW + o + 1] - qy[q];
                }
                State lo, hi;
                cell_faces<0, HLL>(qy, dm, dp, true, true, lo, hi);
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
                const double limd = THICK ? dmax(pc[4 * FPHW + o - 1], pc[4 * FPHW + o]) : kInf;
                riemann<HLL>(L, lo, limd, fl);
                if (CURVI) {
#pragma unroll
                    for (int q = 0; q < 4; ++q) fl[q] *= wx;
                }
                const double cx = kx * g.cg[0][2][c];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const double fu = __shfl_down_sync(0xffffffffu, fl[q], 1);
                    acc[q] = fma(-cx, fu - fl[q], acc[q]);
                }
                if (CURVI) {
                    const double E2 = qy[0] * qy[0];
                    const double F2 = fma(qy[3], qy[3], fma(qy[2], qy[2], qy[1] * qy[1]));
                    const Closure cl = closure_of(qy[0], E2, F2);
                    const double s = dtc * g.invr[ic];
                    if (g.geometry == 1) {
                        acc[1] = fma(s, fma(cl.gE * qy[2], qy[2], cl.dE), acc[1]);
                        acc[2] = fma(-s, cl.gE * qy[1] * qy[2], acc[2]);
                    } else {
                        const double ct = g.cot[jc];
                        const double Ptt = fma(cl.gE * qy[2], qy[2], cl.dE);
                        const double Ppp = fma(cl.gE * qy[3], qy[3], cl.dE);
                        const double Prt = cl.gE * qy[1] * qy[2];
                        const double Prp = cl.gE * qy[1] * qy[3];
                        const double Ptp = cl.gE * qy[2] * qy[3];
                        acc[1] = fma(s, Ptt + Ppp, acc[1]);
                        acc[2] = fma(s, fma(ct, Ppp, -Prt), acc[2]);
                        acc[3] = fma(-s, fma(ct, Ptp, Prp), acc[3]);
                    }
                }
            }
        }
    }
    implicit_warp_epilogue<true>(a.im, rate, nfloor, nclip);
}

}  // namespace rtm1
