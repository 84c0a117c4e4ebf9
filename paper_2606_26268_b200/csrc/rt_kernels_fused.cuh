// rt_kernels_fused.cuh — ONE kernel for the whole sub-step on 3-D (and, without its x3 phase, 2-D) grids
// (SURVEY.md Sect. 8(f) NEXT-1):
// steps 3-8 and the rate of step 10 in a single pass over U^n.
//
// Design (DESIGN.md Sect. 5 "Fused sub-step kernel").  A CTA of 32 x FTY threads owns an x1-x2 tile of
// 30 x FTY cells and marches along x3 through a segment [ka, kb).  The x1-x2 planes of U^n (and of the
// thick-limit array) it needs — tile + 2 ghost cells on each side — are staged in shared memory by TMA (one
// cp.async.bulk.tensor.3d box of 34 x (FTY+4) x 1 doubles per field and plane, issued by one thread,
// completion on an mbarrier) into a ring of four planes (c-1, c, c+1 in use, c+2 in flight): every
// stencil value is read from HBM/L2 once per CTA, the loads occupy no registers and no issue slots, and
// boxes hanging over the array edge are zero-filled by the hardware.  Arrays the TMA cannot address
// (odd x1 extent => row pitch not a multiple of 16 B, or a base pointer not 16-B aligned) take an
// 8-byte cp.async loop instead.  Thread (lx, ly) owns cell (i0+lx, j0+ly): every lane owns an output cell.  The
// fluxes through the two OUTER x1 faces of a row (lower face of lane 0, upper face of lane 31) need the face states of
// the cells i0-1 and i0+32: the 2 x FTY such faces of a plane are one half-filled warp task ("edge task": both face
// states + Riemann flux of the face), done one step ahead by the warp whose turn it is (rows 1, 2, 5, 6 take turns:
// rows 0 and FTY-1 already carry the tile's extra x2 face work, and rows 4 and 3 share their schedulers) and handed
// over through shared memory.  That costs 3.6 % more warp instructions than the rows
// alone; halo lanes (30 useful lanes of 32, and a ragged ninth tile on a 256-cell row) cost 12.5 %.
// Per plane c, every thread:
//   Z  : both x3 face states of cell c (Eq. 17-21 + closure + speeds), Riemann flux at face c-1/2 against
//        the upper-face state of cell c-1 kept in this thread's shared-memory slot;
//   FIN: cell c-1 is complete: U* = acc - dt/V [A F]_z, then floor/clip, opacities, implicit coupling
//        (Eq. 29-33, 30, 28), stores, CFL rate of the updated state (a8-a11); its rho, T, m were
//        prefetched into L2 one plane earlier;
//   X  : x1 face states; exchanged by warp shuffles; + geometric sources;
//   Y  : x2 face states; the upper-face state goes to the row above through the thread's shared-memory slot,
//        guarded by a 64-thread named barrier per row pair (producer bar.arrive, consumer bar.sync); the row
//        above computes the flux through that face and writes it back INTO THE SAME SLOT, where the owner picks
//        it up one plane later (after the per-plane __syncthreads).  The bottom row builds the upper-face state
//        of the cell below the tile itself, the top row the lower-face state of the cell above and that flux.
//   acc = U^n - dt/V([AF]_x + [AF]_y) + dt S_geo.
// One __syncthreads per plane, no idle warps, no idle lanes.  Every closure, wave speed and Riemann flux is evaluated
// once per face inside the tile; the tile boundary costs the edge task in x1 and one extra face state + flux per edge
// row in x2.  Face states, fluxes and U* never touch HBM.
#pragma once
#include <cuda.h>  // CUtensorMap (type only: the encoder is fetched through cudaGetDriverEntryPoint)

#include "rt_kernels_step.cuh"

namespace rtm1 {

constexpr int FTX = 32;           // output cells per CTA along x1 = lanes: no halo lanes (the fluxes through the two outer
                                  // x1 faces of a row come from the edge task below)
constexpr int FTY = 8;            // output cells per CTA along x2 = thread rows (no halo rows: rows 0 and FTY-1
                                  // build the face states of the cells below / above the tile themselves)
constexpr int FNY = FTY;          // thread rows
constexpr int FNT = 32 * FNY;     // threads per CTA
constexpr int FPW = FTX + 4;      // staged plane width  (cells i0-2 .. i0+33)
constexpr int FPH = FTY + 4;      // staged plane height (cells j0-2 .. j0+FTY+1)
constexpr int FPHW = FPW * FPH;
constexpr int FPS = (FPHW + 15) / 16 * 16;  // doubles between staged arrays: every TMA destination 128-B aligned
constexpr int FNARR = 5;          // E, F1, F2, F3, lim
constexpr int FNSLOT = 4;
#ifndef FUSED_MINB
#define FUSED_MINB 2
#endif
constexpr int FNST = 10;          // doubles of an exchanged face state: U[4], G[4], lm, lp
constexpr int FNEDGE = 2 * FNY;   // x1 edge tasks per plane: (lower, upper) outer face of every row
// staged planes | zhi[FNST][FNT] | yex[FNST][FNT] | xedge[2][4][FNEDGE] | mbarriers
constexpr size_t kFusedSmemBytes =
    sizeof(double) * (size_t)(FNSLOT * FNARR * FPS + 2 * FNST * FNT + 2 * 4 * FNEDGE) + FNSLOT * sizeof(unsigned long long);
static_assert(FTY <= 15, "one named barrier per row pair");

struct FusedArgs {
    const double* src[FNARR];  // U_in[4], lim (or nullptr)
    const double* kpr;         // rho kappa_P per cell from the pre-pass (with lim), or nullptr
    ImplicitArgs im;           // U = U_out, rho, T, mom, dt / dt_dev, scratch, counters
    double chat;
    int use_tma;
    int fix;                   // RT_FIX_* (read only by the VMODE = 2 instantiations)
};
struct alignas(64) FusedMaps {
    CUtensorMap m[FNARR];      // ghosted (nt1, nt2, nt3) fp64 tensors, box 34 x FPH x 1
};

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned bar_smem, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar_smem), "r"(parity)
        : "memory");
    return ok != 0;
}
// Wait for a phase of an mbarrier.  A bulk copy that never completes (a descriptor the hardware rejects) would spin
// here for ever: after 2^24 failed tries (seconds) the kernel traps instead, and the next API call reports RT_ERR_CUDA.
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    const unsigned b = (unsigned)__cvta_generic_to_shared(bar);
    unsigned spins = 0;
    while (!mbar_try_wait(b, parity)) {
        if (++spins > (1u << 24)) __trap();  // each failed try already waits a hardware time slice: seconds in total
    }
}
__device__ __forceinline__ void tma_load_3d(double* smem_dst, const CUtensorMap* map, int x, int y, int z, unsigned long long* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            (unsigned)__cvta_generic_to_shared(smem_dst)),
        "l"(map), "r"(x), "r"(y), "r"(z), "r"((unsigned)__cvta_generic_to_shared(bar))
        : "memory");
}
// 64-thread named barriers: the producer warp arrives, the consumer warp waits
__device__ __forceinline__ void pair_arrive(int id) { asm volatile("bar.arrive %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void pair_sync(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// a face state in shared memory: component-major, N slots per component (conflict-free)
template <bool HLL, int N>
__device__ __forceinline__ void state_store(double* buf, int t, const State& s) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        buf[q * N + t] = s.U[q];
        buf[(4 + q) * N + t] = s.G[q];
    }
    if (HLL) {
        buf[8 * N + t] = s.lm;
        buf[9 * N + t] = s.lp;
    }
}
template <bool HLL, int N>
__device__ __forceinline__ void state_load(const double* buf, int t, State& s) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        s.U[q] = buf[q * N + t];
        s.G[q] = buf[(4 + q) * N + t];
    }
    if (HLL) {
        s.lm = buf[8 * N + t];
        s.lp = buf[9 * N + t];
    } else {
        s.lm = 0.0;
        s.lp = 0.0;
    }
}



// RUS (with HLL = true): RT_SOLVER_RUSANOV, compile-time so that the HLL faces do not pay for the test
// HASZ = false: 2-D grids (n3 = 1, x3 inactive): one staged plane, no x3 phase; the march degenerates to the steps
// c = 0 (X, Y) and 1 (FIN, which reads nothing but the thick-limit value of plane 0).
// VMODE = 0: the paper's f-preserving scheme compiled in, T and m updated through a.im.Tout / mout, no other option
// (the path of rt_substep).  1: the same plus the RK2 average of the second stage (rt_rk2_step) behind one
// launch-uniform test per cell (a.im.avgU[0] != nullptr); the values to average with are prefetched into L2 one plane
// ahead.  2: 1 plus the comparison face fixes of rt_set_face_fix (flat fallback L136 / clip Eq. 36-38) selected by
// the launch-uniform a.fix.
template <bool HLL, bool THICK, bool CURVI, bool FEEDBACK, bool RUS, bool HASZ, int VMODE = 0>
__global__ void __launch_bounds__(FNT, FUSED_MINB)
    k_substep_fused(const __grid_constant__ GridDev g, const __grid_constant__ ParamsDev par, const __grid_constant__ OpacDev oP,
                    const __grid_constant__ OpacDev oR, const __grid_constant__ OpacDev oS, const __grid_constant__ FusedArgs a,
                    const __grid_constant__ FusedMaps maps, int seglen) {
    extern __shared__ __align__(128) double sm[];
    double* const planes = sm;
    double* const zhi = planes + FNSLOT * FNARR * FPS;  // [FNST][FNT] own slot: upper x3 face state of the previous plane
    double* const yex = zhi + FNST * FNT;               // [FNST][FNT] x2 exchange, one slot per thread: its upper x2 face
                                                        // state on the way up, then (components 0-3) the flux through
                                                        // that face on the way back down
    double* const xedge = yex + FNST * FNT;             // [2 (plane parity)][4][FNEDGE] area-weighted fluxes through the
                                                        // outer x1 faces: task t = side * FNY + row
    unsigned long long* const mbar = (unsigned long long*)(xedge + 2 * 4 * FNEDGE);  // [FNSLOT]

    const int lx = threadIdx.x, ly = threadIdx.y;
    const int tid = ly * 32 + lx;
    const int i0 = blockIdx.x * FTX, j0 = blockIdx.y * FTY;
    const int ka = blockIdx.z * seglen;
    const int kb = min(ka + seglen, g.n[2]);
    const int i = i0 + lx, j = j0 + ly;
    const bool writer = i < g.n[0] && j < g.n[1];
    const int ic = min(i, g.n[0] - 1), jc = min(j, g.n[1] - 1);
    const int o = (ly + 2) * FPW + lx + 2;  // this thread's cell inside a staged plane
    const bool tma = a.use_tma != 0;
    constexpr bool rus = HLL && RUS;
    const int fix = VMODE == 2 ? a.fix : 0;
    const double dt = a.im.dt_dev ? __ldg(a.im.dt_dev) : a.im.dt;
    const double dtc = dt * a.chat;

    constexpr int NA = THICK ? 5 : 4;
    if (tma) {
        if (tid == 0) {
#pragma unroll
            for (int s = 0; s < FNSLOT; ++s) mbar_init(mbar + s, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("fence.proxy.async;" ::: "memory");
        }
        __syncthreads();
    }
    // stage plane cc (x3 cell index, -2 .. n3+1) into ring slot (cc + 4) & 3
    auto load_plane = [&](int cc) {
        const int slot = (cc + 4) & 3;
        double* dst = planes + slot * (FNARR * FPS);
        if (tma) {
            if (tid == 0) {
                mbar_expect_tx(mbar + slot, (unsigned)(NA * FPHW * sizeof(double)));
#pragma unroll
                for (int arr = 0; arr < NA; ++arr) tma_load_3d(dst + arr * FPS, &maps.m[arr], i0, j0, cc + g.gh[2], mbar + slot);
            }
        } else {
            const long long zoff = (long long)min(max(cc + g.gh[2], 0), g.nt[2] - 1) * g.stride[2];
            for (int e = tid; e < NA * FPHW; e += FNT) {
                const int arr = e / FPHW, r = e - arr * FPHW;
                const int row = r / FPW, col = r - row * FPW;
                const int gi = min(i0 + col, g.nt[0] - 1), gj = min(j0 + row, g.nt[1] - 1);
                cp_async8(dst + arr * FPS + r, a.src[arr] + zoff + (long long)gj * g.stride[1] + gi);
            }
            cp_async_commit();
        }
    };
    // plane p of this segment is the ((p - ka + 2) >> 2)-th use of its slot
    auto wait_plane = [&](int p) {
        if (tma) mbar_wait(mbar + ((p + 4) & 3), (unsigned)(((p - ka + 2) >> 2) & 1));
    };
    if (HASZ) {
        load_plane(ka - 2);
        load_plane(ka - 1);
        load_plane(ka);
        wait_plane(ka - 2);
        wait_plane(ka - 1);
    } else {
        load_plane(0);  // the only plane of a 2-D grid; it is waited for at the top of step 0
    }

    const double kx = dtc * g.cg[0][0][ic] * g.cg[0][1][jc];
    const double ky = dtc * g.cg[1][0][ic] * g.cg[1][1][jc];
    const double kz = HASZ ? dtc * g.cg[2][0][ic] * g.cg[2][1][jc] : 0.0;
    double wx = 1.0, wylo = 1.0, wyhi = 1.0;  // face-area weights of this cell's lower x1 face, lower / upper x2 faces
    if (CURVI) {
        wx = g.wf[0][min(i, g.n[0])];
        wylo = g.wf[1][min(j, g.n[1])];
        wyhi = g.wf[1][min(j + 1, g.n[1])];
    }
    const int id0 = (ic + g.gh[0]) + (jc + g.gh[1]) * (int)g.stride[1] + g.gh[2] * (int)g.stride[2];  // cell (i, j, 0)
    const int zstride = (int)g.stride[2];
    double ilxy[3];  // x1-x2 part of 1/dl_d (CFL)
#pragma unroll
    for (int d = 0; d < 3; ++d) ilxy[d] = (d < 2 || HASZ) ? g.ilen[d][0][ic] * g.ilen[d][1][jc] : 0.0;

    double acc[4] = {0.0, 0.0, 0.0, 0.0};  // U^n - dt/V ([AF]_x + [AF]_y) + dt S_geo of the previous plane's cell,
                                           // still missing the flux through its upper x2 face (held by the row above)
    double Fz[4] = {0.0, 0.0, 0.0, 0.0};   // area-weighted flux through the lower x3 face of that cell
    int nfloor = 0, nclip = 0;             // cells of this thread whose floor / clip fired
    double rate = 0.0;

    // Edge task of plane cc (staged at pe): lanes 0 .. FNEDGE-1 of the calling warp; task t = side * FNY + row computes
    // the flux through the lower (side 0: cells i0-1 | i0) or upper (side 1: cells i0+31 | i0+32) outer x1 face of that
    // row from scratch and leaves it, area-weighted, in xedge[cc & 1].  Faces outside the grid produce unused numbers.
    auto edge_task = [&](int cc, const double* pe) {
        if (lx < FNEDGE) {
            const int row = lx % FNY, side = lx / FNY;
            const int ob = (row + 2) * FPW + 2 + side * FTX;  // cell b = the upper cell of the face; a = b - 1
            double qa[4], qb[4], dma[4], dpa[4], dpb[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                qa[q] = pe[q * FPS + ob - 1];
                qb[q] = pe[q * FPS + ob];
                dma[q] = qa[q] - pe[q * FPS + ob - 2];
                dpa[q] = qb[q] - qa[q];
                dpb[q] = pe[q * FPS + ob + 1] - qb[q];
            }
            State loa, hia, lob, hib;
            cell_faces<0, HLL>(qa, dma, dpa, false, true, loa, hia, 0.0, 0.0, 0.0, fix);
            cell_faces<0, HLL>(qb, dpa, dpb, true, false, lob, hib, 0.0, 0.0, 0.0, fix);
            const double limd = THICK ? dmax(pe[4 * FPS + ob - 1], pe[4 * FPS + ob]) : kInf;
            double fe[4];
            riemann<HLL>(hia, lob, limd, fe, rus);
            const double w = CURVI ? g.wf[0][min(i0 + side * FTX, g.n[0])] : 1.0;
            double* dst = xedge + (cc & 1) * (4 * FNEDGE) + lx;
#pragma unroll
            for (int q = 0; q < 4; ++q) dst[q * FNEDGE] = fe[q] * w;
        }
    };

#pragma unroll 1
    for (int c = HASZ ? ka - 1 : 0; c <= kb; ++c) {
        if (HASZ || c == 0) {
            if (tma) wait_plane(HASZ ? c + 1 : 0); else cp_async_wait_all();
        }
        __syncthreads();  // plane c+1 visible to all; every warp is done with step c-1
        if (HASZ && c + 2 <= kb + 1) load_plane(c + 2);
        const double* pc = planes + ((c + 4) & 3) * (FNARR * FPS);
        if (HASZ) {
            // outer x1 faces of plane c+1, consumed by the X phase of the next step (behind its barrier); the buffer
            // written here was last read in the X phase of step c-1, before this step's barrier
            // the task rotates over the warps of rows 1, 2, 5, 6: rows 0 and FTY-1 carry the extra x2 face work of the tile's
            // edge and share their schedulers (warp id mod 4) with rows 4 and 3
            if (c + 1 < kb && ly == (((c + 1) & 1) + 1 + ((c + 1) & 2) * 2)) edge_task(c + 1, planes + ((c + 5) & 3) * (FNARR * FPS));
        } else if (c == 0) {
            if (ly == 0) edge_task(0, pc);   // 2-D: the only plane; one extra barrier
            __syncthreads();
        }
        if (writer && c < kb) {  // inputs of the implicit half of cell c, needed one step from now
            const int idn = id0 + c * zstride;
            prefetch_l2(a.im.rho + idn);
            prefetch_l2(a.im.T + idn);
            if (THICK) prefetch_l2(a.kpr + idn);
            if (FEEDBACK) {
#pragma unroll
                for (int q = 0; q < 3; ++q) prefetch_l2(a.im.mom[q] + idn);
            }
            if (VMODE != 0 && a.im.avgU[0] != nullptr) {  // launch-uniform: the second RK2 stage averages with U^n, T^n, m^n
#pragma unroll
                for (int q = 0; q < 4; ++q) prefetch_l2(a.im.avgU[q] + idn);
                prefetch_l2(a.im.avgT + idn);
                if (FEEDBACK) {
#pragma unroll
                    for (int q = 0; q < 3; ++q) prefetch_l2(a.im.avgm[q] + idn);
                }
            }
        }
        // gas state of cell c-1 for FIN: issued here so that the x3 phase hides what is left of its latency
        double rho_f = 1.0, T_f = 1.0, kpr_f = 0.0;
        double m_f[3] = {0.0, 0.0, 0.0};
        if (writer && c > ka) {
            const int id = id0 + (c - 1) * zstride;
            rho_f = __ldg(a.im.rho + id);
            T_f = a.im.T[id];
            if (THICK) kpr_f = __ldg(a.kpr + id);
            if (FEEDBACK) {
#pragma unroll
                for (int q = 0; q < 3; ++q) m_f[q] = a.im.mom[q][id];
            }
        }
        double invEc, Ec2, F2c;
        // ---------------------------------------------------------------- Z
        {
            const double* pm = planes + ((c + 3) & 3) * (FNARR * FPS);
            const double* pp = planes + ((c + 5) & 3) * (FNARR * FPS);
            double q0[4], dm[4], dp[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                // 2-D grids stage plane 0 only: step 1 (their FIN step) has no plane of its own to read
                q0[q] = (HASZ || c == 0) ? pc[q * FPS + o] : 1.0;
                dm[q] = HASZ ? q0[q] - pm[q * FPS + o] : 0.0;
                dp[q] = HASZ ? pp[q * FPS + o] - q0[q] : 0.0;
            }
            State lo, hi;
            invEc = frcp(q0[0]);  // 1/E_c, E_c^2, |F_c|^2: shared by the three directions of this cell
            Ec2 = q0[0] * q0[0];
            F2c = fma(q0[3], q0[3], fma(q0[2], q0[2], q0[1] * q0[1]));
            if (HASZ) cell_faces<2, HLL, true>(q0, dm, dp, true, true, lo, hi, invEc, Ec2, F2c, fix);  // both always: one basic block, two independent chains
            double flz[4] = {0.0, 0.0, 0.0, 0.0};
            if (HASZ && c >= ka) {
                State L;
                state_load<HLL, FNT>(zhi, tid, L);
                const double limd = THICK ? dmax(pm[4 * FPS + o], pc[4 * FPS + o]) : kInf;
                riemann<HLL>(L, lo, limd, flz, rus);
                if (CURVI) {
                    const double w = g.wf[2][c];
#pragma unroll
                    for (int q = 0; q < 4; ++q) flz[q] *= w;
                }
            }
            if (HASZ) state_store<HLL, FNT>(zhi, tid, hi);
            // ------------------------------------------------------------ FIN (cell c-1): a8-a11
            if (c > ka) {
                const double coef = HASZ ? kz * g.cg[2][2][c - 1] : 0.0;
                const double cyp = ky * g.cg[1][2][c - 1];
                double U4[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) U4[q] = fma(-coef, flz[q] - Fz[q], fma(-cyp, yex[q * FNT + tid], acc[q]));
                if (writer) {
                    const int id = id0 + (c - 1) * zstride;
                    const double rho = rho_f, T0 = T_f;
                    const double m[3] = {m_f[0], m_f[1], m_f[2]};
                    double F[3] = {U4[1], U4[2], U4[3]};
                    const double il[3] = {ilxy[0] * g.ilen[0][2][c - 1], ilxy[1] * g.ilen[1][2][c - 1],
                                          HASZ ? ilxy[2] * g.ilen[2][2][c - 1] : 0.0};
                    bool floored = false, clipped = false;
                    // rho chi of the cell from the thick-limit array of this sub-step: lim = 4/(3 rho chi dx), dx = the
                    // cell's largest extent = 1/min_d(1/dl_d); lim = +inf stands for rho chi dx <= 1e-100
                    double rhochi = 0.0;
                    if (THICK) {
                        const double lim = pm[4 * FPS + o];
                        const double ilmin = HASZ ? dmin(il[0], dmin(il[1], il[2])) : dmin(il[0], il[1]);  // active directions
                        rhochi = lim > 1.0e300 ? 0.0 : (4.0 / 3.0) * ilmin * frcp(lim);
                    }
                    const double r = implicit_cell<FEEDBACK, true, THICK, VMODE != 0>(g, par, oP, oR, oS, a.im, dt, (long long)id, il, U4[0],
                                                                                  F, rho, T0, m, floored, clipped, rhochi, kpr_f);
                    rate = dmax(rate, r);
                    nfloor += floored ? 1 : 0;
                    nclip += clipped ? 1 : 0;
                }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) Fz[q] = flz[q];
        }
        if (c < ka || c >= kb) continue;  // block-uniform

        double qc[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) qc[q] = pc[q * FPS + o];
        // ---------------------------------------------------------------- X
        {
            double dm[4], dp[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                dm[q] = qc[q] - pc[q * FPS + o - 1];
                dp[q] = pc[q * FPS + o + 1] - qc[q];
            }
            State lo, hi;
            cell_faces<0, HLL, true>(qc, dm, dp, true, true, lo, hi, invEc, Ec2, F2c, fix);
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
            const double limd = THICK ? dmax(pc[4 * FPS + o - 1], pc[4 * FPS + o]) : kInf;
            riemann<HLL>(L, lo, limd, fl, rus);
            if (CURVI) {
#pragma unroll
                for (int q = 0; q < 4; ++q) fl[q] *= wx;
            }
            const double cx = kx * g.cg[0][2][c];
            const double* xe = xedge + (c & 1) * (4 * FNEDGE);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (lx == 0) fl[q] = xe[q * FNEDGE + ly];                    // lower outer face of the row
                double fu = __shfl_down_sync(0xffffffffu, fl[q], 1);
                if (lx == 31) fu = xe[q * FNEDGE + FNY + ly];                // upper outer face of the row
                acc[q] = fma(-cx, fu - fl[q], qc[q]);
            }
            if (CURVI) {
                const double E2 = qc[0] * qc[0];
                const double F2 = fma(qc[3], qc[3], fma(qc[2], qc[2], qc[1] * qc[1]));
                const Closure cl = closure_of(qc[0], E2, F2);
                const double s = dtc * g.invr[ic];
                if (g.geometry == 1) {
                    acc[1] = fma(s, fma(cl.gE * qc[2], qc[2], cl.dE), acc[1]);
                    acc[2] = fma(-s, cl.gE * qc[1] * qc[2], acc[2]);
                } else {
                    const double ct = g.cot[jc];
                    const double Ptt = fma(cl.gE * qc[2], qc[2], cl.dE);
                    const double Ppp = fma(cl.gE * qc[3], qc[3], cl.dE);
                    const double Prt = cl.gE * qc[1] * qc[2];
                    const double Prp = cl.gE * qc[1] * qc[3];
                    const double Ptp = cl.gE * qc[2] * qc[3];
                    acc[1] = fma(s, Ptt + Ppp, acc[1]);
                    acc[2] = fma(s, fma(ct, Ppp, -Prt), acc[2]);
                    acc[3] = fma(-s, fma(ct, Ptp, Prp), acc[3]);
                }
            }
        }
        // ---------------------------------------------------------------- Y: face states; the upper one to the row above
        State ylo;
        {
            double dm[4], dp[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                dm[q] = qc[q] - pc[q * FPS + o - FPW];
                dp[q] = pc[q * FPS + o + FPW] - qc[q];
            }
            State hi;
            cell_faces<1, HLL, true>(qc, dm, dp, true, true, ylo, hi, invEc, Ec2, F2c, fix);
            if (ly < FTY - 1) {
                state_store<HLL, FNT>(yex, tid, hi);
                pair_arrive(1 + ly);
            } else {
                // top row: the lower-face state of the cell above the tile, and the flux through the face between them
                double qa[4], dma[4], dpa[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    qa[q] = pc[q * FPS + o + FPW];
                    dma[q] = qa[q] - qc[q];
                    dpa[q] = pc[q * FPS + o + 2 * FPW] - qa[q];
                }
                State loa, hia;
                cell_faces<1, HLL>(qa, dma, dpa, true, false, loa, hia, 0.0, 0.0, 0.0, fix);
                const double limd = THICK ? dmax(pc[4 * FPS + o], pc[4 * FPS + o + FPW]) : kInf;
                double fup[4];
                riemann<HLL>(hi, loa, limd, fup, rus);
#pragma unroll
                for (int q = 0; q < 4; ++q) yex[q * FNT + tid] = CURVI ? fup[q] * wyhi : fup[q];
            }
        }
        // ---------------------------------------------------------------- Y: flux through the lower x2 face
        {
            State L;
            if (ly > 0) {
                pair_sync(ly);  // the row below has stored its upper-face state
                state_load<HLL, FNT>(yex, tid - 32, L);
            } else {
                // bottom row: the upper-face state of the cell below the tile
                double qb[4], dmb[4], dpb[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    qb[q] = pc[q * FPS + o - FPW];
                    dmb[q] = qb[q] - pc[q * FPS + o - 2 * FPW];
                    dpb[q] = qc[q] - qb[q];
                }
                State lob;
                cell_faces<1, HLL>(qb, dmb, dpb, false, true, lob, L, 0.0, 0.0, 0.0, fix);
            }
            const double limd = THICK ? dmax(pc[4 * FPS + o - FPW], pc[4 * FPS + o]) : kInf;
            double fly[4];
            riemann<HLL>(L, ylo, limd, fly, rus);
            const double cy = ky * g.cg[1][2][c];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (CURVI) fly[q] *= wylo;
                // back down to the row below, which reads it at the start of the next step, into the slot its state came
                // from: that row wrote the slot BEFORE its pair_arrive, this store comes AFTER the pair_sync on it
                if (ly > 0) yex[q * FNT + tid - 32] = fly[q];
                acc[q] = fma(cy, fly[q], acc[q]);
            }
        }
    }
    implicit_warp_epilogue<true>(a.im, rate, nfloor, nclip);
}

}  // namespace rtm1
