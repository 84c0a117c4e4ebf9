// rt_math.cuh — fp64 device arithmetic of the gray-M1 sub-step (sm_100a).
//
// The sweeps sit at the fp64-pipe ridge of B200, so the formulas of
// PAPER.md Sect. 2.1/2.6 are restated in a division-lean form.  With s = sqrt(4 - 3 f^2) (Eq. 13,
// L75) the Levermore factor is xi = (3 + 4f^2)/(5 + 2s) = (5 - 2s)/3, hence
//     (1 - xi)/2 = (s - 1)/3,     (3 xi - 1)/(2 f^2) = 3/(2 + s),
//     P^{ij} = (s-1)/3 E delta^{ij} + 3/(2+s) F^i F^j / E                       (Eq. 11-12)
//     zeta^2 = 2/3 (s - 1)(s - 3 mu^2/(2+s)),  mu = F^d/E,  lambda_{1,3} = (mu -+ zeta)/s   (Eq. 22, 24)
// and everything is carried multiplied by E ("E-scaled": sE = sqrt(4E^2 - 3|F|^2) = E s) so that no
// 1/E is needed:  P^{id} = (sE - E)/3 delta^{id} + gE F^i F^d,  gE = 3/(2E + sE),
//                 zE^2 = 2/3 (sE - E)(sE - gE (F^d)^2),  lambda_{1,3} = (F^d -+ zE)/sE.
// Reciprocals / square roots are MUFU seeds (rcp.approx / rsqrt.approx, ~20 bits) plus one third-order
// step (and a residual step for the square root): <= ~1-1.3 ulp, no slow path.  Valid for NORMAL-range operands whose squares are
// normal too (|x| in ~[1e-150, 1e150]); include/rt.h states that as the field range.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rtm1 {

__device__ __forceinline__ double rcp_seed(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    return r;
}
__device__ __forceinline__ double rsqrt_seed(double x) {
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    return r;
}

// 1/x: seed (relative error <= 2^-19.9, measured) + ONE third-order step r (1 + e + e^2), e = 1 - x r: 3 dependent
// DFMA instead of the 4 of two Newton steps (the kernels are bound by the number of instructions issued).  Measured on
// B200 over 2^30 inputs: <= 1 ulp.
__device__ __forceinline__ double frcp(double x) {
    const double r = rcp_seed(x);
    const double e = fma(-x, r, 1.0);
    const double t = fma(e, e, e);
    return fma(r, t, r);
}

// y/2 of a NORMAL positive double whose half is normal too (the MUFU seeds below): one integer subtraction on the
// exponent field instead of a multiplication in the fp64 pipe, which is the unit this library is short of
__device__ __forceinline__ double half_of_normal(double y) {
    return __hiloint2double(__double2hiint(y) - 0x00100000, __double2loint(y));
}

// s = sqrt(x) and hrs = 1/(2 sqrt(x)) together (one third-order coupled step + residual step, 7 fp64 ops;
// measured on B200 over 2^30 inputs: s correctly rounded, 2 hrs <= 1.3 ulp).
__device__ __forceinline__ void fsqrt_hrsqrt(double x, double& s, double& hrs) {
    const double y = rsqrt_seed(x);
    double g = x * y, h = half_of_normal(y);
    // one third-order step: with 2t = 1 - x y^2,  1/sqrt(1 - 2t) = 1 + t + 3/2 t^2 + O(t^3)
    const double t = fma(-h, g, 0.5);
    const double p = fma(1.5 * t, t, t);
    g = fma(g, p, g);
    h = fma(h, p, h);
    // residual step: makes s exact for perfect squares (x = E^2/4 at f = 1 gives s = E/2, hence
    // (1 - xi)/2 = 0 and zeta = 0 exactly: the lambda -> cos(theta) limit of L167)
    const double d = fma(-g, g, x);
    s = fma(d, h, g);
    hrs = h;
}

// sqrt(x) alone (5 fp64 ops): one third-order step, no residual step (<= ~1 ulp; exactness for perfect squares is
// not needed where this is used: zeta and the CFL rate); x must be > 0 (callers add a tiny positive number).
__device__ __forceinline__ double fsqrt(double x) {
    const double y = rsqrt_seed(x);
    const double g = x * y, h = half_of_normal(y);
    const double t = fma(-h, g, 0.5);
    const double p = fma(1.5 * t, t, t);
    return fma(g, p, g);
}

// log10(x) and 10^v for the opacity tables (L375; R-G14), written out because the pre-pass and the implicit half were
// spending most of their issue slots inside the library versions (their polynomial coefficients arrive as pairs of
// 32-bit immediates: two register moves per coefficient).  Same recipe as any libm, no special cases:
// x = 2^e m, m in [sqrt(1/2), sqrt(2)), log m = 2 atanh(s), s = (m-1)/(m+1), |s| <= 0.1716, series to s^21/21 (next term
// < 1e-18); 10^v = 2^n 10^r, n = round(v log2 10), |r| <= 0.1506 (two-piece log10 2), 10^r = exp(r ln 10), Taylor to
// t^13/13! (next term < 5e-18).  <= ~2 ulp each against libm over the table ranges; x must be positive and normal
// (zero gives -308, below any table edge, like the -inf of the exact function), |v| < 300.
__device__ __forceinline__ double flog10(double x) {
    int hi = __double2hiint(x);
    int e = (hi >> 20) - 1023;
    hi = (hi & 0x000fffff) | 0x3ff00000;  // m in [1, 2)
    if (hi >= 0x3ff6a09f) {                // m > sqrt(2): halve it
        hi -= 0x00100000;
        e += 1;
    }
    const double m = __hiloint2double(hi, __double2loint(x));
    const double s = (m - 1.0) * frcp(m + 1.0);
    const double z = s * s;
    double p = 1.0 / 21.0;
    p = fma(p, z, 1.0 / 19.0);
    p = fma(p, z, 1.0 / 17.0);
    p = fma(p, z, 1.0 / 15.0);
    p = fma(p, z, 1.0 / 13.0);
    p = fma(p, z, 1.0 / 11.0);
    p = fma(p, z, 1.0 / 9.0);
    p = fma(p, z, 1.0 / 7.0);
    p = fma(p, z, 1.0 / 5.0);
    p = fma(p, z, 1.0 / 3.0);
    p = fma(p * z, s, s);                                          // s (1 + z/3 + z^2/5 + ...)
    return fma((double)e, 0.3010299956639812, 0.8685889638065036 * p);  // e log10 2 + (2 / ln 10) atanh s
}
__device__ __forceinline__ double fexp10(double v) {
    const double sh = fma(v, 3.321928094887362, 6755399441055744.0);   // round(v log2 10) in the low word
    const int n = __double2loint(sh);
    const double nf = sh - 6755399441055744.0;
    double r = fma(-nf, 0.3010299955494702, v);       // log10 2 in two pieces: the first has 21 trailing zero bits
    r = fma(-nf, 1.1451100898021838e-10, r);
    const double t = r * 2.302585092994046;
    double p = 1.0 / 6227020800.0;
    p = fma(p, t, 1.0 / 479001600.0);
    p = fma(p, t, 1.0 / 39916800.0);
    p = fma(p, t, 1.0 / 3628800.0);
    p = fma(p, t, 1.0 / 362880.0);
    p = fma(p, t, 1.0 / 40320.0);
    p = fma(p, t, 1.0 / 5040.0);
    p = fma(p, t, 1.0 / 720.0);
    p = fma(p, t, 1.0 / 120.0);
    p = fma(p, t, 1.0 / 24.0);
    p = fma(p, t, 1.0 / 6.0);
    p = fma(p, t, 0.5);
    p = fma(p, t, 1.0);
    p = fma(p, t, 1.0);
    return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));  // times 2^n: p in [0.7, 1.42]
}

__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

constexpr double kTiny = 1.0e-200;  // positive clamp under square roots (zeta^2 = 0 at f = 1)
constexpr double kTinySpeed = 1.0e-30;  // HLL: S_R >= +tiny, S_L <= -tiny  ==> den > 0 always (R-G8)

// One face (or cell) state with what the Riemann solver needs from it.
struct State {
    double U[4];   // E, F1, F2, F3
    double G[4];   // physical flux through direction D divided by chat: (F^D, P^{1D}, P^{2D}, P^{3D})
    double lm, lp; // lambda_1 (minus) and lambda_3 (plus) along D, in units of chat (HLL only)
};

// E-scaled closure pieces shared by flux, wave speeds and sources.
struct Closure {
    double sE;   // E sqrt(4 - 3 f^2)
    double rsE;  // 1 / sE
    double gE;   // 3 / (2E + sE)
    double dE;   // (sE - E)/3   = (1 - xi)/2 E
};

// E2 = E*E and F2 = |F|^2 are passed in because the callers have them already.
// f is capped at 1 (Eq. 14; round-off guard, R-G4): |F|^2 enters as min(F2, E2).
// The square root is taken of (4 E^2 - 3 |F|^2)/4 = E^2 - 3/4 |F|^2 (the scaling by a power of two commutes with every
// rounding): sE = 2 sqrt(.), 1/sE = the routine's 1/(2 sqrt(.)) as it stands.
__device__ __forceinline__ Closure closure_of(double E, double E2, double F2) {
    Closure c;
    const double m = dmin(F2, E2);
    const double w = fma(-0.75, m, E2);
    double hs;
    fsqrt_hrsqrt(w, hs, c.rsE);
    c.sE = hs + hs;
    c.gE = 1.5 * frcp(E + hs);               // 3 / (2E + sE)
    c.dE = fma(2.0, hs, -E) * (1.0 / 3.0);   // (sE - E)/3
    return c;
}

// Flux through direction D (Eq. 5-6, without the factor chat) and, for HLL, lambda_{1,3}.
template <int D, bool WAVES>
__device__ __forceinline__ void flux_and_speeds(State& st, double E2, double F2) {
    const double E = st.U[0];
    const Closure c = closure_of(E, E2, F2);
    const double Fd = st.U[1 + D];
    const double b = c.gE * Fd;
    st.G[0] = Fd;
    st.G[1] = b * st.U[1];
    st.G[2] = b * st.U[2];
    st.G[3] = b * st.U[3];
    st.G[1 + D] += c.dE;
    if (WAVES) {
        // 2/3 (sE - E)(sE - gE Fd^2) >= 0 up to rounding: it can come out a rounding error below zero only where
        // sE - E itself is at round-off (f = 1 to the last bits), and it is exactly 0 for f = 1 exactly; |.| + tiny keeps
        // the square root's argument positive with ONE fp64 operation (a max costs a compare and a chain of selects)
        const double z2 = (2.0 * c.dE) * fma(-b, Fd, c.sE);
        const double z = fsqrt(fabs(z2) + kTiny);
        st.lm = (Fd - z) * c.rsE;
        st.lp = (Fd + z) * c.rsE;
    } else {
        st.lm = 0.0;
        st.lp = 0.0;
    }
}

// PLM + van Leer limiter (Eq. 17-18; R-G3): HALF slope  h = dm dp/(dm + dp) if dm dp > 0.
__device__ __forceinline__ double half_slope(double dm, double dp) {
    double pr = dm * dp;
    double h = pr * frcp(dm + dp);
    return pr > 0.0 ? h : 0.0;
}

// LimO3 (L132; Cada & Torrilhon 2009; DESIGN R-G22): phi(dnum/dden) dden without the quotient.  With s = sign(dden),
// a = |dden|, b = s dnum and P = s (2 dden + dnum)/3 = a phi_3:  a phi_L = max(0, min(P, max(-b/2, min(2b, P, 1.6a)))),
// which is 0 for dden = 0 as the limit demands.  eta < 0: no smoothness switch (phi = phi_L); else phi_3 below
// eta = 1 - eps, phi_L above 1 + eps, their blend in between (eps = 1e-12).
__device__ __forceinline__ double limo3_times(double dnum, double dden, double eta) {
    const double p3 = (2.0 * dden + dnum) * (1.0 / 3.0);
    // the sign folds are multiplications by s = +-1 (exact) instead of selects, and the min / max chain is split by the
    // sign of b, which leaves three of its five: for b >= 0 every candidate is >= 0 and P >= the others' minimum, so
    // a phi_L = min(P, 2b, 1.6a); for b < 0 the inner minimum is <= 2b < 0 < -b/2, so a phi_L = max(0, min(P, -b/2)).
    // Both are max(0, min(P, c, d)) with (c, d) = (2b, 1.6a) or (-b/2, +inf): the same VALUE as the chain, bit for bit
    // (min and max round nothing; 2b and -b/2 are exact).
    const double s = __hiloint2double((__double2hiint(dden) & (int)0x80000000) | 0x3ff00000, 0);
    const double a = fabs(dden), b = s * dnum, P = s * p3;
    const bool pos = b >= 0.0;
    const double c = b * (pos ? 2.0 : -0.5);
    const double d = pos ? 1.6 * a : __builtin_huge_val();
    const double pl = dmax(0.0, dmin(dmin(P, c), d));
    const double pL = s * pl;
    if (eta < 0.0) return pL;
    constexpr double eps = 1.0e-12;
    if (eta <= 1.0 - eps) return p3;
    if (eta >= 1.0 + eps) return pL;
    return 0.5 * ((1.0 - (eta - 1.0) / eps) * p3 + (1.0 + (eta - 1.0) / eps) * pL);
}
// the smoothness indicator (d-^2 + d+^2)/(r dx)^2, rounded operation by operation: it DECIDES which branch a face
// takes, so it is evaluated exactly as the oracle evaluates it (no contraction into fused multiply-adds)
__device__ __forceinline__ double limo3_eta(double dm, double dp, double rdx) {
    return __ddiv_rn(__dadd_rn(__dmul_rn(dm, dm), __dmul_rn(dp, dp)), __dmul_rn(rdx, rdx));
}

// f-preserving face state (Eq. 19-21; R-G4).  Uc = cell value, invEc = 1/E_c,
// Ec2 = E_c^2, F2c = |F_c|^2; on entry st.U holds the reconstructed R(U) = Uc + sh (sh = the signed half slope, of
// which dE = sh[0] is passed in); on exit the face state.  Returns through E2f/F2f the squares of the final face state.
__device__ __forceinline__ void fpreserve(State& st, const double Uc[4], double dE, double invEc, double Ec2, double F2c,
                                          double& E2f, double& F2f) {
    const double Ef = st.U[0];
    E2f = Ef * Ef;
    double F2r = fma(st.U[3], st.U[3], fma(st.U[2], st.U[2], st.U[1] * st.U[1]));
    bool keep = (F2r <= E2f) && (F2r * Ec2 > F2c * E2f);
    // E_f/E_c = 1 + dE/E_c in ONE operation (E_f = E_c + dE up to its own rounding: 1-2 ulp on the quotient): a zero
    // slope gives r = 1 EXACTLY, so a cell with f = 1 and zero slopes keeps f_face = 1 exactly (the zeta = 0 limit, L167)
    const double r = fma(dE, invEc, 1.0);
    st.U[1] = keep ? st.U[1] : Uc[1] * r;
    st.U[2] = keep ? st.U[2] : Uc[2] * r;
    st.U[3] = keep ? st.U[3] : Uc[3] * r;
    F2f = keep ? F2r : F2c * (r * r);
}

// The two comparison schemes of Sect. 2.5 / 3.2 (rt_set_face_fix; per-direction kernels only), same contract as fpreserve.
// fix == 1, "PLUTO reconstruction" (L136): U_f = U_c, E included, whenever |R(F)| > R(E).
// fix == 2, clip (Eq. 36-38): F_f = R(F) R(E)/|R(F)| whenever |R(F)| > R(E); IEEE sqrt and division (a rare path).
__device__ __forceinline__ void facefix_variant(int fix, State& st, const double Uc[4], double Ec2, double F2c, double& E2f,
                                                double& F2f) {
    const double Ef = st.U[0];
    E2f = Ef * Ef;
    F2f = fma(st.U[3], st.U[3], fma(st.U[2], st.U[2], st.U[1] * st.U[1]));
    if (F2f <= E2f) return;
    if (fix == 1) {
#pragma unroll
        for (int q = 0; q < 4; ++q) st.U[q] = Uc[q];
        E2f = Ec2;
        F2f = F2c;
    } else {
        const double r = Ef / sqrt(F2f);
#pragma unroll
        for (int q = 1; q < 4; ++q) st.U[q] *= r;
        F2f = fma(st.U[3], st.U[3], fma(st.U[2], st.U[2], st.U[1] * st.U[1]));
    }
}

// Riemann flux (L150; R-G5, G6, G8) divided by chat, from left state L and right state R.
// limd = 4/(3 tau_face) (Eq. 25-26 in units of chat; +inf when the thick limit is off).
// rusanov (launch-uniform, HLL instantiation only): the local Lax-Friedrichs bound alpha = max |lambda_{1,3}| of the
// two states, clamped by limd: S_R = -S_L = alpha turns the two-wave formula into 1/2(F_L+F_R) - 1/2 alpha (U_R-U_L).
template <bool HLL>
__device__ __forceinline__ void riemann(const State& L, const State& R, double limd, double flux[4], bool rusanov = false) {
    double sR, sL;
    if (HLL) {
        // S_L = min(lm_L, lm_R, 0), S_R = max(lp_L, lp_R, 0) (R-G6), clamped by -+limd (Eq. 25-26), then kept off zero
        // (R-G8).  The last clamp subsumes the "0" of the first (a positive min ends at -tiny either way), so the
        // comparison against 0 is not spelled out.
        sL = dmin(L.lm, R.lm);
        sR = dmax(L.lp, R.lp);
        if (rusanov) {  // kept a real (uniform) branch: if-converted it costs every HLL face a compare and two selects
            sR = dmax(-sL, sR);
            sL = -sR;
            asm volatile("");
        }
        sL = dmax(sL, -limd);
        sR = dmin(sR, limd);
        sL = dmin(sL, -kTinySpeed);
        sR = dmax(sR, kTinySpeed);
    } else {
        sR = dmax(dmin(1.0, limd), kTinySpeed);  // GLF: alpha = min(chat, 4 chat/(3 tau))
        sL = -sR;
    }
    if (!HLL) {
        // alpha = sR = -sL: 1/2 (G_L + G_R) - 1/2 alpha (U_R - U_L) as it is written (L150), no reciprocal
        const double ha = 0.5 * sR;
#pragma unroll
        for (int q = 0; q < 4; ++q) flux[q] = fma(-ha, R.U[q] - L.U[q], 0.5 * (L.G[q] + R.G[q]));
        return;
    }
    const double rden = frcp(sR - sL);
    const double sRL = sR * sL;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        double num = fma(sR, L.G[q], fma(-sL, R.G[q], sRL * (R.U[q] - L.U[q])));
        flux[q] = num * rden;
    }
}

// Both face states of one cell along D from the cell value q0 and the two one-sided differences.
// lo = state at the cell's lower face (RIGHT state of face c-1/2), hi = state at its upper face
// (LEFT state of face c+1/2).  WANT_LO / WANT_HI are warp-uniform run-time flags.
// KNOWN: the caller passes 1/E_c, E_c^2 and |F_c|^2 (the three directions of one cell share them).
// fix (launch-uniform; RT_FIX_*): 0 = the f-preserving scheme; the fused kernel never passes anything else.
// LIMO3: the compact third-order reconstruction instead of PLM; rdx = r x the cell's length along D (<= 0: no
// smoothness switch).  The per-direction kernels and the 1-D kernel only.
template <int D, bool HLL, bool KNOWN = false, bool LIMO3 = false>
__device__ __forceinline__ void cell_faces(const double q0[4], const double dm[4], const double dp[4], bool want_lo,
                                           bool want_hi, State& lo, State& hi, double invEc_known = 0.0,
                                           double Ec2_known = 0.0, double F2c_known = 0.0, int fix = 0, double rdx = 0.0) {
    double hlo[4], hhi[4];  // U at the lower face = q0 - hlo, at the upper face = q0 + hhi
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (LIMO3) {
            const double eta = rdx > 0.0 ? limo3_eta(dm[q], dp[q], rdx) : -1.0;
            hhi[q] = 0.5 * limo3_times(dm[q], dp[q], eta);
            hlo[q] = 0.5 * limo3_times(dp[q], dm[q], eta);
        } else {
            hlo[q] = hhi[q] = half_slope(dm[q], dp[q]);
        }
    }
    const double Ec = q0[0];
    const double Ec2 = KNOWN ? Ec2_known : Ec * Ec;
    const double F2c = KNOWN ? F2c_known : fma(q0[3], q0[3], fma(q0[2], q0[2], q0[1] * q0[1]));
    const double invEc = KNOWN ? invEc_known : frcp(Ec);
    if (want_lo) {
#pragma unroll
        for (int q = 0; q < 4; ++q) lo.U[q] = q0[q] - hlo[q];
        double E2f, F2f;
        if (fix == 0) fpreserve(lo, q0, -hlo[0], invEc, Ec2, F2c, E2f, F2f);
        else facefix_variant(fix, lo, q0, Ec2, F2c, E2f, F2f);
        flux_and_speeds<D, HLL>(lo, E2f, F2f);
    }
    if (want_hi) {
#pragma unroll
        for (int q = 0; q < 4; ++q) hi.U[q] = q0[q] + hhi[q];
        double E2f, F2f;
        if (fix == 0) fpreserve(hi, q0, hhi[0], invEc, Ec2, F2c, E2f, F2f);
        else facefix_variant(fix, hi, q0, Ec2, F2c, E2f, F2f);
        flux_and_speeds<D, HLL>(hi, E2f, F2f);
    }
}

}  // namespace rtm1
