"""Brute-force, index-free restatement of one radiation sub-step for TINY grids (<= ~6^3 cells).

TEST INFRASTRUCTURE (part of the oracle's own pinning): a second, deliberately different writing of
PAPER.md Sect. 2.4-2.8 used to catch indexing / layout / sign slips in oracle/ort.c:
  * cells live in a dict keyed by (i, j, k); there are NO ghost cells and no strides: a neighbour
    outside the domain is resolved by modular arithmetic (periodic), index clamping (outflow),
    mirroring with the normal flux negated (reflect) or a caller-supplied dict (fixed);
  * every cell sums the fluxes through its own six faces, evaluated face by face on demand;
  * vectors are tuples, the closure is written with explicit unit vectors;
  * areas and volumes are written as products of exact 1-D integrals rather than 3-D formulas.
Pure Python floats (IEEE double).  It shares no code with ort.c and none with the CUDA path.
"""
import math

CART, CYL, SPH = 0, 1, 2
PERIODIC, OUTFLOW, REFLECT, FIXED = 0, 1, 2, 3
HLL, GLF = 0, 1


def xi_of(f):                                    # Eq. 13 (L75)
    return (3.0 + 4.0 * f * f) / (5.0 + 2.0 * math.sqrt(4.0 - 3.0 * f * f))


def closure(E, F):                               # Eq. 11-14 (L69-79) -> 3x3 nested tuple
    nF = math.sqrt(sum(c * c for c in F))
    f = min(nF / E, 1.0)
    xi = xi_of(f)
    nhat = tuple(c / nF for c in F) if nF > 0.0 else (0.0, 0.0, 0.0)
    return tuple(tuple(E * (0.5 * (1.0 - xi) * (1.0 if a == b else 0.0) + 0.5 * (3.0 * xi - 1.0) * nhat[a] * nhat[b])
                       for b in range(3)) for a in range(3))


def lam13(E, F, d):                              # Eq. 22, 24 (L156-162)
    nF = math.sqrt(sum(c * c for c in F))
    f = min(nF / E, 1.0)
    mu = F[d] / nF if nF > 0.0 else 0.0
    root = math.sqrt(4.0 - 3.0 * f * f)
    z2 = 2.0 / 3.0 * (4.0 - 3.0 * f * f - root) + 2.0 * mu * mu * (2.0 - f * f - root)
    z = math.sqrt(max(z2, 0.0))
    return (f * mu - z) / root, (f * mu + z) / root


def limited_slope(a, b, c):                      # van Leer (L132, R-G3)
    lo, hi = b - a, c - b
    return 2.0 * lo * hi / (lo + hi) if lo * hi > 0.0 else 0.0


def face_state(Um, U0, Up, sign, fix=0):         # Eq. 17-21 (L128-146); sign = +1 upper face, -1 lower face
    R = tuple(U0[q] + sign * 0.5 * limited_slope(Um[q], U0[q], Up[q]) for q in range(4))
    F2f = R[1] ** 2 + R[2] ** 2 + R[3] ** 2
    if fix == 1:                                 # "PLUTO reconstruction" (L136): flat where ||R(F)|| > R(E)
        return tuple(U0) if F2f > R[0] ** 2 else R
    if fix == 2:                                 # Eq. 36-38 (L272-279): rescale R(F) onto ||F_f|| = R(E)
        if F2f <= R[0] ** 2:
            return R
        return (R[0],) + tuple(R[q] * R[0] / math.sqrt(F2f) for q in (1, 2, 3))
    F2c = U0[1] ** 2 + U0[2] ** 2 + U0[3] ** 2
    if F2f <= R[0] ** 2 and F2f * U0[0] ** 2 > F2c * R[0] ** 2:
        return R
    return (R[0],) + tuple(U0[q] * R[0] / U0[0] for q in (1, 2, 3))


def phys_flux(U, d, chat):                       # Eq. 5-6 (L49-51)
    P = closure(U[0], U[1:])
    return (chat * U[1 + d], chat * P[0][d], chat * P[1][d], chat * P[2][d])


def riemann(UL, UR, d, chat, solver, lim):       # L150, Eq. 25-26
    FL, FR = phys_flux(UL, d, chat), phys_flux(UR, d, chat)
    if solver == GLF:
        al = min(chat, lim)
        return tuple(0.5 * (FL[q] + FR[q]) - 0.5 * al * (UR[q] - UL[q]) for q in range(4))
    l1L, l3L = lam13(UL[0], UL[1:], d)
    l1R, l3R = lam13(UR[0], UR[1:], d)
    SL = max(chat * min(l1L, l1R, 0.0), -lim)
    SR = min(chat * max(l3L, l3R, 0.0), lim)
    if SR - SL > 0.0:
        return tuple((SR * FL[q] - SL * FR[q] + SR * SL * (UR[q] - UL[q])) / (SR - SL) for q in range(4))
    return tuple(0.5 * (FL[q] + FR[q]) for q in range(4))


class Brute:
    def __init__(self, geometry, edges, bc, params, opac_fn, fixed=None):
        """edges: three lists of cell edges; bc: 6 kinds; params: dict(chat,c,a_R,c_v,E_floor,solver,
        thick_limit, feedback_momentum); opac_fn(rho,T) -> (kappa_P, kappa_R, sigma);
        fixed: dict (i,j,k) -> U tuple for out-of-domain cells behind FIXED boundaries."""
        self.geo, self.x, self.bc, self.p, self.opac, self.fixed = geometry, edges, bc, params, opac_fn, fixed or {}
        self.n = tuple(len(e) - 1 for e in edges)
        self.active = tuple(m > 1 for m in self.n)

    # ---- neighbour resolution without ghost cells
    def resolve(self, key):
        """-> (interior key or None, flip vector); flips record which normal flux components change sign"""
        key = list(key)
        flip = [1.0, 1.0, 1.0]
        for d in range(3):
            m = self.n[d]
            if 0 <= key[d] < m:
                continue
            side = 0 if key[d] < 0 else 1
            kind = self.bc[2 * d + side]
            if kind == PERIODIC:
                key[d] %= m
            elif kind == OUTFLOW:
                key[d] = 0 if side == 0 else m - 1
            elif kind == REFLECT:
                key[d] = -1 - key[d] if side == 0 else 2 * m - 1 - key[d]
                flip[d] = -flip[d]
            else:
                return None, flip
        return tuple(key), flip

    def state(self, U, key):
        k2, flip = self.resolve(key)
        if k2 is None:
            return self.fixed[tuple(key)]
        u = U[k2]
        return (u[0], u[1] * flip[0], u[2] * flip[1], u[3] * flip[2])

    # ---- geometry as products of exact 1-D integrals
    def _w(self, d, lo, hi):
        """1-D volume weight of [lo,hi] along d"""
        if self.geo == CYL and d == 0:
            return 0.5 * (hi * hi - lo * lo)
        if self.geo == SPH and d == 0:
            return (hi ** 3 - lo ** 3) / 3.0
        if self.geo == SPH and d == 1:
            return math.cos(lo) - math.cos(hi)
        return hi - lo

    def volume(self, key):
        return math.prod(self._w(d, self.x[d][key[d]], self.x[d][key[d] + 1]) for d in range(3))

    def area(self, d, key):
        """area of the lower d-face of cell `key` (key[d] may be n[d])"""
        x1, x2, x3 = self.x
        i, j, k = key
        if self.geo == CART:
            return math.prod(self.x[a][key[a] + 1] - self.x[a][key[a]] for a in range(3) if a != d)
        if self.geo == CYL:
            if d == 0:
                return x1[i] * (x2[j + 1] - x2[j]) * (x3[k + 1] - x3[k])
            if d == 1:
                return (x1[i + 1] - x1[i]) * (x3[k + 1] - x3[k])
            return 0.5 * (x1[i + 1] ** 2 - x1[i] ** 2) * (x2[j + 1] - x2[j])
        if d == 0:
            return x1[i] ** 2 * (math.cos(x2[j]) - math.cos(x2[j + 1])) * (x3[k + 1] - x3[k])
        if d == 1:
            return 0.5 * (x1[i + 1] ** 2 - x1[i] ** 2) * math.sin(x2[j]) * (x3[k + 1] - x3[k])
        return 0.5 * (x1[i + 1] ** 2 - x1[i] ** 2) * (x2[j + 1] - x2[j])

    def length(self, d, key):
        i, j, k = key
        dx = [self.x[a][key[a] + 1] - self.x[a][key[a]] for a in range(3)]
        if self.geo == CART or d == 0:
            return dx[d]
        rc = 0.5 * (self.x[0][i] + self.x[0][i + 1])
        if self.geo == CYL:
            return rc * dx[1] if d == 1 else dx[2]
        if d == 1:
            return rc * dx[1]
        return rc * math.sin(0.5 * (self.x[1][j] + self.x[1][j + 1])) * dx[2]

    def tau(self, rho, T, key):
        k2, _ = self.resolve(key)
        if k2 is None:  # behind a FIXED boundary: nearest interior cell (R-G7)
            k2 = tuple(min(max(key[d], 0), self.n[d] - 1) for d in range(3))
        kP, kR, sg = self.opac(rho[k2], T[k2])
        ext = max(self.length(d, k2) for d in range(3) if self.active[d])
        return rho[k2] * (kR + sg) * ext

    # ---- one face
    def face_flux(self, U, rho, T, d, key):
        """flux through the lower d-face of cell `key`"""
        e = tuple(1 if a == d else 0 for a in range(3))
        sh = lambda s: tuple(key[a] + s * e[a] for a in range(3))
        A_mm, A_m, A_0, A_p = (self.state(U, sh(s)) for s in (-2, -1, 0, 1))
        fix = self.p.get("face_fix", 0)
        UL = face_state(A_mm, A_m, A_0, +1.0, fix)
        UR = face_state(A_m, A_0, A_p, -1.0, fix)
        lim = math.inf
        if self.p["thick_limit"]:
            tf = min(self.tau(rho, T, sh(-1)), self.tau(rho, T, key))
            lim = 4.0 * self.p["chat"] / (3.0 * tf) if tf > 0.0 else math.inf
        return riemann(UL, UR, d, self.p["chat"], self.p["solver"], lim)

    # ---- steps
    def explicit(self, U, rho, T, dt):
        out = {}
        chat = self.p["chat"]
        for key, u in U.items():
            V = self.volume(key)
            acc = list(u)
            for d in range(3):
                if not self.active[d]:
                    continue
                up = tuple(key[a] + (1 if a == d else 0) for a in range(3))
                Fm, Fp = self.face_flux(U, rho, T, d, key), self.face_flux(U, rho, T, d, up)
                Am, Ap = self.area(d, key), self.area(d, up)
                for q in range(4):
                    acc[q] -= dt * (Ap * Fp[q] - Am * Fm[q]) / V
            if self.geo != CART:
                P = closure(u[0], u[1:])
                r0, r1 = self.x[0][key[0]], self.x[0][key[0] + 1]
                if self.geo == CYL:
                    ir = (r1 - r0) / (0.5 * (r1 * r1 - r0 * r0))
                    acc[1] += dt * chat * P[1][1] * ir
                    acc[2] -= dt * chat * P[0][1] * ir
                else:
                    ir = 0.5 * (r1 * r1 - r0 * r0) / ((r1 ** 3 - r0 ** 3) / 3.0)
                    t0, t1 = self.x[1][key[1]], self.x[1][key[1] + 1]
                    ct = (math.sin(t1) - math.sin(t0)) / (math.cos(t0) - math.cos(t1))
                    acc[1] += dt * chat * (P[1][1] + P[2][2]) * ir
                    acc[2] += dt * chat * (-P[0][1] + ct * P[2][2]) * ir
                    acc[3] += dt * chat * (-P[0][2] - ct * P[1][2]) * ir
            out[key] = tuple(acc)
        return out

    def implicit(self, U, rho, T, mom, dt):
        """returns new (U, T, mom) dicts; Eq. 33 solved by Cramer's rule on the matrix AS PRINTED"""
        p = self.p
        Un, Tn, mn = {}, {}, {}
        for key, u in U.items():
            E = max(u[0], p["E_floor"])
            F = list(u[1:])
            nF = math.sqrt(sum(c * c for c in F))
            if nF > E:
                F = [c * E / nF for c in F]
            kP, kR, sg = self.opac(rho[key], T[key])
            gr, ga, Cv = dt * p["chat"] * kP * rho[key], dt * p["c"] * kP * rho[key], rho[key] * p["c_v"]
            aT3 = p["a_R"] * T[key] ** 3
            a11, a12 = 1.0 + gr, -4.0 * gr * aT3
            a21, a22 = -ga, Cv + 4.0 * ga * aT3
            b1, b2 = E - 3.0 * gr * aT3 * T[key], Cv * T[key] + 3.0 * ga * aT3 * T[key]
            det = a11 * a22 - a12 * a21
            En, Tnew = (b1 * a22 - a12 * b2) / det, (a11 * b2 - a21 * b1) / det
            Fn = [c / (1.0 + dt * p["chat"] * (kR + sg) * rho[key]) for c in F]
            if mom is not None and p["feedback_momentum"]:
                mn[key] = tuple(mom[key][q] - (Fn[q] - F[q]) / p["chat"] for q in range(3))
            Un[key], Tn[key] = (En,) + tuple(Fn), Tnew
        return Un, Tn, (mn if mom is not None and p["feedback_momentum"] else mom)

    def cfl_dt(self, U, cfl):
        worst = 0.0
        for key, u in U.items():
            s = 0.0
            for d in range(3):
                if self.active[d]:
                    l1, l3 = lam13(u[0], u[1:], d)
                    s += self.p["chat"] * max(abs(l1), abs(l3)) / self.length(d, key)
            worst = max(worst, s)
        return cfl / worst
