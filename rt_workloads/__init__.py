"""Seeded synthetic inputs shared by the CPU oracle and the CUDA path.

This module holds NONE of the method's arithmetic: it only draws random numbers
(numpy.random.Generator(PCG64(seed))), shapes them into initial fields and describes a run
(geometry, edges, boundary kinds, parameters, opacity laws/tables).  Both sides translate the
plain-Python description into their own C structs.

The paper measured on its own test problems (Sect. 3-4) and on RADMC3D-derived opacity
tables (L375) that are not available here; these workloads take their shapes, sizes, value ranges
and structure only (BASELINE.json configs 1-5, SURVEY.md Sect. 8(d)).
"""
from dataclasses import dataclass, field

import numpy as np

SEED0 = 2606_26268

CARTESIAN, CYLINDRICAL, SPHERICAL = 0, 1, 2
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT, BC_FIXED = 0, 1, 2, 3
SOLVER_HLL, SOLVER_GLF, SOLVER_RUSANOV = 0, 1, 2
RECON_PLM, RECON_LIMO3 = 0, 1  # reconstruction of the explicit half (rt_set_reconstruction / ort_set_reconstruction)
FIX_FPRESERVING, FIX_PLUTO, FIX_CLIP = 0, 1, 2  # face fix of the explicit half (rt_set_face_fix / ort_set_face_fix)
OPAC_PLANCK, OPAC_ROSSELAND, OPAC_SCATTER = 0, 1, 2
NGHOST = 2


@dataclass
class Workload:
    name: str
    geometry: int
    n: tuple                      # interior cells (n1, n2, n3)
    xf: list                      # three edge arrays (n_d + 1)
    bc: tuple                     # (x1lo, x1hi, x2lo, x2hi, x3lo, x3hi)
    params: dict                  # chat, c, a_R, c_v, E_floor, solver, thick_limit, feedback_momentum
    opacities: dict               # which -> {"kind": "power", ...} | {"kind": "table", ...}
    U: list                       # [E, F1, F2, F3], ghosted (nt3, nt2, nt1) float64
    rho: np.ndarray
    T: np.ndarray
    mom: list = None              # [m1, m2, m3] or None
    nsub: int = 1
    cfl: float = 0.4
    solver_schedule: tuple = None  # per-sub-step solver sequence (cycled); None = params["solver"]
    notes: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def gh(self):
        return tuple(NGHOST if v > 1 else 0 for v in self.n)

    @property
    def shape(self):
        return tuple(v + 2 * g for v, g in zip(self.n[::-1], self.gh[::-1]))

    @property
    def interior(self):
        return tuple(slice(g, g + v) for g, v in zip(self.gh[::-1], self.n[::-1]))

    @property
    def ncells(self):
        return int(self.n[0]) * int(self.n[1]) * int(self.n[2])

    def solver_at(self, step):
        if self.solver_schedule:
            return self.solver_schedule[step % len(self.solver_schedule)]
        return self.params["solver"]


def power_law(kappa0, a=0.0, b=0.0, rho0=1.0, T0=1.0, kmin=0.0, kmax=np.inf):
    return dict(kind="power", kappa0=float(kappa0), a=float(a), b=float(b), rho0=float(rho0), T0=float(T0),
                kmin=float(kmin), kmax=float(kmax))


def table(log10_kappa, lrho_range, lT_range, rho_unit=1.0, T_unit=1.0):
    return dict(kind="table", log10_kappa=np.ascontiguousarray(log10_kappa, dtype=np.float64),
                lrho_range=tuple(map(float, lrho_range)), lT_range=tuple(map(float, lT_range)),
                rho_unit=float(rho_unit), T_unit=float(T_unit))


def default_params(**kw):
    p = dict(chat=1.0, c=1.0, a_R=1.0, c_v=1.5, E_floor=1e-300, solver=SOLVER_HLL, thick_limit=0,
             feedback_momentum=0)
    p.update(kw)
    return p


def ghosted_shape(n):
    return tuple(v + (2 * NGHOST if v > 1 else 0) for v in n[::-1])


def interior_slices(n):
    return tuple(slice(NGHOST if v > 1 else 0, (NGHOST if v > 1 else 0) + v) for v in n[::-1])


def embed(n, interior_values, fill=0.0):
    """ghosted array with `interior_values` (shape n3,n2,n1 or broadcastable) in the interior"""
    a = np.full(ghosted_shape(n), fill, dtype=np.float64)
    a[interior_slices(n)] = interior_values
    return a


def embed_edge(n, interior_values):
    """ghosted array whose ghosts replicate the nearest interior value (for rho, T: never read, but finite)"""
    pads = [(NGHOST, NGHOST) if v > 1 else (0, 0) for v in n[::-1]]
    return np.ascontiguousarray(np.pad(np.asarray(interior_values, dtype=np.float64).reshape(n[::-1]), pads,
                                       mode="edge"))


def centres(xf):
    xf = np.asarray(xf, dtype=np.float64)
    return 0.5 * (xf[1:] + xf[:-1])


# --------------------------------------------------------------------------- random fields
def gaussian_random_field(rng, n, slope):
    """periodic Gaussian random field on an n = (n1,n2,n3) grid: white noise -> FFT -> amplitude
    proportional to k^slope (k = 0 removed) -> unit variance.  slope = -11/6 gives the shell
    spectrum k^(-5/3) in 3-D."""
    shape = n[::-1]
    w = rng.standard_normal(shape)
    wk = np.fft.rfftn(w)
    ks = [np.fft.fftfreq(s) * s for s in shape[:-1]] + [np.fft.rfftfreq(shape[-1]) * shape[-1]]
    kk = np.sqrt(sum(np.square(k).reshape([-1 if a == i else 1 for a in range(len(shape))])
                     for i, k in enumerate(ks)))
    amp = np.zeros_like(kk)
    nz = kk > 0
    amp[nz] = kk[nz] ** slope
    g = np.fft.irfftn(wk * amp, s=shape, axes=(0, 1, 2))
    g -= g.mean()
    g /= g.std()
    return g


def solenoidal_field(rng, n, slope):
    """v = curl A with three independent random fields A (amplitude k^(slope-1)), spectral curl;
    returns (v1, v2, v3) each of shape (n3,n2,n1); divergence-free by construction."""
    shape = n[::-1]
    ks = [np.fft.fftfreq(s) * s for s in shape[:-1]] + [np.fft.rfftfreq(shape[-1]) * shape[-1]]
    k3, k2, k1 = [k.reshape([-1 if a == i else 1 for a in range(3)]) for i, k in enumerate(ks)]
    kk = np.sqrt(k1 ** 2 + k2 ** 2 + k3 ** 2)
    amp = np.zeros_like(kk)
    nz = kk > 0
    amp[nz] = kk[nz] ** (slope - 1.0)
    A = [np.fft.rfftn(rng.standard_normal(shape)) * amp for _ in range(3)]  # A1, A2, A3
    v1 = np.fft.irfftn(1j * (k2 * A[2] - k3 * A[1]), s=shape, axes=(0, 1, 2))
    v2 = np.fft.irfftn(1j * (k3 * A[0] - k1 * A[2]), s=shape, axes=(0, 1, 2))
    v3 = np.fft.irfftn(1j * (k1 * A[1] - k2 * A[0]), s=shape, axes=(0, 1, 2))
    return v1, v2, v3


# --------------------------------------------------------------------------- C1: 1-D diffusion pulse / equilibration
def c1a(n1=256, nsub=100):
    """BASELINE config 1, first case: 1-D Cartesian Gaussian pulse in the diffusion regime."""
    n = (n1, 1, 1)
    xf = [np.linspace(0.0, 1.0, n1 + 1), np.array([0.0, 1.0]), np.array([0.0, 1.0])]
    x = centres(xf[0])
    E = 1.0 + 10.0 * np.exp(-((x - 0.5) ** 2) / 0.01 ** 2)
    U = [embed(n, E.reshape(1, 1, n1)), embed(n, 0.0), embed(n, 0.0), embed(n, 0.0)]
    return Workload(
        name="C1a", geometry=CARTESIAN, n=n, xf=xf, bc=(BC_PERIODIC,) * 2 + (BC_OUTFLOW,) * 4,
        params=default_params(chat=100.0, c=1.0e4, thick_limit=1, E_floor=1e-12),
        opacities={OPAC_PLANCK: power_law(1.0e3), OPAC_ROSSELAND: power_law(1.0e3)},
        U=U, rho=embed(n, 1.0, fill=1.0), T=embed(n, 1.0, fill=1.0), nsub=nsub,
        notes="kappa rho L = 1e3; chat = 100 x unit signal speed (R-G18)")


def c1b(n1=256, nsub=100):
    """BASELINE config 1, second case: uniform gas/radiation out of equilibrium (T^4 = 10 E/a_R)."""
    w = c1a(n1, nsub)
    w.name = "C1b"
    w.U[0][...] = 0.0
    w.U[0][w.interior] = 1.0
    w.T[...] = 10.0 ** 0.25
    return w


# --------------------------------------------------------------------------- C2: 2-D beam / shadow
def c2(n1=512, n2=512, nsub=2000):
    n = (n1, n2, 1)
    xf = [np.linspace(0.0, 1.0, n1 + 1), np.linspace(0.0, 1.0, n2 + 1), np.array([0.0, 1.0])]
    x, y = centres(xf[0]), centres(xf[1])
    floor = 1.0e-10
    X, Y = np.meshgrid(x, y)  # (n2, n1)
    disc = (X - 0.5) ** 2 + (Y - 0.5) ** 2 < 0.1 ** 2
    rho_i = np.where(disc, 1.0e7, 1.0)
    U = [embed(n, floor, fill=floor), embed(n, 0.0), embed(n, 0.0), embed(n, 0.0)]
    # x1-lo ghosts are FIXED: the beam strip |y - 1/2| < 0.2 injects E = 1, F = (1,0,0) (f = 1)
    strip = np.abs(y - 0.5) < 0.2
    g = NGHOST
    U[0][0, g:g + n2, :g] = np.where(strip, 1.0, floor)[:, None]
    U[1][0, g:g + n2, :g] = np.where(strip, 1.0, 0.0)[:, None]
    return Workload(
        name="C2", geometry=CARTESIAN, n=n, xf=xf,
        bc=(BC_FIXED, BC_OUTFLOW, BC_OUTFLOW, BC_OUTFLOW, BC_OUTFLOW, BC_OUTFLOW),
        params=default_params(chat=1.0, c=100.0, solver=SOLVER_GLF, thick_limit=0, E_floor=floor),
        opacities={OPAC_PLANCK: power_law(1.0e-3), OPAC_ROSSELAND: power_law(1.0e-3)},
        U=U, rho=embed_edge(n, rho_i.reshape(1, n2, n1)), T=embed(n, floor ** 0.25, fill=floor ** 0.25),
        nsub=nsub, notes="kappa rho L = 1e-3 outside, 1e4 inside the disc (rho = 1e7 there)")


# --------------------------------------------------------------------------- C3 / C4: 3-D turbulent box
def _turbulent_box(name, nside, sigma, seed, planck, rosseland, nsub, schedule):
    n = (nside, nside, nside)
    rng = np.random.Generator(np.random.PCG64(seed))
    xf = [np.linspace(0.0, 1.0, nside + 1)] * 3
    g = gaussian_random_field(rng, n, -11.0 / 6.0)
    rho_i = np.exp(sigma * g - 0.5 * sigma ** 2)
    T_i = rho_i ** (2.0 / 3.0)
    T_i /= T_i.mean()
    v = solenoidal_field(rng, n, -11.0 / 6.0)
    vrms = np.sqrt(np.mean(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))
    v = [0.3 * c / vrms for c in v]
    vmax = float(np.sqrt(v[0] ** 2 + v[1] ** 2 + v[2] ** 2).max())
    chat = 100.0 * (vmax + 1.0)
    a_R = 1.0
    noise = np.clip(rng.standard_normal((4,) + n[::-1]), -3.0, 3.0)
    Eeq = a_R * T_i ** 4
    U = [embed(n, Eeq * (1.0 + 0.01 * noise[0]))] + [embed(n, 0.01 * Eeq * noise[q]) for q in (1, 2, 3)]
    mom = [embed(n, rho_i * c) for c in v]
    return Workload(
        name=name, geometry=CARTESIAN, n=n, xf=xf, bc=(BC_PERIODIC,) * 6,
        params=default_params(chat=chat, c=100.0 * chat, a_R=a_R, thick_limit=1, feedback_momentum=1,
                              E_floor=1e-30),
        opacities={OPAC_PLANCK: planck, OPAC_ROSSELAND: rosseland},
        U=U, rho=embed_edge(n, rho_i), T=embed_edge(n, T_i), mom=mom, nsub=nsub, solver_schedule=schedule,
        notes="lognormal rho (sigma_ln rho = %g), k^-5/3 fields, Kramers opacities clipped to [1e-4, 1e6]" % sigma)


def c3(nside=128, nsub=100):
    k0 = float(nside)  # kappa0 = 1/dx
    kr = power_law(k0, a=1.0, b=-3.5, kmin=1e-4, kmax=1e6)
    return _turbulent_box("C3", nside, 1.0, SEED0 + 3, dict(kr), kr, nsub, None)


def c4(nside=256, nsub=100):
    k0 = float(nside)
    kr = power_law(k0, a=1.0, b=-3.5, kmin=1e-4, kmax=1e6)
    kp = power_law(3.0 * k0, a=1.0, b=-3.0, kmin=1e-4, kmax=1e6)
    return _turbulent_box("C4", nside, 2.0, SEED0 + 4, kp, kr, nsub, (SOLVER_HLL, SOLVER_GLF))


# --------------------------------------------------------------------------- C5: 3-D spherical irradiated disc
def smooth_table(rng, n_lT=128, n_lrho=128, lrho_range=(-15.0, 0.0), lT_range=(1.0, 6.0), offset=1.5):
    """log10 kappa = Kramers-like plane + a seeded sum of 6 low-order sinusoids, clipped to [-3, 4]."""
    lr = np.linspace(lrho_range[0], lrho_range[1], n_lrho)
    lt = np.linspace(lT_range[0], lT_range[1], n_lT)
    LR, LT = np.meshgrid(lr, lt)  # (n_lT, n_lrho)
    tab = 0.6 * (LR + 12.0) - 1.0 * (LT - 3.5) + offset
    for _ in range(6):
        a = rng.uniform(0.05, 0.3)
        kx, ky = rng.integers(1, 4, size=2)
        ph = rng.uniform(0.0, 2.0 * np.pi, size=2)
        tab = tab + a * np.sin(2 * np.pi * kx * (LR - lrho_range[0]) / (lrho_range[1] - lrho_range[0]) + ph[0]) \
            * np.sin(2 * np.pi * ky * (LT - lT_range[0]) / (lT_range[1] - lT_range[0]) + ph[1])
    return np.clip(tab, -3.0, 4.0)


def c5(n=(256, 128, 256), nsub=50):
    n = tuple(n)
    n1, n2, n3 = n
    rng = np.random.Generator(np.random.PCG64(SEED0 + 5))
    xf = [np.geomspace(1.0, 100.0, n1 + 1), np.linspace(np.pi / 2 - 0.5, np.pi / 2 + 0.5, n2 + 1),
          np.linspace(0.0, 2.0 * np.pi, n3 + 1)]
    r, th = centres(xf[0]), centres(xf[1])
    R = r.reshape(1, 1, n1)
    TH = th.reshape(1, n2, 1)
    rho_i = np.maximum(R ** -1.5 * np.exp(-np.cos(TH) ** 2 / (2 * 0.1 ** 2)), 1e-6) * np.ones((n3, 1, 1))
    T_i = R ** -0.5 * np.ones((n3, n2, 1))
    vphi = R ** -0.5 * (1.0 + 0.01 * np.clip(rng.standard_normal((n3, n2, n1)), -3, 3))
    chat = 100.0 * (float(np.abs(vphi).max()) + 1.0)
    a_R = 1.0
    tabR = smooth_table(rng)
    tabP = np.clip(tabR + 0.2 + 0.1 * np.sin(np.linspace(0, 3, 128))[:, None], -3.0, 4.0)
    E0 = 10.0
    U = [embed(n, a_R * T_i ** 4), embed(n, 0.0), embed(n, 0.0), embed(n, 0.0)]
    g = NGHOST
    U[0][:, :, :g] = E0      # r-lo ghosts FIXED: central irradiation, F = E r^ (f = 1, R-G2)
    U[1][:, :, :g] = E0
    mom = [embed(n, 0.0), embed(n, 0.0), embed(n, rho_i * vphi)]
    return Workload(
        name="C5", geometry=SPHERICAL, n=n, xf=xf,
        bc=(BC_FIXED, BC_OUTFLOW, BC_OUTFLOW, BC_OUTFLOW, BC_PERIODIC, BC_PERIODIC),
        params=default_params(chat=chat, c=100.0 * chat, a_R=a_R, thick_limit=1, feedback_momentum=1,
                              E_floor=1e-30),
        opacities={OPAC_PLANCK: table(tabP, (-15.0, 0.0), (1.0, 6.0), 1e-9, 1e4),
                   OPAC_ROSSELAND: table(tabR, (-15.0, 0.0), (1.0, 6.0), 1e-9, 1e4)},
        U=U, rho=embed_edge(n, rho_i), T=embed_edge(n, T_i), mom=mom, nsub=nsub,
        notes="log-spaced r in [1,100], theta in pi/2 +- 0.5, seeded smooth 128x128 opacity tables")


# --------------------------------------------------------------------------- CP: the paper's performance workload (context)
def cp(nside=256, nsub=20):
    """3-D Cartesian optically thin pulse of PAPER.md L311-321 / L399 in code units."""
    n = (nside,) * 3
    xf = [np.linspace(-50.0, 50.0, nside + 1)] * 3
    x = centres(xf[0])
    r2 = x.reshape(1, 1, -1) ** 2 + x.reshape(1, -1, 1) ** 2 + x.reshape(-1, 1, 1) ** 2
    Tr = 1.0 + 100.0 * np.exp(-r2 / 5.0 ** 2)
    U = [embed_edge(n, Tr ** 4), embed(n, 0.0), embed(n, 0.0), embed(n, 0.0)]
    return Workload(
        name="CP", geometry=CARTESIAN, n=n, xf=xf, bc=(BC_OUTFLOW,) * 6,
        params=default_params(chat=1.0, c=1.0, E_floor=1e-30),
        opacities={OPAC_SCATTER: power_law(1.0e-4)},
        U=U, rho=embed(n, 1.0, fill=1.0), T=embed(n, 1.0, fill=1.0), nsub=nsub,
        notes="kappa = 0, sigma rho L = 1e-2, T_r = T0 (1 + 100 exp(-r^2/w^2)), w = 5")


def random_state(rng, n, fmax=1.0, emin=0.1, emax=10.0):
    """random admissible radiation state on a ghosted grid: E log-uniform, F with f uniform in [0,fmax]"""
    shape = ghosted_shape(n)
    E = np.exp(rng.uniform(np.log(emin), np.log(emax), size=shape))
    dirv = rng.standard_normal((3,) + shape)
    dirv /= np.sqrt((dirv ** 2).sum(axis=0))
    f = rng.uniform(0.0, fmax, size=shape)
    return [np.ascontiguousarray(E)] + [np.ascontiguousarray(E * f * dirv[q]) for q in range(3)]


BY_NAME = {"C1a": c1a, "C1b": c1b, "C2": c2, "C3": c3, "C4": c4, "C5": c5, "CP": cp}
