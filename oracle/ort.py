"""ctypes wrapper of the CPU ORACLE (oracle/ort.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the CUDA
package and the CUDA package imports nothing from here.

All arrays are numpy float64, C-contiguous, ghosted as ort.h describes (shape (nt3, nt2, nt1)).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libort.so")
_lib = None

CARTESIAN, CYLINDRICAL, SPHERICAL = 0, 1, 2
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT, BC_FIXED = 0, 1, 2, 3
SOLVER_HLL, SOLVER_GLF, SOLVER_RUSANOV = 0, 1, 2
FIX_FPRESERVING, FIX_PLUTO, FIX_CLIP = 0, 1, 2
RECON_PLM, RECON_LIMO3 = 0, 1
OPAC_PLANCK, OPAC_ROSSELAND, OPAC_SCATTER = 0, 1, 2

_dp = C.POINTER(C.c_double)


class Params(C.Structure):
    _fields_ = [("chat", C.c_double), ("c", C.c_double), ("a_R", C.c_double), ("c_v", C.c_double),
                ("E_floor", C.c_double), ("solver", C.c_int32), ("thick_limit", C.c_int32),
                ("feedback_momentum", C.c_int32)]


class Opacity(C.Structure):
    _fields_ = [("kind", C.c_int32), ("kappa0", C.c_double), ("rho0", C.c_double), ("T0", C.c_double),
                ("a", C.c_double), ("b", C.c_double), ("kmin", C.c_double), ("kmax", C.c_double),
                ("n_lrho", C.c_int32), ("n_lT", C.c_int32), ("lrho_min", C.c_double), ("lrho_max", C.c_double),
                ("lT_min", C.c_double), ("lT_max", C.c_double), ("rho_unit", C.c_double), ("T_unit", C.c_double),
                ("log10_kappa", _dp)]


def build(force=False):
    """Compile oracle/ort.c -> oracle/libort.so (gcc -O2 -ffp-contract=off -fopenmp)."""
    src = os.path.join(_HERE, "ort.c")
    hdr = os.path.join(_HERE, "ort.h")
    if (not force and os.path.exists(_LIB_PATH)
            and os.path.getmtime(_LIB_PATH) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _LIB_PATH
    tmp = _LIB_PATH + ".tmp%d" % os.getpid()
    subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
                           src, "-o", tmp, "-lm"])
    os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB_PATH)
        L.ort_eddington_factor.restype = C.c_double
        L.ort_eddington_factor.argtypes = [C.c_double]
        L.ort_vanleer_slope.restype = C.c_double
        L.ort_vanleer_slope.argtypes = [C.c_double] * 3
        L.ort_opacity_eval.restype = C.c_double
        L.ort_opacity_eval.argtypes = [C.POINTER(Opacity), C.c_double, C.c_double]
        L.ort_pressure_tensor.restype = None
        L.ort_pressure_tensor.argtypes = [C.c_double, _dp, _dp]
        L.ort_wave_speeds.restype = None
        L.ort_wave_speeds.argtypes = [C.c_double, _dp, C.c_int32, _dp]
        L.ort_fpreserving_face.restype = None
        L.ort_fpreserving_face.argtypes = [_dp, _dp, _dp]
        L.ort_pluto_face.restype = None
        L.ort_pluto_face.argtypes = [_dp, _dp, _dp]
        L.ort_clip_face.restype = None
        L.ort_clip_face.argtypes = [_dp, _dp]
        L.ort_limo3_faces.restype = None
        L.ort_limo3_faces.argtypes = [C.c_double] * 5 + [_dp, _dp]
        L.ort_set_reconstruction.restype = C.c_int32
        L.ort_set_reconstruction.argtypes = [C.c_void_p, C.c_int32, C.c_double]
        L.ort_set_face_fix.restype = C.c_int32
        L.ort_set_face_fix.argtypes = [C.c_void_p, C.c_int32]
        L.ort_riemann_flux.restype = None
        L.ort_riemann_flux.argtypes = [_dp, _dp, C.c_int32, C.c_double, C.c_int32, C.c_double, _dp]
        L.ort_implicit_cell.restype = None
        L.ort_implicit_cell.argtypes = [C.POINTER(Params), C.c_double, C.c_double, C.c_double, C.c_double,
                                        _dp, _dp, _dp, _dp, C.c_double]
        L.ort_irradiation_radial.restype = C.c_int32
        L.ort_irradiation_radial.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, _dp, _dp, _dp]
        L.ort_set_irradiation.restype = C.c_int32
        L.ort_set_irradiation.argtypes = [C.c_void_p, _dp]
        L.ort_grid_create.argtypes = [C.c_int32, C.POINTER(C.c_int32), C.c_int32, _dp, _dp, _dp,
                                      C.POINTER(C.c_int32), C.POINTER(C.c_void_p)]
        L.ort_grid_destroy.argtypes = [C.c_void_p]
        L.ort_grid_get_metrics.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
        L.ort_set_params.argtypes = [C.c_void_p, C.POINTER(Params)]
        L.ort_set_opacity.argtypes = [C.c_void_p, C.c_int32, C.POINTER(Opacity)]
        L.ort_explicit_step.argtypes = [C.c_void_p, C.c_double, _dp, _dp, C.POINTER(_dp), C.POINTER(_dp)]
        L.ort_implicit_step.argtypes = [C.c_void_p, C.c_double, _dp, _dp, C.POINTER(_dp), C.POINTER(_dp)]
        L.ort_cfl_dt.argtypes = [C.c_void_p, C.POINTER(_dp), C.c_double, _dp]
        L.ort_fill_ghosts.argtypes = [C.c_void_p, C.POINTER(_dp)]
        L.ort_get_floor_counts.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.ort_set_num_threads.argtypes = [C.c_int32]
        L.ort_set_num_threads.restype = None
        L.ort_get_max_threads.restype = C.c_int32
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _arr(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


def _ptrs(arrs):
    return (_dp * len(arrs))(*[_p(a) for a in arrs])


def _check64(*arrs):
    for a in arrs:
        if a is None:
            continue
        assert isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous, "float64 C array needed"


# ---------------------------------------------------------------- point-wise pieces
def eddington_factor(f):
    return lib().ort_eddington_factor(float(f))


def pressure_tensor(E, F):
    Fa = _arr(F)
    P = np.empty(9)
    lib().ort_pressure_tensor(float(E), _p(Fa), _p(P))
    return P.reshape(3, 3)


def wave_speeds(E, F, d):
    Fa = _arr(F)
    lam = np.empty(3)
    lib().ort_wave_speeds(float(E), _p(Fa), int(d), _p(lam))
    return lam


def vanleer_slope(qm, q0, qp):
    return lib().ort_vanleer_slope(float(qm), float(q0), float(qp))


def limo3_faces(um, u0, up, dx=1.0, r=0.0):
    """LimO3 (Cada & Torrilhon 2009) face values (lower, upper) of the middle cell"""
    lo, hi = np.empty(1), np.empty(1)
    lib().ort_limo3_faces(float(um), float(u0), float(up), float(dx), float(r), _p(lo), _p(hi))
    return lo[0], hi[0]


def fpreserving_face(Uc, RU):
    a, b = _arr(Uc), _arr(RU)
    out = np.empty(4)
    lib().ort_fpreserving_face(_p(a), _p(b), _p(out))
    return out


def pluto_face(Uc, RU):
    a, b = _arr(Uc), _arr(RU)
    out = np.empty(4)
    lib().ort_pluto_face(_p(a), _p(b), _p(out))
    return out


def clip_face(RU):
    b = _arr(RU)
    out = np.empty(4)
    lib().ort_clip_face(_p(b), _p(out))
    return out


def riemann_flux(UL, UR, d, chat, solver=SOLVER_HLL, lim=np.inf):
    a, b = _arr(UL), _arr(UR)
    out = np.empty(4)
    lib().ort_riemann_flux(_p(a), _p(b), int(d), float(chat), int(solver), float(lim), _p(out))
    return out


def make_params(chat=1.0, c=1.0, a_R=1.0, c_v=1.5, E_floor=0.0, solver=SOLVER_HLL, thick_limit=0,
                feedback_momentum=0):
    return Params(chat, c, a_R, c_v, E_floor, solver, thick_limit, feedback_momentum)


def make_power_law(kappa0, a=0.0, b=0.0, rho0=1.0, T0=1.0, kmin=0.0, kmax=np.inf):
    o = Opacity()
    o.kind = 0
    o.kappa0, o.rho0, o.T0, o.a, o.b, o.kmin, o.kmax = kappa0, rho0, T0, a, b, kmin, kmax
    o.rho_unit = o.T_unit = 1.0
    return o


def make_table(log10_kappa, lrho_range, lT_range, rho_unit=1.0, T_unit=1.0):
    tab = _arr(log10_kappa)
    assert tab.ndim == 2
    o = Opacity()
    o.kind = 1
    o.n_lT, o.n_lrho = tab.shape
    o.lrho_min, o.lrho_max = lrho_range
    o.lT_min, o.lT_max = lT_range
    o.rho_unit, o.T_unit = rho_unit, T_unit
    o.rho0 = o.T0 = 1.0
    o.log10_kappa = _p(tab)
    o._keep = tab
    return o


def opacity_eval(o, rho, T):
    return lib().ort_opacity_eval(C.byref(o), float(rho), float(T))


def implicit_cell(params, dt, rho, kappaP, chi, E, F, T, mom=None, Q=0.0):
    Ea, Ta, Fa = np.array([E], dtype=np.float64), np.array([T], dtype=np.float64), _arr(F).copy()
    ma = _arr(mom).copy() if mom is not None else None
    lib().ort_implicit_cell(C.byref(params), float(dt), float(rho), float(kappaP), float(chi),
                            _p(Ea), _p(Fa), _p(Ta), _p(ma), float(Q))
    return Ea[0], Fa, Ta[0], ma


# ---------------------------------------------------------------- grid object
class Grid:
    def __init__(self, geometry, n, x1f, x2f, x3f, bc, nghost=2):
        self.n = tuple(int(v) for v in n)
        self.gh = tuple(nghost if v > 1 else 0 for v in self.n)
        self.nt = tuple(v + 2 * g for v, g in zip(self.n, self.gh))
        self.shape = (self.nt[2], self.nt[1], self.nt[0])
        self.geometry = geometry
        self.xf = [_arr(x1f), _arr(x2f), _arr(x3f)]
        self.bc = tuple(int(b) for b in bc)
        n_c = (C.c_int32 * 3)(*self.n)
        bc_c = (C.c_int32 * 6)(*self.bc)
        h = C.c_void_p()
        rc = lib().ort_grid_create(int(geometry), n_c, int(nghost), _p(self.xf[0]), _p(self.xf[1]), _p(self.xf[2]),
                                   bc_c, C.byref(h))
        if rc != 0:
            raise ValueError("ort_grid_create failed with status %d" % rc)
        self._h = h
        self._keep = []

    def __del__(self):
        if getattr(self, "_h", None):
            lib().ort_grid_destroy(self._h)
            self._h = None

    @property
    def interior(self):
        return tuple(slice(g, g + n) for g, n in zip(self.gh[::-1], self.n[::-1]))

    def zeros(self):
        return np.zeros(self.shape, dtype=np.float64)

    def set_params(self, params):
        rc = lib().ort_set_params(self._h, C.byref(params))
        if rc != 0:
            raise ValueError("ort_set_params failed with status %d" % rc)
        self.params = params

    def set_opacity(self, which, o):
        rc = lib().ort_set_opacity(self._h, int(which), C.byref(o))
        if rc != 0:
            raise ValueError("ort_set_opacity failed with status %d" % rc)

    def metrics(self):
        n1, n2, n3 = self.n
        vol = np.empty((n3, n2, n1))
        a1 = np.empty((n3, n2, n1 + 1))
        a2 = np.empty((n3, n2 + 1, n1))
        a3 = np.empty((n3 + 1, n2, n1))
        lib().ort_grid_get_metrics(self._h, _p(vol), _p(a1), _p(a2), _p(a3))
        return vol, a1, a2, a3

    def fill_ghosts(self, U):
        _check64(*U)
        rc = lib().ort_fill_ghosts(self._h, _ptrs(U))
        assert rc == 0

    def explicit_step(self, dt, rho, T, U_in, U_out):
        _check64(rho, T, *U_in, *U_out)
        rc = lib().ort_explicit_step(self._h, float(dt), _p(rho), _p(T), _ptrs(U_in), _ptrs(U_out))
        if rc != 0:
            raise ValueError("ort_explicit_step failed with status %d" % rc)

    def implicit_step(self, dt, rho, T, mom, U):
        _check64(rho, T, *U)
        if mom is not None:
            _check64(*mom)
        rc = lib().ort_implicit_step(self._h, float(dt), _p(rho), _p(T), _ptrs(mom) if mom is not None else None,
                                     _ptrs(U))
        if rc != 0:
            raise ValueError("ort_implicit_step failed with status %d" % rc)

    def set_reconstruction(self, kind, r=0.0):
        """RECON_PLM (van Leer, default) or RECON_LIMO3 with its asymptotic-region radius r (<= 0: limiter alone)"""
        rc = lib().ort_set_reconstruction(self._h, int(kind), float(r))
        if rc != 0:
            raise ValueError("ort_set_reconstruction failed with status %d" % rc)

    def set_face_fix(self, mode):
        """FIX_FPRESERVING (Eq. 19-21, default), FIX_PLUTO (flat fallback, L136) or FIX_CLIP (Eq. 36-38)"""
        rc = lib().ort_set_face_fix(self._h, int(mode))
        if rc != 0:
            raise ValueError("ort_set_face_fix failed with status %d" % rc)

    def irradiation_radial(self, L0, kappa_irr, tau_in, rho):
        """gray Eq. 47-48 along x1 rays: returns (tau at each cell's upper face, div F_irr), ghosted arrays, zero outside
        the interior"""
        _check64(rho)
        tau, div = self.zeros(), self.zeros()
        rc = lib().ort_irradiation_radial(self._h, float(L0), float(kappa_irr), float(tau_in), _p(rho), _p(tau), _p(div))
        if rc != 0:
            raise ValueError("ort_irradiation_radial failed with status %d" % rc)
        return tau, div

    def set_irradiation(self, div_firr):
        """div F_irr per cell (ghosted float64 array, kept alive by this object) or None (Sect. 2.9, Eq. 34-35)"""
        if div_firr is not None:
            _check64(div_firr)
        self._div_firr = div_firr
        rc = lib().ort_set_irradiation(self._h, _p(div_firr) if div_firr is not None else None)
        if rc != 0:
            raise ValueError("ort_set_irradiation failed with status %d" % rc)

    def cfl_dt(self, U, cfl):
        _check64(*U)
        out = np.empty(1)
        rc = lib().ort_cfl_dt(self._h, _ptrs(U), float(cfl), _p(out))
        if rc != 0:
            raise ValueError("ort_cfl_dt failed with status %d" % rc)
        return float(out[0])

    def floor_counts(self):
        a, b = C.c_int64(), C.c_int64()
        lib().ort_get_floor_counts(self._h, C.byref(a), C.byref(b))
        return a.value, b.value


def set_num_threads(n):
    lib().ort_set_num_threads(int(n))


def max_threads():
    return int(lib().ort_get_max_threads())


# ---------------------------------------------------------------- driving a described workload (rt_workloads)
def opacity_from_spec(spec):
    if spec["kind"] == "power":
        return make_power_law(spec["kappa0"], spec["a"], spec["b"], spec["rho0"], spec["T0"], spec["kmin"],
                              spec["kmax"])
    return make_table(spec["log10_kappa"], spec["lrho_range"], spec["lT_range"], spec["rho_unit"], spec["T_unit"])


def grid_from_workload(w):
    g = Grid(w.geometry, w.n, w.xf[0], w.xf[1], w.xf[2], w.bc)
    g.set_params(make_params(**w.params))
    for which, spec in w.opacities.items():
        g.set_opacity(which, opacity_from_spec(spec))
    return g


def run_substeps(g, w, nsub, dts=None, state=None):
    """nsub sub-steps (explicit + implicit [+ CFL when dts is None]) of workload w on grid g.
    Returns (U, T, mom, dts).  `state` = (U, T, mom) continues an earlier run; inputs are not modified."""
    if state is None:
        U = [a.copy() for a in w.U]
        T = w.T.copy()
        mom = [a.copy() for a in w.mom] if w.mom is not None else None
    else:
        U, T, mom = state
    U2 = [a.copy() for a in U]  # ghosts of FIXED boundaries must exist in both buffers
    used = []
    for s in range(nsub):
        p = make_params(**dict(w.params, solver=w.solver_at(s)))
        g.set_params(p)
        dt = float(dts[s]) if dts is not None else g.cfl_dt(U, w.cfl)
        used.append(dt)
        g.explicit_step(dt, w.rho, T, U, U2)
        g.implicit_step(dt, w.rho, T, mom, U2)
        U, U2 = U2, U
    return U, T, mom, used


def run_rk2(g, w, nsteps, t_end=None):
    """nsteps RK2 steps (two Euler sub-steps and the average of every evolved variable; DESIGN.md
    R-G10) of workload w on grid g, each with the CFL time step of its starting state.  With t_end the run instead stops
    at that time (the last step shortened to land on it; nsteps is then ignored).  Returns (U, T, mom, dts)."""
    U = [a.copy() for a in w.U]
    T = w.T.copy()
    mom = [a.copy() for a in w.mom] if w.mom is not None else None
    U1 = [a.copy() for a in U]   # ghosts of FIXED boundaries must exist in every buffer
    U2 = [a.copy() for a in U]
    it = g.interior
    g.set_params(make_params(**w.params))
    used = []
    t = 0.0
    while (len(used) < nsteps) if t_end is None else (t < t_end - 1e-12):
        dt = g.cfl_dt(U, w.cfl)
        if t_end is not None:
            dt = min(dt, t_end - t)
        used.append(dt)
        t += dt
        T0 = T.copy()
        m0 = [a.copy() for a in mom] if mom is not None else None
        g.explicit_step(dt, w.rho, T, U, U1)
        g.implicit_step(dt, w.rho, T, mom, U1)
        g.explicit_step(dt, w.rho, T, U1, U2)
        g.implicit_step(dt, w.rho, T, mom, U2)
        for q in range(4):
            U[q][it] = 0.5 * (U[q][it] + U2[q][it])
        T[it] = 0.5 * (T0[it] + T[it])
        if mom is not None and w.params["feedback_momentum"]:
            for q in range(3):
                mom[q][it] = 0.5 * (m0[q][it] + mom[q][it])
    return U, T, mom, used
