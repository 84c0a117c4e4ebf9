"""Pins of the oracle's implicit radiation-matter coupling (Eq. 29-33, 30, 27-28, 41),
opacity evaluation (L299, L375) and CFL (L120) against high-precision solves, closed forms,
invariants and a stiff ODE integration.  No CUDA here."""
import math

import mpmath
import numpy as np
import pytest
from scipy.integrate import solve_ivp
from scipy.optimize import brentq

from oracle import ort

RNG = np.random.default_rng(11)


def eq33_mpmath(p, dt, rho, kP, E, T):
    """Eq. 33 exactly as printed, solved with 50 digits."""
    mpmath.mp.dps = 50
    m = mpmath.mpf
    gr, g, Cv = m(dt) * m(p.chat) * m(kP) * m(rho), m(dt) * m(p.c) * m(kP) * m(rho), m(rho) * m(p.c_v)
    a, T, E = m(p.a_R), m(T), m(E)
    A = mpmath.matrix([[1 + gr, -4 * gr * a * T ** 3], [-g, Cv + 4 * g * a * T ** 3]])
    b = mpmath.matrix([E - 3 * gr * a * T ** 4, Cv * T + 3 * g * a * T ** 4])
    x = mpmath.lu_solve(A, b)
    return x[0], x[1]


def test_closed_form_matches_50_digit_solve_of_eq33_including_stiff_cells():
    for _ in range(300):
        p = ort.make_params(chat=10 ** RNG.uniform(0, 3), c=10 ** RNG.uniform(3, 6), a_R=10 ** RNG.uniform(-3, 3),
                            c_v=10 ** RNG.uniform(-1, 1))
        dt, rho, kP = 10 ** RNG.uniform(-6, 0), 10 ** RNG.uniform(-6, 3), 10 ** RNG.uniform(-4, 8)
        E, T = 10 ** RNG.uniform(-6, 4), 10 ** RNG.uniform(-2, 2)
        En, _, Tn, _ = ort.implicit_cell(p, dt, rho, kP, kP, E, [0, 0, 0], T)
        Ex, Tx = eq33_mpmath(p, dt, rho, kP, E, T)
        assert abs(En - Ex) / abs(Ex) < 5e-15
        assert abs(Tn - Tx) / abs(Tx) < 5e-15


def test_energy_bookkeeping_eq27_per_cell():
    # C_v T + (c/chat) E_r is unchanged by the implicit step (Eq. 27)
    for _ in range(200):
        p = ort.make_params(chat=10 ** RNG.uniform(0, 2), c=10 ** RNG.uniform(2, 4), a_R=1.0, c_v=1.5)
        dt, rho, kP = 10 ** RNG.uniform(-5, -1), 10 ** RNG.uniform(-2, 2), 10 ** RNG.uniform(-2, 4)
        E, T = 10 ** RNG.uniform(-2, 2), 10 ** RNG.uniform(-1, 1)
        En, _, Tn, _ = ort.implicit_cell(p, dt, rho, kP, kP, E, [0, 0, 0], T)
        tot0 = rho * p.c_v * T + p.c / p.chat * E
        tot1 = rho * p.c_v * Tn + p.c / p.chat * En
        assert tot1 == pytest.approx(tot0, rel=4e-15)


def test_fixed_point_iff_equilibrium_and_one_step_identity():
    p = ort.make_params(chat=100.0, c=1e4, a_R=2.0, c_v=1.5)
    T = 1.3
    Eeq = p.a_R * T ** 4
    En, _, Tn, _ = ort.implicit_cell(p, 1e-3, 0.7, 50.0, 50.0, Eeq, [0, 0, 0], T)
    assert En == pytest.approx(Eeq, rel=1e-15) and Tn == pytest.approx(T, rel=1e-15)
    # linearised departure from equilibrium shrinks by 1/(1 + g_r + 4 g a T^3/C_v)
    E = 3.0 * Eeq
    dt, rho, kP = 1e-3, 0.7, 50.0
    En, _, Tn, _ = ort.implicit_cell(p, dt, rho, kP, kP, E, [0, 0, 0], T)
    gr, g, Cv = dt * p.chat * kP * rho, dt * p.c * kP * rho, rho * p.c_v
    lhs = En - p.a_R * (T ** 4 + 4 * T ** 3 * (Tn - T))
    rhs = (E - p.a_R * T ** 4) / (1 + gr + 4 * g * p.a_R * T ** 3 / Cv)
    assert lhs == pytest.approx(rhs, rel=1e-12)


def test_absorption_only_limit_eq41():
    # a_R -> 0 removes emission: E' = E/(1 + gamma_abs,red)   (Eq. 41)
    p = ort.make_params(chat=7.0, c=700.0, a_R=0.0, c_v=1.5)
    dt, rho, kP, E = 0.01, 2.0, 30.0, 5.0
    En, _, _, _ = ort.implicit_cell(p, dt, rho, kP, kP, E, [0, 0, 0], 1.0)
    assert En == pytest.approx(E / (1 + dt * p.chat * kP * rho), rel=1e-15)


def test_flux_damping_eq30_and_momentum_eq28():
    p = ort.make_params(chat=5.0, c=500.0, feedback_momentum=1)
    dt, rho, chi = 0.02, 3.0, 11.0
    F, m = np.array([0.3, -0.2, 0.1]), np.array([1.0, 2.0, 3.0])
    _, Fn, _, mn = ort.implicit_cell(p, dt, rho, 0.0, chi, 1.0, F, 1.0, m)
    assert np.allclose(Fn, F / (1 + dt * p.chat * chi * rho), rtol=1e-15)
    assert np.allclose(mn + Fn / p.chat, m + F / p.chat, rtol=1e-15)        # Eq. 28 conserved


def test_config1b_relaxes_to_the_root_of_the_conserved_energy():
    """BASELINE config 1b: T^4 = 10 E/a_R.  Long-time limit = root of C_v T + (c/chat) a_R T^4 = const."""
    p = ort.make_params(chat=100.0, c=1e4, a_R=1.0, c_v=1.5)
    E, T, rho, kP = 1.0, 10 ** 0.25, 1.0, 1e3
    tot = rho * p.c_v * T + p.c / p.chat * E
    Teq = brentq(lambda t: rho * p.c_v * t + p.c / p.chat * p.a_R * t ** 4 - tot, 0.5, 2.0, xtol=1e-15, rtol=1e-15)
    for _ in range(60):
        E, _, T, _ = ort.implicit_cell(p, 2.7e-5, rho, kP, kP, E, [0, 0, 0], T)
    assert T == pytest.approx(Teq, rel=1e-12)
    assert E == pytest.approx(p.a_R * Teq ** 4, rel=1e-12)


def test_first_order_convergence_to_the_stiff_ode():
    """dE_r/dt = chat kappa rho (a T^4 - E_r), C_v dT/dt = c kappa rho (E_r - a T^4)  (Eq. 5, 15, 31)"""
    p = ort.make_params(chat=10.0, c=100.0, a_R=1.0, c_v=1.5)
    rho, kP, E0, T0, tend = 1.0, 2.0, 1.0, 1.5, 0.02

    def rhs(t, y):
        d = p.a_R * y[1] ** 4 - y[0]
        return [p.chat * kP * rho * d, -p.c * kP * rho * d / (rho * p.c_v)]

    sol = solve_ivp(rhs, [0, tend], [E0, T0], method="Radau", rtol=1e-12, atol=1e-14)
    Eref, Tref = sol.y[:, -1]
    errs = []
    for nstep in (400, 800, 1600, 3200):
        E, T = E0, T0
        for _ in range(nstep):
            E, _, T, _ = ort.implicit_cell(p, tend / nstep, rho, kP, kP, E, [0, 0, 0], T)
        errs.append(abs(T - Tref) + abs(E - Eref))
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    assert all(1.85 < r < 2.15 for r in ratios), (errs, ratios)


# ----------------------------------------------------------------------------- opacity
def test_power_law_against_numpy_and_clipping():
    o = ort.make_power_law(0.1, a=1.0, b=-3.5, rho0=2.0, T0=290.0, kmin=1e-4, kmax=1e6)   # Kramers, L299
    for _ in range(100):
        rho, T = 10 ** RNG.uniform(-3, 3), 10 ** RNG.uniform(1, 4)
        want = np.clip(0.1 * (rho / 2.0) * np.float64(T / 290.0) ** -3.5, 1e-4, 1e6)
        assert ort.opacity_eval(o, rho, T) == pytest.approx(want, rel=1e-14)
    assert ort.opacity_eval(o, 1e9, 1.0) == 1e6 and ort.opacity_eval(o, 1e-9, 1e6) == 1e-4
    assert ort.opacity_eval(ort.make_power_law(5.0), 3.0, 7.0) == 5.0


def test_table_reproduces_a_bilinear_in_log_function_exactly_and_clamps():
    lr = np.linspace(-15, 0, 31)
    lt = np.linspace(1, 6, 21)
    LR, LT = np.meshgrid(lr, lt)
    fn = lambda x, y: 0.4 * x - 1.3 * y + 0.05 * x * y + 2.0           # bilinear in (log rho, log T)
    o = ort.make_table(fn(LR, LT), (-15, 0), (1, 6), rho_unit=1e-3, T_unit=10.0)
    for _ in range(200):
        x, y = RNG.uniform(-15, 0), RNG.uniform(1, 6)
        got = ort.opacity_eval(o, 10 ** x / 1e-3, 10 ** y / 10.0)
        assert math.log10(got) == pytest.approx(fn(x, y), abs=1e-11)
    # clamped to the table edges
    assert math.log10(ort.opacity_eval(o, 1e10, 1e10)) == pytest.approx(fn(0, 6), abs=1e-12)
    assert math.log10(ort.opacity_eval(o, 1e-30, 1e-30)) == pytest.approx(fn(-15, 1), abs=1e-12)
    # grid nodes are returned exactly
    got = ort.opacity_eval(o, 10 ** lr[7] / 1e-3, 10 ** lt[5] / 10.0)
    assert math.log10(got) == pytest.approx(fn(lr[7], lt[5]), abs=1e-12)


def test_table_1d_in_temperature_paper_form():
    # the paper's own tables are 1-D in T (L375): n_lrho = 1
    lt = np.linspace(1, 4, 16)
    o = ort.make_table((2.0 - 0.5 * lt).reshape(-1, 1), (0, 0), (1, 4))
    for y in RNG.uniform(1, 4, 50):
        assert math.log10(ort.opacity_eval(o, 123.0, 10 ** y)) == pytest.approx(2.0 - 0.5 * y, abs=1e-12)


def test_table_piecewise_linear_between_nodes():
    # a non-linear table: the value midway between two nodes is the mean of the node values
    tab = RNG.uniform(-2, 2, (6, 5))
    o = ort.make_table(tab, (0, 4), (0, 5))
    got = ort.opacity_eval(o, 10 ** 2.5, 10 ** 3.5)
    want = 0.25 * (tab[3, 2] + tab[3, 3] + tab[4, 2] + tab[4, 3])
    assert math.log10(got) == pytest.approx(want, abs=1e-13)
    got = ort.opacity_eval(o, 10 ** 2.0, 10 ** 3.25)                      # on a rho node, 1/4 along T
    assert math.log10(got) == pytest.approx(0.75 * tab[3, 2] + 0.25 * tab[4, 2], abs=1e-13)


# ----------------------------------------------------------------------------- CFL
def _cart_grid(n, L=(1.0, 1.0, 1.0), bc=None):
    xf = [np.linspace(0, L[d], n[d] + 1) for d in range(3)]
    return ort.Grid(ort.CARTESIAN, n, xf[0], xf[1], xf[2], bc or (0,) * 6)


def test_cfl_closed_forms(golden):
    Ca = golden["courant"]["C_a"]
    n, L, chat = (8, 4, 2), (1.0, 2.0, 3.0), 7.0
    g = _cart_grid(n, L)
    g.set_params(ort.make_params(chat=chat))
    U = [g.zeros() for _ in range(4)]
    U[0][...] = 1.0
    # f = 0 everywhere: max|lambda| = 1/sqrt(3) in every direction
    inv = sum(n[d] / L[d] for d in range(3))
    assert g.cfl_dt(U, Ca) == pytest.approx(Ca * math.sqrt(3) / (chat * inv), rel=1e-14)
    # 1-D, f = 1 along x: dt = C_a dx / chat
    g = _cart_grid((16, 1, 1))
    g.set_params(ort.make_params(chat=chat))
    U = [g.zeros() for _ in range(4)]
    U[0][...] = 2.0
    U[1][...] = 2.0
    assert g.cfl_dt(U, Ca) == pytest.approx(Ca / 16 / chat, rel=1e-14)


def test_cfl_takes_the_worst_cell_and_curvilinear_lengths():
    # spherical: lengths dr, r_c dth, r_c sin(th_c) dphi (R-G9); f = 0 so the rate is geometry only
    r = np.geomspace(1, 10, 9)
    th = np.linspace(0.4, 2.0, 7)
    ph = np.linspace(0, 2 * np.pi, 5)
    g = ort.Grid(ort.SPHERICAL, (8, 6, 4), r, th, ph, (1, 1, 1, 1, 0, 0))
    g.set_params(ort.make_params(chat=1.0))
    U = [g.zeros() for _ in range(4)]
    U[0][...] = 1.0
    rc, thc = 0.5 * (r[1:] + r[:-1]), 0.5 * (th[1:] + th[:-1])
    rate = 0.0
    for i in range(8):
        for j in range(6):
            s = (1 / (r[i + 1] - r[i]) + 1 / (rc[i] * (th[1] - th[0])) + 1 / (rc[i] * math.sin(thc[j]) * (ph[1] - ph[0])))
            rate = max(rate, s / math.sqrt(3))
    assert g.cfl_dt(U, 0.4) == pytest.approx(0.4 / rate, rel=1e-14)


# ----------------------------------------------------------------------------- RK2 composition (L107, L256)
def test_rk2_composition_conserves_the_coupled_energy_and_keeps_a_uniform_state_uniform():
    """ort.run_rk2 = two Euler sub-steps at one dt and the average of E, F, T, m.  Each sub-step conserves
    C_v T + (c/chat) E per cell exactly for a uniform state (no transport), so the average does; a uniform state
    stays uniform."""
    import rt_workloads as W
    w = W.c1b()
    g = ort.grid_from_workload(w)
    p = w.params
    it = g.interior
    tot0 = w.rho[it] * p["c_v"] * w.T[it] + (p["c"] / p["chat"]) * w.U[0][it]
    U, T, mom, dts = ort.run_rk2(g, w, 5)
    tot = w.rho[it] * p["c_v"] * T[it] + (p["c"] / p["chat"]) * U[0][it]
    assert np.all(np.abs(tot - tot0) <= 1e-13 * np.abs(tot0))
    for a in (U[0][it], T[it]):
        assert np.ptp(a) <= 1e-14 * np.abs(a).max()
    assert len(dts) == 5 and all(d > 0 for d in dts)


# ----------------------------------------------------------------------------- irradiation (Sect. 2.9, Eq. 34-35)
def test_irradiation_source_is_the_solution_of_eq33_with_eq35():
    """Q = -div F_irr dt enters S_1 of Eq. 33 (Eq. 35).  Independent pin: the 2x2 system written out from
    Eq. 29-32 with the linearised T^4 and solved by numpy.linalg.solve; plus Eq. 34: the coupled energy
    C_v T + (c/chat) E grows by exactly Q, and Q = 0 changes nothing."""
    rng = np.random.default_rng(12)
    for _ in range(200):
        chat, c = np.exp(rng.uniform(0, 3)), np.exp(rng.uniform(3, 6))
        p = ort.make_params(chat=chat, c=c, a_R=np.exp(rng.uniform(-2, 2)), c_v=1.5)
        dt, rho, kP = np.exp(rng.uniform(-4, 1)), np.exp(rng.uniform(-2, 2)), np.exp(rng.uniform(-3, 3))
        E, T = np.exp(rng.uniform(-2, 2)), np.exp(rng.uniform(-1, 1))
        Q = rng.uniform(-0.2, 2.0) * rho * 1.5 * T                     # up to twice the gas energy, either sign
        gr, g, Cv, a = dt * chat * kP * rho, dt * c * kP * rho, rho * 1.5, p.a_R
        M = np.array([[1 + gr, -4 * gr * a * T ** 3], [-g, Cv + 4 * g * a * T ** 3]])
        S = np.array([E - 3 * gr * a * T ** 4, Cv * T + 3 * g * a * T ** 4 + Q])
        En_ref, Tn_ref = np.linalg.solve(M, S)
        En, _, Tn, _ = ort.implicit_cell(p, dt, rho, kP, 0.0, E, [0.0, 0.0, 0.0], T, Q=Q)
        assert En == pytest.approx(En_ref, rel=1e-11) and Tn == pytest.approx(Tn_ref, rel=1e-11)
        assert Cv * Tn + (c / chat) * En == pytest.approx(Cv * T + (c / chat) * E + Q, rel=1e-12)          # Eq. 34
        E0, _, T0, _ = ort.implicit_cell(p, dt, rho, kP, 0.0, E, [0.0, 0.0, 0.0], T)
        E1, _, T1, _ = ort.implicit_cell(p, dt, rho, kP, 0.0, E, [0.0, 0.0, 0.0], T, Q=0.0)
        assert (E0, T0) == (E1, T1)


def test_irradiation_array_reaches_the_grid_level_implicit_step():
    import rt_workloads as W
    w = W.c1b()
    g = ort.grid_from_workload(w)
    it = g.interior
    p = w.params
    div = np.zeros(g.shape)
    div[it] = -0.3 * (1.0 + np.arange(w.n[0]))[None, None, :] / w.n[0]          # heating, growing along x1
    U = [a.copy() for a in w.U]
    T = w.T.copy()
    tot0 = w.rho[it] * p["c_v"] * T[it] + (p["c"] / p["chat"]) * U[0][it]
    dt = 0.01
    g.set_irradiation(div)
    g.implicit_step(dt, w.rho, T, None, U)
    g.set_irradiation(None)
    tot1 = w.rho[it] * p["c_v"] * T[it] + (p["c"] / p["chat"]) * U[0][it]
    assert np.allclose(tot1 - tot0, -div[it] * dt, rtol=1e-10, atol=1e-13)


# ----------------------------------------------------------------------------- radial irradiation (Sect. 3.7, Eq. 47-48)
def _sph_grid(n=(40, 6, 5), rin=1.0, rout=50.0):
    xf = [np.geomspace(rin, rout, n[0] + 1), np.linspace(np.pi / 2 - 0.4, np.pi / 2 + 0.3, n[1] + 1), np.linspace(0.0, 2 * np.pi, n[2] + 1)]
    return ort.Grid(ort.SPHERICAL, n, xf[0], xf[1], xf[2], (1, 1, 1, 1, 0, 0)), xf


def test_irradiation_radial_optical_depth_is_the_analytic_integral_of_eq48():
    """rho(r) = C(theta, phi) / r^2, fed as its exact cell average in r: Eq. 48 gives tau(r) = tau_in + kappa C (1/r_in - 1/r)
    at every radial face, per ray; and the flux divergence equals [A+ F+ - A- F-]/V with F = L0 e^{-tau}/r^2 (Eq. 47, gray)
    built in numpy from the ANALYTIC tau and the oracle's quadrature-pinned face areas and volumes."""
    g, xf = _sph_grid()
    r = xf[0]
    rng = np.random.default_rng(5)
    Cray = rng.uniform(0.5, 30.0, size=(g.n[2], g.n[1], 1))
    rho = g.zeros()
    rho[g.interior] = Cray * ((1.0 / r[:-1] - 1.0 / r[1:]) / np.diff(r))[None, None, :]
    L0, kap, tau_in = 7.0, 0.8, 0.05
    tau, div = g.irradiation_radial(L0, kap, tau_in, rho)
    tau_face = tau_in + kap * Cray * (1.0 / r[0] - 1.0 / r)[None, None, :]          # all n1 + 1 faces
    assert np.allclose(tau[g.interior], tau_face[..., 1:], rtol=1e-13, atol=0)
    vol, a1, _, _ = g.metrics()
    F = L0 * np.exp(-tau_face) / r[None, None, :] ** 2
    ref = (a1[..., 1:] * F[..., 1:] - a1[..., :-1] * F[..., :-1]) / vol
    assert np.all(div[g.interior] < 0.0)
    assert np.allclose(div[g.interior], ref, rtol=2e-12, atol=0)          # the reference differences e^{-tau}: ~1e-14 / dtau
    # nothing outside the interior is written
    mask = np.ones(g.shape, bool)
    mask[g.interior] = False
    assert not div[mask].any() and not tau[mask].any()


def test_irradiation_radial_deposits_exactly_the_luminosity_it_removes():
    """sum_i div_i V_i over a ray bundle = -(L_in - L_out): the solid angle of the bundle times L0 (e^{-tau_in} - e^{-tau_out}),
    tau_out from numpy's cumulative sum; and the optically thin limit is div -> -kappa rho F_irr (the continuum equation)."""
    g, xf = _sph_grid()
    r = xf[0]
    rng = np.random.default_rng(6)
    rho = g.zeros()
    rho[g.interior] = np.exp(rng.uniform(-3, 1, size=rho[g.interior].shape))
    L0, kap, tau_in = 3.0, 0.4, 0.0
    tau, div = g.irradiation_radial(L0, kap, tau_in, rho)
    vol, _, _, _ = g.metrics()
    tau_out = tau_in + kap * np.cumsum(rho[g.interior] * np.diff(r)[None, None, :], axis=-1)[..., -1]
    omega = (np.cos(xf[1][:-1]) - np.cos(xf[1][1:]))[None, :] * np.diff(xf[2])[:, None]      # solid angle per ray
    assert (div[g.interior] * vol).sum(axis=-1) == pytest.approx(-(L0 * omega * (np.exp(-tau_in) - np.exp(-tau_out))), rel=1e-12)
    eps = 1e-9
    _, thin = g.irradiation_radial(L0, eps, 0.0, rho)
    rc2 = 3.0 * np.diff(r) / np.diff(r ** 3)                                               # <1/r^2> of a shell
    assert np.allclose(thin[g.interior], -eps * rho[g.interior] * L0 * rc2[None, None, :], rtol=1e-6, atol=0)


def test_irradiation_radial_cartesian_slab_and_errors():
    """plane-parallel rays along x1 on a Cartesian grid, uniform rho: F = L0 e^{-kappa rho x}, cell-averaged dF/dx"""
    n = (30, 3, 1)
    xf = [np.linspace(0.0, 2.0, n[0] + 1) ** 1.3, np.linspace(0, 1, n[1] + 1), np.array([0.0, 1.0])]
    g = ort.Grid(ort.CARTESIAN, n, xf[0], xf[1], xf[2], (1, 1, 0, 0, 0, 0))
    rho = np.full(g.shape, 2.5)
    tau, div = g.irradiation_radial(4.0, 1.2, 0.3, rho)
    x = xf[0]
    F = 4.0 * np.exp(-(0.3 + 1.2 * 2.5 * x))
    assert np.allclose(div[g.interior], (np.diff(F) / np.diff(x))[None, None, :], rtol=1e-12, atol=0)
    assert np.allclose(tau[g.interior], (0.3 + 3.0 * x[1:])[None, None, :], rtol=1e-14, atol=0)
    gc = ort.Grid(ort.CYLINDRICAL, (4, 4, 1), np.linspace(1, 2, 5), np.linspace(0, 1, 5), np.array([0.0, 1.0]), (1, 1, 1, 1, 0, 0))
    with pytest.raises(ValueError):
        gc.irradiation_radial(1.0, 1.0, 0.0, gc.zeros() + 1.0)
    with pytest.raises(ValueError):
        g.irradiation_radial(1.0, -1.0, 0.0, rho)
