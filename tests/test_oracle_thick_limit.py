"""Pins of the oracle's optically-thick wave-speed limit: `tau_cell` and the Eq. 25-26 wiring inside
`ort_explicit_step` (Sect. 2.6; DESIGN.md R-G7).  No CUDA here.

Every expected value below is worked out by hand IN THE TEST from the paper's statements:
  * Eq. 25-26 (L171-173): S_R = min(S_R, 4 chat/(3 tau)), S_L = max(S_L, -4 chat/(3 tau));
  * L175: tau_cell = rho chi dx of "the cell of maximum size dx" (R-G7: the cell's largest physical extent over the
    active dimensions; tau_face = the smaller tau of the two adjacent cells);
  * L150 (two-wave HLL / Lax-Friedrichs) for two f = 0 states with F = 0: the energy flux through the face is
        F*_E = -1/2 S (E_R - E_L),   S = min(chat/sqrt(3), 4 chat/(3 tau_face)),
    because the physical energy flux chat F^d vanishes on both sides and S_R = -S_L = S (L167: lambda = -+1/sqrt(3));
  * L169-175: with the limit the scheme diffuses at the physical rate D = chat/(3 chi rho); without it the HLL
    dissipation chat dx/(2 sqrt(3)) swamps D as soon as tau_cell > 1.
A mutation of ort.c:503-565 (min -> max over the two cells, largest -> smallest extent, 4/3 -> 1, limit not applied in
one direction) turns at least one of these tests red; DESIGN.md Sect. 7 lists which.
"""
import math

import numpy as np
import pytest

from oracle import ort


def _slab_grid(geometry, n, xf, bc, chat, solver, thick=1):
    g = ort.Grid(geometry, n, xf[0], xf[1], xf[2], bc)
    g.set_params(ort.make_params(chat=chat, solver=solver, thick_limit=thick, E_floor=1e-30))
    return g


# --------------------------------------------------------------------------- (b) hand-worked face flux, Cartesian
@pytest.mark.parametrize("solver", [ort.SOLVER_HLL, ort.SOLVER_GLF, ort.SOLVER_RUSANOV])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_interface_flux_between_two_slabs_on_anisotropic_cells(d, solver):
    """two slabs of different rho chi along direction d, piecewise-constant E (so every van Leer slope next to the jump
    is zero and the face states ARE the cell values), F = 0, cells 0.1 x 0.3 x 0.2: the largest extent is dy = 0.3
    whichever direction the flux crosses."""
    n = (8, 6, 4)
    dx = (0.1, 0.3, 0.2)
    xf = [np.arange(n[e] + 1) * dx[e] for e in range(3)]
    chat = 2.5
    g = _slab_grid(ort.CARTESIAN, n, xf, (0,) * 6, chat, solver)
    rho_a, rho_b = 1.0, 3.0
    k0 = 20.0                                  # sigma = k0 rho: chi = 20 in slab a, 60 in slab b
    chi_a, chi_b = k0 * rho_a, k0 * rho_b
    E_a, E_b = 2.0, 0.5
    half = n[d] // 2
    idx = np.arange(n[d])
    shape1 = [1, 1, 1]
    shape1[2 - d] = n[d]
    left = (idx < half).reshape(shape1)         # interior-shaped mask, broadcast over the other two axes
    it = g.interior
    rho, T = np.ones(g.shape), np.ones(g.shape)
    U = [g.zeros() for _ in range(4)]
    rho[it] = np.where(left, rho_a, rho_b) * np.ones(g.shape)[it]
    U[0][it] = np.where(left, E_a, E_b) * np.ones(g.shape)[it]
    g.set_opacity(ort.OPAC_SCATTER, ort.make_power_law(k0, a=1.0))
    dt = 1.0e-3
    out = [a.copy() for a in U]
    g.explicit_step(dt, rho, T, U, out)

    dmax = max(dx)
    tau_a, tau_b = rho_a * chi_a * dmax, rho_b * chi_b * dmax                     # L175, R-G7
    S = min(chat / math.sqrt(3.0), 4.0 * chat / (3.0 * min(tau_a, tau_b)))         # Eq. 25-26 + L167
    assert S < chat / math.sqrt(3.0)                                               # the clamp is active
    # interface inside the box (cells half-1 | half): flux = -1/2 S (E_b - E_a); periodic wrap (cells n-1 | 0): b -> a
    F_mid = -0.5 * S * (E_b - E_a)
    F_wrap = -0.5 * S * (E_a - E_b)
    E = np.moveaxis(out[0][it], 2 - d, 0)        # axis 0 = direction d
    exp = {half - 1: E_a - dt / dx[d] * (F_mid - 0.0), half: E_b - dt / dx[d] * (0.0 - F_mid),
           n[d] - 1: E_b - dt / dx[d] * (F_wrap - 0.0), 0: E_a - dt / dx[d] * (0.0 - F_wrap)}
    for c in range(n[d]):
        want = exp.get(c, E_a if c < half else E_b)
        assert np.allclose(E[c], want, rtol=2e-15, atol=0), (c, E[c].ravel()[0], want)
    # the normal flux component sees the plain average of the two pressures chat E/3 (F = 0 on both sides, S_R = -S_L)
    Fd = np.moveaxis(out[1 + d][it], 2 - d, 0)
    P_mid = 0.5 * chat * (E_a / 3.0 + E_b / 3.0)
    assert np.allclose(Fd[half - 1], -dt / dx[d] * (P_mid - chat * E_a / 3.0), rtol=1e-13, atol=1e-18)
    assert np.allclose(Fd[half], -dt / dx[d] * (chat * E_b / 3.0 - P_mid), rtol=1e-13, atol=1e-18)


def test_interface_flux_clamp_uses_the_thinner_of_the_two_cells_and_switches_off_when_thin():
    """tau_face = min(tau_a, tau_b) (R-G7): making the THIN side thinner changes the flux, making the thick side
    thicker does not; once 4/(3 tau_face) >= 1/sqrt(3) the clamp is inactive and the flux is the f = 0 HLL value."""
    n = (8, 1, 1)
    xf = [np.linspace(0.0, 0.8, 9), np.array([0.0, 1.0]), np.array([0.0, 1.0])]
    chat, dx, dt = 1.0, 0.1, 1e-3

    def energy_flux(chi_a, chi_b):
        g = _slab_grid(ort.CARTESIAN, n, xf, (1, 1, 1, 1, 1, 1), chat, ort.SOLVER_HLL)
        g.set_opacity(ort.OPAC_ROSSELAND, ort.make_power_law(1.0, a=1.0))          # chi = rho: tau_cell = rho^2 dx
        rho, T = np.ones(g.shape), np.ones(g.shape)
        U = [g.zeros() for _ in range(4)]
        it = g.interior
        rho[it][0, 0, :4], rho[it][0, 0, 4:] = math.sqrt(chi_a), math.sqrt(chi_b)
        U[0][it][0, 0, :4], U[0][it][0, 0, 4:] = 2.0, 0.5
        out = [a.copy() for a in U]
        g.explicit_step(dt, rho, T, U, out)
        return (2.0 - out[0][it][0, 0, 3]) * dx / dt                                # flux through the face 3|4

    base = energy_flux(50.0, 400.0)
    assert base == pytest.approx(-0.5 * (4.0 / (3.0 * 50.0 * dx)) * (0.5 - 2.0), rel=1e-12)
    assert energy_flux(50.0, 4000.0) == pytest.approx(base, rel=1e-12)              # thick side irrelevant
    assert energy_flux(25.0, 400.0) == pytest.approx(2.0 * base, rel=1e-12)         # thin side sets it
    assert energy_flux(400.0, 50.0) == pytest.approx(base, rel=1e-12)               # either order
    thin = energy_flux(1.0, 2.0)                                                    # 4/(3 * 0.1) > 1/sqrt(3): no clamp
    assert thin == pytest.approx(-0.5 / math.sqrt(3.0) * (0.5 - 2.0), rel=1e-12)


# --------------------------------------------------------------------------- (c) spherical: r_c dtheta is the largest extent
def test_interface_flux_on_a_spherical_grid_where_the_polar_extent_is_largest():
    """(r, theta) grid, r in [10, 10.8] in 8 cells (dr = 0.1), theta in [1.2, 1.8] in 4 cells (r_c dtheta ~ 1.5): the
    cell's largest physical extent is r_c dtheta (R-G9 lengths), so tau_i = rho chi r_c,i dtheta depends on the cell
    through r_c.  Jump of E across r = 10.4, uniform in theta, F = 0.  Finite-volume update of E (R-G9 metrics):
    dE_i = -dt [r_+^2 F_+ - r_-^2 F_-] 3/(r_+^3 - r_-^3)."""
    n = (8, 4, 1)
    r = np.linspace(10.0, 10.8, 9)
    th = np.linspace(1.2, 1.8, 5)
    chat = 1.7
    g = _slab_grid(ort.SPHERICAL, n, [r, th, np.array([0.0, 0.5])], (1, 1, 1, 1, 1, 1), chat, ort.SOLVER_HLL)
    chirho = 4.0
    g.set_opacity(ort.OPAC_SCATTER, ort.make_power_law(chirho))
    rho, T = np.ones(g.shape), np.ones(g.shape)
    U = [g.zeros() for _ in range(4)]
    it = g.interior
    E_a, E_b = 3.0, 1.0
    U[0][it][0, :, :4], U[0][it][0, :, 4:] = E_a, E_b
    dt = 1e-3
    out = [a.copy() for a in U]
    g.explicit_step(dt, rho, T, U, out)
    rc = 0.5 * (r[1:] + r[:-1])
    dth = th[1] - th[0]
    assert rc[3] * dth > 0.1 and rc[3] * dth > rc[3] * math.sin(1.5) * 0.0         # x3 inactive: not a candidate
    tau3, tau4 = chirho * rc[3] * dth, chirho * rc[4] * dth
    S = 4.0 * chat / (3.0 * min(tau3, tau4))
    assert S < chat / math.sqrt(3.0)
    Fface = -0.5 * S * (E_b - E_a)
    rf = r[4]
    want3 = E_a - dt * (rf ** 2 * Fface) * 3.0 / (r[4] ** 3 - r[3] ** 3)
    want4 = E_b + dt * (rf ** 2 * Fface) * 3.0 / (r[5] ** 3 - r[4] ** 3)
    E = out[0][it][0]
    assert np.allclose(E[:, 3], want3, rtol=1e-14, atol=0), (E[:, 3], want3)
    assert np.allclose(E[:, 4], want4, rtol=1e-14, atol=0), (E[:, 4], want4)
    for c in (0, 1, 2):
        assert np.allclose(E[:, c], E_a, rtol=1e-15, atol=0)
    for c in (5, 6, 7):
        assert np.allclose(E[:, c], E_b, rtol=1e-15, atol=0)


# --------------------------------------------------------------------------- (a) the diffusion limit, clamp ACTIVE
def _gaussian_variance_growth(N, chirho, thick, nstep, chat=1.0, w=0.05):
    """scattering-only Gaussian (kappa_P = 0): returns (variance(t) - variance(0)) / (2 D t), D = chat/(3 chi rho)"""
    xf = [np.linspace(0.0, 1.0, N + 1), np.array([0.0, 1.0]), np.array([0.0, 1.0])]
    g = _slab_grid(ort.CARTESIAN, (N, 1, 1), xf, (0,) * 6, chat, ort.SOLVER_HLL, thick=thick)
    g.set_opacity(ort.OPAC_SCATTER, ort.make_power_law(chirho))
    x = 0.5 * (xf[0][1:] + xf[0][:-1])
    U = [g.zeros() for _ in range(4)]
    E0 = 1e-6 + np.exp(-((x - 0.5) ** 2) / (2 * w ** 2))
    U[0][g.interior] = E0[None, None, :]
    U[1][g.interior] = (-(1.0 / (3 * chirho)) * np.gradient(E0, x))[None, None, :]   # the diffusion flux: no transient
    rho, T = np.ones(g.shape), np.ones(g.shape)
    U2 = [a.copy() for a in U]

    def variance(E):
        m = E - 1e-6
        mu = (m * x).sum() / m.sum()
        return (m * (x - mu) ** 2).sum() / m.sum()

    dt = 0.4 / N / chat
    for _ in range(nstep):
        g.explicit_step(dt, rho, T, U, U2)
        g.implicit_step(dt, rho, T, None, U2)
        U, U2 = U2, U
    D = chat / (3 * chirho)
    return (variance(U[0][g.interior][0, 0]) - variance(E0)) / (2 * D * nstep * dt)


@pytest.mark.parametrize("chirho,off_min", [(5.0e3, 1.12), (2.0e4, 1.8)])
def test_diffusion_rate_needs_the_thick_limit_when_tau_cell_is_large(chirho, off_min):
    """N = 256, a narrow pulse (w = 0.02, 5 cells): tau_cell = chi rho / 256 = 19.5 and 78, so 4/(3 tau) = 0.068 and
    0.017 clamp the 1/sqrt(3) speed (L171-175).  With the limit the Gaussian's variance grows as 2 D t within a few
    per cent (L169: "in order to recover the diffusion limit": measured 1.042 and 1.059); without it the HLL dissipation
    chat dx/(2 sqrt 3) over-diffuses (measured 1.18 and 2.04).  (At tau_cell = 3.9 and a resolved pulse the clamp fires
    too but PLM keeps both answers within 0.3 % of each other: that regime pins nothing and is not used.)"""
    on = _gaussian_variance_growth(256, chirho, 1, 6000, w=0.02)
    off = _gaussian_variance_growth(256, chirho, 0, 6000, w=0.02)
    assert 0.98 < on < 1.08, on
    assert off > off_min and off > on + 0.1, (on, off)
