"""Pins of the oracle's point-wise formulas against what PAPER.md and the mathematics fix
(closure Eq. 11-14, wave speeds Eq. 22-24, PLM, f-preserving fix Eq. 19-21, Riemann flux L150).
None of these tests calls the CUDA path."""
import math

import numpy as np
import pytest

from oracle import ort

RNG = np.random.default_rng(7)


def random_states(n, fmax=1.0):
    out = []
    for _ in range(n):
        E = math.exp(RNG.uniform(-3, 3))
        v = RNG.standard_normal(3)
        v /= np.linalg.norm(v)
        out.append((E, E * RNG.uniform(0, fmax) * v))
    return out


# ----------------------------------------------------------------------------- closure
def test_eddington_factor_limits(golden):
    g = golden["eddington_factor"]                      # PAPER.md:L75 Eq. 13
    assert ort.eddington_factor(0.0) == pytest.approx(g["xi_at_f0"], abs=1e-16)
    assert ort.eddington_factor(1.0) == pytest.approx(g["xi_at_f1"], abs=1e-16)


def test_eddington_factor_monotone_and_alternative_form():
    # Levermore's closure has the equivalent textbook form xi = 1/3 + 2 f^2 / (2 + sqrt(4 - 3 f^2))
    fs = np.linspace(0, 1, 201)
    xi = np.array([ort.eddington_factor(f) for f in fs])
    assert np.all(np.diff(xi) > 0)
    alt = 1.0 / 3.0 + 2.0 * fs ** 2 / (2.0 + np.sqrt(4.0 - 3.0 * fs ** 2))
    assert np.max(np.abs(xi - alt)) < 1e-15


def test_pressure_tensor_trace_symmetry_and_eigenvector():
    for E, F in random_states(200):
        P = ort.pressure_tensor(E, F)
        assert np.trace(P) == pytest.approx(E, rel=1e-14)               # trace D = 1 (Eq. 12)
        assert np.allclose(P, P.T, rtol=0, atol=1e-16 * E)
        f = np.linalg.norm(F) / E
        n = F / np.linalg.norm(F)
        assert np.allclose(P @ n, ort.eddington_factor(f) * E * n, rtol=1e-13, atol=1e-15 * E)  # P n = xi E n
        # any direction perpendicular to F has eigenvalue (1 - xi)/2 E
        t = np.cross(n, [0.3, -0.5, 0.8])
        t /= np.linalg.norm(t)
        assert np.allclose(P @ t, 0.5 * (1 - ort.eddington_factor(f)) * E * t, rtol=1e-13, atol=1e-15 * E)


def test_pressure_tensor_limits():
    P = ort.pressure_tensor(3.0, [0.0, 0.0, 0.0])                      # Eddington limit: P = E/3 I
    assert np.allclose(P, np.eye(3), atol=1e-15)
    P = ort.pressure_tensor(2.0, [0.0, 2.0, 0.0])                      # free streaming: P = E n n
    want = np.zeros((3, 3))
    want[1, 1] = 2.0
    assert np.allclose(P, want, atol=1e-15)


# ----------------------------------------------------------------------------- wave speeds
def test_wave_speed_limits(golden):
    g = golden["wave_speed_limits"]
    lam = ort.wave_speeds(1.0, [0, 0, 0], 0)
    assert lam[0] == pytest.approx(-g["f0_lambda13"], abs=1e-15)
    assert lam[2] == pytest.approx(+g["f0_lambda13"], abs=1e-15)
    assert lam[1] == g["f0_lambda2"]
    for ang in np.linspace(0, math.pi, 13):                            # f -> 1: all -> cos(theta)
        F = [math.cos(ang), math.sin(ang), 0.0]
        for d, want in ((0, math.cos(ang)), (1, math.sin(ang)), (2, 0.0)):
            lam = ort.wave_speeds(1.0, F, d)
            assert np.allclose(lam, want, atol=2e-8)  # sqrt of a round-off-sized zeta^2


def test_wave_speeds_bounded_and_ordered():
    for E, F in random_states(300):
        for d in range(3):
            l1, l2, l3 = ort.wave_speeds(E, F, d)
            assert -1.0 - 1e-14 <= l1 <= l2 + 1e-14 and l2 <= l3 + 1e-14 and l3 <= 1.0 + 1e-14


def _phys_flux(U, d, chat=1.0):
    # HLL with identical states returns the physical flux (consistency), see test below
    return ort.riemann_flux(U, U, d, chat)


def test_wave_speeds_are_eigenvalues_of_the_flux_jacobian():
    """Independent pin of Eq. 22-24 AND of the closure: lambda_1, lambda_2 (double), lambda_3 must be
    the eigenvalues of d(F^d, P^{.d})/d(E, F) -- computed here by central differences and numpy."""
    for E, F in random_states(40, fmax=0.97):
        if np.linalg.norm(F) / E < 0.02:
            continue
        U = np.concatenate([[E], F])
        for d in range(3):
            J = np.zeros((4, 4))
            for q in range(4):
                h = 1e-6 * E
                up, um = U.copy(), U.copy()
                up[q] += h
                um[q] -= h
                J[:, q] = (_phys_flux(up, d) - _phys_flux(um, d)) / (2 * h)
            ev = np.sort(np.linalg.eigvals(J).real)
            l1, l2, l3 = ort.wave_speeds(E, F, d)
            assert np.allclose(ev, [l1, l2, l2, l3], atol=2e-6), (E, F, d, ev, (l1, l2, l3))


# ----------------------------------------------------------------------------- reconstruction
def test_vanleer_limiter_textbook_form_and_tvd():
    for _ in range(500):
        a, b, c = RNG.standard_normal(3)
        s = ort.vanleer_slope(a, b, c)
        dm, dp = b - a, c - b
        if dm * dp <= 0:
            assert s == 0.0
        else:
            r = dm / dp                                    # van Leer: phi(r) = (r + |r|)/(1 + |r|)
            assert s == pytest.approx((r + abs(r)) / (1 + abs(r)) * dp, rel=1e-13)
            assert abs(s) <= 2 * min(abs(dm), abs(dp)) * (1 + 1e-15)
    assert ort.vanleer_slope(1.0, 2.0, 3.0) == 1.0         # linear data reproduced exactly
    assert ort.vanleer_slope(1.0, 2.0, 1.5) == 0.0         # extremum -> flat


def test_fpreserving_face_cases():
    # (i) face f <= 1 and larger than the cell's: reconstruction kept (Eq. 20)
    Uc = [1.0, 0.2, 0.0, 0.0]
    RU = [1.0, 0.3, 0.1, 0.0]
    assert np.array_equal(ort.fpreserving_face(Uc, RU), RU)
    # (ii) face f > 1: flux rescaled so that f_face = f_cell (Eq. 21), all three components
    RU = [0.5, 0.6, 0.1, 0.0]
    out = ort.fpreserving_face(Uc, RU)
    assert out[0] == 0.5 and np.allclose(out[1:], [0.1, 0.0, 0.0], atol=1e-16)
    # (iii) face f smaller than the cell's ("beam widening", L148): also Eq. 21
    Uc = [1.0, 0.0, 0.9, 0.0]
    RU = [1.2, 0.0, 0.9, 0.05]
    out = ort.fpreserving_face(Uc, RU)
    assert out[0] == 1.2 and np.allclose(out[1:], [0.0, 1.08, 0.0], atol=1e-15)


def test_fpreserving_face_invariant():
    # whatever the reconstruction gives, f_cell <= f_face <= 1 afterwards
    for E, F in random_states(300):
        Uc = np.concatenate([[E], F])
        RU = Uc * (1 + 0.5 * RNG.uniform(-1, 1, 4))
        RU[0] = abs(RU[0]) + 1e-3
        out = ort.fpreserving_face(Uc, RU)
        ff = np.linalg.norm(out[1:]) / out[0]
        fc = np.linalg.norm(F) / E
        assert fc * (1 - 1e-14) <= ff <= 1 + 1e-14


def test_pluto_and_clip_face_cases():
    """The two comparison schemes of Sect. 2.5 / 3.2: flat fallback (L136) and clip-only (Eq. 36-38)."""
    Uc = [1.0, 0.2, 0.0, 0.0]
    # f_face <= 1: both keep the reconstruction (Eq. 37; L136 "whenever ||R(F)|| > R(E)" not met) -- also where the
    # f-preserving scheme would NOT keep it (f_face < f_cell)
    for RU in ([1.0, 0.3, 0.1, 0.0], [1.2, 0.1, 0.0, 0.05]):
        assert np.array_equal(ort.pluto_face(Uc, RU), RU)
        assert np.array_equal(ort.clip_face(RU), RU)
    # f_face > 1 (3-4-5 triangle: ||R(F)|| = 1 exactly, R(E) = 0.5)
    RU = [0.5, 0.6, 0.0, 0.8]
    assert np.array_equal(ort.pluto_face(Uc, RU), Uc)                       # E_f = E_c AND F_f = F_c (L136)
    out = ort.clip_face(RU)
    assert out[0] == 0.5 and np.allclose(out[1:], [0.3, 0.0, 0.4], rtol=0, atol=1e-16)   # Eq. 38
    # the three schemes are three different answers on this input (a swapped branch in the grid-level switch shows)
    fp = ort.fpreserving_face(Uc, RU)
    assert np.allclose(fp, [0.5, 0.1, 0.0, 0.0], atol=1e-16)
    # equality ||R(F)|| = R(E) belongs to the "keep" side of Eq. 37 and of L136 (strict ">")
    RU = [1.0, 0.6, 0.0, 0.8]
    assert np.array_equal(ort.pluto_face(Uc, RU), RU) and np.array_equal(ort.clip_face(RU), RU)


def test_pluto_and_clip_face_invariants():
    # f_face <= 1 afterwards; clip keeps E_f = R(E) and the direction of R(F); PLUTO returns one of its two inputs
    ncl = 0
    for E, F in random_states(300):
        Uc = np.concatenate([[E], F])
        RU = Uc * (1 + 0.5 * RNG.uniform(-1, 1, 4))
        RU[0] = abs(RU[0]) + 1e-3
        over = np.linalg.norm(RU[1:]) > RU[0]
        ncl += over
        c = ort.clip_face(RU)
        assert c[0] == RU[0]
        assert np.linalg.norm(c[1:]) <= c[0] * (1 + 2e-15)
        if over:
            assert np.linalg.norm(c[1:]) == pytest.approx(c[0], rel=2e-15)
            assert np.allclose(np.cross(c[1:], RU[1:]), 0.0, atol=1e-15 * np.linalg.norm(c[1:]) * np.linalg.norm(RU[1:]))
            assert np.dot(c[1:], RU[1:]) > 0
        p = ort.pluto_face(Uc, RU)
        assert np.array_equal(p, Uc if over else RU)
    assert 20 < ncl < 280                                                    # both branches were exercised


# ----------------------------------------------------------------------------- Riemann flux
def test_riemann_consistency_and_closure_flux():
    for E, F in random_states(100):
        U = np.concatenate([[E], F])
        P = ort.pressure_tensor(E, F)
        for d in range(3):
            for solver in (ort.SOLVER_HLL, ort.SOLVER_GLF):
                fl = ort.riemann_flux(U, U, d, 2.5, solver)
                want = 2.5 * np.array([F[d], P[0, d], P[1, d], P[2, d]])    # Eq. 5-6: chat (F^d, P^{.d})
                assert np.allclose(fl, want, rtol=1e-13, atol=1e-15 * E)


def test_hll_upwinds_a_free_streaming_beam():
    # f = 1 along +x on both sides: S_L = 0, S_R = chat => flux = F(U_L) exactly (R-G8)
    UL, UR = [2.0, 2.0, 0, 0], [0.5, 0.5, 0, 0]
    fl = ort.riemann_flux(UL, UR, 0, 3.0)
    assert np.allclose(fl, [6.0, 6.0, 0, 0], atol=1e-15)
    # same beam seen by a face normal to y: lambda = 0 both ways -> den = 0 -> average (R-G8), finite
    fl = ort.riemann_flux(UL, UR, 1, 3.0)
    assert np.all(np.isfinite(fl)) and np.allclose(fl, [0, 0, 0, 0], atol=1e-15)


def test_hll_equals_glf_when_speeds_are_symmetric():
    # f = 0 both sides, thick limit with 4/(3 tau) < 1/sqrt(3): both solvers use alpha = lim
    UL, UR = [1.0, 0, 0, 0], [3.0, 0, 0, 0]
    lim = 0.2
    a = ort.riemann_flux(UL, UR, 0, 1.0, ort.SOLVER_HLL, lim)
    b = ort.riemann_flux(UL, UR, 0, 1.0, ort.SOLVER_GLF, lim)
    assert np.allclose(a, b, rtol=1e-14, atol=1e-16)
    # closed form: energy flux = -alpha/2 (E_R - E_L), momentum flux = average pressure
    assert a[0] == pytest.approx(-0.5 * lim * 2.0, rel=1e-14)
    assert a[1] == pytest.approx(0.5 * (1.0 / 3 + 1.0), rel=1e-14)


def test_rusanov_is_local_lax_friedrichs():
    """RT/ORT_SOLVER_RUSANOV (L150 "Lax-Friedrichs-Rusanov"; R-G5): 1/2(F_L+F_R) - 1/2 alpha (U_R-U_L) with the LOCAL
    alpha = chat max |lambda_{1,3}| of the two states.  Pins: consistency; equals GLF when some |lambda| = 1 (a state
    streaming along the face normal); equals HLL when the speeds are symmetric (f = 0 on both sides); never more
    diffusive than GLF; alpha recovered from the flux equals max |lambda| of ort.wave_speeds; obeys the thick limit."""
    chat = 3.0
    rng = np.random.default_rng(5)
    for E, F in random_states(40):
        U = [E] + list(F)
        for d in range(3):
            assert np.allclose(ort.riemann_flux(U, U, d, chat, ort.SOLVER_RUSANOV), _phys_flux(U, d, chat), rtol=1e-14, atol=1e-15)
    states = random_states(40)
    for (EL, FL), (ER, FR) in zip(states[::2], states[1::2]):
        UL, UR = [EL] + list(FL), [ER] + list(FR)
        for d in range(3):
            fr = np.array(ort.riemann_flux(UL, UR, d, chat, ort.SOLVER_RUSANOV))
            fg = np.array(ort.riemann_flux(UL, UR, d, chat, ort.SOLVER_GLF))
            avg = 0.5 * (np.array(_phys_flux(UL, d, chat)) + np.array(_phys_flux(UR, d, chat)))
            dU = np.array(UR) - np.array(UL)
            lam = [abs(v) for U in (UL, UR) for v in (ort.wave_speeds(U[0], U[1:], d)[0], ort.wave_speeds(U[0], U[1:], d)[2])]
            alpha = chat * max(lam)
            assert np.allclose(fr, avg - 0.5 * alpha * dU, rtol=1e-13, atol=1e-14)
            assert np.all(np.abs(fr - avg) <= np.abs(fg - avg) + 1e-14)
            lim = 0.3 * alpha                                  # thick limit below the local speed: alpha = lim
            fl = np.array(ort.riemann_flux(UL, UR, d, chat, ort.SOLVER_RUSANOV, lim=lim))
            assert np.allclose(fl, avg - 0.5 * lim * dU, rtol=1e-13, atol=1e-14)
    # |lambda| = 1: a beam along +x on the left
    UL, UR = [2.0, 2.0, 0.0, 0.0], [0.7, 0.1, -0.2, 0.05]
    assert np.allclose(ort.riemann_flux(UL, UR, 0, chat, ort.SOLVER_RUSANOV), ort.riemann_flux(UL, UR, 0, chat, ort.SOLVER_GLF), rtol=1e-14)
    # symmetric speeds: f = 0 on both sides -> HLL with S_R = -S_L = chat/sqrt(3) is the same formula
    UL, UR = [1.3, 0.0, 0.0, 0.0], [0.4, 0.0, 0.0, 0.0]
    assert np.allclose(ort.riemann_flux(UL, UR, 1, chat, ort.SOLVER_RUSANOV), ort.riemann_flux(UL, UR, 1, chat, ort.SOLVER_HLL), rtol=1e-14)


def test_riemann_mirror_symmetry():
    for _ in range(50):
        (E1, F1), (E2, F2) = random_states(2)
        UL, UR = np.concatenate([[E1], F1]), np.concatenate([[E2], F2])
        m = np.array([1.0, -1.0, 1.0, 1.0])               # x -> -x
        for solver in (0, 1):
            a = ort.riemann_flux(UL, UR, 0, 1.0, solver, 0.7)
            b = ort.riemann_flux(UR * m, UL * m, 0, 1.0, solver, 0.7)
            # flux of E and of tangential F flips sign, flux of F_x keeps it
            assert np.allclose(a, b * np.array([-1.0, 1.0, -1.0, -1.0]), rtol=1e-12, atol=1e-14)


def test_hll_single_contact_is_resolved_at_rest():
    """lambda_2 = 0 for F perpendicular to the face: two states with equal Pi=(1-xi)E/2 and equal
    normal flux 0 differ only by a contact; HLL still diffuses it, but the momentum flux must
    equal the common pressure."""
    UL = np.array([1.0, 0.0, 0.0, 0.0])
    UR = np.array([1.0, 0.0, 0.0, 0.0])
    fl = ort.riemann_flux(UL, UR, 0, 1.0)
    assert fl[1] == pytest.approx(1.0 / 3.0, rel=1e-15)
