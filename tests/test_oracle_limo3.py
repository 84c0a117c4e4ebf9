"""Pins of the oracle's LimO3 reconstruction (Sect. 2.5: "compact third-order reconstruction (LimO3; Cada &
Torrilhon 2009)", the scheme of the paper's Fig. 1-5).  The formula is not printed in PAPER.md; DESIGN.md R-G22 restates
it.  What pins it here is mathematics, not the oracle: exactness on quadratics, third-order convergence, the limiter's
closed forms on worked cases, symmetries, and the order of accuracy of the whole spatial operator.  No CUDA here."""
import math

import numpy as np
import pytest

import rt_workloads as W
from oracle import ort


def quad_avg(a, b, c, x, h):
    """cell average over [x - h/2, x + h/2] of a + b x + c x^2"""
    return a + b * x + c * (x * x + h * h / 12.0)


@pytest.mark.parametrize("r", [0.0, 1.0])
def test_exact_on_quadratics_where_the_limiter_is_inactive(r):
    """phi_3(theta) = (2 + theta)/3 is the quadratic through the three cell AVERAGES evaluated at the face; the limiter
    leaves it alone for 0.4 <= theta <= 2.8 (2 theta >= phi_3 and phi_3 <= 1.6)"""
    rng = np.random.default_rng(1)
    n = 0
    for _ in range(400):
        a, b, c = rng.uniform(-2, 2, 3)
        x, h = rng.uniform(-1, 1), rng.uniform(0.05, 0.5)
        um, u0, up = (quad_avg(a, b, c, x + s * h, h) for s in (-1, 0, 1))
        if not (up - u0) != 0.0:
            continue
        theta = (u0 - um) / (up - u0)
        if not (0.45 < theta < 2.7 and 0.45 < 1 / theta < 2.7):
            continue
        n += 1
        lo, hi = ort.limo3_faces(um, u0, up, dx=h, r=r)
        q = lambda y: a + b * y + c * y * y
        scale = abs(a) + abs(b) + abs(c)                          # the terms that cancel in q and in the averages
        assert abs(hi - q(x + h / 2)) <= 2e-15 * scale and abs(lo - q(x - h / 2)) <= 2e-15 * scale
    assert n > 50


def test_worked_cases_of_the_limiter():
    """phi_L(theta) = max(0, min(phi_3, max(-theta/2, min(2 theta, phi_3, 1.6)))) by hand (r = 0: no smoothness switch)"""
    # theta = 1/3 < 0.4: phi = 2 theta -> upper face = u0 + d-
    lo, hi = ort.limo3_faces(0.0, 1.0, 4.0)
    assert hi == pytest.approx(1.0 + 1.0, rel=1e-15)
    # seen from the lower face 1/theta = 3 > 2.8: phi = 1.6 -> u0 - 0.8 d-
    assert lo == pytest.approx(1.0 - 0.8 * 1.0, rel=1e-15)
    # theta = 10: phi_3 = 4 is cut at 1.6
    lo, hi = ort.limo3_faces(-9.0, 1.0, 2.0)
    assert hi == pytest.approx(1.0 + 0.8 * 1.0, rel=1e-15)
    # local maximum, theta = -1: phi = min(phi_3, -theta/2) = 1/3 (LimO3 does not flatten mild extrema)
    lo, hi = ort.limo3_faces(1.0, 2.0, 1.0)
    assert hi == pytest.approx(2.0 - 0.5 / 3.0, rel=1e-15) and lo == pytest.approx(2.0 - 0.5 / 3.0, rel=1e-15)
    # sharp extremum, theta = -4 <= -2: phi_3 < 0 -> flat
    lo, hi = ort.limo3_faces(5.0, 1.0, 2.0)
    assert hi == 1.0
    # zero differences: flat, no division by zero
    assert ort.limo3_faces(1.0, 1.0, 1.0) == (1.0, 1.0)
    lo, hi = ort.limo3_faces(1.0, 1.0, 3.0)       # d- = 0: theta = 0 -> phi = 0 at the upper face; lower face: d- = 0
    assert hi == 1.0 and lo == 1.0


def test_symmetries_and_bounds():
    rng = np.random.default_rng(2)
    for _ in range(300):
        um, u0, up = rng.normal(size=3)
        lo, hi = ort.limo3_faces(um, u0, up)
        lo2, hi2 = ort.limo3_faces(up, u0, um)                 # mirror image: the faces swap
        assert lo2 == hi and hi2 == lo
        s, t = rng.uniform(0.1, 10), rng.normal()
        lo3, hi3 = ort.limo3_faces(s * um + t, s * u0 + t, s * up + t)
        assert lo3 == pytest.approx(s * lo + t, rel=1e-13, abs=1e-13) and hi3 == pytest.approx(s * hi + t, rel=1e-13, abs=1e-13)
        if (u0 - um) * (up - u0) > 0:                          # monotone data: face values stay between the neighbours
            assert min(um, up) - 1e-15 <= lo <= max(um, up) + 1e-15 and min(um, up) - 1e-15 <= hi <= max(um, up) + 1e-15
            assert (hi - u0) * (up - u0) >= 0 and (u0 - lo) * (u0 - um) >= 0


def test_smoothness_switch_keeps_smooth_extrema_third_order():
    """eta = (d-^2 + d+^2)/(r dx)^2 <= 1: the unlimited phi_3, even where theta < 0 (a resolved maximum); r = 0 limits it"""
    h = 0.05
    avg = lambda x: (math.sin(x + h / 2) - math.sin(x - h / 2)) / h         # cell average of cos
    x0 = 0.01                                                             # next to the maximum of cos at 0
    um, u0, up = avg(x0 - h), avg(x0), avg(x0 + h)
    lo, hi = ort.limo3_faces(um, u0, up, dx=h, r=1.0)
    assert abs(hi - math.cos(x0 + h / 2)) < 2e-6 and abs(lo - math.cos(x0 - h / 2)) < 2e-6      # O(h^3)
    lo0, hi0 = ort.limo3_faces(um, u0, up, dx=h, r=0.0)
    assert abs(hi0 - math.cos(x0 + h / 2)) > 1e-4                                                # clipped: O(h^2)


def test_face_value_converges_at_third_order():
    err = []
    for N in (16, 32, 64, 128):
        h = 2.0 / N
        x = 0.3
        avg = lambda y: (math.cos(y - h / 2) - math.cos(y + h / 2)) / h     # cell average of sin
        lo, hi = ort.limo3_faces(avg(x - h), avg(x), avg(x + h), dx=h, r=1.0)
        err.append(abs(hi - math.sin(x + h / 2)))
    ratios = [a / b for a, b in zip(err[:-1], err[1:])]
    assert all(7.0 < q < 9.5 for q in ratios), (err, ratios)


def _operator_error(recon, N, fix=ort.FIX_CLIP):
    """L1 error of the E equation's discrete right-hand side against the exact finite-volume one, -chat [F_x]/dx, for smooth
    periodic cell averages (E = 2 + 0.5 sin 2 pi x, F_x = 0.4 + 0.3 cos 2 pi x: f <= 0.47)"""
    n = (N, 1, 1)
    xf = [np.linspace(0.0, 1.0, N + 1), np.array([0.0, 1.0]), np.array([0.0, 1.0])]
    h = 1.0 / N
    k = 2 * np.pi
    xl, xr = xf[0][:-1], xf[0][1:]
    Eavg = 2.0 + 0.5 * (np.cos(k * xl) - np.cos(k * xr)) / (k * h)
    Favg = 0.4 + 0.3 * (np.sin(k * xr) - np.sin(k * xl)) / (k * h)
    U = [W.embed(n, Eavg.reshape(1, 1, N)), W.embed(n, Favg.reshape(1, 1, N)), W.embed(n, 0.0), W.embed(n, 0.0)]
    g = ort.Grid(ort.CARTESIAN, n, xf[0], xf[1], xf[2], (0, 0, 1, 1, 1, 1))
    chat = 1.3
    g.set_params(ort.make_params(chat=chat, solver=ort.SOLVER_HLL, E_floor=1e-30))
    g.set_reconstruction(recon, 1.0)
    # the f-preserving fix replaces R(F) by F_c R(E)/E_c on every face where f would fall below the cell's (Eq. 21): a
    # first-order face value by construction.  The order of R() itself shows with the clip-only fix (Eq. 36-38), which
    # leaves R(F) alone as long as |R(F)| <= R(E) (here f <= 0.47 everywhere)
    g.set_face_fix(fix)
    out = [a.copy() for a in U]
    dt = 1e-7
    g.explicit_step(dt, np.ones(g.shape), np.ones(g.shape), U, out)
    rhs = (out[0][g.interior][0, 0] - Eavg) / dt
    Fx = lambda x: 0.4 + 0.3 * np.cos(k * x)
    exact = -chat * (Fx(xr) - Fx(xl)) / h
    return np.abs(rhs - exact).mean()


def test_spatial_operator_is_third_order_with_limo3_and_second_order_with_plm():
    """the whole chain reconstruct -> closure -> HLL -> divergence (face fix: clip-only, inactive here): its truncation
    error falls by ~8 per doubling with LimO3 and by ~4 with PLM (measured on the E equation, whose exact finite-volume
    right-hand side is known from F_x at the faces).  With the f-preserving fix both are first order where Eq. 21
    applies: that is the scheme, and it is checked too."""
    e3 = [_operator_error(ort.RECON_LIMO3, N) for N in (32, 64, 128)]
    e2 = [_operator_error(ort.RECON_PLM, N) for N in (32, 64, 128)]
    assert 6.0 < e3[0] / e3[1] < 10.0 and 6.0 < e3[1] / e3[2] < 10.0, e3
    assert 3.0 < e2[0] / e2[1] < 5.5 and 3.0 < e2[1] / e2[2] < 5.5, e2
    assert e3[2] < 0.05 * e2[2]
    e1 = [_operator_error(ort.RECON_LIMO3, N, ort.FIX_FPRESERVING) for N in (32, 64, 128)]
    assert 1.7 < e1[0] / e1[1] < 2.3 and 1.7 < e1[1] / e1[2] < 2.3, e1


@pytest.mark.parametrize("solver", [ort.SOLVER_HLL, ort.SOLVER_GLF])
def test_limo3_step_preserves_uniform_states_and_conserves(solver):
    n = (12, 10, 8)
    xf = [np.linspace(0.0, 1.0, v + 1) for v in n]
    g = ort.Grid(ort.CARTESIAN, n, xf[0], xf[1], xf[2], (0,) * 6)
    g.set_params(ort.make_params(chat=2.0, solver=solver))
    g.set_reconstruction(ort.RECON_LIMO3, 0.5)
    U = [np.full(g.shape, v) for v in (1.7, 0.3, -0.4, 0.5)]
    out = [a.copy() for a in U]
    g.explicit_step(0.01, np.ones(g.shape), np.ones(g.shape), U, out)
    for q in range(4):
        assert np.array_equal(out[q][g.interior], U[q][g.interior])
    U = W.random_state(np.random.default_rng(5), n)
    dt = g.cfl_dt(U, 0.4)
    out = [a.copy() for a in U]
    g.explicit_step(dt, np.ones(g.shape), np.ones(g.shape), U, out)
    for q in range(4):
        s0, s1 = U[q][g.interior].sum(), out[q][g.interior].sum()
        assert abs(s1 - s0) < 1e-14 * np.abs(U[q][g.interior]).sum()
    # and it is not PLM
    g.set_reconstruction(ort.RECON_PLM)
    out2 = [a.copy() for a in U]
    g.explicit_step(dt, np.ones(g.shape), np.ones(g.shape), U, out2)
    assert np.abs(out2[0] - out[0]).max() > 1e-4


def test_shock_tube_1_with_limo3_keeps_the_fronts(golden):
    """Fig. 1 (L246-248) is drawn with PLM and with LimO3: the outer fronts sit at x ~ 11.2 with either"""
    st = golden["shock_tube_1"]
    N = 512
    n = (N, 1, 1)
    xf = [np.linspace(-20.0, 20.0, N + 1), np.array([0.0, 1.0]), np.array([0.0, 1.0])]
    x = 0.5 * (xf[0][1:] + xf[0][:-1])
    U = [W.embed(n, np.where(x < 0, st["left"][q], st["right"][q]).reshape(1, 1, N)) for q in range(4)]
    w = W.Workload(name="tube", geometry=W.CARTESIAN, n=n, xf=xf, bc=(W.BC_OUTFLOW,) * 6,
                   params=W.default_params(chat=1.0, E_floor=1e-30), opacities={}, U=U,
                   rho=W.embed(n, 1.0, fill=1.0), T=W.embed(n, 1.0, fill=1.0), cfl=golden["courant"]["C_a"])
    g = ort.grid_from_workload(w)
    g.set_reconstruction(ort.RECON_LIMO3, 1.0)
    Uo, _, _, dts = ort.run_rk2(g, w, None, t_end=st["t_end"])
    E = Uo[0][g.interior][0, 0]
    Ep = E[np.argmin(np.abs(x - 5.0))]
    right = x > 5.0
    xr = x[right][np.argmin(np.abs(E[right] - 0.5 * (Ep + 1.0)))]
    assert xr == pytest.approx(st["front_x"], abs=0.25)
    assert E.sum() * (40.0 / N) == pytest.approx(40.0, rel=1e-12)
    assert E.min() > 0.85 and E.max() < 1.2                      # no spurious over/undershoots beyond the plateaus
