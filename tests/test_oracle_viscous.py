"""Pins for the viscous terms, stretched-y metrics and wall ghosts."""
import numpy as np
import pytest
import sympy as sp

import workloads as W
from oracle import oracle as O

GAMMA, RGAS, PR, MU0, SUTH = 1.4, 1.0, 0.72, 0.05, 110.4 / 288.15


def _manufactured():
    """Symbolic viscous right-hand sides d_j sigma_ij and d_j(sigma_ij u_i) + d_j(lambda d_j T)
    (the governing equations as SURVEY 8(c) states them) for trigonometric fields."""
    x, y, z = sp.symbols("x y z")
    u = sp.sin(x) * sp.cos(2 * y) * sp.cos(z) * sp.Rational(3, 10) + sp.Rational(1, 10) * sp.sin(y)
    v = sp.cos(x) * sp.sin(y) * sp.cos(2 * z) * sp.Rational(1, 5)
    w = sp.sin(2 * x) * sp.sin(y) * sp.sin(z) * sp.Rational(1, 4)
    T = 1 + sp.Rational(1, 5) * sp.cos(x) * sp.cos(y) * sp.sin(z)
    rho = 1 + sp.Rational(1, 10) * sp.sin(x + y + z)
    t = T                                                   # T_ref = 1
    mu = MU0 * t * sp.sqrt(t) * (1 + SUTH) / (t + SUTH)
    cp = GAMMA * RGAS / (GAMMA - 1)
    lam = cp * mu / PR
    X = (x, y, z)
    vel = (u, v, w)
    div = sum(sp.diff(vel[a], X[a]) for a in range(3))
    sig = [[mu * (sp.diff(vel[a], X[b]) + sp.diff(vel[b], X[a]) - (sp.Rational(2, 3) * div if a == b else 0))
            for b in range(3)] for a in range(3)]
    mom = [sum(sp.diff(sig[a][b], X[b]) for b in range(3)) for a in range(3)]
    ene = sum(sp.diff(sum(sig[a][b] * vel[a] for a in range(3)), X[b]) for b in range(3)) + \
        sum(sp.diff(lam * sp.diff(T, X[b]), X[b]) for b in range(3))
    f = lambda e: sp.lambdify((x, y, z), e, "numpy")
    return dict(u=f(u), v=f(v), w=f(w), T=f(T), rho=f(rho), mom=[f(m) for m in mom], ene=f(ene))


MF = _manufactured()


def _visc_error(n, stretched, order=6):
    L = 2 * np.pi
    x = np.arange(n) * L / n
    z = np.arange(n) * L / n
    eta = np.arange(n) * L / n
    y = eta + 0.25 * np.sin(eta) if stretched else eta       # periodic stretching, dy/deta in [0.75, 1.25]
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    rho, T = MF["rho"](X, Y, Z), MF["T"](X, Y, Z)
    p = rho * RGAS * T
    case = W.Case(name="mms", nx=n, ny=n, nz=n, lx=L, ly=L, lz=L, y_nodes=y if stretched else None,
                  gamma=GAMMA, rgas=RGAS, prandtl=PR, visc_law=W.VISC_SUTHERLAND, mu_ref=MU0, t_ref=1.0,
                  central_order=order, visc_order=order,
                  w0=W.conserved_from_primitive(rho, MF["u"](X, Y, Z), MF["v"](X, Y, Z), MF["w"](X, Y, Z), p, GAMMA))
    R = O.Oracle(case).rhs(parts=O.PART_VISC)
    ref = [np.zeros_like(X)] + [m(X, Y, Z) for m in MF["mom"]] + [MF["ene"](X, Y, Z)]
    assert np.all(R[0] == 0.0)
    return [np.max(np.abs(R[q] - ref[q])) / np.max(np.abs(ref[q])) for q in range(1, 5)]


@pytest.mark.parametrize("stretched", [False, True])
def test_viscous_terms_match_symbolic_navier_stokes_at_design_order(stretched):
    """O4 / S10 pin: manufactured fields, order 2L on uniform and on stretched y."""
    e1 = _visc_error(32, stretched)
    e2 = _visc_error(64, stretched)
    for a, b in zip(e1, e2):
        assert b < 2e-6 and np.log2(a / b) > 6 - 0.3, (e1, e2)


@pytest.mark.parametrize("order", [2, 4])
def test_viscous_other_orders(order):
    e1 = _visc_error(32, True, order)
    e2 = _visc_error(64, True, order)
    for a, b in zip(e1, e2):
        assert np.log2(a / b) > order - 0.3, (order, e1, e2)


def test_metrics_of_a_known_mapping():
    """O4 / S3: eta_y = 1/(dy/deta), eta_yy = -(d2y/deta2) eta_y^3 for y = eta + 0.25 sin(eta)."""
    n = 64
    L = 2 * np.pi
    eta = np.arange(n) * L / n
    y = eta + 0.25 * np.sin(eta)
    one = np.ones((4, n, 4))
    case = W.Case(name="met", nx=4, ny=n, nz=4, lx=1.0, ly=L, lz=1.0, y_nodes=y, visc_law=W.VISC_SUTHERLAND,
                  mu_ref=0.1, w0=W.conserved_from_primitive(one, 0 * one, 0 * one, 0 * one, one, GAMMA))
    eyc, eyv, eyyv, ypad = O.Oracle(case).metrics()
    h = L / n                                   # oracle's eta has unit spacing: eta_oracle = eta / h
    yp = (1 + 0.25 * np.cos(eta)) * h
    ypp = (-0.25 * np.sin(eta)) * h * h
    assert np.allclose(eyc, 1 / yp, rtol=1e-8) and np.allclose(eyv, 1 / yp, rtol=1e-8)
    assert np.allclose(eyyv, -ypp / yp ** 3, rtol=1e-6, atol=1e-8)
    assert np.allclose(ypad[:3], y[-3:] - L) and np.allclose(ypad[-3:], y[:3] + L)


def _wall_case(ny=24, shear=0.0, tgrad=0.0, top=W.BC_FREESTREAM, visc=W.VISC_POWER, tw=1.3):
    nx, nz = 6, 5
    ly = 1.0
    eta = (np.arange(ny) + 0.5) / ny
    y = ly * (1 - np.tanh(1.5 * (1 - eta)) / np.tanh(1.5)) if top != W.BC_WALL_ISOTHERMAL else \
        ly * 0.5 * (1 + np.tanh(1.5 * (2 * eta - 1)) / np.tanh(1.5))
    Y = np.broadcast_to(y[None, :, None], (nz, ny, nx))
    T = tw + tgrad * Y
    p = 0.8 * np.ones_like(Y)
    rho = p / (RGAS * T)
    u = shear * Y
    zero = np.zeros_like(Y)
    case = W.Case(name="wall", nx=nx, ny=ny, nz=nz, lx=1.0, ly=ly, lz=1.0, y_nodes=y, y_wall_lo=0.0, y_wall_hi=ly,
                  bc_y_lo=W.BC_WALL_ISOTHERMAL, bc_y_hi=top, t_wall_lo=tw, t_wall_hi=tw,
                  gamma=GAMMA, rgas=RGAS, prandtl=PR, visc_law=visc, pow_exp=0.0, mu_ref=0.03, t_ref=1.0,
                  freestream=(0.8 / (RGAS * (tw + tgrad * ly)), 0, 0, 0, 0.8 / (GAMMA - 1)),
                  w0=W.conserved_from_primitive(rho, u, zero, zero, p, GAMMA))
    return case, y


@pytest.mark.parametrize("top", [W.BC_WALL_ISOTHERMAL, W.BC_FREESTREAM])
def test_fluid_at_rest_at_wall_temperature_stays_at_rest(top):
    """O6 / S15 pin: u = 0, T = T_w, uniform p  =>  R = 0 to round-off (rho_ghost is recomputed)."""
    case, _ = _wall_case(top=top, visc=W.VISC_SUTHERLAND)
    R = O.Oracle(case).rhs()
    scale = 0.8 * 24            # p / dy_min-ish
    assert np.max(np.abs(R)) < 1e-12 * scale


def test_wall_ghosts_are_the_odd_reflection():
    """O6: u_i(-1-m) = -u_i(m), T(-1-m) = 2 T_w - T(m), p(-1-m) = p(m), rho = p / (R T)."""
    case, y = _wall_case(shear=0.7, tgrad=0.4)
    o = O.Oracle(case)
    o.rhs()
    pad = [o.padded(q) for q in range(5)]
    g = o.ng
    w0 = case.w0
    for m in range(g):
        rho_i, ru_i, E_i = w0[0][:, m, :], w0[1][:, m, :], w0[4][:, m, :]
        u_i = ru_i / rho_i
        p_i = (GAMMA - 1) * (E_i - 0.5 * rho_i * u_i ** 2)
        T_i = p_i / (RGAS * rho_i)
        sl = (slice(g, -g), g - 1 - m, slice(g, -g))
        rho_g = pad[0][sl]
        u_g = pad[1][sl] / rho_g
        p_g = (GAMMA - 1) * (pad[4][sl] - 0.5 * rho_g * u_g ** 2)
        assert np.allclose(u_g, -u_i, rtol=1e-14)
        assert np.allclose(p_g, p_i, rtol=1e-13)
        assert np.allclose(p_g / (RGAS * rho_g), 2 * 1.3 - T_i, rtol=1e-13)
    ypad = o.metrics()[3]
    assert np.allclose(ypad[:g], -y[:g][::-1])           # node array reflected about the wall plane y = 0


def test_linear_shear_and_temperature_at_a_wall():
    """O6 pin: u = S y, T = T_w + G y (the odd reflection is their exact continuation), constant mu:
    viscous x-momentum = 0, energy = mu S^2 (dissipation), conduction = 0, right up to the wall."""
    S, G, mu = 0.7, 0.0, 0.03
    case, y = _wall_case(shear=S, tgrad=G)
    R = O.Oracle(case).rhs(parts=O.PART_VISC)
    near = slice(0, 12)                                     # the wall-side half, away from the top boundary
    assert np.max(np.abs(R[1][:, near, :])) < 1e-10
    assert np.allclose(R[4][:, near, :], mu * S * S, rtol=1e-10)
    # with a temperature gradient and constant mu: lambda lap(T) = 0, still only dissipation
    case, y = _wall_case(shear=S, tgrad=0.4)
    R = O.Oracle(case).rhs(parts=O.PART_VISC)
    assert np.allclose(R[4][:, near, :], mu * S * S, rtol=1e-9)


def test_poiseuille_balance_away_from_the_walls():
    """O6 pin: parabolic profile, constant mu: mu u_yy = -2 mu U / h^2 to round-off wherever the
    stencil does not reach the reflected ghosts (a parabola is not odd about the wall)."""
    ny, U, mu = 32, 1.1, 0.03
    nx, nz = 5, 4
    eta = -1 + (2 * np.arange(ny) + 1) / ny
    y = np.tanh(1.5 * eta) / np.tanh(1.5)
    Y = np.broadcast_to(y[None, :, None], (nz, ny, nx))
    one = np.ones_like(Y)
    case = W.Case(name="pois", nx=nx, ny=ny, nz=nz, lx=1.0, ly=2.0, lz=1.0, y_nodes=y, y_wall_lo=-1.0, y_wall_hi=1.0,
                  bc_y_lo=W.BC_WALL_ISOTHERMAL, bc_y_hi=W.BC_WALL_ISOTHERMAL, visc_law=W.VISC_POWER, pow_exp=0.0,
                  mu_ref=mu, w0=W.conserved_from_primitive(one, U * (1 - Y * Y), 0 * one, 0 * one, one, GAMMA))
    R = O.Oracle(case).rhs(parts=O.PART_VISC)
    inner = slice(3, ny - 3)
    assert np.allclose(R[1][:, inner, :], -2 * mu * U, rtol=1e-5)      # 6th-order metric error of the tanh map
    assert np.max(np.abs(R[1][:, 0, :] + 2 * mu * U)) > 1e-3           # and the wall node does see the kink
