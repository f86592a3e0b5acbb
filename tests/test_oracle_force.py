"""Pins of the oracle's body force (reading S17; "forcing term evaluations"): a uniform acceleration g adds
rho g to the momentum equations and its work (rho u).g to the total energy.  Checked against what the mathematics fixes:
the exact right-hand side of a uniform state, the momentum and energy budgets of a periodic box, and the Poiseuille
flow that g = 2 mu U / (rho h^2) holds steady."""
import numpy as np

import workloads as W
from oracle import oracle as O
from tests.helpers import random_periodic_case

GAMMA = 1.4


def test_uniform_state_gives_exactly_rho_g_and_its_work():
    rho0, vel, p0, g = 1.3, (0.4, -0.2, 0.7), 0.9, (0.05, -0.11, 0.23)
    shape = (7, 9, 8)
    one = np.ones(shape)
    case = W.Case(name="uni", nx=8, ny=9, nz=7, lx=1.0, ly=1.3, lz=0.8, gamma=GAMMA, flux_mode=W.FLUX_CENTRAL, accel=g,
                  w0=W.conserved_from_primitive(rho0 * one, vel[0] * one, vel[1] * one, vel[2] * one, p0 * one, GAMMA))
    R = O.Oracle(case).rhs()
    assert np.max(np.abs(R[0])) == 0.0                                   # free stream: the fluxes cancel exactly
    for a in range(3):
        assert np.allclose(R[1 + a], rho0 * g[a], rtol=0, atol=1e-15)
    work = rho0 * (vel[0] * g[0] + vel[1] * g[1] + vel[2] * g[2])
    assert np.allclose(R[4], work, rtol=0, atol=1e-15)
    # the force-only part of the right-hand side, and nothing else, changes with g
    R_only = O.Oracle(case).rhs(parts=O.PART_FORCE)
    assert np.array_equal(R_only[0], np.zeros(shape)) and np.allclose(R_only[1], rho0 * g[0], atol=1e-15)
    assert np.max(np.abs(O.Oracle(case.replace(accel=(0.0, 0.0, 0.0))).rhs()[1:])) < 1e-13


def test_force_is_additive_and_budgets_of_a_periodic_box():
    """sum R(rho u_a) = g_a sum rho and sum R(rho E) = g . sum(rho u) on any periodic field (the fluxes telescope)."""
    g = (0.3, 0.0, -0.2)
    case, (rho, u, v, w, p) = random_periodic_case(12, 10, 11, seed=4, flux_mode=W.FLUX_CENTRAL)
    R0 = O.Oracle(case).rhs()
    R1 = O.Oracle(case.replace(accel=g)).rhs()
    w0 = case.w0
    for a in range(3):
        assert np.allclose(R1[1 + a] - R0[1 + a], w0[0] * g[a], rtol=1e-12, atol=1e-14)
    assert np.allclose(R1[4] - R0[4], w0[1] * g[0] + w0[2] * g[1] + w0[3] * g[2], rtol=1e-12, atol=1e-14)
    assert np.array_equal(R1[0], R0[0])
    for a in range(3):
        assert abs(R1[1 + a].sum() - g[a] * w0[0].sum()) < 1e-10
    assert abs(R1[4].sum() - (g[0] * w0[1].sum() + g[2] * w0[3].sum())) < 1e-10


def test_poiseuille_flow_is_held_steady_by_its_force():
    """u = U (1 - y^2), constant mu, uniform rho and p: the viscous x-momentum term is -2 mu U, so g = 2 mu U / rho balances
    it (away from the wall nodes, whose stencil sees the reflected ghosts), and the transverse momenta stay zero."""
    ny, U, mu = 32, 1.1, 0.03
    nx, nz = 5, 4
    eta = -1 + (2 * np.arange(ny) + 1) / ny
    y = np.tanh(1.5 * eta) / np.tanh(1.5)
    Y = np.broadcast_to(y[None, :, None], (nz, ny, nx))
    one = np.ones_like(Y)
    case = W.Case(name="pois_g", nx=nx, ny=ny, nz=nz, lx=1.0, ly=2.0, lz=1.0, y_nodes=y, y_wall_lo=-1.0, y_wall_hi=1.0,
                  bc_y_lo=W.BC_WALL_ISOTHERMAL, bc_y_hi=W.BC_WALL_ISOTHERMAL, visc_law=W.VISC_POWER, pow_exp=0.0,
                  mu_ref=mu, accel=(2 * mu * U, 0.0, 0.0), flux_mode=W.FLUX_CENTRAL,
                  w0=W.conserved_from_primitive(one, U * (1 - Y * Y), 0 * one, 0 * one, one, GAMMA))
    R = O.Oracle(case).rhs()
    inner = slice(3, ny - 3)
    assert np.max(np.abs(R[1][:, inner, :])) < 1e-5 * 2 * mu * U * 10      # 6th-order metric error of the tanh map
    assert np.max(np.abs(R[2])) < 1e-12 and np.max(np.abs(R[3])) < 1e-12
    # without the force the same nodes decelerate at -2 mu U
    R0 = O.Oracle(case.replace(accel=(0.0, 0.0, 0.0))).rhs()
    assert np.allclose(R0[1][:, inner, :], -2 * mu * U, rtol=1e-4)
