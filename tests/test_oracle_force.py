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


# ---- S18: the bulk-flow controller (PAPER:377, 386 force_rhs); the paper prints no formula, the pins are its properties
def test_controller_is_deadbeat_on_a_frictionless_uniform_flow():
    """Uniform state in a periodic inviscid box: the right-hand side is the body force alone, so a force g acting for
    one step changes the bulk momentum P by exactly g M dt.  Started 10 % below its target, P is on target after the
    first controlled step (to round-off), the force that brought it there was (P_target - P0) / (M dt), and from then on
    the force returns to zero and P stays put."""
    n = 8
    one = np.ones((n, n, n))
    rho0, u0, p0 = 1.3, 0.5, 1.1
    case = W.Case(name="ctrl", nx=n, ny=n, nz=n, lx=1.0, ly=1.0, lz=1.0, dt_fixed=1e-2,
                  w0=W.conserved_from_primitive(rho0 * one, u0 * one, 0 * one, 0 * one, p0 * one, 1.4))
    o = O.Oracle(case, kind="serial")
    mass, mom0 = o.bulk_sums(0)
    assert np.isclose(mass, rho0, rtol=1e-14) and np.isclose(mom0, rho0 * u0, rtol=1e-14)      # unit volume
    target = 1.1 * mom0
    dt, t, g = o.step_forced(1, 0, target)           # step 1 runs unforced, then the controller sets g
    assert np.isclose(o.bulk_sums(0)[1], mom0, rtol=1e-14)
    assert np.isclose(g[0], (target - mom0) / (mass * dt), rtol=1e-12) and g[1] == 0.0 and g[2] == 0.0
    dt, t, g = o.step_forced(1, 0)                   # step 2 under that force lands on the target
    assert np.isclose(o.bulk_sums(0)[1], target, rtol=1e-13)
    assert abs(g[0]) <= 1e-10 * abs(target - mom0) / (mass * dt)
    for _ in range(3):
        dt, t, g = o.step_forced(1, 0)
        assert np.isclose(o.bulk_sums(0)[1], target, rtol=1e-13)
    # the energy integral has grown by the work of the force, the mass is untouched
    assert np.isclose(o.bulk_sums(0)[0], mass, rtol=1e-14)


def test_controller_holds_a_laminar_channel_against_wall_friction():
    """Poiseuille-like profile between isothermal walls: without a force the bulk momentum decays (wall friction);
    under the controller it is back on target after every step to 1e-6 of the drift an unforced step leaves, and the
    force settles near the friction it balances, tau_w * wall area / mass."""
    case = W.channel(24, 24, 12, seed=3)
    case = case.replace(flux_mode=W.FLUX_CENTRAL, dt_fixed=0.0)
    free = O.Oracle(case, kind="serial")
    m0, p0 = free.bulk_sums(0)
    free.step(6)
    drift = p0 - free.bulk_sums(0)[1]
    assert drift > 0
    o = O.Oracle(case, kind="serial")
    gs = []
    for _ in range(6):
        dt, t, g = o.step_forced(1, 0)
        gs.append(g[0])
    # P one step after an update: the controller corrected the previous deviation; what remains is the change of the
    # friction over one step, far below the unforced drift
    o.step_forced(1, 0)
    assert abs(o.bulk_sums(0)[1] - p0) < 0.05 * drift / 6
    assert gs[-1] > 0 and abs(gs[-1] - gs[-2]) < 0.2 * abs(gs[-1])
