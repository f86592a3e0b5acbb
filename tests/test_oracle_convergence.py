"""T4: design order of convergence on a smooth advected density wave with a closed-form
solution, and O5 pins for the RK3 scheme and the time step."""
import numpy as np
import pytest

import workloads as W
from oracle import oracle as O

GAMMA = 1.4


def _wave_case(n, kvec, u0, tfinal, steps, mode=W.FLUX_CENTRAL, order=6, weno_order=5, amp=0.2):
    """rho = 1 + amp sin(k.(x - u0 t)), uniform velocity u0 and pressure: an exact solution of the
    Euler equations.  Grid has n nodes along every direction with k != 0 and 4 along the others."""
    dims = [n if kvec[a] != 0 else 4 for a in range(3)]
    nx, ny, nz = dims
    L = 2 * np.pi
    x = np.arange(nx) * L / nx
    y = np.arange(ny) * L / ny
    z = np.arange(nz) * L / nz
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    phase = kvec[0] * X + kvec[1] * Y + kvec[2] * Z
    one = np.ones_like(X)
    rho0 = 1 + amp * np.sin(phase)
    case = W.Case(name="wave", nx=nx, ny=ny, nz=nz, lx=L, ly=L, lz=L, flux_mode=mode, central_order=order,
                  weno_order=weno_order, dt_fixed=tfinal / steps,
                  w0=W.conserved_from_primitive(rho0, u0[0] * one, u0[1] * one, u0[2] * one, one, GAMMA))
    o = O.Oracle(case)
    o.step(steps)
    w = o.get_fields()
    exact = 1 + amp * np.sin(phase - np.dot(kvec, u0) * tfinal)
    return w[0] - exact, w


def _orders(errs):
    return [np.log2(errs[i] / errs[i + 1]) for i in range(len(errs) - 1)]


@pytest.mark.parametrize("kvec,u0", [((1, 0, 0), (1.0, 0.3, -0.2)), ((0, 1, 0), (0.3, 1.0, -0.2)),
                                     ((0, 0, 1), (0.3, -0.2, 1.0)), ((1, 1, 0), (0.7, 0.5, 0.1))])
def test_central_scheme_reaches_design_order_6(kvec, u0):
    errs = []
    for n in (16, 32, 64):
        steps = max(4, int(round(4 * (n / 16) ** 2)))      # dt ~ dx^2 keeps the RK3 error below the spatial one
        e, _ = _wave_case(n, kvec, np.array(u0), 0.1, steps)
        errs.append(np.sqrt(np.mean(e * e)))
    od = _orders(errs)
    assert od[-1] >= 6 - 0.3, (errs, od)


@pytest.mark.parametrize("order", [2, 4, 8])
def test_central_scheme_other_orders(order):
    errs = []
    for n in (16, 32, 64):
        steps = max(8, int(round(8 * (n / 16) ** 3)))
        e, _ = _wave_case(n, (1, 0, 0), np.array([1.0, 0.0, 0.0]), 0.05, steps, order=order)
        errs.append(np.sqrt(np.mean(e * e)))
    od = _orders(errs)
    assert od[-1] >= order - 0.3, (errs, od)


def test_momentum_flux_is_u0_times_mass_flux_on_the_density_wave():
    """With uniform u0 and p the cubic split gives R^{rho u_i} = u0_i R^{rho} (the triple average
    reduces to u0 times the mass flux and the pressure flux is uniform), to round-off."""
    n = 24
    L = 2 * np.pi
    x = np.arange(n) * L / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    one = np.ones_like(X)
    u0 = (1.0, 0.3, -0.2)
    rho = 1 + 0.2 * np.sin(X + 2 * Y - Z)
    case = W.Case(name="w", nx=n, ny=n, nz=n, lx=L, ly=L, lz=L,
                  w0=W.conserved_from_primitive(rho, u0[0] * one, u0[1] * one, u0[2] * one, one, GAMMA))
    R = O.Oracle(case).rhs()
    for a in range(3):
        assert np.max(np.abs(R[1 + a] - u0[a] * R[0])) < 1e-13 * np.max(np.abs(R[0]))
    # and the mass equation is the plain advection operator: R^rho = -u0 . grad(rho) to 6th order
    exact = -0.2 * np.cos(X + 2 * Y - Z) * (u0[0] + 2 * u0[1] - u0[2])
    assert np.max(np.abs(R[0] - exact)) < 2e-5


@pytest.mark.parametrize("weno_order,expect", [(3, 1.8), (5, 4.5), (7, 6.0)])
def test_weno_only_mode_order_in_l1(weno_order, expect):
    """O3 pin (vi): WENO everywhere on the smooth wave, order ~ 2r-1 in L1 (JS weights lose
    accuracy only at the critical points)."""
    errs = []
    ns = (16, 32, 64) if weno_order < 7 else (12, 24, 48)
    for n in ns:
        steps = max(8, int(round(8 * (n / 16) ** 3)))
        e, _ = _wave_case(n, (1, 0, 0), np.array([1.0, 0.0, 0.0]), 0.05, steps, mode=W.FLUX_WENO,
                          weno_order=weno_order, order=8, amp=0.2)
        errs.append(np.mean(np.abs(e)))
    od = _orders(errs)
    assert od[-1] >= expect, (errs, od)


# ------------------------------------------------------------------ RK3
def test_rk3_amplification_factor_is_the_cubic_taylor_polynomial():
    """O5 pin: on the density wave the mass equation is linear (u stays uniform), so one RK3 step
    multiplies the Fourier mode e^{ikx} by 1 + z + z^2/2 + z^3/6, z = -i u0 k_eff dt, where
    k_eff = (2/dx) sum_l a_l sin(l k dx) is the symbol of the 6th-order central difference."""
    n, k, u0, dt = 32, 3, 0.9, 0.02
    L = 2 * np.pi
    x = np.arange(n) * L / n
    amp = 1e-3
    rho0 = 1 + amp * np.cos(k * x)
    shp = (4, 4, n)
    b = lambda a: np.broadcast_to(a, shp).copy()
    case = W.Case(name="lin", nx=n, ny=4, nz=4, lx=L, ly=L, lz=L, dt_fixed=dt,
                  w0=W.conserved_from_primitive(b(rho0), b(u0 * np.ones(n)), b(0 * x), b(0 * x), b(np.ones(n)), GAMMA))
    o = O.Oracle(case)
    o.step(1)
    rho1 = o.get_fields()[0][0, 0]
    dx = L / n
    a = [3 / 4, -3 / 20, 1 / 60]
    keff = (2 / dx) * sum(a[l - 1] * np.sin(l * k * dx) for l in (1, 2, 3))
    z = -1j * u0 * keff * dt
    G = 1 + z + z * z / 2 + z ** 3 / 6
    c0 = np.fft.fft(rho0)[k]
    c1 = np.fft.fft(rho1)[k]
    assert abs(c1 / c0 - G) < 1e-11
    # a second-order or mis-weighted scheme would miss the z^3/6 term by ~ |z|^3/6
    assert abs(z) ** 3 / 6 > 1e-6


def test_rk3_third_order_in_time():
    """O5 pin: temporal order 3 on a fixed grid (difference to a 8x finer time step)."""
    def run(steps):
        _, w = _wave_case(16, (1, 0, 0), np.array([1.0, 0.2, 0.0]), 0.4, steps, amp=0.2)
        return w
    ref = run(64)
    e = [np.max(np.abs(run(s) - ref)) for s in (4, 8, 16)]
    od = _orders(e)
    assert 2.7 < od[0] < 3.4 and 2.7 < od[1] < 3.6, (e, od)


# ------------------------------------------------------------------ time step
def test_dt_closed_form_convective_and_viscous_limits():
    """O5 / S13: dt = CFL / max{(|u_d|+c) m_d, nu m_d^2, gamma nu m_d^2 / Pr}."""
    nx, ny, nz = 8, 6, 10
    lx, ly, lz = 1.0, 0.3, 2.0
    one = np.ones((nz, ny, nx))
    rho, p = 1.2, 0.9
    vel = (0.3, -0.8, 0.5)
    w0 = W.conserved_from_primitive(rho * one, vel[0] * one, vel[1] * one, vel[2] * one, p * one, GAMMA)
    c = np.sqrt(GAMMA * p / rho)
    m = (nx / lx, ny / ly, nz / lz)
    conv = max((abs(vel[d]) + c) * m[d] for d in range(3))
    case = W.Case(name="dt", nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz, cfl=0.7, w0=w0)
    assert abs(O.Oracle(case).compute_dt() - 0.7 / conv) < 1e-15
    # viscous-limited: power law with exponent 0 -> mu = mu_ref
    mu = 5.0
    case = case.replace(visc_law=W.VISC_POWER, pow_exp=0.0, mu_ref=mu, prandtl=0.5)
    visc = max(GAMMA * (mu / rho) / 0.5 * m[d] ** 2 for d in range(3))
    assert visc > conv
    assert abs(O.Oracle(case).compute_dt() - 0.7 / visc) < 1e-12 * (0.7 / visc)
    # stretched y: the largest eta_y rules
    y = np.cumsum(np.array([0.02, 0.03, 0.05, 0.07, 0.08, 0.05]))
    case = W.Case(name="dt", nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz, cfl=0.7, w0=w0, y_nodes=y,
                  bc_y_lo=W.BC_FREESTREAM, bc_y_hi=W.BC_FREESTREAM, y_wall_lo=0.0, y_wall_hi=0.33)
    o = O.Oracle(case)
    eta_y = o.metrics()[0]
    conv = max((abs(vel[0]) + c) * m[0], (abs(vel[1]) + c) * eta_y.max(), (abs(vel[2]) + c) * m[2])
    assert abs(o.compute_dt() - 0.7 / conv) < 1e-14


def test_dt_every_reuses_the_time_step():
    case = W.config(0).replace(dt_every=3)
    o = O.Oracle(case)
    dts = [o.step(1)[0] for _ in range(4)]
    assert dts[0] == dts[1] == dts[2] and dts[3] != dts[0]
    o2 = O.Oracle(W.config(0).replace(dt_fixed=1e-3))
    dt, t = o2.step(3)
    assert dt == 1e-3 and abs(t - 3e-3) < 1e-18
