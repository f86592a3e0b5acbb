"""Pins for the oracle's central convective flux (tests T1, T2, T3, T5)."""
from fractions import Fraction
import os

import numpy as np
import pytest

import workloads as W
from oracle import oracle as O
from tests.helpers import random_periodic_case

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden_coeffs():
    out = {}
    for line in open(os.path.join(GOLD, "fd_coefficients.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        out[(int(t[0]), t[1])] = [float(Fraction(x)) for x in t[2:]]
    return out


def test_fd_coefficients_match_golden_and_taylor():
    gold = _golden_coeffs()
    for order in (2, 4, 6, 8):
        a, b = O.fd_coeffs(order)
        assert np.array_equal(a, np.array(gold[(order, "a")]))
        assert np.array_equal(b, np.array(gold[(order, "b")]))
        # Taylor conditions: sum 2 l a_l = 1, sum l^(2m+1) a_l = 0 (m = 1..L-1);
        # sum l^2 b_l = 1, sum l^(2m) b_l = 0 (m = 2..L)
        ls = np.arange(1, order // 2 + 1, dtype=float)
        assert abs(np.sum(2 * ls * a) - 1) < 1e-14
        assert abs(np.sum(ls ** 2 * b) - 1) < 1e-14
        for m in range(1, order // 2):
            assert abs(np.sum(ls ** (2 * m + 1) * a)) < 1e-12
            assert abs(np.sum(ls ** (2 * m + 2) * b)) < 1e-12


def _D(f, axis, order, h):
    """Plain central difference of order `order` on a periodic array (numpy reference)."""
    gold = _golden_coeffs()[(order, "a")]
    out = np.zeros_like(f)
    for l, a in enumerate(gold, start=1):
        out += a * (np.roll(f, -l, axis=axis) - np.roll(f, l, axis=axis))
    return out / h


@pytest.mark.parametrize("order", [2, 4, 6, 8])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_flux_difference_equals_expanded_split_form(order, d):
    """O1 pin (i): -(f_{i+1/2} - f_{i-1/2})/h equals the seven-term split form
    1/4 [D(rho u phi) + rho D(u phi) + u D(rho phi) + phi D(rho u) + rho u D phi + rho phi D u + u phi D rho]
    plus D(p) on the d-momentum, D the plain central difference."""
    case, (rho, u, v, w, p) = random_periodic_case(9, 10, 11, seed=order + d, central_order=order)
    o = O.Oracle(case, kind="serial")
    R = o.rhs(parts=1 << d)
    axis = 2 - d                      # arrays are [z, y, x]
    h = (case.lx / case.nx, case.ly / case.ny, case.lz / case.nz)[d]
    ud = (u, v, w)[d]
    gamma = case.gamma
    H = (p / (gamma - 1) + 0.5 * rho * (u * u + v * v + w * w) + p) / rho
    D = lambda f: _D(f, axis, order, h)
    for q, phi in enumerate([np.ones_like(rho), u, v, w, H]):
        split = 0.25 * (D(rho * ud * phi) + rho * D(ud * phi) + ud * D(rho * phi) + phi * D(rho * ud)
                        + rho * ud * D(phi) + rho * phi * D(ud) + ud * phi * D(rho))
        if q == 1 + d:
            split = split + D(p)
        err = np.max(np.abs(R[q] + split)) / np.max(np.abs(split))
        assert err < 5e-14, (q, err)
    # the other directions contribute nothing when their part bit is off
    assert np.all(np.isfinite(R))


def test_pressure_flux_stencil_L3():
    """O1 pin (iv): p^_{i+1/2} has stencil (1,-8,37,37,-8,1)/60 for L=3.  With u = 0 only the
    pressure flux survives; an impulse in p shows the differences of that stencil."""
    n = 16
    rho = np.ones((4, 4, n))
    z = np.zeros_like(rho)
    p = np.ones_like(rho)
    p[:, :, 8] += 1.0
    case = W.Case(name="imp", nx=n, ny=4, nz=4, lx=float(n), ly=4.0, lz=4.0,
                  w0=W.conserved_from_primitive(rho, z, z, z, p, 1.4))
    R = O.Oracle(case, kind="serial").rhs(parts=1)
    resp = -R[1][0, 0, :]            # (p^_{i+1/2} - p^_{i-1/2}) / 1
    # interface i+1/2 sees node 8 with coefficient c[8 - i + 2], c = stencil over nodes i-2..i+3
    c = np.array([1, -8, 37, 37, -8, 1]) / 60.0
    phat = np.zeros(n + 1)           # phat[i+1] = impulse part of p^_{i+1/2}
    for i in range(-1, n):
        k = 8 - i + 2
        if 0 <= k < 6:
            phat[i + 1] = c[k]
    assert np.allclose(resp, phat[1:] - phat[:-1], atol=1e-15)
    assert np.all(R[0] == 0) and np.all(R[4] == 0)


@pytest.mark.parametrize("mode", [W.FLUX_CENTRAL, W.FLUX_WENO, W.FLUX_HYBRID])
def test_conservation_telescoping(mode):
    """T2: sum_i R_i * volume = 0 to round-off in a periodic box without viscosity."""
    case, _ = random_periodic_case(12, 10, 9, seed=3, flux_mode=mode, sensor_threshold=0.05,
                                   u_ref=1.0, l_ref=10.0)
    R = O.Oracle(case).rhs()
    for q in range(5):
        assert abs(R[q].sum()) <= 1e-12 * np.abs(R[q]).sum()


def test_mass_conserved_with_viscosity():
    case, _ = random_periodic_case(12, 10, 9, seed=4, visc_law=W.VISC_SUTHERLAND, mu_ref=0.01)
    R = O.Oracle(case).rhs()
    assert abs(R[0].sum()) <= 1e-12 * np.abs(R[0]).sum()


@pytest.mark.parametrize("order", [2, 6, 8])
def test_kinetic_energy_identity(order):
    """O1 pin (iii) / T3: sum_i [u . C^{rho u} - 1/2 |u|^2 C^{rho}] = 0 for the convective part
    without pressure: the split form conserves kinetic energy discretely."""
    case, (rho, u, v, w, p) = random_periodic_case(10, 9, 8, seed=5, central_order=order)
    R = O.Oracle(case, kind="serial", dbg_flags=O.DBG_NO_PRESSURE).rhs()
    ke_rate = u * R[1] + v * R[2] + w * R[3] - 0.5 * (u * u + v * v + w * w) * R[0]
    assert abs(ke_rate.sum()) <= 1e-13 * np.abs(ke_rate).sum()
    # with pressure the identity must NOT hold (the flag really removes a term)
    R2 = O.Oracle(case, kind="serial").rhs()
    ke2 = u * R2[1] + v * R2[2] + w * R2[3] - 0.5 * (u * u + v * v + w * w) * R2[0]
    assert abs(ke2.sum()) > 1e-6 * np.abs(ke2).sum()


def _stretched_periodic_y(ny, ly):
    eta = np.arange(ny) * (ly / ny)
    return eta + 0.08 * ly / (2 * np.pi) * np.sin(2 * np.pi * eta / ly)


@pytest.mark.parametrize("mode", [W.FLUX_CENTRAL, W.FLUX_WENO, W.FLUX_HYBRID])
@pytest.mark.parametrize("visc", [W.VISC_NONE, W.VISC_SUTHERLAND])
@pytest.mark.parametrize("stretched", [False, True])
def test_free_stream_preserved_bitwise(mode, visc, stretched):
    """T1: a uniform state gives R == 0.0 exactly in every mode, uniform or stretched y."""
    nx, ny, nz = 8, 9, 7
    one = np.ones((nz, ny, nx))
    w0 = W.conserved_from_primitive(1.3 * one, 0.37 * one, -0.21 * one, 0.11 * one, 0.9 * one, 1.4)
    case = W.Case(name="fs", nx=nx, ny=ny, nz=nz, lx=1.0, ly=1.7, lz=0.9, flux_mode=mode, visc_law=visc,
                  mu_ref=0.01, y_nodes=_stretched_periodic_y(ny, 1.7) if stretched else None, w0=w0)
    R = O.Oracle(case).rhs()
    assert np.all(R == 0.0)


def test_tgv_kinetic_energy_initial_value_and_drift():
    """T3: config 0 mean kinetic energy starts at exactly 1/8 (closed form of the TGV field) and,
    for the inviscid central scheme, its change over 10 steps is tiny (pressure-dilatation work)."""
    case = W.config(0)
    w0 = case.w0
    ke0 = float(np.mean(0.5 * (w0[1] ** 2 + w0[2] ** 2 + w0[3] ** 2) / w0[0]))
    assert abs(ke0 - 0.125) < 1e-15
    o = O.Oracle(case)
    dt, t = o.step(10)
    assert abs(dt - 0.5 / ((1.0 + np.sqrt(1.4 * case.rgas)) * 32 / (2 * np.pi))) < 2e-4   # CFL dt, |u|max ~ 1
    w1 = o.get_fields()
    ke1 = float(np.mean(0.5 * (w1[1] ** 2 + w1[2] ** 2 + w1[3] ** 2) / w1[0]))
    assert abs(ke1 - ke0) < 2e-6
    for q in range(5):   # conservation over the run
        assert abs(w1[q].sum() - w0[q].sum()) <= 1e-12 * np.abs(w0[q]).sum() + 1e-9


def test_serial_and_openmp_builds_bit_identical():
    """T6: threading invariance."""
    case, _ = random_periodic_case(12, 11, 10, seed=7, flux_mode=W.FLUX_HYBRID, sensor_threshold=0.05,
                                   visc_law=W.VISC_SUTHERLAND, mu_ref=0.01, u_ref=1.0, l_ref=10.0,
                                   dt_fixed=1e-3)
    a, b = O.Oracle(case, kind="serial"), O.Oracle(case, kind="omp")
    assert np.array_equal(a.rhs(), b.rhs())
    a.step(2)
    b.step(2)
    assert np.array_equal(a.get_fields(), b.get_fields())
