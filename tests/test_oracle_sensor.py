"""Pins for the shock sensor, node mask and interface flags."""
import numpy as np
import pytest

import workloads as W
from oracle import oracle as O


def _linear_case(grad, stretched=False, n=(14, 13, 12), eps_ul=(1.0, 100.0)):
    """Velocity field u_a = sum_b grad[a][b] x_b on a box with free-stream ghosts; only nodes
    at least ng away from every face see exact central differences (linear data)."""
    nx, ny, nz = n
    lx, ly, lz = 1.4, 1.3, 1.2
    x = np.arange(nx) * lx / nx
    z = np.arange(nz) * lz / nz
    if stretched:
        eta = (np.arange(ny) + 0.5) / ny
        y = ly * (eta + 0.15 * np.sin(2 * np.pi * eta) / (2 * np.pi))
    else:
        y = (np.arange(ny) + 0.5) * ly / ny
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    g = np.asarray(grad, dtype=float)
    vel = [g[a, 0] * X + g[a, 1] * Y + g[a, 2] * Z for a in range(3)]
    one = np.ones_like(X)
    case = W.Case(name="lin", nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz,
                  y_nodes=y if stretched else None, y_wall_lo=0.0, y_wall_hi=ly,
                  bc_x=W.BC_FREESTREAM, bc_y_lo=W.BC_FREESTREAM, bc_y_hi=W.BC_FREESTREAM, bc_z=W.BC_FREESTREAM,
                  flux_mode=W.FLUX_HYBRID, u_ref=eps_ul[0], l_ref=eps_ul[1], sensor_threshold=0.5,
                  w0=W.conserved_from_primitive(one, vel[0], vel[1], vel[2], one, 1.4))
    o = O.Oracle(case, kind="serial")
    o.rhs()
    th, mk, dv = o.sensor()
    s = (slice(3, -3),) * 3
    return th[s], mk[s], dv[s]


@pytest.mark.parametrize("stretched", [False, True])
def test_sensor_closed_forms(stretched):
    eps = (1.0 / 100.0) ** 2
    # solid-body rotation about z: theta = 0, div = 0
    th, mk, dv = _linear_case([[0, -2, 0], [2, 0, 0], [0, 0, 0]], stretched)
    assert np.all(th == 0.0) and np.all(mk == 0) and np.max(np.abs(dv)) < 1e-12
    # isotropic compression u = -alpha x: theta = 3 alpha / sqrt(9 alpha^2 + eps)
    al = 0.7
    th, mk, dv = _linear_case(-al * np.eye(3), stretched)
    assert np.allclose(dv, -3 * al, rtol=1e-12)
    assert np.allclose(th, 3 * al / np.sqrt(9 * al * al + eps), rtol=1e-12)
    assert np.all(mk == 1)
    # pure expansion: theta = 0
    th, mk, dv = _linear_case(al * np.eye(3), stretched)
    assert np.all(th == 0.0) and np.all(mk == 0)
    # compression in y only plus shear du/dz = s (vorticity magnitude s): theta = a / sqrt(a^2 + s^2 + eps)
    a, s = 0.9, 1.7
    th, mk, dv = _linear_case([[0, 0, s], [0, -a, 0], [0, 0, 0]], stretched)
    assert np.allclose(th, a / np.sqrt(a * a + s * s + eps), rtol=1e-12)
    # every component of the curl enters: shear dw/dx and dv/dz
    th, _, _ = _linear_case([[0, 0, 0], [0, -a, 1.1], [0.6, 0, 0]], stretched)
    assert np.allclose(th, a / np.sqrt(a * a + 1.1 ** 2 + 0.6 ** 2 + eps), rtol=1e-12)
    assert np.all((th >= 0) & (th <= 1))


def test_theta_tends_to_one_as_regulariser_vanishes():
    th, _, _ = _linear_case(-0.3 * np.eye(3), eps_ul=(1e-9, 1.0))
    assert np.allclose(th, 1.0, atol=1e-12)


def test_threshold_is_strict_and_mask_matches_theta():
    rng = np.random.default_rng(0)
    n = 12
    f = lambda: rng.uniform(-1, 1, (n, n, n))
    one = np.ones((n, n, n))
    case = W.Case(name="thr", nx=n, ny=n, nz=n, lx=1.0, ly=1.0, lz=1.0, flux_mode=W.FLUX_HYBRID,
                  sensor_threshold=0.3, u_ref=1.0, l_ref=1.0,
                  w0=W.conserved_from_primitive(one, f(), f(), f(), one, 1.4))
    o = O.Oracle(case)
    o.rhs()
    th, mk, _ = o.sensor()
    assert np.array_equal(mk, (th > 0.3).astype(np.uint8))
    assert 0 < mk.mean() < 1


@pytest.mark.parametrize("weno_order,r", [(3, 2), (5, 3), (7, 4)])
def test_interface_flags_are_the_2r_dilation_of_the_node_mask(weno_order, r):
    """O2 / S5 brute force: interface i+1/2 flagged iff any node in {i-r+1..i+r} is flagged,
    periodic wrap."""
    rng = np.random.default_rng(1)
    nx, ny, nz = 13, 11, 12
    mask = (rng.uniform(size=(nz, ny, nx)) < 0.04).astype(np.uint8)
    one = np.ones((nz, ny, nx))
    case = W.Case(name="dil", nx=nx, ny=ny, nz=nz, lx=1.0, ly=1.0, lz=1.0, flux_mode=W.FLUX_HYBRID,
                  weno_order=weno_order, central_order=8,
                  w0=W.conserved_from_primitive(one, 0 * one, 0 * one, 0 * one, one, 1.4))
    o = O.Oracle(case, kind="serial")
    o.set_mask_override(mask)
    o.rhs()
    _, mk, _ = o.sensor()
    assert np.array_equal(mk, mask)
    for d in range(3):
        axis = 2 - d
        n = mask.shape[axis]
        flags = o.interface_flags(d)
        expect = np.zeros_like(mask)
        for m in range(-r + 1, r + 1):
            expect |= np.roll(mask, -m, axis=axis)     # expect[i] = OR mask[i+m]
        # flags index s <-> interface (s-1)+1/2 ; s = 1..n is interface i = s-1
        got = np.take(flags, np.arange(1, n + 1), axis=axis)
        assert np.array_equal(got, expect)
        first = np.take(flags, [0], axis=axis)          # interface -1/2 == interface n-1/2 (periodic)
        last = np.take(flags, [n], axis=axis)
        assert np.array_equal(first, last)


def test_central_and_weno_modes_ignore_the_mask():
    one = np.ones((8, 8, 8))
    base = dict(name="m", nx=8, ny=8, nz=8, lx=1.0, ly=1.0, lz=1.0,
                w0=W.conserved_from_primitive(one, 0 * one, 0 * one, 0 * one, one, 1.4))
    o = O.Oracle(W.Case(flux_mode=W.FLUX_WENO, **base), kind="serial")
    o.rhs()
    assert all(o.interface_flags(d).all() for d in range(3))
    o = O.Oracle(W.Case(flux_mode=W.FLUX_CENTRAL, **base), kind="serial")
    o.rhs()
    assert not any(o.interface_flags(d).any() for d in range(3))
