"""Pins for the three oracle branches that the other pin files do not reach:

  * fill_scalar_ghosts, non-periodic side (constant extrapolation of theta / div / mask),
  * viscosity(), power-law branch with a non-zero exponent,
  * wall_image, the T_ghost >= 0.1 T_w clamp.

None of them retypes the oracle's own formula: the flags are compared with a brute-force dilation written with
clamped indices; the dilatation ghosts with the exact continuation of a field whose dilatation is constant, and with
golden-coefficient differences of the oracle's interior dilatation extended by hand; the power law with
sympy-differentiated Navier-Stokes terms; the clamp with the thermodynamic state read back from the conserved ghost
values.  Each was checked to fail under the matching mutation of the oracle (mirrored / shifted / wrapped source index,
div ghosts not filled, clamp removed, T_ref dropped).
"""
import numpy as np
import pytest
import sympy as sp

import workloads as W
from oracle import oracle as O

GAMMA, RGAS, PR = 1.4, 1.0, 0.72


# ------------------------------------------------------------------------------------------------
# S6: node-mask ghosts beyond a non-periodic face = the nearest interior value
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("weno_order,r", [(3, 2), (5, 3), (7, 4)])
@pytest.mark.parametrize("bcs", ["freestream_all", "wall_lo_free_hi", "periodic_x_only"])
def test_interface_flags_next_to_nonperiodic_faces_use_the_clamped_mask(weno_order, r, bcs):
    """Interface n+1/2 is flagged iff any node of {n-r+1 .. n+r} is; where that window leaves the domain through a
    non-periodic face the node it sees is the nearest interior one (clamped index), through a periodic face the
    wrapped one.  The imposed mask is dense in the three planes next to every face, so ghosts that are wrapped
    across a non-periodic face, left unset, or not filled for the mask at all change some flag.  (A mirrored ghost
    cannot be told from a clamped one here: the window always holds the interior nodes a mirror would copy.  WHICH
    interior value a ghost takes is pinned on the dilatation, below, through the same fill routine.)"""
    rng = np.random.default_rng(7)
    nx, ny, nz = 12, 11, 10
    mask = (rng.uniform(size=(nz, ny, nx)) < 0.03).astype(np.uint8)
    for ax in range(3):
        for side in (slice(0, 3), slice(-3, None)):
            sl = [slice(None)] * 3
            sl[ax] = side
            mask[tuple(sl)] = (rng.uniform(size=mask[tuple(sl)].shape) < 0.3).astype(np.uint8)
    bc_x = W.BC_PERIODIC if bcs == "periodic_x_only" else W.BC_FREESTREAM
    bc_y_lo = W.BC_WALL_ISOTHERMAL if bcs == "wall_lo_free_hi" else W.BC_FREESTREAM
    one = np.ones((nz, ny, nx))
    case = W.Case(name="clamp", nx=nx, ny=ny, nz=nz, lx=1.0, ly=1.0, lz=1.0, y_wall_lo=0.0, y_wall_hi=1.0,
                  bc_x=bc_x, bc_y_lo=bc_y_lo, bc_y_hi=W.BC_FREESTREAM, bc_z=W.BC_FREESTREAM,
                  flux_mode=W.FLUX_HYBRID, weno_order=weno_order, central_order=8,
                  freestream=(1.0, 0.0, 0.0, 0.0, 1.0 / (GAMMA - 1)),
                  w0=W.conserved_from_primitive(one, 0 * one, 0 * one, 0 * one, one, GAMMA))
    o = O.Oracle(case, kind="serial")
    o.set_mask_override(mask)
    o.rhs()
    for d in range(3):
        axis = 2 - d
        n = mask.shape[axis]
        periodic = (d == 0 and bc_x == W.BC_PERIODIC)
        flags = o.interface_flags(d)                       # entry s <-> interface (s - 1) + 1/2, s = 0 .. n
        for s in range(n + 1):
            expect = np.zeros(np.take(mask, 0, axis=axis).shape, dtype=np.uint8)
            for m in range(-r + 1, r + 1):
                src = (s - 1) + m
                src = src % n if periodic else min(max(src, 0), n - 1)
                expect |= np.take(mask, src, axis=axis)
            assert np.array_equal(np.take(flags, s, axis=axis), expect), (d, s)


# ------------------------------------------------------------------------------------------------
# S6: dilatation ghosts beyond a wall feed the (mu/3) grad(div) term of the Laplacian form
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("visc_order", [2, 4, 6, 8])
def test_uniform_compression_towards_a_wall_has_no_dilatation_gradient(visc_order):
    """v = -alpha (y - y_wall), u = w = 0, T = T_w, p uniform: the wall image (v -> -v about the wall plane) is the
    exact continuation of v, so div u = -alpha at every node including j = 0, 1, 2, and the constant extrapolation of
    div into the ghosts is exact.  Then every viscous momentum term vanishes: lap v = 0 (linear), grad mu = 0 (uniform
    T), and (mu/3) d(div)/dy = 0 -- the last one only if the ghost values of div really are div(j = 0): wrapping
    them (the free-stream top has div != -alpha) or leaving them unset leaves an O(alpha mu / dy) residue at the three
    nodes next to the wall.  Energy: mu (4/3) alpha^2 of dissipation."""
    al, mu, tw = 0.8, 0.05, 1.2
    nx, ny, nz = 5, 20, 4
    y = (np.arange(ny) + 0.5) / ny
    Y = np.broadcast_to(y[None, :, None], (nz, ny, nx))
    p = 0.9 * np.ones_like(Y)
    rho = p / (RGAS * tw)
    zero = np.zeros_like(Y)
    case = W.Case(name="compress", nx=nx, ny=ny, nz=nz, lx=1.0, ly=1.0, lz=1.0, y_nodes=y, y_wall_lo=0.0, y_wall_hi=1.0,
                  bc_y_lo=W.BC_WALL_ISOTHERMAL, bc_y_hi=W.BC_FREESTREAM, t_wall_lo=tw, t_wall_hi=tw,
                  gamma=GAMMA, rgas=RGAS, prandtl=PR, visc_law=W.VISC_POWER, pow_exp=0.0, mu_ref=mu, t_ref=1.0,
                  central_order=visc_order, visc_order=visc_order, flux_mode=W.FLUX_HYBRID, weno_order=visc_order - 1,
                  sensor_threshold=0.5, u_ref=1e-6, l_ref=1.0,
                  freestream=(float(rho[0, 0, 0]), 0, 0, 0, 0.9 / (GAMMA - 1)),
                  w0=W.conserved_from_primitive(rho, zero, -al * Y, zero, p, GAMMA))
    o = O.Oracle(case, kind="serial")
    R = o.rhs(parts=O.PART_VISC)
    th, mk, dv = o.sensor()
    near = slice(0, 6)
    assert np.allclose(dv[:, near, :], -al, rtol=1e-12)
    assert np.allclose(th[:, near, :], 1.0, atol=1e-9) and np.all(mk[:, near, :] == 1)
    scale = mu * al * ny                                   # what a wrong div ghost would leave behind
    assert np.max(np.abs(R[2][:, near, :])) < 1e-11 * scale
    assert np.max(np.abs(R[1][:, near, :])) < 1e-11 * scale and np.max(np.abs(R[3][:, near, :])) < 1e-11 * scale
    # energy = dissipation mu (2 S:S - 2/3 div^2) = mu alpha^2 (2 - 2/3), plus v * (momentum residue ~ 0)
    assert np.allclose(R[4][:, near, :], mu * al * al * (4.0 / 3.0), rtol=1e-9)
    # and the check does bite: at the free-stream top the ghost velocities are not the continuation
    assert np.max(np.abs(R[2][:, -3:, :])) > 1e-3 * scale


def _golden_fd(order):
    import os
    from fractions import Fraction
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "fd_coefficients.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            t = line.split()
            if int(t[0]) == order:
                out[t[1]] = np.array([float(Fraction(c)) for c in t[2:]])
    return out["a"], out["b"]


@pytest.mark.parametrize("order", [4, 6, 8])
def test_dilatation_ghosts_at_a_wall_are_the_first_interior_value(order):
    """Which interior value the div ghosts take is visible where div varies next to the wall.  1-D flow between two
    walls, v = A sin(pi y) (odd about both wall planes, so the wall image IS its continuation), T = T_w, uniform p,
    constant mu: the viscous y-momentum is mu D2(v) + (mu/3) D1(div) and nothing else.  D2(v) is formed here from the
    analytic continuation of v with the golden second-derivative coefficients; D1(div) from the oracle's own nodal
    dilatation (interior values, streams_get_sensor's third output) extended by the CLAMPED index, with the golden
    first-derivative coefficients.  The mirrored and the wrapped extension are shown to give a different answer."""
    A, mu, tw = 0.4, 0.05, 1.1
    nx, ny, nz = 4, 24, 3
    L = order // 2
    dy = 1.0 / ny
    jj = np.arange(-L, ny + L)
    yext = (jj + 0.5) * dy
    vext = A * np.sin(np.pi * yext)
    v = vext[L:-L]
    V = np.broadcast_to(v[None, :, None], (nz, ny, nx))
    p = 0.9 * np.ones_like(V)
    rho = p / (RGAS * tw)
    case = W.Case(name="divghost", nx=nx, ny=ny, nz=nz, lx=1.0, ly=1.0, lz=1.0, y_wall_lo=0.0, y_wall_hi=1.0,
                  bc_y_lo=W.BC_WALL_ISOTHERMAL, bc_y_hi=W.BC_WALL_ISOTHERMAL, t_wall_lo=tw, t_wall_hi=tw,
                  gamma=GAMMA, rgas=RGAS, prandtl=PR, visc_law=W.VISC_POWER, pow_exp=0.0, mu_ref=mu, t_ref=1.0,
                  central_order=order, visc_order=order,
                  w0=W.conserved_from_primitive(rho, 0 * V, V, 0 * V, p, GAMMA))
    o = O.Oracle(case, kind="serial")
    R = o.rhs(parts=O.PART_VISC)
    dv = o.sensor()[2][0, :, 0]
    a, b = _golden_fd(order)
    # the dilatation itself: first derivative of the continued v (checks the premise)
    d1v = sum(a[l - 1] * (vext[L + l:L + l + ny] - vext[L - l:L - l + ny]) for l in range(1, L + 1)) / dy
    assert np.allclose(dv, d1v, rtol=1e-12)
    d2v = sum(b[l - 1] * (vext[L + l:L + l + ny] - 2 * v + vext[L - l:L - l + ny]) for l in range(1, L + 1)) / dy ** 2

    def grad_div(src):
        ext = dv[np.array([src(j) for j in jj])]
        return sum(a[l - 1] * (ext[L + l:L + l + ny] - ext[L - l:L - l + ny]) for l in range(1, L + 1)) / dy

    clamp = grad_div(lambda j: min(max(j, 0), ny - 1))
    mirror = grad_div(lambda j: -1 - j if j < 0 else (2 * ny - 1 - j if j >= ny else j))
    wrap = grad_div(lambda j: j % ny)
    expect = mu * d2v + (mu / 3.0) * clamp
    scale = np.max(np.abs(expect))
    assert np.max(np.abs(R[2][0, :, 0] - expect)) < 1e-12 * scale
    assert np.all(R[2] == R[2][:1, :, :1])                 # and the same in every column
    for other in (mirror, wrap):
        assert np.max(np.abs((mu / 3.0) * (other - clamp))) > 1e-3 * scale


# ------------------------------------------------------------------------------------------------
# O4: power-law viscosity with a non-zero exponent
# ------------------------------------------------------------------------------------------------
def test_power_law_viscosity_of_a_uniform_state():
    """mu = mu_ref (T / T_ref)^n on uniform states, read back through the oracle's primitive field; the exponent
    and the reference temperature both matter (T / T_ref != 1, n = 0.76), and n = 0.5, 1, 2 reduce to sqrt, the
    identity and a square."""
    one = np.ones((4, 4, 4))
    for T, t_ref, n in [(1.7, 0.9, 0.76), (0.6, 1.3, 0.76), (2.25, 1.0, 0.5), (1.3, 0.5, 1.0), (0.8, 1.6, 2.0)]:
        p = 1.1
        rho = p / (RGAS * T)
        case = W.Case(name="pow", nx=4, ny=4, nz=4, lx=1.0, ly=1.0, lz=1.0, gamma=GAMMA, rgas=RGAS, prandtl=PR,
                      visc_law=W.VISC_POWER, pow_exp=n, mu_ref=0.037, t_ref=t_ref,
                      w0=W.conserved_from_primitive(rho * one, 0.1 * one, 0 * one, 0 * one, p * one, GAMMA))
        o = O.Oracle(case, kind="serial")
        o.rhs()
        mu = o.prim(6)
        t = T / t_ref
        expect = {0.5: 0.037 * np.sqrt(t), 1.0: 0.037 * t, 2.0: 0.037 * t * t}.get(n, 0.037 * np.exp(n * np.log(t)))
        assert np.allclose(mu, expect, rtol=1e-14), (T, t_ref, n)


def _manufactured_power(n_exp, t_ref, mu0):
    x, y, z = sp.symbols("x y z")
    u = sp.sin(x) * sp.cos(2 * y) * sp.cos(z) * sp.Rational(3, 10) + sp.Rational(1, 10) * sp.sin(y)
    v = sp.cos(x) * sp.sin(y) * sp.cos(2 * z) * sp.Rational(1, 5)
    w = sp.sin(2 * x) * sp.sin(y) * sp.sin(z) * sp.Rational(1, 4)
    T = 1 + sp.Rational(3, 10) * sp.cos(x) * sp.cos(y) * sp.sin(z)
    rho = 1 + sp.Rational(1, 10) * sp.sin(x + y + z)
    mu = mu0 * (T / t_ref) ** n_exp
    lam = GAMMA * RGAS / (GAMMA - 1) * mu / PR
    X, vel = (x, y, z), (u, v, w)
    div = sum(sp.diff(vel[a], X[a]) for a in range(3))
    sig = [[mu * (sp.diff(vel[a], X[b]) + sp.diff(vel[b], X[a]) - (sp.Rational(2, 3) * div if a == b else 0))
            for b in range(3)] for a in range(3)]
    mom = [sum(sp.diff(sig[a][b], X[b]) for b in range(3)) for a in range(3)]
    ene = sum(sp.diff(sum(sig[a][b] * vel[a] for a in range(3)), X[b]) for b in range(3)) + \
        sum(sp.diff(lam * sp.diff(T, X[b]), X[b]) for b in range(3))
    f = lambda e: sp.lambdify((x, y, z), e, "numpy")
    return dict(u=f(u), v=f(v), w=f(w), T=f(T), rho=f(rho), mom=[f(m) for m in mom], ene=f(ene))


def test_power_law_viscous_terms_match_symbolic_navier_stokes():
    """The manufactured-solution pin of test_oracle_viscous.py with mu = mu_ref (T / T_ref)^0.76, T_ref = 0.8: the
    variable-viscosity terms (grad mu . strain, grad mu . grad T) carry d mu / dT = n mu / T, so a wrong exponent, a
    missing T_ref or T_ref applied on the wrong side shows at leading order; design order 6 confirms the wiring."""
    n_exp, t_ref, mu0 = 0.76, 0.8, 0.05
    mf = _manufactured_power(sp.Rational(19, 25), sp.Rational(4, 5), sp.Rational(1, 20))
    errs = []
    for n in (32, 64):
        L = 2 * np.pi
        x = np.arange(n) * L / n
        y = x + 0.25 * np.sin(x)
        Z, Y, X = np.meshgrid(x, y, x, indexing="ij")
        rho, T = mf["rho"](X, Y, Z), mf["T"](X, Y, Z)
        case = W.Case(name="mms_pow", nx=n, ny=n, nz=n, lx=L, ly=L, lz=L, y_nodes=y, gamma=GAMMA, rgas=RGAS,
                      prandtl=PR, visc_law=W.VISC_POWER, pow_exp=n_exp, mu_ref=mu0, t_ref=t_ref,
                      w0=W.conserved_from_primitive(rho, mf["u"](X, Y, Z), mf["v"](X, Y, Z), mf["w"](X, Y, Z),
                                                    rho * RGAS * T, GAMMA))
        R = O.Oracle(case).rhs(parts=O.PART_VISC)
        ref = [m(X, Y, Z) for m in mf["mom"]] + [mf["ene"](X, Y, Z)]
        errs.append([np.max(np.abs(R[q + 1] - ref[q])) / np.max(np.abs(ref[q])) for q in range(4)])
    for a, b in zip(*errs):
        assert b < 2e-6 and np.log2(a / b) > 6 - 0.3, errs


# ------------------------------------------------------------------------------------------------
# O6 / S15: the clamp of the ghost temperature at an isothermal wall
# ------------------------------------------------------------------------------------------------
def test_wall_ghost_temperature_is_clamped_at_a_tenth_of_the_wall_temperature():
    """T(m) = 2.5 T_w > 1.9 T_w makes 2 T_w - T(m) negative: the ghost takes T = 0.1 T_w exactly, keeps p and -u, and
    its density follows from the gas law; the second row (T = 1.5 T_w) is below the limit and is reflected as usual."""
    tw, p0 = 0.9, 1.3
    nx, ny, nz = 4, 8, 3
    g = 3
    y = (np.arange(ny) + 0.5) / ny
    T = np.full((nz, ny, nx), 1.0 * tw)
    T[:, 0, :] = 2.5 * tw
    T[:, 1, :] = 1.5 * tw
    T[:, 2, :] = 1.95 * tw                                  # just past the limit 1.9 T_w: clamped too
    rho = p0 / (RGAS * T)
    u = 0.3 * np.ones_like(T)
    v = -0.2 * np.ones_like(T)
    case = W.Case(name="clampT", nx=nx, ny=ny, nz=nz, lx=1.0, ly=1.0, lz=1.0, y_nodes=y, y_wall_lo=0.0, y_wall_hi=1.0,
                  bc_y_lo=W.BC_WALL_ISOTHERMAL, bc_y_hi=W.BC_WALL_ISOTHERMAL, t_wall_lo=tw, t_wall_hi=tw,
                  gamma=GAMMA, rgas=RGAS, w0=W.conserved_from_primitive(rho, u, v, 0 * u, p0 * np.ones_like(T), GAMMA))
    o = O.Oracle(case, kind="serial")
    o.rhs()
    pad = [o.padded(q) for q in range(5)]
    assert o.ng == g
    expect_T = {0: 0.1 * tw, 1: 0.5 * tw, 2: 0.1 * tw}
    for m in range(g):
        sl = (slice(g, -g), g - 1 - m, slice(g, -g))
        rho_g = pad[0][sl]
        u_g, v_g = pad[1][sl] / rho_g, pad[2][sl] / rho_g
        p_g = (GAMMA - 1) * (pad[4][sl] - 0.5 * rho_g * (u_g ** 2 + v_g ** 2))
        T_g = p_g / (RGAS * rho_g)
        assert np.allclose(T_g, expect_T[m], rtol=1e-13), (m, T_g)
        assert np.allclose(p_g, p0, rtol=1e-13)
        assert np.allclose(u_g, -0.3, rtol=1e-14) and np.allclose(v_g, 0.2, rtol=1e-14)
    # the upper wall sees T = T_w: ghost T = T_w, nothing clamped
    sl = (slice(g, -g), g + ny, slice(g, -g))
    rho_g = pad[0][sl]
    p_g = (GAMMA - 1) * (pad[4][sl] - 0.5 * (pad[1][sl] ** 2 + pad[2][sl] ** 2) / rho_g)
    assert np.allclose(p_g / (RGAS * rho_g), tw, rtol=1e-13)
