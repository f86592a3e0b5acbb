"""GPU-vs-oracle parity through the C ABI (BASELINE north_star tolerances):
max field-normalised error <= 1e-11 after one RHS, <= 1e-9 after 10 RK steps, bit-identical mask."""
import numpy as np
import pytest

import workloads as W
from tests import helpers
from tests.helpers import field_err, natural_scales

pytestmark = pytest.mark.gpu

TOL_RHS = 1e-11
TOL_STEP = 1e-9


@pytest.fixture(scope="module")
def S():
    from paper_2304_05494_b200 import build, binding
    build.build()
    return binding.Streams


def _oracle(case):
    from oracle.oracle import Oracle
    return Oracle(case)


def check_case(S, case, nsteps, tol_rhs=TOL_RHS, tol_step=TOL_STEP, expect_activation=None):
    gpu = S(case)
    ora = _oracle(case)
    floor_w, floor_r = natural_scales(case)
    hits0 = len(helpers.FLOOR_HITS)
    # one RHS
    r_gpu = gpu.rhs().cpu().numpy()
    r_ora = ora.rhs()
    errs = [field_err(r_gpu[q], r_ora[q], floor_r[q], "rhs", q, tol_rhs) for q in range(5)]
    assert max(errs) <= tol_rhs, ("rhs", case.name, errs)
    # streams_rhs must not change the interior
    assert np.array_equal(gpu.get_fields(), case.w0)
    # sensor mask, bit-identical
    if case.flux_mode == W.FLUX_HYBRID:
        th_g, mk_g = gpu.get_sensor()
        th_o, mk_o, _ = ora.sensor()
        assert np.array_equal(th_g, th_o), ("theta", float(np.max(np.abs(th_g - th_o))))
        assert np.array_equal(mk_g, mk_o)
        frac = float(mk_o.mean())
        if expect_activation is not None:
            assert expect_activation[0] <= frac <= expect_activation[1], frac
        flagged, shock, ifaces = gpu.get_activation()
        assert flagged == int(mk_o.sum())
        # every flagged interface is on exactly one work list (oracle: nd + 1 interfaces per pencil)
        assert ifaces == [int(ora.interface_flags(d).sum()) for d in range(3)]
    # nsteps RK3 steps
    dt_g, t_g = gpu.step(nsteps)
    dt_o, t_o = ora.step(nsteps)
    assert abs(dt_g - dt_o) <= 1e-12 * dt_o and abs(t_g - t_o) <= 1e-12 * t_o
    w_g, w_o = gpu.get_fields(), ora.get_fields()
    errs = [field_err(w_g[q], w_o[q], floor_w[q], "state", q, tol_step) for q in range(5)]
    assert max(errs) <= tol_step, ("step", case.name, errs)
    helpers.check_floor_hits(case, hits0)        # the floor was used only where DESIGN.md says a field is at round-off
    # mask of the evolved state (S14): may differ only at nodes whose theta sits within 1e-10 of the
    # threshold, because the two states now differ by round-off
    if case.flux_mode == W.FLUX_HYBRID:
        th_g, mk_g = gpu.get_sensor()
        ora.rhs()
        th_o, mk_o, _ = ora.sensor()
        near = np.abs(th_o - case.sensor_threshold) < 1e-10
        assert np.array_equal(mk_g[~near], mk_o[~near])
        assert np.max(np.abs(th_g - th_o)) < 1e-9
    gpu.destroy()
    return errs


def test_purely_solenoidal_start_then_shocklets_form(S):
    """configs 1/4 as specified start solenoidal (theta = 0); the sensor wakes up as the flow evolves."""
    case = W.isotropic_turbulence(nx=40, ny=40, nz=40, mach_t=0.8, k0=4.0, kmax=12, seed=4)
    check_case(S, case, 10, expect_activation=(0.0, 0.05))


def test_config0_taylor_green_full_size(S):
    check_case(S, W.config(0), 10)


@pytest.mark.parametrize("shape", [(40, 36, 33), (35, 67, 20)])
def test_periodic_inviscid_central_ragged(S, shape):
    case = W.isotropic_turbulence(nx=shape[0], ny=shape[1], nz=shape[2], mach_t=0.3, k0=3.0, kmax=8, seed=11,
                                  flux_mode=W.FLUX_CENTRAL, viscous=False)
    check_case(S, case, 10)


def test_periodic_viscous_central(S):
    case = W.isotropic_turbulence(nx=37, ny=34, nz=41, mach_t=0.3, k0=3.0, kmax=8, seed=12, flux_mode=W.FLUX_CENTRAL)
    check_case(S, case, 10)


def test_periodic_full_weno_inviscid(S):
    case = W.isotropic_turbulence(nx=34, ny=33, nz=35, mach_t=0.5, k0=3.0, kmax=8, seed=13,
                                  flux_mode=W.FLUX_WENO, viscous=False)
    check_case(S, case, 10)


def test_config1_replica_hybrid_viscous(S):
    case = W.isotropic_turbulence(nx=48, ny=44, nz=41, mach_t=0.6, k0=4.0, kmax=12, seed=1, dilatational=0.5)
    check_case(S, case, 10, expect_activation=(0.005, 0.6))


def test_config2_replica_channel(S):
    case = W.channel(48, 40, 36, seed=2)
    check_case(S, case, 10)


def test_config3_replica_boundary_layer(S):
    case = W.boundary_layer(96, 40, 36, seed=3, nblobs=6)
    check_case(S, case, 10, expect_activation=(0.0005, 0.5))


def test_config4_replica(S):
    case = W.isotropic_turbulence(nx=40, ny=40, nz=40, mach_t=0.8, k0=8.0, kmax=16, seed=4, dilatational=0.3)
    check_case(S, case, 10, expect_activation=(0.01, 0.8))


def test_state_errors(S):
    from paper_2304_05494_b200 import binding
    case = W.config(0)
    gpu = S(case.replace(w0=None))
    with pytest.raises(binding.StreamsError) as e:
        gpu.rhs()
    assert e.value.code == binding.STREAMS_ESTATE
    with pytest.raises(binding.StreamsError):
        gpu.step(1)
    bad = case.w0.copy()
    bad[0, 3, 3, 3] = np.nan
    gpu.set_fields(bad)
    with pytest.raises(binding.StreamsError) as e:
        gpu.step(1)
    assert e.value.code == binding.STREAMS_ENAN


# ---- the other instantiated order families: central / WENO / viscous = 2/1/2 and 4/3/4
def _with_orders(case, m):
    return case.replace(central_order=2 * m, weno_order=2 * m - 1, visc_order=2 * m, name=f"{case.name}_m{m}")


@pytest.mark.parametrize("m", [1, 2])
def test_order_family_hybrid_viscous_periodic(S, m):
    case = W.isotropic_turbulence(nx=40, ny=37, nz=35, mach_t=0.6, k0=3.0, kmax=8, seed=31, dilatational=0.5)
    check_case(S, _with_orders(case, m), 10, expect_activation=(0.002, 0.8))


@pytest.mark.parametrize("m", [1, 2])
def test_order_family_channel_walls(S, m):
    check_case(S, _with_orders(W.channel(40, 36, 34, seed=32), m), 6)


@pytest.mark.parametrize("m", [1, 2])
def test_order_family_full_weno_and_central(S, m):
    base = W.isotropic_turbulence(nx=34, ny=33, nz=36, mach_t=0.4, k0=3.0, kmax=8, seed=33, viscous=False,
                                  flux_mode=W.FLUX_WENO)
    check_case(S, _with_orders(base, m), 6)
    check_case(S, _with_orders(base.replace(flux_mode=W.FLUX_CENTRAL), m), 6)


# ---- order 8 / WENO 7 / viscous 8 (four ghost layers) and mixed orders
def test_order_family_8_7_8_hybrid_viscous_periodic(S):
    case = W.isotropic_turbulence(nx=40, ny=37, nz=35, mach_t=0.6, k0=3.0, kmax=8, seed=31, dilatational=0.5)
    check_case(S, _with_orders(case, 4), 10, expect_activation=(0.002, 0.8))


def test_order_family_8_7_8_channel_walls(S):
    check_case(S, _with_orders(W.channel(40, 36, 34, seed=32), 4), 6)


def test_order_family_8_7_8_boundary_layer(S):
    check_case(S, _with_orders(W.boundary_layer(72, 40, 36, seed=34, nblobs=5), 4), 6, expect_activation=(0.0005, 0.5))


def test_order_family_8_7_8_full_weno_and_central(S):
    base = W.isotropic_turbulence(nx=34, ny=33, nz=36, mach_t=0.4, k0=3.0, kmax=8, seed=33, viscous=False,
                                  flux_mode=W.FLUX_WENO)
    check_case(S, _with_orders(base, 4), 6)
    check_case(S, _with_orders(base.replace(flux_mode=W.FLUX_CENTRAL), 4), 6)
    # ragged and narrow: extents that are not multiples of any tile, one of them below two ghost widths
    small = W.isotropic_turbulence(nx=35, ny=7, nz=21, mach_t=0.4, k0=2.0, kmax=3, seed=35, dilatational=0.4)
    check_case(S, _with_orders(small, 4), 4)


@pytest.mark.parametrize("orders", [(6, 3, 4), (4, 5, 6), (2, 7, 2), (8, 3, 6), (6, 5, 8), (2, 1, 8), (8, 1, 2)])
def test_mixed_orders_hybrid_viscous(S, orders):
    """Any mix of central / WENO / viscous orders runs on the covering instance with zero-padded coefficients and
    must give the oracle's numbers for exactly that mix."""
    co, wo, vo = orders
    case = W.isotropic_turbulence(nx=36, ny=34, nz=33, mach_t=0.6, k0=3.0, kmax=8, seed=36, dilatational=0.5)
    check_case(S, case.replace(central_order=co, weno_order=wo, visc_order=vo, name=f"mix_{co}_{wo}_{vo}"), 6,
               expect_activation=(0.002, 0.8))


@pytest.mark.parametrize("orders", [(6, 3, 6), (4, 7, 4)])
def test_mixed_orders_channel(S, orders):
    co, wo, vo = orders
    check_case(S, W.channel(40, 36, 34, seed=37).replace(central_order=co, weno_order=wo, visc_order=vo), 6)


def test_invalid_orders_are_rejected_at_init(S):
    from paper_2304_05494_b200 import binding
    for bad in (dict(central_order=10), dict(central_order=5), dict(weno_order=9), dict(visc_order=3)):
        case = W.isotropic_turbulence(nx=16, ny=16, nz=16, mach_t=0.3, k0=2.0, kmax=4, seed=1).replace(**bad)
        with pytest.raises(binding.StreamsError) as e:
            S(case)
        assert e.value.code == binding.STREAMS_EINVAL


# ---- WENO-Z weights (S19)
@pytest.mark.parametrize("m", [2, 3, 4])
def test_weno_z_hybrid_and_full_weno(S, m):
    case = W.isotropic_turbulence(nx=40, ny=37, nz=35, mach_t=0.6, k0=3.0, kmax=8, seed=81, dilatational=0.5)
    case = _with_orders(case, m).replace(weno_variant=1)
    check_case(S, case, 8, expect_activation=(0.002, 0.8))
    check_case(S, case.replace(flux_mode=W.FLUX_WENO, visc_law=W.VISC_NONE, name=case.name + "_dense"), 4)


def test_weno_z_channel_mixed_orders(S):
    check_case(S, W.channel(40, 36, 34, seed=82).replace(weno_variant=1, central_order=6, weno_order=3), 6)


# ---- branches the round-1 suite did not reach on the GPU
def test_power_law_viscosity(S):
    """STREAMS_VISC_POWER with a non-zero exponent and T_ref != 1 (device pow vs the oracle's std::pow)."""
    case = W.isotropic_turbulence(nx=40, ny=36, nz=34, mach_t=0.6, k0=3.0, kmax=8, seed=41, dilatational=0.5)
    case = case.replace(visc_law=W.VISC_POWER, pow_exp=0.76, t_ref=0.8, mu_ref=4 * case.mu_ref, name="power_law")
    check_case(S, case, 10, expect_activation=(0.002, 0.8))
    ch = W.channel(40, 36, 34, seed=42)
    check_case(S, ch.replace(visc_law=W.VISC_POWER, pow_exp=0.7, t_ref=1.3, name="power_law_channel"), 6)


def test_wall_ghost_temperature_clamp(S):
    """Fluid hotter than 1.9 T_w next to an isothermal wall: the ghost temperature is clamped at 0.1 T_w (O6 / S15)."""
    case = W.channel(40, 36, 34, seed=43)
    w0 = case.w0.copy()
    g = case.gamma
    rho, ru, rv, rw, E = w0
    p = (g - 1) * (E - 0.5 * (ru ** 2 + rv ** 2 + rw ** 2) / rho)
    T = p / (case.rgas * rho)
    for j, fac in ((0, 2.5), (1, 2.0), (case.ny - 1, 2.2)):          # rows 0, 1 at the lower wall, the last row at the upper
        Tn = fac * case.t_wall_lo * np.ones_like(T[:, j, :])
        rn = p[:, j, :] / (case.rgas * Tn)
        sc = rn / rho[:, j, :]
        for q in range(4):
            w0[q][:, j, :] *= sc                                       # same velocities, same pressure, hotter and lighter
        w0[4][:, j, :] = p[:, j, :] / (g - 1) + 0.5 * (w0[1][:, j, :] ** 2 + w0[2][:, j, :] ** 2 + w0[3][:, j, :] ** 2) / rn
    check_case(S, case.replace(w0=w0, name="hot_wall"), 4)


@pytest.mark.parametrize("flux_mode", [W.FLUX_HYBRID, W.FLUX_WENO, W.FLUX_CENTRAL])
def test_freestream_faces_in_x_y_and_z(S, flux_mode):
    """STREAMS_BC_FREESTREAM on all six faces, hybrid + viscous: the x-column and z-slab segments of the ghost fill and
    the constant extrapolation of div / mask beyond non-periodic x and z faces."""
    base = W.isotropic_turbulence(nx=37, ny=35, nz=33, mach_t=0.5, k0=3.0, kmax=8, seed=44, dilatational=0.5)
    w0 = base.w0
    fs = tuple(float(w0[q].mean()) for q in range(5))
    case = base.replace(bc_x=W.BC_FREESTREAM, bc_y_lo=W.BC_FREESTREAM, bc_y_hi=W.BC_FREESTREAM, bc_z=W.BC_FREESTREAM,
                        y_wall_lo=0.0, y_wall_hi=base.ly, freestream=fs, flux_mode=flux_mode, name="freestream_box")
    check_case(S, case, 6, expect_activation=(0.002, 0.9) if flux_mode == W.FLUX_HYBRID else None)
    # periodic x, free-stream z only; and the reverse
    check_case(S, case.replace(bc_x=W.BC_PERIODIC, name="fs_z"), 3)
    check_case(S, case.replace(bc_z=W.BC_PERIODIC, name="fs_x"), 3)


def test_blow_up_mid_run_is_reported(S):
    """A state that goes non-finite in the middle of a multi-step call: STREAMS_ENAN, with the CFL time step (the rate
    of the last stage's epilogue must keep a NaN) and with a fixed one (finiteness check of the updated state)."""
    from paper_2304_05494_b200 import binding
    base = W.isotropic_turbulence(nx=32, ny=32, nz=32, mach_t=0.6, k0=3.0, kmax=8, seed=45, dilatational=0.5)
    gpu = S(base)
    dt, _ = gpu.step(2)                                   # healthy
    assert np.isfinite(gpu.get_fields()).all()
    gpu.destroy()
    for case in (base.replace(cfl=40.0, name="cfl40"), base.replace(dt_fixed=60 * dt, name="dtfixed")):
        gpu = S(case)
        with pytest.raises(binding.StreamsError) as e:
            gpu.step(60)
        assert e.value.code == binding.STREAMS_ENAN
        gpu.destroy()
    # one node with a negative pressure, reached after a healthy step: the sound speed of that node is NaN while every
    # conserved value stays finite; the very next dt must not come from the healthy nodes alone
    gpu = S(base)
    gpu.step(1)
    w = gpu.get_fields()
    w[4, 5, 6, 7] = 0.4 * (w[1, 5, 6, 7] ** 2 + w[2, 5, 6, 7] ** 2 + w[3, 5, 6, 7] ** 2) / w[0, 5, 6, 7]   # E < kinetic energy
    gpu.set_fields(w)
    with pytest.raises(binding.StreamsError) as e:
        gpu.step(3)
    assert e.value.code == binding.STREAMS_ENAN
    gpu.destroy()


# ---- uniform body acceleration (S17; PAPER:377 forcing)
def test_body_force_periodic_hybrid(S):
    case = W.isotropic_turbulence(nx=40, ny=38, nz=36, mach_t=0.5, k0=3.0, kmax=8, seed=51, dilatational=0.4)
    check_case(S, case.replace(accel=(0.3, -0.2, 0.15), name="forced_box"), 10, expect_activation=(0.001, 0.8))


def test_body_force_drives_the_channel(S):
    case = W.channel(48, 40, 36, seed=52)
    check_case(S, case.replace(accel=(0.02, 0.0, 0.0), name="forced_channel"), 10)


def test_body_force_momentum_budget_with_the_library_sums(S):
    """Inviscid periodic box: d/dt sum(rho u) = g sum(rho) exactly, so after time t the momentum integral has grown by
    g M t and the energy integral by g . (P(0) t + g M t^2 / 2), whatever the flow does (checked with streams_get_sums)."""
    g = np.array([0.25, 0.0, -0.1])
    case = W.isotropic_turbulence(nx=36, ny=34, nz=32, mach_t=0.4, k0=3.0, kmax=8, seed=53, viscous=False,
                                  dilatational=0.3).replace(accel=tuple(g), dt_fixed=2e-3)
    gpu = S(case)
    s0 = gpu.get_sums(0)
    _, t = gpu.step(15)
    s1 = gpu.get_sums(0)
    mass = s0[0]
    assert abs(s1[0] - mass) <= 1e-13 * mass
    assert np.all(np.abs((s1[1:4] - s0[1:4]) - g * mass * t) <= 1e-12 * mass)
    # RK3 integrates the quadratic-in-time energy growth exactly (third order)
    de = float(g @ s0[1:4]) * t + 0.5 * float(g @ g) * mass * t * t
    assert abs((s1[4] - s0[4]) - de) <= 1e-11 * abs(s0[4])
    gpu.destroy()
