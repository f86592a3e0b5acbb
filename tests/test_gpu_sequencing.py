"""Call sequences through the C ABI against the oracle: the library keeps two primitive buffers (the fused RHS
epilogue writes the primitives of the updated state into the other one), a "rate ready" state for the time step and
owner-written periodic ghosts, so every order of calls a user can make must still give the oracle's numbers."""
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


def _cmp_fields(gpu, ora, case, tol=TOL_STEP):
    floor_w, _ = natural_scales(case)
    w_g, w_o = gpu.get_fields(), ora.get_fields()
    errs = [field_err(w_g[q], w_o[q], floor_w[q]) for q in range(5)]
    assert max(errs) <= tol, errs


def _cmp_rhs(gpu, ora, case):
    _, floor_r = natural_scales(case)
    r_g, r_o = gpu.rhs().cpu().numpy(), ora.rhs()
    errs = [field_err(r_g[q], r_o[q], floor_r[q]) for q in range(5)]
    assert max(errs) <= TOL_RHS, errs


def test_dt_every_three(S):
    """dt recomputed every third step: the last stage of steps 2, 5, ... reduces the rate of the state it produces."""
    case = W.isotropic_turbulence(nx=40, ny=36, nz=33, mach_t=0.5, k0=3.0, kmax=8, seed=21, dilatational=0.4).replace(dt_every=3)
    gpu, ora = S(case), _oracle(case)
    for n in (1, 1, 2, 3, 1):
        dt_g, t_g = gpu.step(n)
        dt_o, t_o = ora.step(n)
        assert abs(dt_g - dt_o) <= 1e-12 * dt_o and abs(t_g - t_o) <= 1e-12 * t_o
    _cmp_fields(gpu, ora, case)
    gpu.destroy()


def test_rhs_and_sensor_calls_between_steps(S):
    """streams_rhs / streams_get_sensor between steps neither change the state nor confuse the buffer bookkeeping."""
    case = W.channel(48, 40, 36, seed=7)
    gpu, ora = S(case), _oracle(case)
    _cmp_rhs(gpu, ora, case)
    gpu.step(2); ora.step(2)
    w_before = gpu.get_fields()
    _cmp_rhs(gpu, ora, case)                       # RHS of the evolved state
    gpu.get_sensor()
    _cmp_rhs(gpu, ora, case)                       # twice in a row
    assert np.array_equal(gpu.get_fields(), w_before)
    gpu.step(3); ora.step(3)
    _cmp_fields(gpu, ora, case)
    gpu.destroy()


def test_set_fields_mid_run_restarts_cleanly(S):
    case = W.isotropic_turbulence(nx=36, ny=34, nz=38, mach_t=0.6, k0=3.0, kmax=8, seed=22, dilatational=0.5)
    gpu, ora = S(case), _oracle(case)
    gpu.step(3)
    gpu.set_fields(case.w0)                        # back to the initial state: stale primitives / rate must not be used
    dt_g, t_g = gpu.step(4)
    dt_o, t_o = ora.step(4)
    assert abs(dt_g - dt_o) <= 1e-12 * dt_o and abs(t_g - t_o) <= 1e-12 * t_o
    _cmp_fields(gpu, ora, case)
    gpu.destroy()


@pytest.mark.parametrize("shape", [(40, 36, 5), (5, 34, 37), (38, 4, 33), (3, 3, 3)])
def test_narrow_periodic_extents(S, shape):
    """Extents below 2 ng: a node has two periodic images in the ghost layers, which the owner-writes path does not
    cover; the library must fall back to the ghost kernels for that direction."""
    nx, ny, nz = shape
    rng = np.random.default_rng(5)
    rho = 1.0 + 0.1 * rng.uniform(-1, 1, (nz, ny, nx))
    u, v, w = (0.3 * rng.uniform(-1, 1, (nz, ny, nx)) for _ in range(3))
    p = 1.0 + 0.1 * rng.uniform(-1, 1, (nz, ny, nx))
    base = W.isotropic_turbulence(nx=12, ny=12, nz=12, mach_t=0.3, k0=2.0, kmax=3, seed=1)
    case = base.replace(name="narrow", nx=nx, ny=ny, nz=nz, w0=W.conserved_from_primitive(rho, u, v, w, p, base.gamma),
                        sensor_threshold=0.05)
    gpu, ora = S(case), _oracle(case)
    _cmp_rhs(gpu, ora, case)
    th_g, mk_g = gpu.get_sensor()
    th_o, mk_o, _ = ora.sensor()
    assert np.array_equal(th_g, th_o) and np.array_equal(mk_g, mk_o)
    gpu.step(3); ora.step(3)
    _cmp_fields(gpu, ora, case)
    gpu.destroy()


def test_fixed_dt_and_central_inviscid(S):
    """dt_fixed: no rate is ever reduced; the lean (central, inviscid) variant with its L2 prefetch."""
    case = W.config(0).replace(dt_fixed=2e-3)
    gpu, ora = S(case), _oracle(case)
    dt_g, t_g = gpu.step(6)
    dt_o, t_o = ora.step(6)
    assert dt_g == 2e-3 and abs(t_g - t_o) <= 1e-12 * t_o
    _cmp_fields(gpu, ora, case)
    gpu.destroy()


@pytest.mark.parametrize("kind", ["slab", "random", "all", "none"])
def test_mask_override_matches_the_oracle(S, kind):
    """streams_set_mask_override (the activation-sweep hook): WENO exactly where the mask says."""
    case = W.isotropic_turbulence(nx=40, ny=36, nz=34, mach_t=0.5, k0=3.0, kmax=8, seed=41, dilatational=0.3)
    rng = np.random.default_rng(3)
    shape = (case.nz, case.ny, case.nx)
    if kind == "slab":
        mask = np.zeros(shape, np.uint8); mask[: case.nz // 3] = 1
    elif kind == "random":
        mask = (rng.uniform(size=shape) < 0.03).astype(np.uint8)
    elif kind == "all":
        mask = np.ones(shape, np.uint8)
    else:
        mask = np.zeros(shape, np.uint8)
    gpu, ora = S(case), _oracle(case)
    gpu.set_mask_override(mask)
    ora.set_mask_override(mask)
    _cmp_rhs(gpu, ora, case)
    th_g, mk_g = gpu.get_sensor()
    th_o, mk_o, _ = ora.sensor()
    assert np.array_equal(mk_g, mask) and np.array_equal(mk_o, mask) and np.array_equal(th_g, th_o)
    flagged, _, ifaces = gpu.get_activation()
    assert flagged == int(mask.sum())
    assert ifaces == [int(ora.interface_flags(d).sum()) for d in range(3)]
    gpu.step(3); ora.step(3)
    _cmp_fields(gpu, ora, case)
    # back to the sensor's own decision
    gpu.set_mask_override(None); ora.set_mask_override(None)
    _cmp_rhs(gpu, ora, case)
    gpu.destroy()


def _volume_weights(case):
    """dV(j) of the oracle's reading S3: dx dz / (d eta/dy)(j), from the oracle's own metrics."""
    ora = _oracle(case)
    eta_y_c, _, _, _ = ora.metrics()
    ora.close()
    return (case.lx / case.nx) * (case.lz / case.nz) / eta_y_c


def test_sum_reductions_match_plain_sums(S):
    """streams_get_sums against the definitions written out with numpy on the oracle's numbers."""
    from paper_2304_05494_b200 import binding
    case = W.channel(48, 40, 36, seed=9)
    gpu, ora = S(case), _oracle(case)
    dv = _volume_weights(case)
    state = gpu.get_sums(0)
    ref = np.array([np.sum(case.w0[q] * dv[None, :, None]) for q in range(5)])
    assert np.all(np.abs(state - ref) <= 1e-12 * np.maximum(np.abs(ref), 1.0)), (state, ref)
    with pytest.raises(binding.StreamsError) as e:      # no streams_rhs yet
        gpu.get_sums(1)
    assert e.value.code == binding.STREAMS_ESTATE
    gpu.rhs()
    r_o = ora.rhs()
    res = gpu.get_sums(1)
    ref = np.array([np.sum(r_o[q] ** 2) for q in range(5)])
    assert np.all(np.abs(res - ref) <= 1e-10 * ref), (res, ref)
    assert np.array_equal(res, gpu.get_sums(1))         # fixed summation order: bit-reproducible
    gpu.step(1)
    with pytest.raises(binding.StreamsError):            # the state moved on: R is no longer its right-hand side
        gpu.get_sums(1)
    gpu.destroy()


def test_discrete_conservation_on_the_gpu(S):
    """Periodic box: mass is conserved to round-off by the hybrid viscous scheme, and so are momentum and total energy
    without the (Laplacian-form, non-conservative) viscous terms (S11) -- measured with the library's own sums."""
    for viscous in (True, False):
        case = W.isotropic_turbulence(nx=48, ny=44, nz=40, mach_t=0.6, k0=3.0, kmax=8, seed=23, dilatational=0.4,
                                      viscous=viscous)
        gpu = S(case)
        s0 = gpu.get_sums(0)
        gpu.step(20)
        s1 = gpu.get_sums(0)
        scale = np.array([s0[0], s0[0], s0[0], s0[0], s0[4]])     # momentum sums are ~0: measure against the mass
        drift = np.abs(s1 - s0) / scale
        assert drift[0] <= 1e-13, drift
        if not viscous:
            assert np.all(drift <= 1e-12), drift
        gpu.destroy()


def test_bulk_flow_controller_against_the_oracle(S):
    """streams_step_forced (device-side sums + one-thread controller, no host round trip per step) against the oracle's
    controller (reading S18) on a channel: same fields, same force, step by step and in one multi-step call."""
    case = W.channel(48, 40, 36, seed=61)
    free = S(case)
    p0 = free.get_sums(0)[1]
    free.step(20)
    loss = 1.0 - free.get_sums(0)[1] / p0
    free.destroy()
    assert loss > 1e-4                                   # friction is at work
    gpu, ora = S(case), _oracle(case)
    for n in (1, 1, 3, 15):
        dt_g, t_g, g_g = gpu.step_forced(n)
        dt_o, t_o, g_o = ora.step_forced(n)
        assert abs(dt_g - dt_o) <= 1e-12 * dt_o and abs(t_g - t_o) <= 1e-12 * t_o
        assert abs(g_g[0] - g_o[0]) <= 1e-8 * abs(g_o[0]) and g_g[1] == 0.0 and g_g[2] == 0.0, (g_g, g_o)
    _cmp_fields(gpu, ora, case)
    assert g_g[0] > 0.0
    assert abs(gpu.get_sums(0)[1] / p0 - 1.0) < 0.02 * loss            # held at its target
    # a target given later moves the bulk momentum there within a step (deadbeat up to the change of the friction)
    gpu.step_forced(1, 0, 1.01 * p0); ora.step_forced(1, 0, 1.01 * p0)
    gpu.step_forced(2); ora.step_forced(2)
    assert abs(gpu.get_sums(0)[1] / (1.01 * p0) - 1.0) < 1e-4
    _cmp_fields(gpu, ora, case)
    # streams_set_body_force takes the acceleration back to the host
    gpu.set_body_force((0.0, 0.0, 0.0)); ora.close()
    gpu.step(1)
    gpu.destroy()


def test_bulk_flow_controller_is_deadbeat_without_friction(S):
    """Uniform flow in an inviscid periodic box: on target one step after the controller saw the deviation."""
    one = np.ones((16, 16, 16))
    case = W.Case(name="ctrl", nx=16, ny=16, nz=16, lx=1.0, ly=1.0, lz=1.0, dt_fixed=1e-2,
                  w0=W.conserved_from_primitive(1.3 * one, 0.5 * one, 0 * one, 0 * one, 1.1 * one, 1.4))
    gpu = S(case)
    p0 = gpu.get_sums(0)[1]
    gpu.step_forced(1, 0, 1.1 * p0)
    assert abs(gpu.get_sums(0)[1] / p0 - 1.0) < 1e-13
    _, _, g = gpu.step_forced(1)
    assert abs(gpu.get_sums(0)[1] / (1.1 * p0) - 1.0) < 1e-12 and abs(g[0]) < 1e-8
    gpu.destroy()


def test_runs_are_bit_reproducible(S):
    """The work lists are filled in atomic (run-dependent) order, but every flagged interface writes its own slot and
    every reduction has a fixed order (or is a max): two runs of the same problem give the same bits."""
    case = W.isotropic_turbulence(nx=44, ny=40, nz=36, mach_t=0.6, k0=3.0, kmax=8, seed=71, dilatational=0.5)
    out = []
    for _ in range(2):
        gpu = S(case)
        dt, t = gpu.step(6)
        out.append((dt, t, gpu.get_fields(), gpu.get_sums(0)))
        gpu.destroy()
    assert out[0][0] == out[1][0] and out[0][1] == out[1][1]
    assert np.array_equal(out[0][2], out[1][2]) and np.array_equal(out[0][3], out[1][3])


@pytest.mark.parametrize("visc", [W.VISC_SUTHERLAND, W.VISC_POWER])
def test_restart_through_get_fields_set_fields_is_bit_reproducible(S, visc):
    """The primitives of a state carry the same bits whether the fused RHS epilogue or the fill kernel produced them
    (prims_from_state is contraction-independent), so stopping, copying the state out and in again and continuing
    gives exactly the uninterrupted run.  dt_fixed: the restart also resets time and the step counter."""
    case = W.channel(48, 40, 36, seed=61).replace(dt_fixed=2e-3, visc_law=visc, pow_exp=0.76, t_ref=0.9)
    a = S(case)
    a.step(6)
    w_a = a.get_fields()
    b = S(case)
    b.step(3)
    w_mid = b.get_fields()
    b.set_fields(w_mid)
    b.step(3)
    w_b = b.get_fields()
    assert np.array_equal(w_a, w_b)
    a.destroy(); b.destroy()


def test_graph_replay_is_taken_and_changes_nothing(S, monkeypatch):
    """streams_step replays every step after the first from a CUDA graph (two graphs, one per primitive buffer the step
    starts from; the first step runs the full ghost + primitive pass and is launched kernel by kernel): the count of
    graph submissions says so, and STREAMS_NO_GRAPH=1 -- every kernel launched on its own -- gives the same bits and the
    same number of kernels.  A capture that silently fell back to direct launches would show up as a count of zero."""
    for dt_every, calls in ((1, (2, 4)), (3, (1, 1, 5))):
        case = W.isotropic_turbulence(nx=44, ny=40, nz=36, mach_t=0.6, k0=3.0, kmax=8, seed=73, dilatational=0.5).replace(dt_every=dt_every)
        out = []
        for no_graph in (False, True):
            if no_graph:
                monkeypatch.setenv("STREAMS_NO_GRAPH", "1")
            else:
                monkeypatch.delenv("STREAMS_NO_GRAPH", raising=False)
            gpu = S(case)
            for n in calls:
                dt, t = gpu.step(n)
            out.append((dt, t, gpu.get_fields(), gpu.graph_launches(), gpu.kernel_launches()))
            gpu.destroy()
        monkeypatch.delenv("STREAMS_NO_GRAPH", raising=False)
        assert out[0][3] == sum(calls) - 1 and out[1][3] == 0, (out[0][3], out[1][3])
        assert out[0][4] == out[1][4]
        assert out[0][0] == out[1][0] and out[0][1] == out[1][1] and np.array_equal(out[0][2], out[1][2])
