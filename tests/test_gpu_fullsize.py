"""GPU-vs-oracle parity at the FULL sizes of BASELINE.json configs 1-4, in the launch configuration bench.py times.

configs 1, 2 and 3 are small enough for the oracle (OpenMP build) to evaluate the whole grid, ten RK3 steps, every
output compared (config 3: 67 M points, about two minutes of oracle time -- marked slow, still part of -m gpu).
config 4 (262 M points) is compared on SAMPLED outputs: the oracle evaluates sub-boxes cut out of the full-size
field (periodic wrap where the box crosses the domain edge), and only the nodes further than the method's dependency
radius from the artificial sub-box faces are compared.  Dependency radius of one RHS: the fused pass reads
primitives at +-3 and the dilatation at +-3 (itself a +-3 stencil), and an interface flag looks at mask nodes up
to 3 away whose theta is a +-3 stencil: 6 nodes; three RK stages: 18 per step.  Margins used: 8 (one RHS), 20 (one
step), 60 (three steps), 182 (ten steps: a 384^3 box of which the central 20^3 nodes are compared).
Plus properties that hold at any size (discrete conservation in the periodic box).

Inputs are the seeded workloads; for the periodic boxes the `dilatational` knob keeps part of the compressive
component so that the sensor fires at step 0 (the BASELINE fields are solenoidal and theta = 0 initially); no
oracle input comes from the GPU except (i) the scalar dt of the full grid's CFL reduction, which a sub-box cannot
know and which is checked separately against the whole-grid oracle on configs 1-3, and (ii) in
test_config4_as_benchmarked_three_steps, which the round-1 review asked for, the state bench.py times: the seeded
config-4 field advanced by the bench's warm-up steps on the GPU (the oracle cannot advance 262 M points); that test
checks the steps FROM that state, every other test starts both sides from the seeded field.
"""
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
    return Oracle(case, kind="omp")


def _take(a, i0, j0, k0, mx, my, mz, wrap_y):
    """a[..., k0:k0+mz, j0:j0+my, i0:i0+mx] with periodic wrap in x and z (and y if wrap_y)."""
    nz, ny, nx = a.shape[-3:]
    kz = (k0 + np.arange(mz)) % nz
    ix = (i0 + np.arange(mx)) % nx
    jy = (j0 + np.arange(my)) % ny if wrap_y else j0 + np.arange(my)
    return a[..., kz[:, None, None], jy[None, :, None], ix[None, None, :]]


def subbox_case(case, i0, j0, k0, mx, my, mz, dt_fixed):
    """The same problem on a sub-box: same spacings, same gas / scheme numbers, the full grid's dt."""
    per_y = case.bc_y_lo == W.BC_PERIODIC
    kw = dict(name=f"{case.name}_box", nx=mx, ny=my, nz=mz, lx=case.lx * mx / case.nx, lz=case.lz * mz / case.nz,
              dt_fixed=dt_fixed, w0=np.ascontiguousarray(_take(case.w0, i0, j0, k0, mx, my, mz, per_y)))
    if per_y:
        kw["ly"] = case.ly * my / case.ny
    else:
        y = np.asarray(case.y_nodes)
        ys = y[j0:j0 + my].copy()
        lo_wall = j0 == 0
        hi_wall = j0 + my == case.ny
        kw["y_nodes"] = ys
        kw["y_wall_lo"] = case.y_wall_lo if lo_wall else 0.5 * (y[j0 - 1] + y[j0])
        kw["y_wall_hi"] = case.y_wall_hi if hi_wall else 0.5 * (y[j0 + my - 1] + y[j0 + my])
        kw["bc_y_lo"] = case.bc_y_lo if lo_wall else W.BC_FREESTREAM
        kw["bc_y_hi"] = case.bc_y_hi if hi_wall else W.BC_FREESTREAM
    return case.replace(**kw)


def compare_box(case, gpu_rhs, gpu_w1, gpu_mask, gpu_theta, box, dt, floors, margin_rhs=8, margin_step=20):
    """Oracle on one sub-box vs the GPU's full-grid outputs restricted to it."""
    i0, j0, k0, mx, my, mz = box
    sub = subbox_case(case, i0, j0, k0, mx, my, mz, dt)
    ora = _oracle(sub)
    per_y = case.bc_y_lo == W.BC_PERIODIC
    lo_wall = (not per_y) and j0 == 0
    hi_wall = (not per_y) and j0 + my == case.ny

    def inner(a, m):
        jl = 0 if lo_wall else m
        jh = my if hi_wall else my - m
        return a[..., m:mz - m, jl:jh, m:mx - m]

    floor_w, floor_r = floors
    r_o = ora.rhs()
    r_g = _take(gpu_rhs, i0, j0, k0, mx, my, mz, per_y)
    errs = [field_err(inner(r_g[q], margin_rhs), inner(r_o[q], margin_rhs), floor_r[q], "rhs", q, TOL_RHS) for q in range(5)]
    assert max(errs) <= TOL_RHS, ("rhs", case.name, box, errs)
    flagged = 0
    if case.flux_mode == W.FLUX_HYBRID:
        th_o, mk_o, _ = ora.sensor()
        m = 4     # theta is a +-3 stencil of the primitives
        assert np.array_equal(inner(_take(gpu_theta, i0, j0, k0, mx, my, mz, per_y), m), inner(th_o, m)), ("theta", box)
        assert np.array_equal(inner(_take(gpu_mask, i0, j0, k0, mx, my, mz, per_y), m), inner(mk_o, m)), ("mask", box)
        flagged = int(inner(mk_o, margin_rhs).sum())
    ora.step(1)
    w_o = ora.get_fields()
    w_g = _take(gpu_w1, i0, j0, k0, mx, my, mz, per_y)
    errs = [field_err(inner(w_g[q], margin_step), inner(w_o[q], margin_step), floor_w[q], "state", q, TOL_STEP) for q in range(5)]
    assert max(errs) <= TOL_STEP, ("step", case.name, box, errs)
    ora.close()
    return flagged


def run_sampled(S, case, boxes, need_flagged=True):
    import torch
    floors = natural_scales(case)
    gpu = S(case)
    rhs = gpu.rhs()
    # properties at any size: finite everywhere; in a periodic box the RHS sums to zero (mass always;
    # momentum and energy up to the non-conservative Laplacian-form viscous terms, S11)
    assert bool(torch.isfinite(rhs).all())
    if case.bc_y_lo == W.BC_PERIODIC:
        s_mass = float(rhs[0].sum())
        s_abs = float(rhs[0].abs().sum())
        assert abs(s_mass) <= 1e-9 * max(s_abs, 1.0), (s_mass, s_abs)
    theta, mask = gpu.get_sensor() if case.flux_mode == W.FLUX_HYBRID else (None, None)
    # the box with the strongest sensor response is always sampled
    if theta is not None:
        k, j, i = np.unravel_index(int(np.argmax(theta)), theta.shape)
        mx, my, mz = boxes[0][3:]
        jj = min(max(j - my // 2, 0), case.ny - my) if case.bc_y_lo != W.BC_PERIODIC else j - my // 2
        boxes = list(boxes) + [(i - mx // 2, jj, k - mz // 2, mx, my, mz)]
    rhs_h = rhs.cpu().numpy()
    del rhs
    sums0 = gpu.get_sums(0)
    dt, _ = gpu.step(1)
    sums1 = gpu.get_sums(0)
    if case.bc_y_lo == W.BC_PERIODIC:          # mass is conserved to round-off at any size (library's own fixed-order sums)
        assert abs(sums1[0] - sums0[0]) <= 1e-13 * abs(sums0[0]), (sums0, sums1)
    w1 = gpu.get_fields()
    gpu.destroy()
    flagged = 0
    for box in boxes:
        flagged += compare_box(case, rhs_h, w1, mask, theta, box, dt, floors)
    if need_flagged:
        assert flagged > 0, "no sampled box exercised the WENO branch"


def check_whole_grid(S, case, nsteps):
    """Every output of the full grid against the oracle (configs 1, 2)."""
    gpu = S(case)
    ora = _oracle(case)
    floor_w, floor_r = natural_scales(case)
    hits0 = len(helpers.FLOOR_HITS)
    r_g, r_o = gpu.rhs().cpu().numpy(), ora.rhs()
    errs = [field_err(r_g[q], r_o[q], floor_r[q], "rhs", q, TOL_RHS) for q in range(5)]
    assert max(errs) <= TOL_RHS, ("rhs", case.name, errs)
    th_g, mk_g = gpu.get_sensor()
    th_o, mk_o, _ = ora.sensor()
    assert np.array_equal(th_g, th_o) and np.array_equal(mk_g, mk_o)
    flagged, _, ifaces = gpu.get_activation()
    assert flagged == int(mk_o.sum())
    assert ifaces == [int(ora.interface_flags(d).sum()) for d in range(3)]
    dt_g, t_g = gpu.step(nsteps)
    dt_o, t_o = ora.step(nsteps)
    assert abs(dt_g - dt_o) <= 1e-12 * dt_o and abs(t_g - t_o) <= 1e-12 * t_o
    w_g, w_o = gpu.get_fields(), ora.get_fields()
    errs = [field_err(w_g[q], w_o[q], floor_w[q], "state", q, TOL_STEP) for q in range(5)]
    assert max(errs) <= TOL_STEP, ("step", case.name, errs)
    helpers.check_floor_hits(case, hits0)
    gpu.destroy()
    ora.close()
    return int(mk_o.sum())


def test_config1_full_size_as_benchmarked(S):
    """128^3 exactly as bench.py builds it (solenoidal start: theta ~ 0 at step 0, 10 RK3 steps)."""
    import bench
    check_whole_grid(S, bench.make_case(1), 10)


def test_config1_full_size_sensor_active(S):
    case = W.isotropic_turbulence(n=128, mach_t=0.6, k0=4.0, kmax=32, seed=1, dilatational=0.5)
    assert check_whole_grid(S, case, 10) > 1000


def test_config2_full_size_as_benchmarked(S):
    import bench
    check_whole_grid(S, bench.make_case(2), 10)


@pytest.mark.slow
def test_config3_full_size_whole_grid_ten_steps(S):
    """1024 x 256 x 256 exactly as bench.py builds it, every node, ten RK3 steps (oracle: OpenMP build, ~15 GB)."""
    import bench
    assert check_whole_grid(S, bench.make_case(3), 10) > 0


def test_config3_full_size_sampled(S):
    import bench
    case = bench.make_case(3)            # 1024 x 256 x 256, wall below, free stream above, seeded shocklets
    boxes = [(1024 - 32, 0, 256 - 24, 64, 56, 56),      # wraps in x and z, includes the wall
             (300, 256 - 56, 100, 64, 56, 56)]          # includes the free-stream boundary
    run_sampled(S, case, boxes)


def test_config4_full_size_sampled(S):
    case = W.isotropic_turbulence(n=640, mach_t=0.8, k0=8.0, kmax=64, seed=4, nsteps=10, name="cfg4_iso_640_dil",
                                  dilatational=0.3)
    boxes = [(640 - 30, 640 - 28, 640 - 26, 60, 56, 56),   # the periodic corner
             (200, 311, 421, 60, 56, 56)]
    run_sampled(S, case, boxes)


def _steps_on_boxes(S, case, w_start, nsteps, boxes, margin, dt):
    """GPU: the full grid from w_start, nsteps RK3 steps with the fixed step dt.  Oracle: the same steps on sub-boxes
    cut out of w_start; compared further than `margin` from the box faces.  Returns the flagged nodes the oracle saw
    in the compared regions (evolved state)."""
    floor_w, _ = natural_scales(case)
    fixed = case.replace(dt_fixed=dt, w0=w_start)
    gpu = S(fixed)
    dt_g, t_g = gpu.step(nsteps)
    assert dt_g == dt and abs(t_g - nsteps * dt) <= 1e-12 * t_g
    w_g = gpu.get_fields()
    th_g, mk_g = gpu.get_sensor()
    gpu.destroy()
    flagged = 0
    for (i0, j0, k0, mx, my, mz) in boxes:
        sub = subbox_case(fixed, i0, j0, k0, mx, my, mz, dt)
        ora = _oracle(sub)
        ora.step(nsteps)
        w_o = ora.get_fields()
        sl = (slice(margin, mz - margin), slice(margin, my - margin), slice(margin, mx - margin))
        w_b = _take(w_g, i0, j0, k0, mx, my, mz, True)
        errs = [field_err(w_b[q][sl], w_o[q][sl], floor_w[q], "state", q, TOL_STEP) for q in range(5)]
        assert max(errs) <= TOL_STEP, ("steps", nsteps, (i0, j0, k0), errs)
        # the evolved sensor: theta to round-off of the evolved state, mask equal away from the threshold (S14)
        ora.rhs()
        th_o, mk_o, _ = ora.sensor()
        m2 = margin + 8
        s2 = (slice(m2, mz - m2), slice(m2, my - m2), slice(m2, mx - m2))
        th_b, mk_b = _take(th_g, i0, j0, k0, mx, my, mz, True)[s2], _take(mk_g, i0, j0, k0, mx, my, mz, True)[s2]
        assert np.max(np.abs(th_b - th_o[s2])) < 1e-9
        near = np.abs(th_o[s2] - case.sensor_threshold) < 1e-10
        assert np.array_equal(mk_b[~near], mk_o[s2][~near])
        flagged += int(mk_o[s2].sum())
        ora.close()
    return flagged


def test_config4_as_benchmarked_three_steps(S):
    """bench.make_case(4) itself, from the state bench.py times: the seeded field advanced by the bench's three
    warm-up steps on the GPU, then three more steps with the step size the CFL reduction gives for that state, on
    both sides (GPU: all 640^3 nodes in the launch geometry of the bench; oracle: two 144^3 boxes, margin 60).
    The box around the node with the strongest sensor response is always one of them."""
    import bench
    case = bench.make_case(4)
    gpu = S(case)
    gpu.step(3)
    w_start = gpu.get_fields()
    theta, _ = gpu.get_sensor()
    dt, _ = gpu.step(1)
    gpu.destroy()
    k, j, i = np.unravel_index(int(np.argmax(theta)), theta.shape)
    del theta
    boxes = [(640 - 70, 640 - 72, 640 - 74, 144, 144, 144), (i - 72, j - 72, k - 72, 144, 144, 144)]
    _steps_on_boxes(S, case, w_start, 3, boxes, 60, dt)


@pytest.mark.slow
def test_config4_full_size_ten_steps_sampled(S):
    """Ten RK3 steps at 640^3 from the seeded field (with part of the compressive component kept, so that the WENO
    branch is active from the start): the oracle advances a 384^3 box that wraps around the periodic corner; the
    20^3 nodes further than 182 from its faces (10 steps x 18 nodes of dependency) are compared."""
    case = W.isotropic_turbulence(n=640, mach_t=0.8, k0=8.0, kmax=64, seed=4, nsteps=10, name="cfg4_iso_640_dil",
                                  dilatational=0.3)
    gpu = S(case)
    dt, _ = gpu.step(1)                     # the CFL step of the seeded field, used as the fixed step of both sides
    gpu.destroy()
    _steps_on_boxes(S, case, case.w0, 10, [(640 - 200, 640 - 190, 640 - 180, 384, 384, 384)], 182, 0.8 * dt)
