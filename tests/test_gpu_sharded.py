"""The sharded step on ONE GPU: the z slabs of a run live in one process and are stepped in lockstep on one stream
(nothing waits on anything else: the phases of all slabs are enqueued in order), their halo planes moved by device
copies through the same exchange routine that moves them over NCCL between processes.  Every node is computed by the
same arithmetic as in a single context, so the result must equal the single-context run BIT FOR BIT -- fields, time
step and time -- whatever the number of slabs."""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    from paper_2304_05494_b200 import build, binding, sharded
    build.build()
    return binding, sharded


def _single(binding, case, nsteps):
    g = binding.Streams(case)
    dt, t = g.step(nsteps)
    w = g.get_fields()
    g.destroy()
    return dt, t, w


def _sharded(sharded, case, world, nsteps, chunks=(None,)):
    s = sharded.ShardedStreams(case, world, list(range(world)))
    dt = t = None
    n = nsteps
    for c in chunks:
        k = n if c is None else c
        dt, t = s.step(k)
        n -= k
    w = s.get_fields()
    launches = s.kernel_launches()
    s.destroy()
    return dt, t, w, launches


@pytest.mark.parametrize("world", [1, 2, 3])
def test_hybrid_viscous_box_equals_the_single_context_run(mods, world):
    binding, sharded = mods
    case = W.isotropic_turbulence(nx=40, ny=36, nz=41, mach_t=0.6, k0=3.0, kmax=8, seed=91, dilatational=0.5)
    dt0, t0, w0 = _single(binding, case, 6)
    dt1, t1, w1, launches = _sharded(sharded, case, world, 6, chunks=(2, 1, 3))
    assert launches > 0
    assert dt1 == dt0 and t1 == t0
    assert np.array_equal(w1, w0)


def test_channel_with_walls_and_dt_every(mods):
    """Walls in y (ghost fill of the other directions inside each slab), dt recomputed every third step."""
    binding, sharded = mods
    case = W.channel(48, 40, 36, seed=92).replace(dt_every=3)
    dt0, t0, w0 = _single(binding, case, 7)
    dt1, t1, w1, _ = _sharded(sharded, case, 3, 7)
    assert dt1 == dt0 and t1 == t0 and np.array_equal(w1, w0)


@pytest.mark.parametrize("mode", [W.FLUX_CENTRAL, W.FLUX_WENO])
def test_other_flux_modes_and_four_ghost_layers(mods, mode):
    binding, sharded = mods
    case = W.isotropic_turbulence(nx=34, ny=33, nz=30, mach_t=0.4, k0=3.0, kmax=8, seed=93, flux_mode=mode,
                                  viscous=(mode == W.FLUX_CENTRAL))
    case = case.replace(central_order=8, weno_order=7, visc_order=8)
    dt0, t0, w0 = _single(binding, case, 4)
    dt1, t1, w1, _ = _sharded(sharded, case, 2, 4)
    assert dt1 == dt0 and t1 == t0 and np.array_equal(w1, w0)


def test_snapshot_restore_repeats_the_same_steps(mods):
    """bench.py --sharded times every region from one state: restore must bring all slabs back to it."""
    _, sharded = mods
    case = W.isotropic_turbulence(nx=40, ny=36, nz=41, mach_t=0.6, k0=3.0, kmax=8, seed=93, dilatational=0.5)
    s = sharded.ShardedStreams(case, 2, [0, 1])
    s.step(2)
    snap = s.snapshot()
    dt1, t1 = s.step(3)
    w1 = s.get_fields()
    s.restore(snap)
    dt2, _ = s.step(3)
    w2 = s.get_fields()
    s.destroy()
    assert dt1 == dt2 and np.array_equal(w1, w2)


def test_sharded_run_against_the_oracle(mods):
    """The sharded step compared with the oracle itself, not only through the single-context run: three slabs of a
    channel with walls (hybrid, viscous, stretched y), six steps with dt recomputed every other step; fields to the step
    tolerance of the parity tests (1e-9), time step and time to 1e-12."""
    from oracle.oracle import Oracle
    from tests.helpers import field_err, natural_scales
    _, sharded = mods
    case = W.channel(48, 40, 36, seed=93).replace(dt_every=2)
    ora = Oracle(case)
    dt_o, t_o = ora.step(6)
    w_o = ora.get_fields()
    ora.close()
    dt_s, t_s, w_s, _ = _sharded(sharded, case, 3, 6, chunks=(4, 2))
    assert abs(dt_s - dt_o) <= 1e-12 * dt_o and abs(t_s - t_o) <= 1e-12 * t_o
    floor_w, _ = natural_scales(case)
    errs = [field_err(w_s[q], w_o[q], floor_w[q]) for q in range(5)]
    assert max(errs) <= 1e-9, errs
