"""The host logic of the sharded path (paper_2304_05494_b200/sharded.py) on CPU: slab ranges, the halo exchange over
torch.distributed (two gloo ranks, one slab each; several slabs in one process only without torch.distributed), the
bit-pattern max of the time-step rate, and ShardedStreams.step end to end on a stub solver (phase order, rate reduce,
buffer swap, failure on one rank).  The slabs here are plain padded arrays laid out as the library lays out a field ([k][j][i], `ng` ghost
planes in z): after one exchange every ghost plane must hold the periodic neighbour's interior plane."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2304_05494_b200 import sharded as SH


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _global_fields(nz, ny, nx, nf):
    rng = np.random.default_rng(5)
    return rng.standard_normal((nf, nz, ny, nx))


def _make_slab(glob, k0, k1, ng):
    """Padded copy of planes [k0, k1) of every field, ghosts poisoned; returns (array, slab views as the ABI gives them)."""
    nf, nz, ny, nx = glob.shape
    a = torch.full((nf, (k1 - k0) + 2 * ng, ny, nx), float("nan"), dtype=torch.float64)
    a[:, ng:ng + (k1 - k0)] = torch.from_numpy(glob[:, k0:k1])
    n = k1 - k0
    flat = [a[f].reshape(-1).view(torch.uint8) for f in range(nf)]
    plane = ny * nx * 8
    v = dict(lo_recv=[t[:ng * plane] for t in flat], lo_send=[t[ng * plane:2 * ng * plane] for t in flat],
             hi_send=[t[n * plane:(n + ng) * plane] for t in flat], hi_recv=[t[(n + ng) * plane:(n + 2 * ng) * plane] for t in flat])
    return a, v


def _check_slab(a, glob, k0, k1, ng):
    nf, nz = glob.shape[:2]
    for m in range(ng):
        assert np.array_equal(a[:, ng - 1 - m].numpy(), glob[:, (k0 - 1 - m) % nz]), ("lower ghost", m)
        assert np.array_equal(a[:, ng + (k1 - k0) + m].numpy(), glob[:, (k1 + m) % nz]), ("upper ghost", m)
    assert np.array_equal(a[:, ng:ng + (k1 - k0)].numpy(), glob[:, k0:k1])


def test_slab_ranges_cover_the_domain():
    assert SH.slab_ranges(41, 3) == [(0, 14), (14, 28), (28, 41)]
    assert SH.slab_ranges(640, 8) == [(80 * r, 80 * r + 80) for r in range(8)]
    for nz, world in ((7, 2), (128, 5), (33, 4)):
        r = SH.slab_ranges(nz, world)
        assert r[0][0] == 0 and r[-1][1] == nz and all(a[1] == b[0] for a, b in zip(r, r[1:]))
        assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1


def test_slab_case_keeps_spacings_and_marks_the_halo():
    import workloads as W
    case = W.isotropic_turbulence(nx=16, ny=12, nz=21, mach_t=0.3, k0=2.0, kmax=4, seed=1)
    s = SH.slab_case(case, 1, 2, 3)
    assert (s.nz, s.nz_global, s.bc_z, s.lz) == (10, 21, W.BC_HALO, case.lz)
    assert np.array_equal(s.w0, case.w0[:, 11:21])
    with pytest.raises(ValueError):
        SH.slab_case(case, 7, 8, 3)                       # the last slabs have two planes: thinner than the ghost width
    with pytest.raises(ValueError):
        SH.slab_case(case.replace(bc_z=W.BC_FREESTREAM), 0, 2, 3)


@pytest.mark.parametrize("world", [1, 2, 3])
def test_exchange_inside_one_process(world):
    """All slabs local (the one-GPU emulation, and the periodic self-exchange of a single slab)."""
    ng, glob = 3, _global_fields(13, 4, 5, 2)
    ranges = SH.slab_ranges(13, world)
    arrs, views = {}, {}
    for r, (k0, k1) in enumerate(ranges):
        arrs[r], views[r] = _make_slab(glob, k0, k1, ng)
    SH.exchange(views, world, None)
    for r, (k0, k1) in enumerate(ranges):
        _check_slab(arrs[r], glob, k0, k1, ng)


def test_rate_max_on_bit_patterns_keeps_a_nan():
    a, b, c = (torch.tensor([x], dtype=torch.float64).view(torch.uint8) for x in (3.5, 7.25, 0.0))
    SH.rate_bits_max([a, b, c])
    assert [t.view(torch.float64).item() for t in (a, b, c)] == [7.25, 7.25, 7.25]
    n = torch.tensor([float("nan")], dtype=torch.float64).view(torch.uint8)
    SH.rate_bits_max([a, n])
    assert np.isnan(a.view(torch.float64).item()) and np.isnan(n.view(torch.float64).item())


def _worker(rank, nproc, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(nproc))
    dist.init_process_group("gloo", rank=rank, world_size=nproc)
    try:
        ng, nz = 4, 19
        glob = _global_fields(nz, 3, 6, 3)
        # (a) one slab per process
        k0, k1 = SH.slab_ranges(nz, nproc)[rank]
        a, v = _make_slab(glob, k0, k1, ng)
        SH.exchange({rank: v}, nproc, dist)
        _check_slab(a, glob, k0, k1, ng)
        # (b) the time-step rate: every rank ends with the global maximum; a NaN on one rank reaches all
        r = torch.tensor([1.0 + rank], dtype=torch.float64).view(torch.uint8)
        SH.rate_bits_max([r], dist)
        assert r.view(torch.float64).item() == float(nproc)
        r = torch.tensor([float("nan") if rank == 1 else 2.0], dtype=torch.float64).view(torch.uint8)
        SH.rate_bits_max([r], dist)
        assert np.isnan(r.view(torch.float64).item())
        out.put((rank, "ok"))
    except Exception as e:                                 # report instead of hanging the peer
        out.put((rank, repr(e)))
    dist.barrier()
    dist.destroy_process_group()


def test_exchange_between_two_gloo_ranks():
    nproc, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, nproc, port, q)) for r in range(nproc)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(nproc))
    for p in procs:
        p.join(timeout=60)
    assert res == [(0, "ok"), (1, "ok")], res


# ---- ShardedStreams.step end to end with a stub solver (no GPU): the phase order, the HALO_RATE reduce, the exchanges
# of every phase and the primitive-buffer swap are exercised by a toy update whose every phase READS the ghost planes
# the preceding exchange must have filled (they are poisoned with NaN before each phase).  Whatever the cut, the result
# must carry the bits of the uncut run.
class _StubSolver:
    NG = 3

    def __init__(self, case, device="cpu", stream=None):
        assert case.bc_z == SH.BC_HALO
        self.case, self.shape = case, (case.nz, case.ny, case.nx)
        self.w = torch.from_numpy(np.ascontiguousarray(case.w0[0])).clone()          # one scalar field as the state
        nzp = case.nz + 2 * self.NG
        self.q = [torch.full((10, nzp, case.ny, case.nx), float("nan"), dtype=torch.float64) for _ in range(2)]
        self.div = torch.full((1, nzp, case.ny, case.nx), float("nan"), dtype=torch.float64)
        self.mask = torch.full((1, nzp, case.ny, case.nx), 255, dtype=torch.uint8)
        self.rate = torch.zeros(1, dtype=torch.float64)
        self.cur, self.time, self.dt, self.log, self.fail = 0, 0.0, 0.0, [], False

    def _inner(self, a):
        return a[:, self.NG:self.NG + self.case.nz]

    def _poison(self, a, value):
        a[:, :self.NG] = value
        a[:, self.NG + self.case.nz:] = value

    def _zsum(self, plane_stack):                       # sum over the 2 NG + 1 planes around every interior plane
        n, g = self.case.nz, self.NG
        out = plane_stack[g - g:n + g - g].clone()
        for m in range(1, 2 * g + 1):
            out = out + plane_stack[m:n + m]
        return out

    def shard_fill(self, stage):
        self.log.append(("fill", stage))
        q = self.q[self.cur]
        self._poison(q, float("nan"))
        for f in range(10):
            self._inner(q)[f] = self.w * (1.0 + 0.125 * f)
        if stage == 0:
            self.rate[0] = float(self.w.abs().max())
            return True
        return False

    def shard_sensor(self, stage):
        self.log.append(("sensor", stage))
        q = self.q[self.cur]
        assert not torch.isnan(q[[0, 1, 2, 3, 4, 5, 9]]).any(), "primitive ghosts missing before the sensor"
        self._poison(self.div, float("nan"))
        self._poison(self.mask, 255)
        self._inner(self.div)[0] = self._zsum(q[1])
        self._inner(self.mask)[0] = (self._inner(self.div)[0] > 7.0).to(torch.uint8)
        if stage == 0:
            self.dt = 1e-3 / float(self.rate[0])        # the rate must be the global one by now
            self.time += self.dt

    def shard_rhs(self, stage):
        self.log.append(("rhs", stage))
        assert not torch.isnan(self.div).any() and int(self.mask.max()) <= 1, "div / mask ghosts missing before the RHS"
        q = self.q[self.cur]
        self.w = self.w + self.dt * (self._zsum(self.div[0] * self.mask[0].to(torch.float64)) + self._zsum(q[3]))
        self.cur ^= 1                                   # like the library: the other primitive buffer is current now

    def shard_finish(self):
        if self.fail:
            raise RuntimeError("stub: non-finite state")
        return self.dt, self.time

    def halo_slabs(self, what):
        g, n = self.NG, self.case.nz
        if what == SH.HALO_RATE:
            return dict(lo_send=[self.rate.view(torch.uint8)], lo_recv=[], hi_send=[], hi_recv=[])
        a = {SH.HALO_PRIMS: self.q[self.cur], SH.HALO_DIV: self.div, SH.HALO_MASK: self.mask}[what]
        flat = [a[f].reshape(-1).view(torch.uint8) for f in range(a.shape[0])]
        plane = self.case.ny * self.case.nx * a.element_size()
        return dict(lo_recv=[t[:g * plane] for t in flat], lo_send=[t[g * plane:2 * g * plane] for t in flat],
                    hi_send=[t[n * plane:(n + g) * plane] for t in flat], hi_recv=[t[(n + g) * plane:(n + 2 * g) * plane] for t in flat])

    def get_fields(self, out=None):
        return self.w.numpy()[None]

    def kernel_launches(self):
        return len(self.log)

    def destroy(self):
        pass


def _stub_case():
    import workloads as W
    return W.isotropic_turbulence(nx=6, ny=5, nz=17, mach_t=0.3, k0=2.0, kmax=3, seed=4).replace(flux_mode=W.FLUX_HYBRID)


def _stub_run(world, ranks, d=None, steps=3):
    sh = SH.ShardedStreams(_stub_case(), world, ranks, device="cpu", dist=d, solver_cls=_StubSolver)
    dt, t = sh.step(steps)
    logs = [g.log for g in sh.slabs.values()]
    return sh, dt, t, sh.get_fields()[0], logs


def test_sharded_step_on_a_stub_solver_in_one_process():
    """One slab (periodic self-exchange), two and three local slabs: same bits, and the phases in the documented order."""
    _, dt1, t1, w1, logs = _stub_run(1, [0])
    per_stage = [("fill",), ("sensor",), ("rhs",)]
    assert logs[0] == [(p[0], s) for _ in range(3) for s in range(3) for p in per_stage]
    assert np.isfinite(w1).all() and not np.array_equal(w1, _stub_case().w0[0])
    for world in (2, 3):
        sh, dt, t, w, _ = _stub_run(world, list(range(world)))
        assert (dt, t) == (dt1, t1) and np.array_equal(w, w1)
        assert sh.halo_bytes_per_stage() == 2 * 3 * 5 * 6 * (8 * 9 + 8 + 1)      # 9 primitive fields, div, mask; two sides


def _stub_worker(rank, nproc, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(nproc))
    dist.init_process_group("gloo", rank=rank, world_size=nproc)
    try:
        _, dt1, t1, w1, _ = _stub_run(1, [0])                        # the uncut run, locally
        sh, dt, t, w, _ = _stub_run(nproc, [rank], dist)
        k0, k1 = SH.slab_ranges(17, nproc)[rank]
        assert (dt, t) == (dt1, t1) and np.array_equal(w, w1[k0:k1])
        with pytest.raises(ValueError):                              # several slabs per process need no torch.distributed
            SH.ShardedStreams(_stub_case(), 4, [2 * rank, 2 * rank + 1], device="cpu", dist=dist, solver_cls=_StubSolver)
        # a failure on one rank is raised on every rank (nobody is left waiting in the next exchange)
        next(iter(sh.slabs.values())).fail = rank == 1
        with pytest.raises(RuntimeError):
            sh.step(1)
        out.put((rank, "ok"))
    except BaseException as e:                                       # report instead of hanging the peer
        out.put((rank, repr(e)))
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_step_on_a_stub_solver_between_two_gloo_ranks():
    nproc, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_stub_worker, args=(r, nproc, port, q)) for r in range(nproc)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(nproc))
    for p in procs:
        p.join(timeout=60)
    assert res == [(0, "ok"), (1, "ok")], res
