"""The host logic of the sharded path (paper_2304_05494_b200/sharded.py) on CPU: slab ranges, the halo exchange over
torch.distributed (two gloo ranks, and three slabs of which two share a process) and the bit-pattern max of the
time-step rate.  The slabs here are plain padded arrays laid out as the library lays out a field ([k][j][i], `ng` ghost
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
