"""The N > 1 path of bench.py on CPU: two gloo ranks, independent replicas, max-over-ranks timing
("replicas only", no data-path collective)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    from paper_2304_05494_b200 import replicas as R
    import workloads as W
    assert R.rank_info() == (rank, world, rank)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rep = R.Replicas(dist, torch.device("cpu"))
    assert (rep.rank, rep.world) == (rank, world)
    # each rank builds ITS replica of the workload: same recipe, its own seed, no exchange of field data
    case = W.isotropic_turbulence(n=16, mach_t=0.3, k0=2.0, kmax=4, seed=R.replica_seed(1, rank))
    checksum = float(np.abs(case.w0).sum())
    rep.barrier()
    ms = 10.0 * (rank + 1)                       # rank 1 is the slow one
    units = 1000.0 * (rank + 1)
    out.put((rank, checksum, rep.max_over_ranks(ms), rep.throughput(units, ms)))
    rep.barrier()
    dist.destroy_process_group()


def test_two_rank_replicas_timing_and_seeds():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, c0, m0, t0), (r1, c1, m1, t1) = res
    assert (r0, r1) == (0, 1)
    assert c0 != c1                               # replicas differ by seed
    assert m0 == m1 == 20.0                       # the slowest rank's time, seen by every rank
    assert t0 == t1 == (1000.0 + 2000.0) / 20e-3  # all units / max time


def test_single_rank_needs_no_process_group():
    from paper_2304_05494_b200 import replicas as R
    rep = R.Replicas(None)
    assert rep.world == 1 and rep.max_over_ranks(3.0) == 3.0 and rep.throughput(50.0, 10.0) == 5000.0
    assert R.replica_seed(4, 0) == 4 and R.replica_seed(4, 3) == 304
