"""Sharded stepping: the domain cut into z slabs, one libstreams context per slab ("GPU-aware
halo communication", PAPER:507 synchronous mode).

Host logic only: every step of the path still runs in the kernels of libstreams.so through the C ABI
(`streams_shard_fill / _sensor / _rhs`, include/streams.h); this module decides who owns which planes, moves the halo
planes between the slabs after each phase and max-reduces the time-step rate.  Two transports:

  * `torch.distributed` point-to-point operations (one process per GPU, backend "nccl": over NVLink the send of a
    slab's first / last `ng` planes lands directly in the neighbour's ghost planes; backend "gloo" on CPU tensors for the
    tests of this logic), one `batch_isend_irecv` per phase;
  * direct copies between slabs that live in the same process (several slabs on one GPU, used by the one-GPU test that
    checks a sharded run against the single-context run bit for bit; also the periodic self-exchange of a single slab).

Only z is cut and z must be periodic in the whole domain (all five BASELINE configs are).  The exchange is synchronous:
it is enqueued on the slab's stream between two phases (the paper's asynchronous mode gains 1.4-2.5 %; the
interior-first split that would overlap it is not built).

With torch.distributed every process holds exactly ONE slab and the slab index is the process rank (`exchange` uses it
as the peer of its sends and receives); several slabs per process exist only without torch.distributed (one GPU).
"""
from __future__ import annotations

import numpy as np

HALO_PRIMS, HALO_DIV, HALO_MASK, HALO_RATE = 0, 1, 2, 3
BC_PERIODIC, BC_HALO = 0, 3
Q_T, Q_MU, Q_DIV, Q_C = 6, 7, 8, 9          # slots of the primitive buffer that not every mode uses


def slab_ranges(nz: int, world: int):
    """[k0, k1) of every rank: contiguous, as even as possible, the first nz % world slabs one plane thicker."""
    base, rem = divmod(nz, world)
    out, k = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((k, k + n))
        k += n
    return out


def slab_case(case, rank: int, world: int, ng_needed: int = 4):
    """The sub-problem of one slab: same spacings and parameters, nz planes of the field, halo boundaries in z."""
    if case.bc_z != BC_PERIODIC:
        raise ValueError("the sharded path cuts a periodic z direction")
    k0, k1 = slab_ranges(case.nz, world)[rank]
    if k1 - k0 < ng_needed:
        raise ValueError(f"slab of rank {rank} has {k1 - k0} planes: fewer than the ghost width")
    w0 = None if case.w0 is None else np.ascontiguousarray(case.w0[:, k0:k1])
    return case.replace(name=f"{case.name}_slab{rank}of{world}", nz=k1 - k0, nz_global=case.nz, bc_z=BC_HALO, w0=w0)


def rate_bits_max(tensors, dist=None):
    """Max of non-negative doubles (or NaN) over slabs and ranks, in place, on their bit patterns viewed as int64: the
    order of the patterns is the order of the values and a NaN (0x7ff8...) is the largest, as in the kernels' own
    reduction; MAX on the floating values would leave NaN propagation to the backend."""
    import torch
    bits = [t.view(torch.int64) for t in tensors]
    m = bits[0].clone()
    for b in bits[1:]:
        m = torch.maximum(m, b)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(m, op=dist.ReduceOp.MAX)
    for b in bits:
        b.copy_(m)


def exchange(slabs, world: int, dist=None):
    """One halo exchange.  slabs: {rank: dict(lo_send, lo_recv, hi_send, hi_recv -> list of 1-D tensors, one per
    field)} for the ranks that live in this process.  A slab's lo_send goes to the hi_recv of the slab below
    (rank - 1, periodic), its hi_send to the lo_recv of the slab above; copies inside the process are direct, the
    others one batch of point-to-point operations."""
    if dist is not None and world > 1 and len(slabs) != 1:
        raise ValueError("with torch.distributed a process holds exactly one slab (slab index = process rank)")
    ops = []
    for r, s in slabs.items():
        lo, hi = (r - 1) % world, (r + 1) % world
        for mine, peer, theirs in (("lo_send", lo, "hi_recv"), ("hi_send", hi, "lo_recv")):
            if peer in slabs:
                for src, dst in zip(s[mine], slabs[peer][theirs]):
                    dst.copy_(src)
            else:
                ops += [dist.P2POp(dist.isend, t, peer) for t in s[mine]]
        # Messages between one pair of ranks match in posting order (NCCL has no tags).  With two ranks both neighbours
        # are the same peer: its first messages are its lo_send, which belong in this slab's hi_recv -- so the upper
        # ghosts are posted first, mirroring the order of the sends above.
        for mine, peer in (("hi_recv", hi), ("lo_recv", lo)):
            if peer not in slabs:
                ops += [dist.P2POp(dist.irecv, t, peer) for t in s[mine]]
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()


class ShardedStreams:
    """The slabs of this process stepped in lockstep.  ranks: the global slab indices held here (one per process with
    torch.distributed; all of them for an in-process run on one device)."""

    def __init__(self, case, world: int, ranks, device="cuda:0", dist=None, solver_cls=None):
        import torch
        from . import binding
        self.torch = torch
        self.case, self.world, self.dist = case, int(world), dist
        self.ranges = slab_ranges(case.nz, world)
        self.device = torch.device(device)
        cls = solver_cls or binding.Streams
        ng = 4 if max(case.central_order, case.visc_order if case.visc_law else 0, case.weno_order + 1) >= 8 else 3
        if dist is not None and world > 1 and len(list(ranks)) != 1:
            raise ValueError("with torch.distributed a process holds exactly one slab (slab index = process rank)")
        self.stream = None                                      # CPU tensors (stub solvers in the gloo tests): no stream
        if self.device.type == "cuda":
            with torch.cuda.device(self.device):
                self.stream = torch.cuda.Stream(self.device)    # one stream for all local slabs: phases stay ordered
        self.slabs = {r: cls(slab_case(case, r, world, ng), device=device, stream=self.stream) for r in ranks}
        self.hybrid = case.flux_mode == 2
        self.visc = case.visc_law != 0
        self.weno = case.flux_mode != 0

    def _views(self, what):
        out = {}
        for r, g in self.slabs.items():
            v = g.halo_slabs(what)
            if what == HALO_PRIMS:                              # only the slots this mode reads (div travels on its own)
                keep = [f for f in range(10) if f not in (Q_DIV,) and (self.visc or f not in (Q_T, Q_MU))
                        and (self.weno or f != Q_C)]
                v = {k: [t[f] for f in keep] for k, t in v.items()}
            out[r] = v
        return out

    def _on_stream(self):
        import contextlib
        return self.torch.cuda.stream(self.stream) if self.stream is not None else contextlib.nullcontext()

    def _exchange(self, what):
        with self._on_stream():
            exchange(self._views(what), self.world, self.dist)

    def halo_bytes_per_stage(self):
        """Bytes one slab SENDS per RK stage (both neighbours, every exchange of the stage), from the slab sizes the
        library reports (streams_halo_slabs) and the fields this mode exchanges."""
        r = next(iter(self.slabs))
        total = 0
        for what in [HALO_PRIMS] + ([HALO_DIV] if (self.hybrid or self.visc) else []) + ([HALO_MASK] if self.hybrid else []):
            v = self._views(what)[r]
            total += sum(int(t.numel()) * t.element_size() for k in ("lo_send", "hi_send") for t in v[k])
        return total

    def step(self, nsteps: int):
        for _ in range(int(nsteps)):
            for stage in range(3):
                local_rate = [g.shard_fill(stage) for g in self.slabs.values()]
                if any(local_rate):
                    with self._on_stream():
                        rate_bits_max([g.halo_slabs(HALO_RATE)["lo_send"][0] for g in self.slabs.values()], self.dist)
                self._exchange(HALO_PRIMS)
                for g in self.slabs.values():
                    g.shard_sensor(stage)
                if self.hybrid or self.visc:
                    self._exchange(HALO_DIV)
                if self.hybrid:
                    self._exchange(HALO_MASK)
                for g in self.slabs.values():
                    g.shard_rhs(stage)
        out, err = [], None
        for g in self.slabs.values():
            try:
                out.append(g.shard_finish())
            except RuntimeError as e:                            # e.g. STREAMS_ENAN on this slab only
                err = e
        # every rank learns of a failure before anybody raises: a rank that raised alone would leave its peers blocked
        # in the next exchange
        d = self.dist
        if d is not None and d.is_initialized() and d.get_world_size() > 1:
            flag_dev = self.device if d.get_backend() == "nccl" else "cpu"
            flag = self.torch.tensor([1 if err is not None else 0], dtype=self.torch.int32, device=flag_dev)
            d.all_reduce(flag, op=d.ReduceOp.MAX)
            if err is None and int(flag.item()):
                err = RuntimeError("the step failed on another rank's slab")
        if err is not None:
            raise err
        return out[0]

    def get_fields(self):
        """The conserved state of the local slabs stacked along z: [5, sum of local nz, ny, nx]."""
        return np.concatenate([self.slabs[r].get_fields() for r in sorted(self.slabs)], axis=1)

    def snapshot(self):
        """The conserved state of every local slab as device tensors (for restore)."""
        out = {}
        for r, g in self.slabs.items():
            t = self.torch.empty((5,) + tuple(g.shape), dtype=self.torch.float64, device=self.device)
            out[r] = g.get_fields(t)
        return out

    def restore(self, snap):
        """Back to a snapshot: the next step starts from it like from streams_set_fields."""
        for r, g in self.slabs.items():
            g.set_fields(snap[r])

    def kernel_launches(self):
        return sum(g.kernel_launches() for g in self.slabs.values())

    def destroy(self):
        for g in self.slabs.values():
            g.destroy()
        self.slabs = {}
