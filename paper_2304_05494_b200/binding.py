"""Thin ctypes binding of include/streams.h: argument marshalling only.

Every step of the path runs in the kernels of libstreams.so.  PyTorch is used for device memory
(the workspace tensor) and the CUDA stream, nothing else.  There is no CPU fallback: if the
library or a CUDA device is missing, construction raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "lib", "libstreams.so")

STREAMS_OK, STREAMS_EINVAL, STREAMS_ENOMEM, STREAMS_ECUDA, STREAMS_ESTATE, STREAMS_ENAN = 0, -1, -2, -3, -4, -5
EXPORTS = ("streams_workspace_bytes", "streams_init", "streams_set_fields", "streams_rhs", "streams_step",
           "streams_step_forced", "streams_shard_fill", "streams_shard_sensor", "streams_shard_rhs",
           "streams_shard_finish", "streams_halo_slabs", "streams_get_fields", "streams_get_sensor", "streams_set_mask_override", "streams_get_sums", "streams_set_body_force", "streams_get_activation", "streams_get_activation_totals",
           "streams_kernel_launches", "streams_graph_launches",
           "streams_profile", "streams_get_profile", "streams_kernel_name", "streams_measure_fp64",
           "streams_measure_fp64_scratch_bytes", "streams_sums_static",
           "streams_last_error", "streams_destroy")
STREAMS_K_COUNT = 8
SUMS_STATIC_MAX_FIELDS = 16          # STREAMS_SUMS_STATIC_MAX_FIELDS

_dp = C.POINTER(C.c_double)


class streams_grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
                ("y_nodes", _dp), ("y_wall_lo", C.c_double), ("y_wall_hi", C.c_double),
                ("bc_x", C.c_int), ("bc_y_lo", C.c_int), ("bc_y_hi", C.c_int), ("bc_z", C.c_int),
                ("t_wall_lo", C.c_double), ("t_wall_hi", C.c_double), ("nz_global", C.c_int)]


class streams_gas(C.Structure):
    _fields_ = [("gamma", C.c_double), ("rgas", C.c_double), ("prandtl", C.c_double),
                ("visc_law", C.c_int), ("mu_ref", C.c_double), ("t_ref", C.c_double),
                ("suth_s_over_tref", C.c_double), ("pow_exp", C.c_double),
                ("u_ref", C.c_double), ("l_ref", C.c_double), ("freestream", C.c_double * 5),
                ("accel", C.c_double * 3)]


class streams_scheme(C.Structure):
    _fields_ = [("central_order", C.c_int), ("weno_order", C.c_int), ("visc_order", C.c_int),
                ("flux_mode", C.c_int), ("sensor_threshold", C.c_double), ("weno_eps", C.c_double),
                ("cfl", C.c_double), ("dt_fixed", C.c_double), ("dt_every", C.c_int), ("weno_variant", C.c_int)]


_lib = None


def load_library(path: str = None):
    """dlopen libstreams.so and declare the prototypes of include/streams.h.  STREAMS_LIB=<path> selects another
    build of the same library (measurement builds of paper_2304_05494_b200.build --tag)."""
    global _lib
    if _lib is not None:
        return _lib
    if path is None:
        path = os.environ.get("STREAMS_LIB") or LIB_PATH
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with `python -m paper_2304_05494_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(path)
    gp, ap, sp = C.POINTER(streams_grid), C.POINTER(streams_gas), C.POINTER(streams_scheme)
    lib.streams_workspace_bytes.restype = C.c_size_t
    lib.streams_workspace_bytes.argtypes = [gp, ap, sp]
    lib.streams_init.argtypes = [C.POINTER(C.c_void_p), gp, ap, sp, C.c_void_p, C.c_size_t, C.c_void_p]
    lib.streams_set_fields.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
    lib.streams_rhs.argtypes = [C.c_void_p, C.c_void_p]
    lib.streams_step.argtypes = [C.c_void_p, C.c_int, _dp, _dp]
    lib.streams_step_forced.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, _dp, _dp, _dp]
    lib.streams_get_fields.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
    lib.streams_shard_fill.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int)]
    lib.streams_shard_sensor.argtypes = [C.c_void_p, C.c_int]
    lib.streams_shard_rhs.argtypes = [C.c_void_p, C.c_int]
    lib.streams_shard_finish.argtypes = [C.c_void_p, _dp, _dp]
    lib.streams_halo_slabs.argtypes = [C.c_void_p, C.c_int] + [C.POINTER(C.c_void_p)] * 4 + [C.POINTER(C.c_size_t), C.POINTER(C.c_int), C.POINTER(C.c_size_t)]
    lib.streams_get_sensor.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
    lib.streams_set_mask_override.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
    lib.streams_get_sums.argtypes = [C.c_void_p, C.c_int, _dp]
    lib.streams_set_body_force.argtypes = [C.c_void_p, _dp]
    lib.streams_get_activation.argtypes = [C.c_void_p] + [C.POINTER(C.c_longlong)] * 3
    lib.streams_get_activation_totals.argtypes = [C.c_void_p] + [C.POINTER(C.c_longlong)] * 4
    lib.streams_kernel_launches.restype = C.c_longlong
    lib.streams_kernel_launches.argtypes = [C.c_void_p]
    lib.streams_graph_launches.restype = C.c_longlong
    lib.streams_graph_launches.argtypes = [C.c_void_p]
    lib.streams_profile.argtypes = [C.c_void_p, C.c_int, C.c_int]
    lib.streams_get_profile.argtypes = [C.c_void_p, _dp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    lib.streams_measure_fp64_scratch_bytes.restype = C.c_size_t
    lib.streams_measure_fp64_scratch_bytes.argtypes = []
    lib.streams_measure_fp64.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_size_t, _dp]
    lib.streams_sums_static.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_void_p,
                                        C.c_void_p, C.c_char_p, C.c_size_t]
    lib.streams_kernel_name.restype = C.c_char_p
    lib.streams_kernel_name.argtypes = [C.c_int]
    lib.streams_last_error.restype = C.c_char_p
    lib.streams_last_error.argtypes = [C.c_void_p]
    lib.streams_destroy.argtypes = [C.c_void_p]
    _lib = lib
    return lib


def structs_from_case(case):
    """workloads.Case -> (streams_grid, streams_gas, streams_scheme, keepalive)."""
    g, a, s = streams_grid(), streams_gas(), streams_scheme()
    for n in ("nx", "ny", "nz", "lx", "ly", "lz", "y_wall_lo", "y_wall_hi", "bc_x", "bc_y_lo", "bc_y_hi", "bc_z",
              "t_wall_lo", "t_wall_hi", "nz_global"):
        setattr(g, n, getattr(case, n))
    keep = None
    if case.y_nodes is not None:
        keep = np.ascontiguousarray(case.y_nodes, dtype=np.float64)
        g.y_nodes = keep.ctypes.data_as(_dp)
    for n in ("gamma", "rgas", "prandtl", "visc_law", "mu_ref", "t_ref", "suth_s_over_tref", "pow_exp", "u_ref", "l_ref"):
        setattr(a, n, getattr(case, n))
    for q in range(5):
        a.freestream[q] = case.freestream[q]
    for d in range(3):
        a.accel[d] = case.accel[d]
    for n in ("central_order", "weno_order", "visc_order", "flux_mode", "sensor_threshold", "weno_eps", "cfl",
              "dt_fixed", "dt_every", "weno_variant"):
        setattr(s, n, getattr(case, n))
    return g, a, s, keep


def measure_fp64(kind: int = 0, repeats: int = 5, stream=None) -> float:
    """streams_measure_fp64 on the current device: 1e9 thread-level fp64 instructions per second
    (kind 0: DFMA chains, kind 1: DADD + DMUL)."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: libstreams has no CPU fallback")
    lib = load_library()
    st = stream if stream is not None else torch.cuda.current_stream()
    out = C.c_double()
    nbytes = lib.streams_measure_fp64_scratch_bytes()
    scratch = torch.empty(max(nbytes, 8), dtype=torch.uint8, device="cuda")
    rc = lib.streams_measure_fp64(C.c_void_p(st.cuda_stream), int(kind), int(repeats), C.c_void_p(scratch.data_ptr()),
                                  C.c_size_t(nbytes), C.byref(out))
    if rc != STREAMS_OK:
        raise StreamsError(rc, lib.streams_last_error(None).decode())
    return out.value


def sums_static(f, kind: int = 0, row_weight=None, out=None, stream=None):
    """streams_sums_static: the sums of streams_get_sums for callers who cannot hand the library device scratch memory
    (a fixed arena, a hook inside another solver's step; include/streams.h says who and why).  The partial sums go to
    an array inside the library's device image, the C call allocates nothing.

    f: CUDA float64 tensor [nfields, nz, ny, nx] (at most 16 fields), contiguous; row_weight: CUDA float64 [ny] or None;
    kind 0: sum of f_q * row_weight[j], kind 1: sum of f_q ** 2.  out: CUDA float64 [nfields], given by the caller (only
    this Python convenience makes one with torch when it is None).  Enqueued on `stream` (default: torch's current
    stream) and not synchronised.  Do not let two calls overlap on the GPU: they share the one static array."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: libstreams has no CPU fallback")
    lib = load_library()
    assert f.is_cuda and f.dtype == torch.float64 and f.is_contiguous() and f.dim() == 4
    nf, nz, ny, nx = (int(n) for n in f.shape)
    if row_weight is not None:
        assert row_weight.is_cuda and row_weight.dtype == torch.float64 and row_weight.is_contiguous()
        assert tuple(row_weight.shape) == (ny,) and row_weight.device == f.device
    if out is None:
        out = torch.empty(max(nf, 1), dtype=torch.float64, device=f.device)[:nf]
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= nf and out.device == f.device
    err = C.create_string_buffer(256)
    with torch.cuda.device(f.device):
        st = stream if stream is not None else torch.cuda.current_stream()
        rc = lib.streams_sums_static(C.c_void_p(f.data_ptr()), nf, nx, ny, nz,
                                     C.c_void_p(row_weight.data_ptr()) if row_weight is not None else None, int(kind),
                                     C.c_void_p(out.data_ptr()), C.c_void_p(st.cuda_stream), err, len(err))
    if rc != STREAMS_OK:
        raise StreamsError(rc, err.value.decode())
    return out


class StreamsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"streams error {code}: {msg}")
        self.code = code


class Streams:
    """One solver context on the current CUDA device.  Method names follow the C ABI."""

    def __init__(self, case, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: libstreams has no CPU fallback")
        self.lib = load_library()
        self.torch = torch
        self.device = torch.device(device)
        self.case = case
        self.shape = (case.nz, case.ny, case.nx)
        g, a, s, self._keep = structs_from_case(case)
        nbytes = self.lib.streams_workspace_bytes(C.byref(g), C.byref(a), C.byref(s))
        if nbytes == 0:
            raise StreamsError(STREAMS_EINVAL, self.lib.streams_last_error(None).decode())
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            # a stream of the context's own unless the caller brings one: the legacy default stream cannot be captured
            # into the CUDA graphs streams_step replays.  Device tensors that cross this boundary are ordered against
            # torch's current stream explicitly (_after_torch / _before_torch).
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
        ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        h = C.c_void_p()
        rc = self.lib.streams_init(C.byref(h), C.byref(g), C.byref(a), C.byref(s), C.c_void_p(ptr), nbytes,
                                   C.c_void_p(self.stream.cuda_stream))
        if rc != STREAMS_OK:
            raise StreamsError(rc, self.lib.streams_last_error(None).decode())
        self.h = h
        self.workspace_bytes = nbytes
        if case.w0 is not None:
            self.set_fields(case.w0)

    # -- helpers
    def _check(self, rc):
        if rc != STREAMS_OK:
            raise StreamsError(rc, self.lib.streams_last_error(self.h).decode())

    @staticmethod
    def _ptr(x):
        """(pointer, is_device) of a numpy array or torch tensor."""
        if isinstance(x, np.ndarray):
            assert x.flags["C_CONTIGUOUS"]
            return C.c_void_p(x.ctypes.data), 0
        assert x.is_contiguous()
        return C.c_void_p(x.data_ptr()), int(x.is_cuda)

    def _after_torch(self):
        """The library's stream waits for what torch has enqueued (a device tensor is about to be read)."""
        self.stream.wait_stream(self.torch.cuda.current_stream(self.device))

    def _before_torch(self):
        """torch's current stream waits for the library's (a device tensor has just been written)."""
        self.torch.cuda.current_stream(self.device).wait_stream(self.stream)

    # -- C ABI
    def set_fields(self, w):
        if isinstance(w, np.ndarray):
            w = np.ascontiguousarray(w, dtype=np.float64)
        assert tuple(w.shape) == (5,) + self.shape
        p, dev = self._ptr(w)
        if dev:
            self._after_torch()
        self._check(self.lib.streams_set_fields(self.h, p, dev))

    def rhs(self, out=None):
        if out is None:
            out = self.torch.empty((5,) + self.shape, dtype=self.torch.float64, device=self.device)
        assert out.is_cuda
        self._after_torch()
        self._check(self.lib.streams_rhs(self.h, C.c_void_p(out.data_ptr())))
        self._before_torch()
        return out

    def step(self, nsteps):
        dt, t = C.c_double(), C.c_double()
        self._check(self.lib.streams_step(self.h, int(nsteps), C.byref(dt), C.byref(t)))
        return dt.value, t.value

    def step_forced(self, nsteps, direction=0, target=float("nan")):
        """nsteps steps under the device-side bulk-flow controller; returns (dt, time, [g_x, g_y, g_z])."""
        dt, t = C.c_double(), C.c_double()
        g = (C.c_double * 3)()
        self._check(self.lib.streams_step_forced(self.h, int(nsteps), int(direction), C.c_double(target), C.byref(dt),
                                                 C.byref(t), C.cast(g, _dp)))
        return dt.value, t.value, list(g)

    # -- sharded stepping (one context per z slab; paper_2304_05494_b200/sharded.py drives these)
    def shard_fill(self, stage):
        flag = C.c_int()
        self._check(self.lib.streams_shard_fill(self.h, int(stage), C.byref(flag)))
        return bool(flag.value)

    def shard_sensor(self, stage):
        self._check(self.lib.streams_shard_sensor(self.h, int(stage)))

    def shard_rhs(self, stage):
        self._check(self.lib.streams_shard_rhs(self.h, int(stage)))

    def shard_finish(self):
        dt, t = C.c_double(), C.c_double()
        self._check(self.lib.streams_shard_finish(self.h, C.byref(dt), C.byref(t)))
        return dt.value, t.value

    def halo_slabs(self, what):
        """Torch views (no copies) of the slabs to exchange: dict lo_send / lo_recv / hi_send / hi_recv, each a list of
        one 1-D uint8 tensor per field, aliasing the workspace."""
        ptrs = [C.c_void_p() for _ in range(4)]
        nbytes, nf, stride = C.c_size_t(), C.c_int(), C.c_size_t()
        self._check(self.lib.streams_halo_slabs(self.h, int(what), *[C.byref(p) for p in ptrs], C.byref(nbytes), C.byref(nf),
                                                C.byref(stride)))
        base = self.workspace.data_ptr()
        out = {}
        for name, p in zip(("lo_send", "lo_recv", "hi_send", "hi_recv"), ptrs):
            if not p.value:
                out[name] = []
                continue
            off = p.value - base
            out[name] = [self.workspace[off + f * stride.value: off + f * stride.value + nbytes.value] for f in range(nf.value)]
        return out

    def get_fields(self, out=None):
        if out is None:
            out = np.empty((5,) + self.shape, dtype=np.float64)
        p, dev = self._ptr(out)
        if dev:
            self._after_torch()
        self._check(self.lib.streams_get_fields(self.h, p, dev))
        if dev:
            self._before_torch()
        return out

    def get_sensor(self):
        theta = np.empty(self.shape, dtype=np.float64)
        mask = np.empty(self.shape, dtype=np.uint8)
        self._check(self.lib.streams_get_sensor(self.h, C.c_void_p(theta.ctypes.data), C.c_void_p(mask.ctypes.data), 0))
        return theta, mask

    def set_mask_override(self, mask):
        """Impose the node mask ([nz, ny, nx] uint8 of 0 / 1, numpy or CUDA tensor); None restores the sensor's own."""
        if mask is None:
            self._check(self.lib.streams_set_mask_override(self.h, None, 0))
            return
        if isinstance(mask, np.ndarray):
            mask = np.ascontiguousarray(mask, dtype=np.uint8)
        assert tuple(mask.shape) == self.shape
        p, dev = self._ptr(mask)
        if dev:
            self._after_torch()
        self._check(self.lib.streams_set_mask_override(self.h, p, dev))

    def set_body_force(self, accel):
        g = (C.c_double * 3)(*[float(x) for x in accel])
        self._check(self.lib.streams_set_body_force(self.h, g))

    def get_sums(self, kind=0):
        """kind 0: volume integrals of the five conserved variables; kind 1: sums of R_q^2 of the last streams_rhs."""
        out = (C.c_double * 5)()
        self._check(self.lib.streams_get_sums(self.h, int(kind), out))
        return np.array(list(out))

    def get_activation(self):
        """(flagged nodes, nodes next to a flagged interface, [flagged interfaces x, y, z]) of the last RHS."""
        a, b = C.c_longlong(), C.c_longlong()
        f = (C.c_longlong * 3)()
        self._check(self.lib.streams_get_activation(self.h, C.byref(a), C.byref(b), f))
        return a.value, b.value, list(f)

    def get_activation_totals(self):
        """(flagged nodes, shock-list nodes, [interfaces x, y, z], sensor evaluations) summed since set_fields."""
        a, b, n = C.c_longlong(), C.c_longlong(), C.c_longlong()
        f = (C.c_longlong * 3)()
        self._check(self.lib.streams_get_activation_totals(self.h, C.byref(a), C.byref(b), f, C.byref(n)))
        return a.value, b.value, list(f), n.value

    def kernel_launches(self):
        return int(self.lib.streams_kernel_launches(self.h))

    def graph_launches(self):
        return int(self.lib.streams_graph_launches(self.h))

    def profile(self, enable=True, max_records=0):
        self._check(self.lib.streams_profile(self.h, int(bool(enable)), int(max_records)))

    def get_profile(self):
        """{kernel class name: (device ms, recorded launch groups)}, and the number of unrecorded launches."""
        ms = (C.c_double * STREAMS_K_COUNT)()
        cnt = (C.c_longlong * STREAMS_K_COUNT)()
        dropped = C.c_longlong()
        self._check(self.lib.streams_get_profile(self.h, ms, cnt, C.byref(dropped)))
        out = {self.lib.streams_kernel_name(k).decode(): (ms[k], cnt[k]) for k in range(STREAMS_K_COUNT)}
        return out, dropped.value

    def destroy(self):
        if getattr(self, "h", None):
            self.lib.streams_destroy(self.h)         # synchronises the stream
            self.h = None
        self.workspace = None                        # the device memory goes back to torch's allocator

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
