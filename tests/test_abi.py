"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/streams.h declares,
validates its inputs, and fails loudly (no CPU fallback) without a CUDA device."""
import ctypes as C
import os
import re

import pytest

import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2304_05494_b200 import build, binding
    build.build()
    return binding.load_library()


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "streams.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(streams_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol(lib):
    from paper_2304_05494_b200 import binding
    names = _declared_symbols()
    assert set(names) == set(binding.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_workspace_bytes_and_validation(lib):
    from paper_2304_05494_b200 import binding
    case = W.config(0)
    g, a, s, keep = binding.structs_from_case(case)
    n = lib.streams_workspace_bytes(C.byref(g), C.byref(a), C.byref(s))
    # 5 conserved + 8 primitive + div padded fields at least
    assert n > 14 * 38 * 38 * 38 * 8
    s.central_order = 5
    assert lib.streams_workspace_bytes(C.byref(g), C.byref(a), C.byref(s)) == 0
    assert b"central_order" in lib.streams_last_error(None)
    s.central_order = 6
    g.bc_x = W.BC_WALL_ISOTHERMAL
    assert lib.streams_workspace_bytes(C.byref(g), C.byref(a), C.byref(s)) == 0
    g.bc_x = W.BC_PERIODIC
    g.nx = 2
    assert lib.streams_workspace_bytes(C.byref(g), C.byref(a), C.byref(s)) == 0
    g.nx = 32
    # every order combination the paper names is accepted ("up to 8th and 7th"); order 8 / WENO 7 widen the
    # ghost shell to four layers, so the workspace grows
    s.flux_mode = W.FLUX_HYBRID
    a.l_ref = 1.0
    sizes = {}
    for co in (2, 4, 6, 8):
        for wo in (1, 3, 5, 7):
            s.central_order, s.weno_order = co, wo
            sizes[(co, wo)] = lib.streams_workspace_bytes(C.byref(g), C.byref(a), C.byref(s))
            assert sizes[(co, wo)] > 0, (co, wo, lib.streams_last_error(None))
    assert sizes[(2, 1)] == sizes[(6, 5)] < sizes[(8, 5)] == sizes[(6, 7)] == sizes[(8, 7)]
    s.weno_order = 4
    assert lib.streams_workspace_bytes(C.byref(g), C.byref(a), C.byref(s)) == 0
    s.weno_order = 5
    g.ny = 70000
    assert lib.streams_workspace_bytes(C.byref(g), C.byref(a), C.byref(s)) == 0


def test_fp64_probe_takes_its_scratch_from_the_caller(lib):
    from paper_2304_05494_b200 import binding
    out = C.c_double()
    rc = lib.streams_measure_fp64(None, 0, 1, None, 0, C.byref(out))
    assert rc in (binding.STREAMS_ENOMEM, binding.STREAMS_ECUDA)       # no device: ECUDA; device but no scratch: ENOMEM
    assert lib.streams_measure_fp64(None, 7, 1, None, 0, C.byref(out)) == binding.STREAMS_EINVAL


def test_static_scratch_sums_refuse_what_the_static_array_cannot_hold(lib):
    """streams_sums_static checks its arguments before it touches CUDA: the field limit of its static scratch array and
    the plain argument errors come back with a message in the caller's buffer, with or without a device."""
    from paper_2304_05494_b200 import binding
    err = C.create_string_buffer(256)
    fake = C.c_void_p(256)
    rc = lib.streams_sums_static(fake, binding.SUMS_STATIC_MAX_FIELDS + 1, 4, 4, 4, None, 0, fake, None, err, len(err))
    assert rc == binding.STREAMS_ENOMEM and b"16" in err.value and b"streams_sums_static" in err.value
    assert lib.streams_sums_static(fake, 0, 4, 4, 4, None, 0, fake, None, err, len(err)) == binding.STREAMS_EINVAL
    assert lib.streams_sums_static(fake, 5, 4, 0, 4, None, 0, fake, None, err, len(err)) == binding.STREAMS_EINVAL
    assert lib.streams_sums_static(fake, 5, 4, 4, 4, None, 2, fake, None, err, len(err)) == binding.STREAMS_EINVAL
    assert lib.streams_sums_static(None, 5, 4, 4, 4, None, 0, fake, None, None, 0) == binding.STREAMS_EINVAL


def test_init_without_device_or_workspace_fails_loudly(lib):
    import torch
    from paper_2304_05494_b200 import binding
    case = W.config(0)
    g, a, s, keep = binding.structs_from_case(case)
    h = C.c_void_p()
    rc = lib.streams_init(C.byref(h), C.byref(g), C.byref(a), C.byref(s), None, 0, None)
    assert rc == binding.STREAMS_ENOMEM and not h
    if not torch.cuda.is_available():
        rc = lib.streams_init(C.byref(h), C.byref(g), C.byref(a), C.byref(s), C.c_void_p(256), 1 << 40, None)
        assert rc == binding.STREAMS_ECUDA and not h
        with pytest.raises(RuntimeError):
            binding.Streams(case)


def test_product_path_never_touches_the_oracle():
    """The package must not import or open anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2304_05494_b200")
    for root, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(root, f)).read()
                assert "oracle" not in txt.lower() or f in ("streams_march.cu", "streams_weno.cu", "streams_canon.cu", "streams_fill.cu", "streams_dev.cuh"), f
                assert "import oracle" not in txt and "from oracle" not in txt
