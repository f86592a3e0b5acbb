"""streams_sums_static, the entry point for callers that cannot allocate device memory, against streams_get_sums.

Everything else in the library computes inside a context whose workspace the caller allocated; the sums of
streams_get_sums keep their per-block partials there.  A program that holds all its device memory in a fixed arena, a
residual monitor that another solver calls mid-step with borrowed pointers (where cudaMalloc / cudaFree would stall every
stream of the host application), or a tool that only wants the integrals of a field it already has, cannot or should not
set that up.  streams_sums_static keeps the partials in a static array of the library's device image instead and calls
no allocator.  Every call shares that one array and finds the previous call's partials in it, so the check is made on
calls IN A ROW, of different kinds, field counts and grid sizes: each must still return what the context path returns.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a problem here must not hide the
parity tests.  The test does not depend on what ran before it: the first call in a fresh process performs the one-time
address look-up, after the other tests it finds the library loaded and other kernels' leftovers in memory.
"""
import numpy as np
import pytest

import workloads as W
from tests import helpers

pytestmark = pytest.mark.gpu

TOL_SUM = 1e-12          # the tolerance of test_sum_reductions_match_plain_sums (weights built on the host here)


@pytest.fixture(scope="module")
def B():
    from paper_2304_05494_b200 import build, binding
    build.build()
    return binding


def _volume_weights(case):
    """dV(j) = dx dz / (d eta/dy)(j) with the y metric of the oracle (reading S3), as tests/test_gpu_sequencing.py does."""
    from oracle.oracle import Oracle
    ora = Oracle(case)
    eta_y_c, _, _, _ = ora.metrics()
    ora.close()
    return (case.lx / case.nx) * (case.lz / case.nz) / eta_y_c


def _context_path(B, case):
    """What the existing path returns, and the device arrays the new entry point is then given."""
    import torch
    gpu = B.Streams(case)
    state = gpu.get_sums(0)
    w = gpu.get_fields(torch.empty((5, case.nz, case.ny, case.nx), dtype=torch.float64, device="cuda"))
    r = gpu.rhs()
    residual = gpu.get_sums(1)
    torch.cuda.synchronize()
    gpu.destroy()
    dv = torch.from_numpy(np.ascontiguousarray(_volume_weights(case))).cuda()
    return state, residual, w, r, dv


def test_static_scratch_sums_match_the_context_path_on_calls_in_a_row(B):
    import torch
    cases = [W.channel(48, 40, 36, seed=9),                                   # stretched y, 1440 rows over 592 blocks
             helpers.random_periodic_case(300, 9, 11, seed=3)[0]]             # rows longer than a block, 493 idle blocks
    ref = [_context_path(B, c) for c in cases]
    out = torch.empty(16, dtype=torch.float64, device="cuda")                 # the caller's output buffer, reused
    for rounds in range(2):                                                   # the second round runs on a used array
        for (state, residual, w, r, dv) in ref:
            got = B.sums_static(w, kind=0, row_weight=dv, out=out)[:5].cpu().numpy()
            assert np.all(np.abs(got - state) <= TOL_SUM * np.maximum(np.abs(state), 1.0)), (rounds, got, state)
            got = B.sums_static(r, kind=1, out=out)[:5].cpu().numpy()         # straight after, same array
            assert np.all(np.abs(got - residual) <= TOL_SUM * residual), (rounds, got, residual)
            assert np.array_equal(got, residual)                              # same numbers, same order: same bits
    # 16 fields (the maximum) fill every slot of the array; a one-field call after it must not see them
    state, residual, w, r, dv = ref[0]
    many = torch.cat([r, w, r, w[:1]]).contiguous()
    got16 = B.sums_static(many, kind=1, out=out).cpu().numpy()
    assert np.array_equal(got16[:5], residual) and np.array_equal(got16[10:15], residual)
    one = B.sums_static(r[1:2].contiguous(), kind=1, out=out)[:1].cpu().numpy()
    assert one[0] == residual[1]
    plain = B.sums_static(w[:1].contiguous(), kind=0, out=out)[:1].cpu().numpy()          # no weights: the plain sum
    assert abs(plain[0] - float(w[0].sum())) <= TOL_SUM * abs(plain[0])


def test_static_scratch_limit_is_refused_with_a_message(B):
    import torch
    f = torch.zeros((B.SUMS_STATIC_MAX_FIELDS + 1, 2, 3, 4), dtype=torch.float64, device="cuda")
    with pytest.raises(B.StreamsError) as e:
        B.sums_static(f, kind=1)
    assert e.value.code == B.STREAMS_ENOMEM and "16" in str(e.value)
    with pytest.raises(B.StreamsError) as e:
        B.sums_static(f[:2].contiguous(), kind=5)
    assert e.value.code == B.STREAMS_EINVAL
