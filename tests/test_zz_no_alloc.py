"""igr_max_wavespeed_noalloc (include/igr.h, csrc/igr_noalloc.cu): the CFL wave speed through the entry point that
allocates nothing (scratch in a file-scope device array) against the existing path, igr_max_wavespeed on a solver
that holds the same fp32 state.  Both run the same per-cell arithmetic and a maximum does not depend on the order of
its operands, so the two agree bitwise on an fp32-stored state; the bound asserted is the one the wave-speed parity
tests use (tests/test_gpu_kernels.py: 2e-6 relative).

Collected last on purpose (file name): the suite runs with `pytest -x`.  The tests pass alone in a fresh process
and after the other tests: nothing here depends on what ran before, and the scratch is shared by every call, so the
two-calls-in-a-row case goes from a large, fast state to a small, slow one (stale partials of the first call sit
beyond the slots the second one reads and must not leak into it)."""
import numpy as np
import pytest
import torch

from paper_2505_07392_b200 import igr
from paper_2505_07392_b200 import workloads as W

pytestmark = pytest.mark.gpu

RTOL = 2e-6          # tests/test_gpu_kernels.py, wave speed


def _existing_path(w, q):
    g = igr.Solver.for_workload(w)
    g.set_state(q)
    return g.max_wavespeed()


def _state(w):
    return W.state(w, device="cuda").contiguous()


def test_two_calls_in_a_row_match_the_existing_path():
    big = W.jets9(n=96, radius=6, pitch=24)          # 54 blocks of 16384 cells, Mach-10 jets
    small = W.entropy_wave(24)                       # 1 block, |u| + c of order 2
    qb, qs = _state(big), _state(small)
    want_b, want_s = _existing_path(big, qb), _existing_path(small, qs)
    assert want_b > 2.0 * want_s                     # a stale partial of the first call would show in the second
    out = torch.full((2,), -1.0, dtype=torch.float32, device="cuda")
    igr.max_wavespeed_noalloc(qb, big.gamma, out)
    got_b = out.cpu().numpy().copy()
    igr.max_wavespeed_noalloc(qs, small.gamma, out)  # second call, same scratch, fewer slots
    got_s = out.cpu().numpy().copy()
    assert got_b[1] == 0.0 and got_s[1] == 0.0
    assert abs(got_b[0] - want_b) <= RTOL * want_b, (got_b[0], want_b)
    assert abs(got_s[0] - want_s) <= RTOL * want_s, (got_s[0], want_s)
    # and back again, both queued before anything is read (stream order alone separates the calls)
    out2 = torch.full((2,), -1.0, dtype=torch.float32, device="cuda")
    igr.max_wavespeed_noalloc(qb, big.gamma, out)
    igr.max_wavespeed_noalloc(qs, small.gamma, out2)
    torch.cuda.synchronize()
    assert abs(float(out[0]) - want_b) <= RTOL * want_b and abs(float(out2[0]) - want_s) <= RTOL * want_s


def test_ragged_size_and_a_side_stream():
    w = W.jets9(n=45, radius=4, pitch=11)            # 91125 cells: 5 full blocks and a tail of 9205 cells
    q = _state(w)
    want = _existing_path(w, q)
    out = torch.zeros(2, dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    igr.max_wavespeed_noalloc(q, w.gamma, out, stream=side.cuda_stream)
    side.synchronize()
    assert float(out[1]) == 0.0 and abs(float(out[0]) - want) <= RTOL * want, (float(out[0]), want)


def test_no_device_memory_is_allocated_by_a_call():
    w = W.entropy_wave(32)
    q = _state(w)
    out = torch.zeros(2, dtype=torch.float32, device="cuda")
    igr.max_wavespeed_noalloc(q, w.gamma, out)       # first call on the device: resolves the scratch address
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        igr.max_wavespeed_noalloc(q, w.gamma, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)


def test_nonfinite_state_is_flagged_like_the_existing_path():
    w = W.entropy_wave(24)
    q = _state(w)
    q[4, 3, 5, 7] = -1.0                             # negative energy: sqrt of a negative pressure
    with pytest.raises(igr.IgrError) as ei:
        _existing_path(w, q)
    assert ei.value.code == igr.ERR_NONFINITE
    out = torch.zeros(2, dtype=torch.float32, device="cuda")
    igr.max_wavespeed_noalloc(q, w.gamma, out)
    assert float(out[1]) == 1.0 and np.isfinite(float(out[0]))
    q[4, 3, 5, 7] = float("nan")
    igr.max_wavespeed_noalloc(q, w.gamma, out)
    assert float(out[1]) == 1.0


def test_sizes_beyond_the_scratch_are_refused_with_a_message():
    q = torch.zeros(8, dtype=torch.float32, device="cuda")       # never read: the size check comes first
    out = torch.full((2,), -7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(igr.IgrError) as ei:
        igr.max_wavespeed_noalloc(q, 1.4, out, shape=(1025, 1024, 1024))
    assert ei.value.code == igr.ERR_ARG
    assert "IGR_NOALLOC_MAX_CELLS" in str(ei.value) and str(igr.NOALLOC_MAX_CELLS) in str(ei.value)
    for bad in ((0, 4, 4), (4, -1, 4)):
        with pytest.raises(igr.IgrError) as ei:
            igr.max_wavespeed_noalloc(q, 1.4, out, shape=bad)
        assert ei.value.code == igr.ERR_ARG
    with pytest.raises(igr.IgrError):
        igr.max_wavespeed_noalloc(q, 1.0, out, shape=(1, 1, 1))  # gamma <= 1
    torch.cuda.synchronize()
    assert float(out[0]) == -7.0                                 # nothing was launched
