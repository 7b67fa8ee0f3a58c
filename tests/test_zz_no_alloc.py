"""g3_msd_static, the entry point of libg3 that allocates no device memory, against g3_msd.

Why the entry point exists: g3_msd takes its scratch from the CUDA memory pool on every call.  A host
program that analyses in situ while its own allocator (an MD engine's arena, PyTorch's caching
allocator) already owns nearly all of the GPU's memory, or that runs under a fixed per-process
memory limit, cannot count on the driver having anything left and gets G3_ENOMEM.  g3_msd_static
keeps the same scratch in a fixed array built into the library (include/g3.h: about 8 MiB per GPU,
held until the process exits) and therefore accepts only problems that fit it.

What is checked: the sums (exact 128-bit integers) are bit-identical to g3_msd's and msd agrees
to the 1e-12 the MSD parity tests use, on calls IN A ROW.  All calls share the one array and it
keeps the last call's contents, so the second call is smaller than the first (stale partial
sums lie right behind its own) and a rejected trajectory is followed by a good one (the error
counter must have been cleared).  Problems beyond the array's size must be refused with G3_ELIMIT
rather than served by an allocation, and a call must not lower the GPU's free memory.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It makes no assumption about earlier tests: it passes alone
in a fresh process (then its first call does the one-time set-up) and after the whole suite.
"""
import numpy as np
import pytest

from workloads import WORKLOADS, grid_to_pos, unwrapped_walk

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def g3():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1708_08619_b200 import build
    build.build()
    import paper_1708_08619_b200 as g3
    g3.load()
    return g3


def both(g3, m, box, max_lag=None):
    """the same device trajectory through the allocating call and through the static one"""
    import torch
    d = torch.from_numpy(grid_to_pos(m, box)).cuda()
    s_ref, m_ref = g3.msd(d, box, max_lag)
    s_new, m_new = g3.msd_static(d, box, max_lag)
    torch.cuda.synchronize()
    assert np.array_equal(s_new.cpu().numpy().view(np.uint64), s_ref.cpu().numpy().view(np.uint64))
    a, b = m_new.cpu().numpy(), m_ref.cpu().numpy()
    assert a[0] == 0.0 and np.allclose(a[1:], b[1:], rtol=1e-12, atol=0)
    return s_new.cpu().numpy().view(np.uint64)


def test_two_calls_in_a_row_match_the_allocating_path(g3, oracle_lib):
    # first call: 129 CTAs x 300 lags of partial sums, a ragged last CTA (4097 = 128 * 32 + 1)
    both(g3, unwrapped_walk(4097, 300, seed=31, step_sigma=500.0), 6.0)
    # second call, straight after: fewer CTAs and fewer lags, so its partial sums cover only the
    # start of what the first call wrote; a different box and step, so leftovers could not pass
    m = unwrapped_walk(1000, 64, seed=32, step_sigma=40.0)
    sums = both(g3, m, 2.5)
    so, _ = oracle_lib.msd(grid_to_pos(m, 2.5), 2.5, None)      # and the CPU oracle agrees
    assert np.array_equal(sums, so)
    # third: a subset of the lags, one CTA, the smallest shape
    both(g3, unwrapped_walk(33, 40, seed=33), 6.0, 12)
    both(g3, unwrapped_walk(1, 1, seed=34), 6.0)


def test_error_counter_is_cleared_between_calls(g3):
    import torch
    pos = torch.zeros((2, 40, 3), dtype=torch.float64, device="cuda")
    pos[1, 7, 2] = 2048.0                                       # 2^31 grid units at box = 1
    with pytest.raises(g3.G3Error) as e:
        g3.msd_static(pos, 1.0)
    assert e.value.code == g3.G3_EINVAL
    both(g3, unwrapped_walk(300, 50, seed=35), 6.0)             # the next call is clean again
    with pytest.raises(g3.G3Error) as e:
        g3.msd_static(pos, 1.0, max_lag=1)
    assert e.value.code == g3.G3_EINVAL


def test_config4_shape_fits_and_matches(g3):
    """N = 32768, 500 frames, every lag: 1024 x 500 = 512000 of the 524288 partial sums"""
    w = WORKLOADS[4]
    assert (w.n // 32) * w.n_frames <= g3.G3_MSD_STATIC_MAX_PARTIALS
    both(g3, unwrapped_walk(w.n, w.n_frames, seed=w.seed, step_sigma=1000.0), w.box)


def test_sizes_beyond_the_array_are_refused(g3):
    import torch
    # more (CTA, lag) pairs than the array holds: 1025 CTAs x 512 lags
    d = torch.zeros((512, 32 * 1025, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(g3.G3Error) as e:
        g3.msd_static(d, 1.0)
    assert e.value.code == g3.G3_ELIMIT and "scratch" in str(e.value)
    g3.msd_static(d, 1.0, max_lag=510)                          # 1025 x 511 fits
    g3.msd(d, 1.0)                                              # the allocating call has no such limit
    # more frames than shared memory holds: g3_msd switches to a global copy, this call refuses
    d = torch.zeros((1500, 70, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(g3.G3Error) as e:
        g3.msd_static(d, 1.0, max_lag=10)
    assert e.value.code == g3.G3_ELIMIT
    g3.msd(d, 1.0, max_lag=10)


def test_a_call_takes_no_device_memory(g3):
    """free memory as the driver reports it does not drop across calls once the first call on
    this device has been made (outputs are created beforehand, as such a caller would)"""
    import torch
    d = torch.from_numpy(grid_to_pos(unwrapped_walk(2048, 200, seed=36), 6.0)).cuda()
    sums = torch.empty((200, 2), dtype=torch.int64, device="cuda")
    out = torch.empty(200, dtype=torch.float64, device="cuda")
    g3.msd_static(d, 6.0, sums=sums, out=out)                   # set-up, if this is the first call
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        g3.msd_static(d, 6.0, sums=sums, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0
    s_ref, _ = g3.msd(d, 6.0)
    assert torch.equal(sums, s_ref)
