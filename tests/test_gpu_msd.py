"""Parity of g3_msd (Eq. 5; Algorithm 11) against the CPU oracle: the exact 128-bit
sums of squared grid displacements bit-exact, msd to relative 1e-12 (one fp64 division and two
multiplications on each side, reading M3)."""
import numpy as np
import pytest

from workloads import GRID, WORKLOADS, grid_to_pos, unwrapped_walk

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


def check(oracle_lib, g3, m, box, max_lag=None):
    import torch
    pos = grid_to_pos(m, box)
    sums, msd = g3.msd(torch.from_numpy(pos).cuda(), box, max_lag)
    so, mo = oracle_lib.msd(pos, box, max_lag)
    assert np.array_equal(sums.cpu().numpy().view(np.uint64), so)
    got = msd.cpu().numpy()
    assert got[0] == 0.0 and np.allclose(got[1:], mo[1:], rtol=1e-12, atol=0)
    return so, got


@pytest.mark.parametrize("n,F,lag", [(1, 1, None), (5, 7, None), (33, 40, 12), (1000, 64, None), (4097, 300, 299)])
def test_small_and_ragged_shapes(oracle_lib, g3, n, F, lag):
    check(oracle_lib, g3, unwrapped_walk(n, F, seed=100 + n), 6.0, lag)


def test_long_trajectory_takes_the_global_path(oracle_lib, g3):
    """F x 384 B exceeds shared memory: snapped copy in global memory, same sums"""
    check(oracle_lib, g3, unwrapped_walk(70, 1500, seed=8, step_sigma=300.0), 6.0, 700)


def test_config4_shape_all_lags(oracle_lib, g3):
    """the headline shape: N = 32768 sites, 500 frames, every lag (4.1e9 displacements)"""
    w = WORKLOADS[4]
    so, got = check(oracle_lib, g3, unwrapped_walk(w.n, w.n_frames, seed=w.seed, step_sigma=1000.0), w.box)
    g = w.box / GRID
    assert abs(got[10] / (3.0 * (1000.0 ** 2 + 1.0 / 12.0) * g * g * 10) - 1.0) < 0.01      # random-walk law


def test_wide_range_and_128_bit_sums(oracle_lib, g3):
    F, n = 3, 70000
    m = np.zeros((F, n, 3), dtype=np.int64)
    m[1:, :, :] = (1 << 29)
    so, _ = check(oracle_lib, g3, m, 1.0)
    assert int(so[1, 1]) > 0                                    # the high word is in use


def test_range_edge_sum_of_squares_exceeds_63_bits(oracle_lib, g3):
    """m = -(2^30 - 1) -> +(2^30 - 1) on all three axes: one squared displacement is
    3 (2^31 - 2)^2 > 2^63 (readings M1, M2); the expected sum is a Python integer"""
    e = (1 << 30) - 1
    n = 67
    m = np.zeros((3, n, 3), dtype=np.int64)
    m[0] = -e
    m[1] = e
    m[2] = -e
    so, _ = check(oracle_lib, g3, m, 1.0)
    d2 = 3 * (2 * e) ** 2
    assert d2 > (1 << 63)
    want = [0, 2 * n * d2, 0]
    assert [int(lo) + (int(hi) << 64) for lo, hi in so] == want


def test_out_of_range_coordinate_is_an_error(g3):
    import torch
    pos = torch.zeros((2, 40, 3), dtype=torch.float64, device="cuda")
    pos[1, 7, 2] = 2048.0                                       # 2^31 grid units at box = 1
    with pytest.raises(g3.G3Error) as e:
        g3.msd(pos, 1.0)
    assert e.value.code == g3.G3_EINVAL
    with pytest.raises(g3.G3Error):
        g3.msd(pos, 1.0, max_lag=2)
