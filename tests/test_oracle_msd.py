"""Pins of the MSD oracle (oracle/g3_oracle.c: g3o_msd; Eq. 5; Algorithm 10,
PAPER.md:642-668) against things other than itself: the closed form for ballistic motion, exact
Python-integer brute force, the hand value of a single jump (no wrapping of unwrapped input),
invariances, and the random-walk law MSD = 3 sigma^2 dt."""
import numpy as np
import pytest

from workloads import GRID, grid_to_pos, unwrapped_walk


def to128(sums):
    return [int(lo) + (int(hi) << 64) for lo, hi in sums]


def test_ballistic_motion_closed_form(oracle_lib):
    """r_i(t) = r_i(0) + v_i t on the grid: |dr|^2 = |v_i|^2 dt^2 for every origin, so
    S[dt] = (F - dt) dt^2 sum_i |v_i|^2 and msd[dt] = g^2 dt^2 <|v|^2>"""
    rng = np.random.default_rng(1)
    n, F, box = 37, 20, 7.5
    r0 = rng.integers(0, GRID, size=(1, n, 3))
    v = rng.integers(-5000, 5000, size=(1, n, 3))
    m = r0 + v * np.arange(F).reshape(F, 1, 1)
    sums, msd = oracle_lib.msd(grid_to_pos(m, box), box)
    v2 = int((v.astype(object) ** 2).sum())
    assert to128(sums) == [(F - dt) * dt * dt * v2 for dt in range(F)]
    g = box / GRID
    assert np.allclose(msd, [g * g * dt * dt * v2 / n for dt in range(F)], rtol=1e-14, atol=0)


def test_python_integer_brute_force_and_max_lag(oracle_lib):
    m = unwrapped_walk(11, 9, seed=3, step_sigma=3.0e5)
    box = 4.0
    want = []
    for dt in range(9):
        s = 0
        for i in range(11):
            for t in range(9 - dt):
                d = m[t + dt, i].astype(object) - m[t, i].astype(object)
                s += int(d[0] * d[0] + d[1] * d[1] + d[2] * d[2])
        want.append(s)
    sums, msd = oracle_lib.msd(grid_to_pos(m, box), box)
    assert to128(sums) == want and want[0] == 0
    s5, m5 = oracle_lib.msd(grid_to_pos(m, box), box, max_lag=5)
    assert np.array_equal(s5, sums[:6]) and np.array_equal(m5, msd[:6])


def test_unwrapped_input_is_not_wrapped_and_128_bit_sums(oracle_lib):
    """one particle jumping 1.5 box lengths along x between two frames counts (1.5 L)^2; many
    particles doing it 2^9 times each overflow 64 bits, the (lo, hi) pair carries on"""
    box = 3.0
    m = np.zeros((2, 1, 3), dtype=np.int64)
    m[1, 0, 0] = 3 * GRID // 2
    sums, msd = oracle_lib.msd(grid_to_pos(m, box), box)
    assert to128(sums) == [0, (3 * GRID // 2) ** 2]
    assert msd[1] == pytest.approx(4.5 ** 2, rel=1e-15)
    F, n = 3, 70000
    m = np.zeros((F, n, 3), dtype=np.int64)
    m[1:, :, :] = (1 << 29)                      # jump of 2^29 in all three coordinates at frame 1
    sums, _ = oracle_lib.msd(grid_to_pos(m, 1.0), 1.0)
    assert to128(sums) == [0, n * 3 * (1 << 58), n * 3 * (1 << 58)]
    assert int(sums[2, 1]) > 0 or n * 3 * (1 << 58) < (1 << 64)
    with pytest.raises(ValueError):
        oracle_lib.msd(np.full((2, 1, 3), 1.0 * (1 << 11)), 1.0)       # 2^31 grid units


def test_range_edge_sum_of_squares_exceeds_63_bits(oracle_lib):
    """the corner of reading M1's range: m = -(2^30 - 1) -> +(2^30 - 1) on all three axes between
    two frames, so one squared displacement is 3 (2^31 - 2)^2 > 2^63 (a signed 64-bit sum would
    wrap); expected values from Python integers (readings M1, M2)"""
    e = (1 << 30) - 1
    n = 5
    m = np.zeros((2, n, 3), dtype=np.int64)
    m[0] = -e
    m[1] = e
    m[1, 3] = (e, -e, e)                       # mixed signs: displacement (2e, 0, 2e)
    m[0, 3] = (-e, -e, -e)
    want1 = (n - 1) * 3 * (2 * e) ** 2 + 2 * (2 * e) ** 2
    assert 3 * (2 * e) ** 2 > (1 << 63)
    sums, msd = oracle_lib.msd(grid_to_pos(m, 1.0), 1.0)
    assert to128(sums) == [0, want1]
    g = 1.0 / GRID
    assert msd[1] == pytest.approx(want1 * g * g / n, rel=1e-15)
    with pytest.raises(ValueError):            # one step further is outside the range
        m[1, 0, 0] = e + 1
        oracle_lib.msd(grid_to_pos(m, 1.0), 1.0)


def test_invariances(oracle_lib):
    m = unwrapped_walk(50, 12, seed=5)
    box = 9.0
    sums, msd = oracle_lib.msd(grid_to_pos(m, box), box)
    shifted = m + np.array([123456, -987654, 5])
    assert np.array_equal(oracle_lib.msd(grid_to_pos(shifted, box), box)[0], sums)
    perm = np.random.default_rng(0).permutation(50)
    assert np.array_equal(oracle_lib.msd(grid_to_pos(m[:, perm], box), box)[0], sums)
    assert np.array_equal(oracle_lib.msd(grid_to_pos(m[::-1].copy(), box), box)[0], sums)      # time reversal
    assert np.array_equal(oracle_lib.msd(grid_to_pos(m[:, :, ::-1].copy(), box), box)[0], sums)
    two = np.concatenate([m, m + 77], axis=1)
    assert to128(oracle_lib.msd(grid_to_pos(two, box), box)[0]) == [2 * v for v in to128(sums)]


def test_random_walk_law(oracle_lib):
    """independent Gaussian steps of variance sigma^2 per coordinate: MSD(dt) = 3 sigma^2 dt"""
    sigma, n, F, box = 2000.0, 4000, 40, 10.0
    m = unwrapped_walk(n, F, seed=9, step_sigma=sigma)
    _, msd = oracle_lib.msd(grid_to_pos(m, box), box)
    g = box / GRID
    dt = np.arange(1, 11)
    want = 3.0 * (sigma * sigma + 1.0 / 12.0) * g * g * dt        # + rounding of the steps to integers
    assert np.abs(msd[1:11] / want - 1.0).max() < 0.02
