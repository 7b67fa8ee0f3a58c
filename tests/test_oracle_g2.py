"""Pins of the g2 oracle (oracle/g3_oracle.c: g3o_g2_frame, g3o_g2_normalise) against things
other than itself: a hand-derived lattice example, a numpy all-pairs count written from the
definition, the neighbour counts behind the g3 oracle's pair statistics, invariances, and the
ideal-gas value (N-1)/N.  PAPER.md:423-429, 513-518 (g2 beside the neighbour vectors)."""
import os

import numpy as np

from workloads import GRID, WORKLOADS, frames, uniform_frame

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def numpy_pair_counts(m, T_r):
    """ordered pairs per shell, from the definition: per-axis separation min(|d|, G - |d|)"""
    m = m.astype(np.int64)
    H2 = np.zeros(T_r.size - 1, dtype=np.uint64)
    k = np.zeros(m.shape[0], dtype=np.int64)
    for i in range(m.shape[0]):
        d = np.abs(m - m[i])
        d = np.minimum(d, GRID - d)
        d2 = (d * d).sum(axis=1)
        d2[i] = np.iinfo(np.int64).max
        inside = d2 < int(T_r[-1])
        k[i] = inside.sum()
        shells = np.searchsorted(T_r.astype(np.int64), d2[inside], side="right") - 1
        H2 += np.bincount(shells, minlength=H2.size).astype(np.uint64)
    return H2, k


def test_lattice_worked_example(oracle_lib):
    g = np.arange(4, dtype=np.int32) << 18
    m = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    T_r, _ = oracle_lib.thresholds(4.0, 1.9, 8, 8)
    H2 = oracle_lib.g2_frame(m, T_r)
    want = np.zeros(8, dtype=np.uint64)
    with open(os.path.join(GOLDEN, "lattice_4x4x4_g2.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                a, c = line.split()
                want[int(a)] = int(c)
    assert np.array_equal(H2, want)


def wide_thresholds(oracle_lib, box, r_max, n_r):
    """squared shell edges b w, b = 0..2 n_r, with the neighbour shells' own width w = r_max / n_r:
    (2 r_max) / (2 n_r) is the same double as r_max / n_r, so the first n_r + 1 edges are T_r itself"""
    T2, _ = oracle_lib.thresholds(box, 2.0 * r_max, 2 * n_r, 1)
    T_r, _ = oracle_lib.thresholds(box, r_max, n_r, 1)
    assert np.array_equal(T2[: n_r + 1], T_r)
    return T2


def test_hand_derived_lattice_over_the_whole_rjk_range(oracle_lib):
    """tests/golden/lattice_8x8x8_g2_wide.txt: g2 counted to 2 r_max (the r_jk axis of g3)"""
    g = np.arange(8, dtype=np.int32) << 17
    m = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    T2 = wide_thresholds(oracle_lib, 8.0, 1.05, 7)
    H2 = oracle_lib.g2_frame(m, T2)
    want = np.zeros(14, dtype=np.uint64)
    with open(os.path.join(GOLDEN, "lattice_8x8x8_g2_wide.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                a, c = line.split()
                want[int(a)] = int(c)
    assert want.sum() == 512 * 32
    assert np.array_equal(H2, want)
    # the lower half is the neighbour-range histogram
    T_r, _ = oracle_lib.thresholds(8.0, 1.05, 7, 1)
    assert np.array_equal(oracle_lib.g2_frame(m, T_r), want[:7])


def test_wide_range_against_numpy_and_ideal_gas(oracle_lib):
    """numpy all-pairs count over [0, 2 r_max) and the ideal-gas value (N-1)/N in every shell"""
    w = WORKLOADS[2]
    m, _ = frames(w, 1)
    m = m[0][:700]
    T2 = wide_thresholds(oracle_lib, w.box, w.r_max, w.n_r)
    ref, _ = numpy_pair_counts(m, T2)
    assert np.array_equal(oracle_lib.g2_frame(m, T2), ref)
    n, box, r_max, n_r = 3000, 10.0, 1.2, 6                  # 2 r_max = 2.4 < box / 2
    H2 = np.zeros(2 * n_r, dtype=np.uint64)
    T2 = wide_thresholds(oracle_lib, box, r_max, n_r)
    for f in range(4):
        oracle_lib.g2_frame(uniform_frame(n, seed=900 + f), T2, H2)
    g2 = oracle_lib.g2_normalise(H2, 2.0 * r_max, 4, n, box)
    z = (g2 / (1.0 - 1.0 / n) - 1.0) * np.sqrt(H2.astype(np.float64) / 2.0)
    assert np.abs(z[1:]).max() < 5.0


def test_against_numpy_definition_and_g3_pair_statistics(oracle_lib):
    for widx, n_take in ((1, 216), (2, 600)):
        w = WORKLOADS[widx]
        m, _ = frames(w, 1)
        m = m[0][:n_take]
        T_r, T_t = oracle_lib.thresholds(w.box, w.r_max, w.n_r, w.n_t)
        H2 = oracle_lib.g2_frame(m, T_r)
        ref, k = numpy_pair_counts(m, T_r)
        assert np.array_equal(H2, ref)
        # the g3 oracle's own pair statistic is sum_i k_i (k_i - 1) over the same neighbour sets
        H = np.zeros((w.n_r, w.n_r, w.n_t), dtype=np.uint64)
        stats = np.zeros(3, dtype=np.uint64)
        oracle_lib.frame_allpairs(m, T_r, T_t, H, stats)
        assert int(H2.sum()) == int(k.sum())
        assert int(stats[1]) == int((k * (k - 1)).sum())
        # shell marginal of the triplet histogram: sum_{b,c} H[a][b][c] = sum_i n_i(a) (k_i - 1);
        # with one shell only (n_r = 1) this is sum_i k_i (k_i - 1) = H.sum(), and H2[0] = sum_i k_i
        T1, Tt1 = oracle_lib.thresholds(w.box, w.r_max, 1, 1)
        assert int(oracle_lib.g2_frame(m, T1)[0]) == int(k.sum())


def test_two_particles_and_boundary(oracle_lib):
    T_r, _ = oracle_lib.thresholds(8.0, 2.0, 4, 4)            # shells of width 0.5
    step = GRID // 8                                          # one length unit
    m = np.array([[3, 3, 3], [3 + step + step // 4, 3, 3]], dtype=np.int32)       # r = 1.25
    assert oracle_lib.g2_frame(m, T_r).tolist() == [0, 0, 2, 0]
    m = np.array([[GRID - step // 2, 9, 9], [step // 4, 9, 9]], dtype=np.int32)   # across the wall, r = 0.75
    assert oracle_lib.g2_frame(m, T_r).tolist() == [0, 2, 0, 0]
    m = np.array([[0, 0, 0], [2 * step, 0, 0]], dtype=np.int32)                   # r = r_max exactly: outside
    assert oracle_lib.g2_frame(m, T_r).tolist() == [0, 0, 0, 0]
    m = np.array([[5, 5, 5], [5, 5, 5]], dtype=np.int32)                          # coincident: shell 0
    assert oracle_lib.g2_frame(m, T_r).tolist() == [2, 0, 0, 0]


def test_invariances(oracle_lib):
    w = WORKLOADS[1]
    m, _ = frames(w, 1)
    m = m[0]
    T_r, _ = oracle_lib.thresholds(w.box, w.r_max, w.n_r, w.n_t)
    H2 = oracle_lib.g2_frame(m, T_r)
    rng = np.random.default_rng(3)
    shifted = ((m.astype(np.int64) + rng.integers(0, GRID, size=3)) % GRID).astype(np.int32)
    assert np.array_equal(oracle_lib.g2_frame(shifted, T_r), H2)
    assert np.array_equal(oracle_lib.g2_frame(m[rng.permutation(m.shape[0])], T_r), H2)
    assert np.array_equal(oracle_lib.g2_frame(np.ascontiguousarray(m[:, ::-1]), T_r), H2)
    twice = oracle_lib.g2_frame(m, T_r, H2.copy())
    assert np.array_equal(twice, 2 * H2)


def test_ideal_gas_is_flat(oracle_lib):
    n, box, r_max, n_r, F = 3000, 10.0, 2.0, 10, 6
    T_r, _ = oracle_lib.thresholds(box, r_max, n_r, n_r)
    H2 = np.zeros(n_r, dtype=np.uint64)
    for f in range(F):
        oracle_lib.g2_frame(uniform_frame(n, seed=700 + f), T_r, H2)
    g2 = oracle_lib.g2_normalise(H2, r_max, F, n, box)
    ideal = 1.0 - 1.0 / n
    z = (g2 / ideal - 1.0) * np.sqrt(H2.astype(np.float64) / 2.0)
    assert np.abs(z[1:]).max() < 5.0                          # shell 0 holds too few pairs
    # normalisation closed form: sum_a g2[a] V_a = H2.sum() / (F N rho), V_a summing to the sphere
    rho = n / box ** 3
    edges = np.arange(n_r + 1) * (r_max / n_r)
    V = 4.0 * np.pi / 3.0 * np.diff(edges ** 3)
    assert np.isclose((g2 * V).sum(), H2.sum() / (F * n * rho), rtol=1e-13)
    assert np.isclose(V.sum(), 4.0 * np.pi / 3.0 * r_max ** 3, rtol=1e-13)
