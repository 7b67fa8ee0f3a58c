"""Pins of the q_tet oracle (oracle/g3_oracle.c: g3o_qtet_frame; Eq. 1; Algorithm 2,
PAPER.md:205-251) against things other than itself: closed forms for hand-built neighbourhoods
(tetrahedron 1, planar square 1/2, collinear -3), the perfect diamond lattice, a numpy
implementation written from the definition with unit vectors, the tie rule, invariances, and
<q> = 0 for uniformly random directions (ideal gas)."""
import numpy as np

from workloads import GRID, WORKLOADS, frames, uniform_frame


def q_of(oracle_lib, m, n_q=8):
    m = np.ascontiguousarray(m, dtype=np.int32)
    q = np.zeros(m.shape[0])
    H, st = oracle_lib.qtet_frame(m, n_q, q_out=q)
    return q, H, st


def far_fillers(k, base):
    """k atoms far from the origin cluster (so that every atom has >= 4 neighbours somewhere)"""
    return [[base + 5000 * i, base + 7000 * i, base] for i in range(k)]


def test_closed_form_neighbourhoods(oracle_lib):
    c = np.array([1000, 1000, 1000])
    a = 300
    cases = {
        # regular tetrahedron directions (1,1,1), (1,-1,-1), (-1,1,-1), (-1,-1,1): cos = -1/3
        1.0: [[a, a, a], [a, -a, -a], [-a, a, -a], [-a, -a, a]],
        # planar square +-x, +-y: two opposite pairs (cos -1), four perpendicular (cos 0):
        # sum = 2 (2/3)^2 + 4 (1/3)^2 = 4/3  ->  q = 1 - (3/8)(4/3) = 1/2
        0.5: [[a, 0, 0], [-a, 0, 0], [0, a, 0], [0, -a, 0]],
        # four collinear neighbours on one side: cos = 1 six times: q = 1 - (3/8) 6 (4/3)^2 = -3
        -3.0: [[a, 0, 0], [2 * a, 0, 0], [3 * a, 0, 0], [4 * a, 0, 0]],
    }
    for want, vecs in cases.items():
        m = np.array([c] + [c + np.array(v) for v in vecs] + far_fillers(4, GRID // 2))
        q, H, st = q_of(oracle_lib, m % GRID, n_q=8)
        assert abs(q[0] - want) < 1e-15 * 8, (want, q[0])
        assert st[0] + st[1] == m.shape[0]
    # bins: 8 bins of width 1/2 on [-3, 1]: q = 1/2 -> bin 7, q = -3 -> bin 0, q = 1 -> last bin
    m = np.array([c] + [c + np.array(v) for v in cases[-3.0]] + far_fillers(4, GRID // 2)) % GRID
    q, H, st = q_of(oracle_lib, m, n_q=8)
    want = np.zeros(8, dtype=np.uint64)
    for v in q[~np.isnan(q)]:
        want[min(7, int(np.floor((v + 3.0) * 2.0)))] += 1
    assert np.array_equal(H, want) and H[0] >= 1


def test_neighbourhood_across_the_periodic_wall(oracle_lib):
    a = 300
    c = np.array([5, GRID - 7, 11])
    vecs = [[a, a, a], [a, -a, -a], [-a, a, -a], [-a, -a, a]]
    m = (np.array([c] + [c + np.array(v) for v in vecs] + far_fillers(4, GRID // 2))) % GRID
    q, _, _ = q_of(oracle_lib, m)
    assert abs(q[0] - 1.0) < 1e-14


def test_tie_rule_is_lexicographic(oracle_lib):
    """4th neighbour tied in d2 between (-3a,0,0) and (0,-3a,0): (d2, dx, dy, dz) order takes the
    first; by hand q = 1 - (3/8)(3/9 + 16/9 + 8/9) = -1/8 (the other choice would give +1/8)."""
    a = 1000
    c = np.array([400000, 400000, 400000])
    vecs = [[a, 0, 0], [0, 0, 3 * a // 2], [2 * a, 0, 0], [-3 * a, 0, 0], [0, -3 * a, 0]]
    m = np.array([c] + [c + np.array(v) for v in vecs] + far_fillers(3, 10))
    q, _, _ = q_of(oracle_lib, m)
    assert abs(q[0] + 0.125) < 1e-15
    q2, _, _ = q_of(oracle_lib, m[::-1].copy())               # independent of particle numbering
    assert abs(q2[-1] + 0.125) < 1e-15


def test_coincident_neighbour_is_skipped(oracle_lib):
    c = np.array([1000, 1000, 1000])
    m = np.array([c, c, c + [300, 0, 0], c + [0, 300, 0], c + [0, 0, 300], c + [300, 300, 300]])
    q, H, st = q_of(oracle_lib, m)
    assert np.isnan(q[0]) and np.isnan(q[1]) and st[1] >= 2 and st[0] + st[1] == 6
    assert int(H.sum()) == int(st[0])


def test_perfect_diamond_lattice(oracle_lib):
    cells, a = 4, GRID // 4
    fcc = np.array([[0, 0, 0], [0, 2, 2], [2, 0, 2], [2, 2, 0]])
    basis = np.concatenate([fcc, fcc + 1]) * (a // 4)
    g = np.arange(cells) * a
    origin = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    m = (origin + basis[None]).reshape(-1, 3) % GRID
    q, H, st = q_of(oracle_lib, m, n_q=100)
    assert st.tolist() == [m.shape[0], 0]
    assert np.abs(q - 1.0).max() < 1e-15 and H[-1] == m.shape[0]


def numpy_q(m):
    m = m.astype(np.int64)
    out = np.zeros(m.shape[0])
    for i in range(m.shape[0]):
        d = m - m[i]
        d = (d + GRID // 2) % GRID - GRID // 2
        d2 = (d * d).sum(axis=1)
        d2[i] = np.iinfo(np.int64).max
        order = np.lexsort((d[:, 2], d[:, 1], d[:, 0], d2))[:4]
        u = d[order] / np.sqrt(d2[order].astype(np.float64))[:, None]
        cosm = u @ u.T
        out[i] = 1.0 - 0.375 * sum((cosm[j, k] + 1.0 / 3.0) ** 2 for j in range(3) for k in range(j + 1, 4))
    return out


def test_against_numpy_definition_and_invariances(oracle_lib):
    w = WORKLOADS[2]
    m, _ = frames(w, 1)
    m = m[0][:700]
    q, H, st = q_of(oracle_lib, m, n_q=64)
    assert np.abs(q - numpy_q(m)).max() < 1e-13
    assert int(H.sum()) == int(st[0]) == 700
    rng = np.random.default_rng(11)
    shifted = ((m.astype(np.int64) + rng.integers(0, GRID, size=3)) % GRID).astype(np.int32)
    assert np.array_equal(q_of(oracle_lib, shifted, 64)[1], H)
    perm = rng.permutation(700)
    qp, Hp, _ = q_of(oracle_lib, m[perm], 64)
    assert np.array_equal(Hp, H) and np.array_equal(qp, q[perm])


def test_ideal_gas_mean_is_zero(oracle_lib):
    """directions of the four nearest neighbours of a Poisson point are independent and uniform:
    E[(cos + 1/3)^2] = 1/3 + 1/9, six pairs -> E[q] = 1 - (3/8)(6)(4/9) = 0"""
    q, _, st = q_of(oracle_lib, uniform_frame(20000, seed=77))
    assert st[1] == 0
    assert abs(q.mean()) < 4.0 * q.std() / np.sqrt(q.size)
