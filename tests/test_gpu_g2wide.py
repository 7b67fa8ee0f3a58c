"""Parity of the pair histogram over the whole r_jk range [0, 2 r_max) (G3_OPT_G2_WIDE; SURVEY.md
8(f) NEXT-1) against the oracle's plain all-pairs count: the 2 n_r shell
counts bit-exact, g2 to 1e-12.  The lower n_r shells come from the neighbour pass, the upper n_r
from g2_wide_kernel's half-stencil pair search."""
import numpy as np
import pytest

from workloads import GRID, WORKLOADS, frames, grid_to_pos, uniform_frame

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


def wide_edges(oracle_lib, box, r_max, n_r):
    return oracle_lib.thresholds(box, 2.0 * r_max, 2 * n_r, 1)[0]


def check(oracle_lib, g3, ms, box, r_max, n_r, n_t, **opts):
    import torch
    ms = np.asarray(ms)
    pos = grid_to_pos(ms, box)
    with g3.Plan(ms.shape[1], box, r_max, n_r, n_t, g2_wide=True, **opts) as plan:
        assert plan.info(g3.G3_INFO_G2_SHELLS) == 2 * n_r
        plan.accumulate_frames(torch.from_numpy(pos).cuda())
        c2, g2 = plan.finalize_g2()
        counts, _, stats = plan.finalize(want_g3=False)
        cells = plan.info(g3.G3_INFO_CELLS_PER_EDGE)
    T2 = wide_edges(oracle_lib, box, r_max, n_r)
    H2 = np.zeros(2 * n_r, dtype=np.uint64)
    for m in ms:
        oracle_lib.g2_frame(m, T2, H2)
    got = c2.cpu().numpy().view(np.uint64)
    assert np.array_equal(got, H2)
    want = oracle_lib.g2_normalise(H2, 2.0 * r_max, ms.shape[0], ms.shape[1], box)
    assert np.allclose(g2.cpu().numpy(), want, rtol=1e-12, atol=0)
    assert int(got[:n_r].sum()) > 0 or ms.shape[1] < 10
    return got, cells


@pytest.mark.parametrize("kernel", [1, 2])
@pytest.mark.parametrize("widx,nf", [(1, 10), (2, 3), (3, 2), (4, 1)])
def test_workload_frames(oracle_lib, g3, widx, nf, kernel):
    w = WORKLOADS[widx]
    ms, _ = frames(w, nf)
    got, _ = check(oracle_lib, g3, ms, w.box, w.r_max, w.n_r, w.n_t, kernel=kernel)
    assert int(got[w.n_r:].sum()) > 0


def test_hand_lattice(oracle_lib, g3):
    """tests/golden/lattice_8x8x8_g2_wide.txt through the CUDA path"""
    g = np.arange(8, dtype=np.int32) << 17
    m = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(1, -1, 3)
    got, cells = check(oracle_lib, g3, m, 8.0, 1.05, 7, 7)
    assert cells >= 5
    want = np.zeros(14, dtype=np.uint64)
    want[[6, 9, 11, 13]] = [3072, 6144, 4096, 3072]
    assert np.array_equal(got, want)


@pytest.mark.parametrize("n,box,r_max,n_r", [
    (3, 1.0, 0.4, 4),               # smallest frame; 2 r_max > box / 2: all-particle scan
    (37, 6.0, 2.9, 8),              # degenerate cell grid
    (1000, 10.0, 2.0, 7),           # exactly five cells per edge: the stencil just does not wrap onto itself
    (1500, 10.0, 2.4, 9),           # four cells per edge: all-particle scan
    (5000, 10.0, 0.35, 33),         # sparse, many cells
])
def test_edge_shapes(oracle_lib, g3, n, box, r_max, n_r):
    m = uniform_frame(n, seed=777 + n)
    if n == 3:
        m = np.array([[5, 5, 5], [5 + GRID // 4, 5, 5], [5, 5 + GRID // 4, 5]], dtype=np.int32)
    check(oracle_lib, g3, m[None], box, r_max, n_r, n_r)


def test_periodic_corner_and_coincident(oracle_lib, g3):
    """a blob straddling the periodic corner (every wrap branch of the stencil) plus coincident sites"""
    rng = np.random.default_rng(5)
    m = uniform_frame(4000, seed=12)
    m[:600] = ((rng.integers(0, GRID // 5, size=(600, 3)) - GRID // 10) % GRID).astype(np.int32)
    m[7] = m[3]
    check(oracle_lib, g3, m[None], 12.0, 1.3, 10, 10, max_neighbours=700)


def test_config5_first_frame_and_ideal_gas(oracle_lib, g3):
    """N = 262144: the oracle's O(N^2) count on one frame; g2 = (N-1)/N within counting error"""
    w = WORKLOADS[5]
    ms, _ = frames(w, 1)
    got, _ = check(oracle_lib, g3, ms, w.box, w.r_max, 32, 32)
    T2 = wide_edges(oracle_lib, w.box, w.r_max, 32)
    g2 = oracle_lib.g2_normalise(got, 2.0 * w.r_max, 1, w.n, w.box)
    z = (g2 / (1.0 - 1.0 / w.n) - 1.0) * np.sqrt(got.astype(np.float64) / 2.0)
    assert np.abs(z[2:]).max() < 6.0


def test_default_is_the_neighbour_range(g3):
    import torch
    w = WORKLOADS[2]
    _, pos = frames(w, 1)
    with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t) as plan:
        assert plan.info(g3.G3_INFO_G2_SHELLS) == w.n_r
        plan.accumulate_frames(torch.from_numpy(pos).cuda())
        c2, g2 = plan.finalize_g2()
        assert c2.numel() == w.n_r and g2.numel() == w.n_r
