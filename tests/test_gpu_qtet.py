"""Parity of the q_tet path (G3_OPT_QTET_BINS, g3_finalize_qtet; Eq. 1) against the
CPU oracle: the uint64 histogram and the (binned, skipped) statistics bit-exact.  Floating point
decides the bin, so both sides evaluate Eq. 1 in fp64 in the operation order of DESIGN.md
reading T2."""
import numpy as np
import pytest

from workloads import GRID, WORKLOADS, frame_iter, frames, grid_to_pos, uniform_frame

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


def gpu_qtet(g3, ms, box, r_max, n_q, **opts):
    import torch
    pos = grid_to_pos(np.stack(ms, axis=0), box)
    with g3.Plan(ms[0].shape[0], box, r_max, 8, 8, qtet_bins=n_q, **opts) as plan:
        plan.accumulate_frames(torch.from_numpy(pos).cuda())
        hist, stats = plan.finalize_qtet()
        cells = plan.info(g3.G3_INFO_CELLS_PER_EDGE)
        return hist.cpu().numpy().view(np.uint64), stats, cells


def oracle_qtet(oracle_lib, ms, n_q):
    H = np.zeros(n_q, dtype=np.uint64)
    st = np.zeros(2, dtype=np.uint64)
    for m in ms:
        oracle_lib.qtet_frame(m, n_q, H, st)
    return H, [int(v) for v in st]


@pytest.mark.parametrize("widx,nf,n_q", [(1, 10, 40), (2, 5, 100), (3, 2, 400), (4, 2, 100)])
def test_workload_frames(oracle_lib, g3, widx, nf, n_q):
    w = WORKLOADS[widx]
    ms = list(frame_iter(w, nf))
    H, st, _ = gpu_qtet(g3, ms, w.box, w.r_max, n_q)
    Ho, so = oracle_qtet(oracle_lib, ms, n_q)
    assert st == so and st[0] == nf * w.n
    assert np.array_equal(H, Ho)


def test_sparse_frame_uses_the_all_particle_path(oracle_lib, g3):
    """fewer than one particle per cell: the fourth neighbour lies beyond the 27 cells"""
    m = uniform_frame(3000, seed=5)
    H, st, cells = gpu_qtet(g3, [m], 20.0, 0.5, 64)
    assert cells >= 16
    Ho, so = oracle_qtet(oracle_lib, [m], 64)
    assert st == so == [3000, 0]
    assert np.array_equal(H, Ho)


def test_smallest_frame_coincident_and_ties(oracle_lib, g3):
    a = 1000
    c = np.array([400000, 400000, 400000])
    # five atoms (the minimum), one pair coincident -> those two are skipped (T4)
    m5 = np.array([c, c, c + [a, 0, 0], c + [0, a, 0], c + [0, 0, a]], dtype=np.int32)
    H, st, _ = gpu_qtet(g3, [m5], 8.0, 1.0, 16)
    Ho, so = oracle_qtet(oracle_lib, [m5], 16)
    assert st == so and st[1] == 2 and np.array_equal(H, Ho)
    # fourth neighbour tied in d2: (d2, dx, dy, dz) order decides (tests/test_oracle_qtet.py)
    vecs = [[a, 0, 0], [0, 0, 3 * a // 2], [2 * a, 0, 0], [-3 * a, 0, 0], [0, -3 * a, 0]]
    m = np.array([c] + [c + np.array(v) for v in vecs] + [[10, 10, 10], [5010, 7010, 10], [10010, 14010, 10]],
                 dtype=np.int32)
    for box, r_max in ((8.0, 3.9), (64.0, 1.0)):              # degenerate grid, and 32 cells per edge
        H, st, _ = gpu_qtet(g3, [m], box, r_max, 32)
        Ho, so = oracle_qtet(oracle_lib, [m], 32)
        assert st == so and np.array_equal(H, Ho)


def test_perfect_diamond_lattice_is_one(g3):
    cells, a = 4, GRID // 4
    fcc = np.array([[0, 0, 0], [0, 2, 2], [2, 0, 2], [2, 2, 0]])
    basis = np.concatenate([fcc, fcc + 1]) * (a // 4)
    g = np.arange(cells) * a
    origin = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    m = ((origin + basis[None]).reshape(-1, 3) % GRID).astype(np.int32)
    H, st, _ = gpu_qtet(g3, [m], 4.0, 0.6, 100)
    assert st == [512, 0] and H[-1] == 512 and H.sum() == 512


def test_config4_whole_trajectory_sampled(oracle_lib, g3):
    """the full 500-frame headline trajectory with q_tet on, in bench.py's launch configuration;
    the oracle checks sampled frames one by one and additivity ties the whole run to them"""
    import torch
    w = WORKLOADS[4]
    ms = list(frame_iter(w, w.n_frames))
    d_pos = torch.from_numpy(grid_to_pos(np.stack(ms, axis=0), w.box)).cuda()
    with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, timing=True, qtet_bins=200) as plan:
        plan.accumulate_frames(d_pos)
        hist, st = plan.finalize_qtet()
        H = hist.cpu().numpy().view(np.uint64).copy()
        Hsum = np.zeros_like(H)
        for f in range(0, w.n_frames):
            plan.reset()
            plan.accumulate_frame(d_pos[f])
            hf, sf = plan.finalize_qtet()
            Hf = hf.cpu().numpy().view(np.uint64)
            Hsum += Hf
            if f in (0, 249, 499):
                Ho, so = oracle_qtet(oracle_lib, [ms[f]], 200)
                assert sf == so and np.array_equal(Hf, Ho), f"frame {f}"
    assert st == [w.n * w.n_frames, 0]
    assert np.array_equal(H, Hsum) and int(H.sum()) == st[0]


def test_option_errors(g3):
    with g3.Plan(1000, 10.0, 1.0, 8, 8) as plan:
        with pytest.raises(g3.G3Error) as e:
            plan.qtet_bins = 10
            plan.finalize_qtet()
        assert e.value.code == g3.G3_ESTATE
    with pytest.raises(g3.G3Error):
        g3.Plan(4, 10.0, 1.0, 8, 8, qtet_bins=10)


def test_capacity_error_reaches_finalize_qtet(oracle_lib, g3):
    """On the tiled path q_tet is read off the capacity-limited neighbour lists: a clumped frame with
    max_neighbours = 64 cuts lists in scan order, the four nearest may be gone, and finalize_qtet
    must say so (G3_ECAPACITY) instead of returning a histogram.  The generic kernel's q_tet scans
    the cells and does not depend on the capacity: it still matches the oracle."""
    import torch
    rng = np.random.default_rng(17)
    m = uniform_frame(6000, seed=3)
    m[:400] = ((rng.integers(0, GRID // 64, size=(400, 3)) + GRID // 3) % GRID).astype(np.int32)   # a blob
    pos = torch.from_numpy(grid_to_pos(m[None], 10.0)).cuda()
    with g3.Plan(6000, 10.0, 1.2, 16, 16, qtet_bins=50, max_neighbours=64, kernel=2) as plan:
        assert plan.info(g3.G3_INFO_KERNEL) == 2
        plan.accumulate_frames(pos)
        with pytest.raises(g3.G3Error) as e:
            plan.finalize_qtet()
        assert e.value.code == g3.G3_ECAPACITY
    with g3.Plan(6000, 10.0, 1.2, 16, 16, qtet_bins=50, max_neighbours=64, kernel=1) as plan:
        plan.accumulate_frames(pos)
        hist, stats = plan.finalize_qtet()
        with pytest.raises(g3.G3Error):
            plan.finalize()                                     # the g(3) counts ARE incomplete
    Ho, so = oracle_qtet(oracle_lib, [m], 50)
    assert stats == so and np.array_equal(hist.cpu().numpy().view(np.uint64), Ho)
    # with room for every neighbour the tiled path gives the same histogram
    with g3.Plan(6000, 10.0, 1.2, 16, 16, qtet_bins=50, max_neighbours=1024, kernel=2) as plan:
        plan.accumulate_frames(pos)
        hist, stats = plan.finalize_qtet()
    assert stats == so and np.array_equal(hist.cpu().numpy().view(np.uint64), Ho)


def test_non_finite_coordinate_reaches_finalize_qtet(g3):
    import torch
    pos = torch.from_numpy(grid_to_pos(uniform_frame(500, seed=9)[None], 5.0)).cuda()
    pos[0, 17, 1] = float("nan")
    with g3.Plan(500, 5.0, 1.0, 8, 8, qtet_bins=20) as plan:
        plan.accumulate_frames(pos)
        with pytest.raises(g3.G3Error) as e:
            plan.finalize_qtet()
        assert e.value.code == g3.G3_EINVAL
