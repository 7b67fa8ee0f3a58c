"""Parity of the CUDA path (through the C ABI) against the CPU oracle: uint64 counts and the
overflow/pair statistics bit-exact, g3 to relative 1e-12 (BASELINE.json north_star)."""
import numpy as np
import pytest

from workloads import GRID, WORKLOADS, frames, grid_to_pos, uniform_frame

pytestmark = pytest.mark.gpu

G3_RTOL = 1e-12


@pytest.fixture(scope="module")
def g3():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1708_08619_b200 import build
    build.build()
    import paper_1708_08619_b200 as g3
    g3.load()
    return g3


def run_gpu(g3, pos, box, r_max, n_r, n_t, **opts):
    import torch
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    if pos.ndim == 2:
        pos = pos[None]
    with g3.Plan(pos.shape[1], box, r_max, n_r, n_t, **opts) as plan:
        d = torch.from_numpy(pos).cuda()
        plan.accumulate_frames(d)
        counts, g3v, stats = plan.finalize()
        c2, g2 = plan.finalize_g2()
        info = {"kernel": plan.info(g3.G3_INFO_KERNEL), "launches": plan.info(g3.G3_INFO_KERNEL_LAUNCHES),
                "counts2": c2.cpu().numpy().view(np.uint64), "g2": g2.cpu().numpy()}
        return counts.cpu().numpy().view(np.uint64), g3v.cpu().numpy(), stats, info


def check(oracle_lib, g3, pos, box, r_max, n_r, n_t, mode="cells", **opts):
    H, G, stats, info = run_gpu(g3, pos, box, r_max, n_r, n_t, **opts)
    pos3 = pos if pos.ndim == 3 else pos[None]
    orc = oracle_lib.Oracle(pos3.shape[1], box, r_max, n_r, n_t, mode=mode)
    orc.accumulate(pos3)
    Ho, Go, so = orc.finalize()
    assert stats == [int(v) for v in so]
    assert np.array_equal(H, Ho)
    nz = Go != 0
    assert np.array_equal(nz, G != 0)
    assert np.allclose(G[nz], Go[nz], rtol=G3_RTOL, atol=0)
    assert info["launches"] > 0
    # g2 from the same neighbour pass: counts bit-exact, g2 to 1e-12.
    # The g2 oracle is a plain O(N^2) loop: all frames for small systems, the first otherwise.
    n = pos3.shape[1]
    T_r, _ = oracle_lib.thresholds(box, r_max, n_r, n_t)
    if n <= 40000:
        H2 = np.zeros(n_r, dtype=np.uint64)
        for f in range(pos3.shape[0]):
            oracle_lib.g2_frame(oracle_lib.quantise(pos3[f], box), T_r, H2)
        assert np.array_equal(info["counts2"], H2)
        g2o = oracle_lib.g2_normalise(H2, r_max, pos3.shape[0], n, box)
        assert np.allclose(info["g2"], g2o, rtol=G3_RTOL, atol=0)
    else:
        H2, _, _, i1 = run_gpu(g3, pos3[:1], box, r_max, n_r, n_t, **opts)
        assert np.array_equal(i1["counts2"], oracle_lib.g2_frame(oracle_lib.quantise(pos3[0], box), T_r))
    return H, stats, info


KERNELS = [1, 2]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("widx,nf", [(1, 10), (2, 3), (3, 2), (4, 2)])
def test_workload_frames(oracle_lib, g3, widx, nf, kernel):
    w = WORKLOADS[widx]
    _, pos = frames(w, nf)
    H, stats, _ = check(oracle_lib, g3, pos, w.box, w.r_max, w.n_r, w.n_t, kernel=kernel)
    assert H.sum() > 0 and stats[2] == 0


@pytest.mark.parametrize("kernel", KERNELS)
def test_config5_one_frame(oracle_lib, g3, kernel):
    w = WORKLOADS[5]
    _, pos = frames(w, 1)
    check(oracle_lib, g3, pos, w.box, w.r_max, w.n_r, w.n_t, kernel=kernel)


@pytest.mark.parametrize("n_r,n_t,max_nb", [(128, 128, None), (100, 200, None), (160, 96, 320)])
def test_slab_passes(oracle_lib, g3, n_r, n_t, max_nb):
    """bin counts whose reachable slots do not fit one shared-memory tile: the tiled kernel runs
    one pass per slab of outer shells.  Water-like and clumped frames, so that
    slab boundaries fall inside 32-blocks, on block edges and on empty shell ranges."""
    import torch
    w = WORKLOADS[2]
    _, pos = frames(w, 3)
    opts = {} if max_nb is None else {"max_neighbours": max_nb}
    r_max = w.r_max if max_nb is None else 1.0
    with g3.Plan(w.n, w.box, r_max, n_r, n_t, kernel=2, **opts) as plan:
        assert plan.info(g3.G3_INFO_KERNEL) == 2 and plan.info(g3.G3_INFO_SLABS) > 1
    check(oracle_lib, g3, pos, w.box, r_max, n_r, n_t, kernel=2, **opts)


def test_config5_uses_slabs(g3):
    w = WORKLOADS[5]
    with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t) as plan:
        assert plan.info(g3.G3_INFO_KERNEL) == 2 and plan.info(g3.G3_INFO_SLABS) > 1


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("n,box,r_max,n_r,n_t", [
    (3, 1.0, 0.4, 4, 4),            # smallest legal frame
    (37, 6.0, 2.9, 8, 16),          # degenerate cell grid (r_max ~ box/2), ragged warp tail
    (1000, 10.0, 2.0, 7, 13),       # odd bin counts, ncell = 4..5
    (5000, 10.0, 0.35, 33, 66),     # sparse: many centres with 0 or 1 neighbours
])
def test_edge_shapes(oracle_lib, g3, n, box, r_max, n_r, n_t, kernel):
    m = uniform_frame(n, seed=4242 + n)
    if n == 3:
        m = np.array([[5, 5, 5], [5 + GRID // 4, 5, 5], [5, 5 + GRID // 4, 5]], dtype=np.int32)
    check(oracle_lib, g3, grid_to_pos(m, box), box, r_max, n_r, n_t, mode="allpairs", kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS)
def test_clumped_and_coincident(oracle_lib, g3, kernel):
    """all particles in a small blob straddling the periodic corner; two coincident particles"""
    rng = np.random.default_rng(99)
    m = ((rng.integers(0, GRID // 16, size=(300, 3)) - GRID // 32) % GRID).astype(np.int32)
    m[1] = m[0]
    check(oracle_lib, g3, grid_to_pos(m, 8.0), 8.0, 0.3, 16, 16, mode="allpairs", kernel=kernel,
          max_neighbours=320)


@pytest.mark.parametrize("kernel", KERNELS)
def test_off_grid_and_unwrapped_inputs(oracle_lib, g3, kernel):
    """any real coordinate is snapped to the grid and wrapped (include/g3.h)"""
    w = WORKLOADS[1]
    _, pos = frames(w, 2)
    rng = np.random.default_rng(5)
    messy = pos + rng.integers(-3, 4, size=pos.shape) * w.box + 0.2 * w.box / GRID
    H1, _, _, _ = run_gpu(g3, pos, w.box, w.r_max, w.n_r, w.n_t, kernel=kernel)
    H2, _, _, _ = run_gpu(g3, messy, w.box, w.r_max, w.n_r, w.n_t, kernel=kernel)
    assert np.array_equal(H1, H2)
    check(oracle_lib, g3, messy, w.box, w.r_max, w.n_r, w.n_t, kernel=kernel)


@pytest.mark.parametrize("kernel", KERNELS)
def test_batching_single_frame_calls_and_reset(oracle_lib, g3, kernel):
    """frame-at-a-time calls, batch sizes that do not divide the frame count, finalize twice, reset"""
    import torch
    w = WORKLOADS[2]
    _, pos = frames(w, 7)
    orc = oracle_lib.Oracle(w.n, w.box, w.r_max, w.n_r, w.n_t, mode="cells")
    orc.accumulate(pos)
    Ho, _, so = orc.finalize()
    d = torch.from_numpy(pos).cuda()
    for batch in (1, 3, 16):
        with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, batch_frames=batch, kernel=kernel) as plan:
            for f in range(4):
                plan.accumulate_frame(d[f])
            c1, _, s1 = plan.finalize(want_g3=False)
            plan.accumulate_frames(d[4:])
            c2, _, s2 = plan.finalize(want_g3=False)
            c3, _, s3 = plan.finalize(want_g3=False)
            assert s1[0] == 4 and s2 == [int(v) for v in so] and s3 == s2
            assert np.array_equal(c2.cpu().numpy().view(np.uint64), Ho)
            assert torch.equal(c2, c3)
            plan.reset()
            plan.accumulate_frames(d[:4])
            c4, _, s4 = plan.finalize(want_g3=False)
            assert torch.equal(c4, c1) and s4 == s1


@pytest.mark.parametrize("kernel", KERNELS)
def test_host_entry_points(oracle_lib, g3, kernel):
    import torch
    w = WORKLOADS[2]
    _, pos = frames(w, 5)
    orc = oracle_lib.Oracle(w.n, w.box, w.r_max, w.n_r, w.n_t, mode="cells")
    orc.accumulate(pos)
    Ho, Go, so = orc.finalize()
    h = torch.from_numpy(pos).pin_memory()
    with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, batch_frames=2, kernel=kernel) as plan:
        plan.accumulate_frames_host(h)
        counts, g3v, stats = plan.finalize_host()
        assert stats == [int(v) for v in so]
        assert np.array_equal(counts.numpy().view(np.uint64), Ho)
        nz = Go != 0
        assert np.allclose(g3v.numpy()[nz], Go[nz], rtol=G3_RTOL, atol=0)
        V = plan.bin_volumes()
        Vo = oracle_lib.volumes(w.r_max, w.n_r, w.n_t)
        assert np.array_equal(V > 0, Vo > 0)
        assert np.allclose(V[V > 0], Vo[V > 0], rtol=5e-13, atol=0)


def test_capacity_error_is_reported(g3):
    import torch
    m = uniform_frame(2000, seed=1)
    pos = grid_to_pos(m, 10.0)
    with g3.Plan(2000, 10.0, 2.0, 8, 8, max_neighbours=32, kernel=1) as plan:
        plan.accumulate_frames(torch.from_numpy(pos[None]).cuda())
        with pytest.raises(g3.G3Error) as e:
            plan.finalize()
        assert e.value.code == g3.G3_ECAPACITY


def test_capacity_error_through_the_tiled_path(g3):
    """kernel 2: a clumped frame with far more than 64 neighbours per centre and max_neighbours = 64
    (the tiled path's smallest capacity) must end in G3_ECAPACITY, on the staged and on the
    crowded (unstaged) route of the neighbour kernel"""
    import torch
    rng = np.random.default_rng(17)
    m = uniform_frame(6000, seed=3)
    m[:400] = ((rng.integers(0, GRID // 64, size=(400, 3)) + GRID // 3) % GRID).astype(np.int32)   # a blob
    pos = grid_to_pos(m, 10.0)
    with g3.Plan(6000, 10.0, 1.2, 16, 16, max_neighbours=64, kernel=2) as plan:
        assert plan.info(g3.G3_INFO_KERNEL) == 2 and plan.info(g3.G3_INFO_MAX_NEIGHBOURS) == 64
        plan.accumulate_frames(torch.from_numpy(pos[None]).cuda())
        with pytest.raises(g3.G3Error) as e:
            plan.finalize()
        assert e.value.code == g3.G3_ECAPACITY


@pytest.mark.parametrize("warps", [8, 12, 16, 20, 24])
def test_triplet_warps_option_full_config2(oracle_lib, g3, warps):
    """G3_OPT_TRIPLET_WARPS instantiates one triplet kernel per value: the whole 100-frame config-2
    trajectory through each, bit-exact against the oracle"""
    w = WORKLOADS[2]
    _, pos = frames(w, w.n_frames)
    H, stats, _ = check(oracle_lib, g3, pos, w.box, w.r_max, w.n_r, w.n_t, kernel=2, triplet_warps=warps)
    assert stats[0] == w.n_frames


def test_two_live_plans_of_different_shape(oracle_lib, g3):
    """distinct plans are independent (include/g3.h): interleave two plans whose kernels need
    different amounts of dynamic shared memory (bins, neighbour capacity, q_tet histogram)"""
    import torch
    wa, wb = WORKLOADS[2], WORKLOADS[1]
    _, pa = frames(wa, 4)
    _, pb = frames(wb, 4)
    da, db = torch.from_numpy(pa).cuda(), torch.from_numpy(pb).cuda()
    with g3.Plan(wa.n, wa.box, wa.r_max, wa.n_r, wa.n_t, batch_frames=1, qtet_bins=300) as A, \
         g3.Plan(wb.n, wb.box, wb.r_max, 8, 8, batch_frames=1, max_neighbours=96, qtet_bins=10) as B, \
         g3.Plan(wa.n, wa.box, 0.9 * wa.r_max, 24, 48, batch_frames=2, kernel=1) as C:
        for f in range(4):
            A.accumulate_frame(da[f])
            B.accumulate_frame(db[f])
            C.accumulate_frame(da[f])
        cb, _, sb = B.finalize(want_g3=False)
        ca, _, sa = A.finalize(want_g3=False)
        cc, _, sc = C.finalize(want_g3=False)
        A.finalize_qtet()
        B.finalize_qtet()
    for (w, pos, n_r, n_t, r_max, c, st) in ((wa, pa, wa.n_r, wa.n_t, wa.r_max, ca, sa), (wb, pb, 8, 8, wb.r_max, cb, sb),
                                             (wa, pa, 24, 48, 0.9 * wa.r_max, cc, sc)):
        orc = oracle_lib.Oracle(w.n, w.box, r_max, n_r, n_t)
        orc.accumulate(pos)
        Ho, _, so = orc.finalize()
        assert st == [int(v) for v in so]
        assert np.array_equal(c.cpu().numpy().view(np.uint64), Ho)


def test_generic_kernel_with_lists_beyond_shared_memory(oracle_lib, g3):
    """the paper's own cut-off r_max = L/4 on a frame large enough that neither the
    tiled path (degenerate cell grid, n > 8192) nor the generic kernel's shared-memory list (capacity
    ~1800) can serve it: the generic kernel keeps its lists in global memory"""
    n, box = 9000, 10.0
    m = uniform_frame(n, seed=2024)
    with g3.Plan(n, box, 0.25 * box, 8, 8) as plan:
        assert plan.info(g3.G3_INFO_KERNEL) == 1 and plan.info(g3.G3_INFO_MAX_NEIGHBOURS) > 1800
    check(oracle_lib, g3, grid_to_pos(m, box), box, 0.25 * box, 8, 8)


def test_non_finite_coordinates_are_an_error(g3):
    """NaN / infinite coordinates have no grid point: sticky G3_EINVAL at finalize, cleared by reset"""
    import torch
    w = WORKLOADS[1]
    _, pos = frames(w, 2)
    d = torch.from_numpy(pos).cuda()
    bad = d.clone()
    bad[1, 17, 2] = float("nan")
    bad[0, 3, 0] = float("inf")
    for kernel in KERNELS:
        with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, kernel=kernel) as plan:
            plan.accumulate_frames(bad)
            with pytest.raises(g3.G3Error) as e:
                plan.finalize()
            assert e.value.code == g3.G3_EINVAL
            plan.reset()
            plan.accumulate_frames(d)
            plan.finalize()


def test_bin_counts_beyond_the_volume_lattice_are_refused(g3):
    """include/g3.h: 2 n_r n_t / gcd(n_t, 2 n_r) <= 2^19, else G3_EINVAL from g3_plan_create"""
    with pytest.raises(g3.G3Error) as e:
        g3.Plan(1000, 10.0, 2.0, 1021, 1023)
    assert e.value.code == g3.G3_EINVAL
    with g3.Plan(1000, 10.0, 2.0, 96, 96) as plan:            # equal counts always qualify
        assert plan.info(g3.G3_INFO_KERNEL) in (1, 2)


def test_normalize_merged_counts(oracle_lib, g3):
    """frame-sharded merge: counts from two plans summed, then g3_normalize"""
    import torch
    w = WORKLOADS[1]
    _, pos = frames(w, 6)
    d = torch.from_numpy(pos).cuda()
    with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t) as pa, g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t) as pb:
        pa.accumulate_frames(d[0::2].contiguous())
        pb.accumulate_frames(d[1::2].contiguous())
        ca, _, sa = pa.finalize(want_g3=False)
        cb, _, sb = pb.finalize(want_g3=False)
        g = pa.normalize(ca + cb, sa[0] + sb[0])
        torch.cuda.synchronize()
    orc = oracle_lib.Oracle(w.n, w.box, w.r_max, w.n_r, w.n_t)
    orc.accumulate(pos)
    Ho, Go, _ = orc.finalize()
    assert np.array_equal((ca + cb).cpu().numpy().view(np.uint64), Ho)
    nz = Go != 0
    assert np.allclose(g.cpu().numpy()[nz], Go[nz], rtol=G3_RTOL, atol=0)


def test_batch_shrinks_when_device_memory_is_short(g3):
    """Config-4 shape with most of the GPU's memory taken by somebody else (an MD engine, other
    plans): the automatic batch is sized from the free memory, an explicit batch that does not
    fit is halved until it does, and the counts are those of the roomy plan."""
    import torch
    w = WORKLOADS[4]
    _, pos = frames(w, 3)
    d = torch.from_numpy(pos).cuda()

    def run(**opts):
        with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, kernel=2, **opts) as plan:
            plan.accumulate_frames(d)
            c, _, st = plan.finalize(want_g3=False)
            return c.clone(), st, plan.info(g3.G3_INFO_BATCH_FRAMES)

    c0, st0, b0 = run()
    assert b0 >= 64                                             # an empty B200: ~2^22 centres per batch
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    hog = torch.empty(free - (6 << 30), dtype=torch.uint8, device="cuda")     # leave 6 GiB
    try:
        c1, st1, b1 = run()                                     # lists <= a quarter of what is free
        assert 1 <= b1 <= 12 and st1 == st0 and torch.equal(c1, c0)
        c2, st2, b2 = run(batch_frames=64)                      # 64 frames of lists need 9.4 GB
        assert 1 <= b2 <= 32 and st2 == st0 and torch.equal(c2, c0)
    finally:
        del hog
        torch.cuda.empty_cache()
    assert run()[2] == b0
