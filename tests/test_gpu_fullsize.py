"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default
batch of 16 frames, event timing on, device and host entry points).

* config 4 (headline, 500 frames) and configs 1-2: the oracle runs the whole trajectory; counts
  and statistics bit-exact, g3 to 1e-12.
* configs 3 and 5 (1.5e10 / 6.7e10 triplets: minutes of oracle time): the whole trajectory goes
  through the library once; the oracle computes SAMPLED frames one by one (the histogram is a
  sum over frames) and the full run is tied to them by properties that hold
  at any size: H(all frames) = sum of per-frame H; sum(H) + overflow = sum_i k_i (k_i - 1);
  H[a][b][c] = H[b][a][c]; H = 0 where V_abc = 0; config 5 (ideal gas): g3 = (1-1/N)(1-2/N)
  within counting error.
"""
import numpy as np
import pytest

from workloads import WORKLOADS, frame_iter, grid_to_pos

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


def oracle_frames(oracle_lib, w, ms):
    T_r, T_t = oracle_lib.thresholds(w.box, w.r_max, w.n_r, w.n_t)
    H = np.zeros((w.n_r, w.n_r, w.n_t), dtype=np.uint64)
    stats = np.zeros(3, dtype=np.uint64)
    for m in ms:
        oracle_lib.frame_cells(m, T_r, T_t, H, stats)
    return H, [int(v) for v in stats]


def check_g3(oracle_lib, w, H, G, n_frames):
    V = oracle_lib.volumes(w.r_max, w.n_r, w.n_t)
    Go = oracle_lib.normalise(H, V, n_frames, w.n, w.box)
    nz = Go != 0
    assert np.array_equal(nz, G != 0)
    assert np.allclose(G[nz], Go[nz], rtol=G3_RTOL, atol=0)


@pytest.mark.parametrize("widx", [1, 2, 4])
def test_full_trajectory_bit_exact(oracle_lib, g3, widx):
    import torch
    w = WORKLOADS[widx]
    ms = list(frame_iter(w, w.n_frames))
    Ho, so = oracle_frames(oracle_lib, w, ms)
    pos = grid_to_pos(np.stack(ms, axis=0), w.box)
    h_pos = torch.from_numpy(pos).pin_memory()
    d_pos = h_pos.cuda()
    with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, timing=True) as plan:      # bench.py's plan
        assert plan.info(g3.G3_INFO_KERNEL) == 2
        plan.accumulate_frames(d_pos)
        counts, G, stats = plan.finalize()
        H = counts.cpu().numpy().view(np.uint64)
        assert stats == so and stats[0] == w.n_frames and stats[2] == 0
        assert np.array_equal(H, Ho)
        assert int(H.sum()) == stats[1]
        check_g3(oracle_lib, w, H, G.cpu().numpy(), w.n_frames)
        plan.reset()                                                         # the e2e leg
        plan.accumulate_frames_host(h_pos)
        hc, hg, hs = plan.finalize_host()
        assert hs == so
        assert np.array_equal(hc.numpy().view(np.uint64), Ho)
        check_g3(oracle_lib, w, Ho, hg.numpy(), w.n_frames)


@pytest.mark.parametrize("widx,sample", [(3, (0, 67, 133, 199)), (5, (0, 41, 99))])
def test_full_trajectory_sampled(oracle_lib, g3, widx, sample):
    import torch
    w = WORKLOADS[widx]
    ms = list(frame_iter(w, w.n_frames))
    d_pos = torch.from_numpy(grid_to_pos(np.stack(ms, axis=0), w.box)).cuda()
    with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, timing=True) as plan:
        assert plan.info(g3.G3_INFO_KERNEL) == 2
        plan.accumulate_frames(d_pos)
        counts, G, stats = plan.finalize()
        H = counts.cpu().numpy().view(np.uint64).copy()
        G = G.cpu().numpy()
        # per-frame histograms from the same plan; sampled ones against the oracle
        Hsum = np.zeros_like(H)
        pairs = 0
        for f in range(w.n_frames):
            plan.reset()
            plan.accumulate_frame(d_pos[f])
            cf, _, sf = plan.finalize(want_g3=False)
            Hf = cf.cpu().numpy().view(np.uint64)
            Hsum += Hf
            pairs += sf[1]
            if f in sample:
                Ho, so = oracle_frames(oracle_lib, w, [ms[f]])
                assert np.array_equal(Hf, Ho), f"frame {f}"
                assert sf == so
    assert stats[0] == w.n_frames and stats[2] == 0
    assert np.array_equal(H, Hsum)                       # additivity over frames and batches
    assert stats[1] == pairs == int(H.sum())             # sum_i k_i (k_i - 1), overflow = 0
    assert np.array_equal(H, H.transpose(1, 0, 2))       # r12 <-> r13
    V = oracle_lib.volumes(w.r_max, w.n_r, w.n_t)
    assert not H[V == 0].any()                           # triangle inequality
    check_g3(oracle_lib, w, H, G, w.n_frames)
    if w.kind == "uniform":                              # ideal gas: flat at (1-1/N)(1-2/N)
        ideal = (1.0 - 1.0 / w.n) * (1.0 - 2.0 / w.n)
        big = H >= 10000
        assert big.sum() > 1000
        z = (G[big] / ideal - 1.0) * np.sqrt(H[big].astype(np.float64) / 2.0)
        # ordered pairs double every count, so the counting error is sqrt(2/H) relative; triplet
        # counts sharing particles are positively correlated, hence the loose 8-sigma bound
        assert np.abs(z).max() < 8.0, np.abs(z).max()
        assert abs(np.average(G[big], weights=H[big]) / ideal - 1.0) < 1e-3
