"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default
batch of ~2^22 centres, event timing on, device and host entry points).

* config 4 (headline, 500 frames) and configs 1-2: the oracle runs the whole trajectory; counts
  and statistics bit-exact, g3 to 1e-12.
* configs 3 and 5 (1.5e10 / 6.7e10 triplets: about one and seven minutes of oracle time on 16
  cores, more than a GPU test session can spare): the oracle's whole-run histogram is stored as a
  digest under tests/golden/ (SHA-256 of the uint64 array, the statistics, the sum and 400 sampled
  bins, written by tests/golden/make_whole_run_digests.py, which calls only oracle/); the library's
  whole-run histogram must hash to it.  The oracle still runs live on sampled frames: the library's
  per-frame histograms are compared with it and tied to the whole run by properties that hold at
  any size:
  H(all frames) = sum of per-frame H; sum(H) + overflow = sum_i k_i (k_i - 1);
  H[a][b][c] = H[b][a][c]; H = 0 where V_abc = 0; config 5 (ideal gas): g3 = (1-1/N)(1-2/N)
  within counting error.
"""
import hashlib
import os

import numpy as np
import pytest

from workloads import WORKLOADS, frame_iter, grid_to_pos

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")

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
        # g2 of the whole trajectory; the O(N^2) oracle runs every frame (every 25th for config 4)
        c2, g2 = plan.finalize_g2()
        c2 = c2.cpu().numpy().view(np.uint64)
        T_r, _ = oracle_lib.thresholds(w.box, w.r_max, w.n_r, w.n_t)
        if widx != 4:
            H2 = np.zeros(w.n_r, dtype=np.uint64)
            for m in ms:
                oracle_lib.g2_frame(m, T_r, H2)
            assert np.array_equal(c2, H2)
            assert np.allclose(g2.cpu().numpy(), oracle_lib.g2_normalise(H2, w.r_max, w.n_frames, w.n, w.box),
                               rtol=G3_RTOL, atol=0)
        else:
            with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t) as p2:
                H2 = np.zeros(w.n_r, dtype=np.uint64)
                for f in range(0, w.n_frames, 25):
                    p2.accumulate_frame(d_pos[f])
                    oracle_lib.g2_frame(ms[f], T_r, H2)
                s2, _ = p2.finalize_g2()
                assert np.array_equal(s2.cpu().numpy().view(np.uint64), H2)
        # sum_a counts2[a] = sum_i k_i; Cauchy-Schwarz ties it to the triplet statistic
        k_sum = int(c2.sum())
        assert stats[1] + k_sum >= k_sum * k_sum // (w.n * w.n_frames)
        plan.reset()                                                         # the e2e leg
        plan.accumulate_frames_host(h_pos)
        hc, hg, hs = plan.finalize_host()
        assert hs == so
        assert np.array_equal(hc.numpy().view(np.uint64), Ho)
        check_g3(oracle_lib, w, Ho, hg.numpy(), w.n_frames)


def whole_run_digest(widx):
    """tests/golden/config<widx>_whole_run.txt -> (shape, sha256, stats, sum, {flat index: count})"""
    shape = sha = stats = total = None
    bins = {}
    for line in open(os.path.join(GOLDEN, f"config{widx}_whole_run.txt")):
        if line.startswith("#") or not line.strip():
            continue
        key, *vals = line.split()
        if key == "shape":
            shape = tuple(int(v) for v in vals)
        elif key == "sha256":
            sha = vals[0]
        elif key == "stats":
            stats = [int(v) for v in vals]
        elif key == "sum":
            total = int(vals[0])
        elif key == "bin":
            bins[int(vals[0])] = int(vals[1])
    assert shape and sha and stats and total is not None and len(bins) >= 300
    return shape, sha, stats, total, bins


@pytest.mark.parametrize("widx,sample", [(3, (0, 67, 133, 199)), (5, (0, 41, 99))])
def test_full_trajectory_configs_3_and_5(oracle_lib, g3, widx, sample):
    import torch
    w = WORKLOADS[widx]
    ms = list(frame_iter(w, w.n_frames))
    shape, sha_all, so_all, sum_all, bins_all = whole_run_digest(widx)   # the oracle over the whole trajectory
    assert shape == (w.n_r, w.n_r, w.n_t) and so_all[0] == w.n_frames
    d_pos = torch.from_numpy(grid_to_pos(np.stack(ms, axis=0), w.box)).cuda()
    with g3.Plan(w.n, w.box, w.r_max, w.n_r, w.n_t, timing=True) as plan:
        assert plan.info(g3.G3_INFO_KERNEL) == 2
        plan.accumulate_frames(d_pos)
        counts, G, stats = plan.finalize()
        H = counts.cpu().numpy().view(np.uint64).copy()
        G = G.cpu().numpy()
        assert stats == so_all
        flat = H.reshape(-1)
        wrong = [(i, int(flat[i]), v) for i, v in bins_all.items() if int(flat[i]) != v]
        assert not wrong, f"whole-run histogram differs from the oracle in sampled bins: {wrong[:5]}"
        assert int(H.sum(dtype=np.uint64)) == sum_all
        assert hashlib.sha256(np.ascontiguousarray(H).astype("<u8").tobytes()).hexdigest() == sha_all, \
            "whole-run histogram differs from the oracle"
        c2all, g2all = plan.finalize_g2()
        c2all = c2all.cpu().numpy().view(np.uint64).copy()
        g2all = g2all.cpu().numpy()
        T_r, _ = oracle_lib.thresholds(w.box, w.r_max, w.n_r, w.n_t)
        # per-frame histograms from the same plan; sampled ones against the oracle
        Hsum = np.zeros_like(H)
        c2sum = np.zeros_like(c2all)
        pairs = 0
        for f in range(w.n_frames):
            plan.reset()
            plan.accumulate_frame(d_pos[f])
            cf, _, sf = plan.finalize(want_g3=False)
            Hf = cf.cpu().numpy().view(np.uint64)
            c2f = plan.finalize_g2()[0].cpu().numpy().view(np.uint64)
            Hsum += Hf
            c2sum += c2f
            pairs += sf[1]
            if f in sample:
                Ho, so = oracle_frames(oracle_lib, w, [ms[f]])
                assert np.array_equal(Hf, Ho), f"frame {f}"
                assert sf == so
                if f == sample[0]:
                    assert np.array_equal(c2f, oracle_lib.g2_frame(ms[f], T_r)), f"g2, frame {f}"
    assert np.array_equal(c2all, c2sum)
    assert np.allclose(g2all, oracle_lib.g2_normalise(c2all, w.r_max, w.n_frames, w.n, w.box),
                       rtol=G3_RTOL, atol=0)
    if w.kind == "uniform":
        z2 = (g2all / (1.0 - 1.0 / w.n) - 1.0) * np.sqrt(c2all.astype(np.float64) / 2.0)
        assert np.abs(z2[4:]).max() < 6.0
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
