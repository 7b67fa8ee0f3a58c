"""Writes tests/golden/config{3,5}_whole_run.txt: the g(3) histogram of the WHOLE config-3 / config-5
trajectory (BASELINE.json configs[2], configs[4]; Algorithm 6/7) as computed by the
CPU oracle, in a form small enough to commit: the SHA-256 of the uint64 [n_r][n_r][n_t] array
(C order, little-endian), the three statistics, the sum, and 400 sampled bins.

Calls ONLY oracle/ and the seeded input generators (workloads/): no value in the files comes from the
CUDA path.  The oracle needs minutes per trajectory (1.5e10 and 6.7e10 triplets), which is why
tests/test_gpu_fullsize.py compares against these files instead of re-running it in every GPU test
session; that test still runs the oracle live on sampled frames of the same trajectories.

    python tests/golden/make_whole_run_digests.py [3] [5]
"""
import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle                                    # noqa: E402
from workloads import WORKLOADS, frame_iter      # noqa: E402

N_SAMPLES = 400


def digest_path(widx: int) -> str:
    return os.path.join(HERE, f"config{widx}_whole_run.txt")


def sample_bins(H: np.ndarray, widx: int) -> np.ndarray:
    """flat indices: 300 drawn from the non-empty bins, 100 from all bins (seeded by the config)"""
    rng = np.random.default_rng(1000 + widx)
    flat = H.reshape(-1)
    nz = np.flatnonzero(flat)
    return np.concatenate([rng.choice(nz, size=min(300, nz.size), replace=False),
                           rng.choice(flat.size, size=N_SAMPLES - min(300, nz.size), replace=False)])


def main(which):
    oracle.build()
    for widx in which:
        w = WORKLOADS[widx]
        T_r, T_t = oracle.thresholds(w.box, w.r_max, w.n_r, w.n_t)
        H = np.zeros((w.n_r, w.n_r, w.n_t), dtype=np.uint64)
        stats = np.zeros(3, dtype=np.uint64)
        t0 = time.time()
        for m in frame_iter(w, w.n_frames):
            oracle.frame_cells(m, T_r, T_t, H, stats)
        secs = time.time() - t0
        sha = hashlib.sha256(np.ascontiguousarray(H).astype("<u8").tobytes()).hexdigest()
        idx = sample_bins(H, widx)
        with open(digest_path(widx), "w") as f:
            f.write(f"# g(3) counts of the whole config-{widx} trajectory ({w.n_frames} frames, N = {w.n}), CPU oracle\n")
            f.write("# (oracle/g3_oracle.c frame_cells; Algorithm 6/7, PAPER.md:411-551; BASELINE.json configs).\n")
            f.write("# Written by tests/golden/make_whole_run_digests.py, which calls only oracle/ and workloads/.\n")
            f.write(f"# oracle wall time {secs:.0f} s on {oracle.num_threads()} threads\n")
            f.write(f"shape {w.n_r} {w.n_r} {w.n_t}\n")
            f.write(f"sha256 {sha}\n")
            f.write(f"stats {int(stats[0])} {int(stats[1])} {int(stats[2])}\n")
            f.write(f"sum {int(H.sum(dtype=np.uint64))}\n")
            for i in idx:
                f.write(f"bin {int(i)} {int(H.reshape(-1)[i])}\n")
        print(f"config {widx}: {secs:.0f} s, sha256 {sha}", flush=True)


if __name__ == "__main__":
    main([int(a) for a in sys.argv[1:]] or [3, 5])
