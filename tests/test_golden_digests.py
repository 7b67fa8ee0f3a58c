"""The stored whole-run digests of configs 3 and 5 (tests/golden/config*_whole_run.txt, written by
tests/golden/make_whole_run_digests.py from the CPU oracle alone) are well-formed and obey what
holds for any g(3) histogram: sum(H) + overflow = sum_i k_i (k_i - 1), the
shape and frame count of the BASELINE.json config, a non-empty sampled bin for each of the 300
drawn from the occupied ones.  The GPU comparison itself is tests/test_gpu_fullsize.py."""
import os
import re

import pytest

from workloads import WORKLOADS

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.mark.parametrize("widx", [3, 5])
def test_digest_is_consistent(widx):
    w = WORKLOADS[widx]
    text = open(os.path.join(GOLDEN, f"config{widx}_whole_run.txt")).read()
    assert "make_whole_run_digests.py" in text and "PAPER.md" in text          # says where it comes from
    shape = tuple(int(v) for v in re.search(r"(?m)^shape (\d+) (\d+) (\d+)$", text).groups())
    sha = re.search(r"(?m)^sha256 ([0-9a-f]{64})$", text).group(1)
    stats = [int(v) for v in re.search(r"(?m)^stats (\d+) (\d+) (\d+)$", text).groups()]
    total = int(re.search(r"(?m)^sum (\d+)$", text).group(1))
    bins = [(int(i), int(v)) for i, v in re.findall(r"(?m)^bin (\d+) (\d+)$", text)]
    assert shape == (w.n_r, w.n_r, w.n_t) and len(sha) == 64
    assert stats[0] == w.n_frames
    assert total + stats[2] == stats[1] and stats[1] % 2 == 0                  # ordered pairs (j, k) and (k, j)
    assert len(bins) == 400 and all(0 <= i < shape[0] * shape[1] * shape[2] for i, _ in bins)
    assert all(v > 0 for _, v in bins[:300])
    # r12 <-> r13 symmetry, wherever both partners of a pair of bins were sampled
    by_index = dict(bins)
    n_r, n_t = shape[0], shape[2]
    for i, v in bins:
        a, b, c = i // (n_r * n_t), (i // n_t) % n_r, i % n_t
        j = (b * n_r + a) * n_t + c
        if j in by_index:
            assert by_index[j] == v
