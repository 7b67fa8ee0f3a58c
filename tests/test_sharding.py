"""Host logic of the frame-sharded multi-GPU path, on CPU with the gloo
backend and world_size 2: each rank accumulates its own block of frames (here with the CPU oracle
standing in for the per-rank histogram producer -- the collective and the shard arithmetic are
what is under test), the uint64 histograms are summed once, and the merged result must equal the
single-process histogram of the whole trajectory bit for bit."""
import os
import socket

import numpy as np
import pytest

from paper_1708_08619_b200.sharding import frame_shard


def test_frame_shard_tiles_the_range():
    for n_frames in (0, 1, 2, 7, 500, 501):
        for world in (1, 2, 3, 8):
            blocks = [frame_shard(n_frames, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == n_frames
            for (b0, e0), (b1, e1) in zip(blocks, blocks[1:]):
                assert e0 == b1
            sizes = [e - b for b, e in blocks]
            assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 0
    with pytest.raises(ValueError):
        frame_shard(10, 2, 2)
    with pytest.raises(ValueError):
        frame_shard(-1, 0, 1)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, n_frames: int, out_dir: str) -> None:
    import torch
    import torch.distributed as dist

    import oracle
    from paper_1708_08619_b200.sharding import frame_shard, merge_counts, merge_frames
    from workloads import WORKLOADS, frames

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = WORKLOADS[1]
        _, pos = frames(w, n_frames)
        b, e = frame_shard(n_frames, rank, world)
        orc = oracle.Oracle(w.n, w.box, w.r_max, w.n_r, w.n_t, mode="allpairs")
        if e > b:
            orc.accumulate(pos[b:e])
        H, _, stats = orc.finalize()
        counts = torch.from_numpy(H.view(np.int64).copy())       # uint64 bit patterns
        merged = merge_counts(counts)
        total_frames = merge_frames(e - b)
        assert counts.equal(torch.from_numpy(H.view(np.int64)))   # input untouched
        np.save(os.path.join(out_dir, f"merged_{rank}.npy"), merged.numpy().view(np.uint64))
        with open(os.path.join(out_dir, f"frames_{rank}.txt"), "w") as f:
            f.write(f"{total_frames} {int(stats[0])}")
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_frames", [5, 1])
def test_two_rank_merge_equals_single_process(oracle_lib, tmp_path, n_frames):
    import torch.multiprocessing as mp

    from workloads import WORKLOADS, frames

    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, n_frames, str(tmp_path)), nprocs=world, join=True)

    w = WORKLOADS[1]
    _, pos = frames(w, n_frames)
    orc = oracle_lib.Oracle(w.n, w.box, w.r_max, w.n_r, w.n_t, mode="allpairs")
    orc.accumulate(pos)
    H, _, _ = orc.finalize()
    local_frames = 0
    for r in range(world):
        merged = np.load(tmp_path / f"merged_{r}.npy")
        assert np.array_equal(merged, H), f"rank {r}: merged histogram differs"
        total, mine = (tmp_path / f"frames_{r}.txt").read_text().split()
        assert int(total) == n_frames
        local_frames += int(mine)
    assert local_frames == n_frames


def test_merge_without_process_group_is_identity():
    import torch

    from paper_1708_08619_b200.sharding import merge_counts, merge_frames
    x = torch.arange(12, dtype=torch.int64).reshape(3, 4)
    y = merge_counts(x)
    assert y.equal(x) and y.data_ptr() != x.data_ptr()
    assert merge_frames(7) == 7


def test_bench_launches_its_own_ranks():
    """`python bench.py --gpus N` (no torchrun, WORLD_SIZE unset) must start N ranks itself
    (PAPER.md:356, 727).  --launch-check runs them on CPU over gloo: every rank reports its rank,
    pid and the frame block --shard-one-trajectory would give it."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "3", "--launch-check",
                          "--frames", "500"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert line["launched"] == 3 and line["ranks"] == [0, 1, 2]
    assert len(set(line["pids"])) == 3
    assert line["shards"] == [list(frame_shard(500, r, 3)) for r in range(3)]
    assert line["shards"][0][0] == 0 and line["shards"][-1][1] == 500
