"""Seeded synthetic inputs shared by the oracle's tests and the CUDA path's tests/bench.
Holds no arithmetic of the g(3) method itself (see frames.py)."""
from .frames import (GRID, GRID_BITS, WORKLOADS, Workload, frame_iter, frames, grid_to_pos,
                     uniform_frame, unwrapped_walk)

__all__ = ["GRID", "GRID_BITS", "WORKLOADS", "Workload", "frame_iter", "frames", "grid_to_pos",
           "uniform_frame", "unwrapped_walk"]
