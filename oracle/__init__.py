"""CPU oracle for g(3) -- TEST INFRASTRUCTURE ONLY (see g3_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_1708_08619_b200."""
from .g3_oracle import (Oracle, accumulate, build, frame_allpairs, frame_cells, g2_frame,
                        g2_normalise, msd, normalise, qtet_frame,
                        num_threads, quantise, set_num_threads, thresholds, volumes)

__all__ = ["Oracle", "accumulate", "build", "frame_allpairs", "frame_cells", "g2_frame",
           "g2_normalise", "msd", "normalise", "qtet_frame",
           "num_threads", "quantise", "set_num_threads", "thresholds", "volumes"]
