"""g(3) triplet correlation function on one B200: Python face of the libg3 C ABI (include/g3.h)."""
from .binding import (BENCH_EXPORTS, BENCH_LIB_PATH, EXPORTS, G3_ECAPACITY, G3_EINTERNAL, G3_ELIMIT, G3_ECUDA, G3_EINVAL, G3_ENOMEM, G3_ESTATE,
                      G3_INFO_BATCH_FRAMES, G3_INFO_CELLS_PER_EDGE, G3_INFO_FRAMES_PENDING,
                      G3_INFO_KERNEL, G3_INFO_KERNEL_LAUNCHES, G3_INFO_MAX_NEIGHBOURS,
                      G3_INFO_G2_SHELLS, G3_INFO_SM_COUNT, G3_INFO_SLABS, G3_INFO_TILE_BINS, G3_INFO_TIMED_LAUNCHES, G3_INFO_TRIPLET_NS,
                      G3_INFO_NEIGHBOUR_NS, G3_OPT_TIMING, G3_OPT_TRIPLET_WARPS, G3_OK, G3_OPT_BATCH_FRAMES,
                      G3_OPT_G2_WIDE, G3_OPT_KERNEL, G3_OPT_MAX_NEIGHBOURS, G3_OPT_QTET_BINS, G3_MSD_STATIC_MAX_PARTIALS, LIB_PATH, G3Error, Plan, load, load_bench, microbench, msd, msd_static,
                      strerror)

__all__ = [n for n in dir() if n.startswith("G3") or n in ("Plan", "load", "microbench", "msd", "msd_static", "strerror", "EXPORTS", "LIB_PATH", "BENCH_EXPORTS", "BENCH_LIB_PATH", "load_bench")]
