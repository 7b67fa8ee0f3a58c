"""Thin ctypes binding of libg3 (include/g3.h).  Argument marshalling only: every step of the
g(3) path runs in the CUDA kernels behind the C ABI.  torch supplies device memory and streams.

There is no CPU fallback: importing works anywhere (so the ABI can be inspected), but creating a
plan without the built library or without a B200 raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Tuple

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libg3.so")

G3_OK, G3_EINVAL, G3_ENOMEM, G3_ECUDA, G3_ECAPACITY, G3_ESTATE, G3_EINTERNAL, G3_ELIMIT = range(8)
G3_OPT_BATCH_FRAMES, G3_OPT_KERNEL, G3_OPT_MAX_NEIGHBOURS, G3_OPT_TIMING, G3_OPT_TRIPLET_WARPS = 1, 2, 3, 4, 5
G3_OPT_QTET_BINS = 6
G3_OPT_G2_WIDE = 7
(G3_INFO_KERNEL_LAUNCHES, G3_INFO_BATCH_FRAMES, G3_INFO_KERNEL, G3_INFO_CELLS_PER_EDGE,
 G3_INFO_MAX_NEIGHBOURS, G3_INFO_TILE_BINS, G3_INFO_SM_COUNT, G3_INFO_FRAMES_PENDING,
 G3_INFO_TRIPLET_NS, G3_INFO_NEIGHBOUR_NS, G3_INFO_TIMED_LAUNCHES, G3_INFO_SLABS, G3_INFO_G2_SHELLS) = range(1, 14)

EXPORTS = [
    "g3_plan_create", "g3_plan_set_option", "g3_plan_get_info", "g3_plan_clear_timing",
    "g3_accumulate_frame",
    "g3_accumulate_frames", "g3_accumulate_frames_host", "g3_finalize", "g3_finalize_host",
    "g3_finalize_g2", "g3_finalize_qtet", "g3_normalize", "g3_bin_volumes", "g3_msd", "g3_msd_static", "g3_plan_reset", "g3_plan_destroy", "g3_strerror",
]


class g3_bins(C.Structure):
    _fields_ = [("n_r", C.c_int32), ("n_t", C.c_int32)]


class G3Error(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {strerror(code)} (g3_status {code})")
        self.code = code


_lib: Optional[C.CDLL] = None


def load() -> C.CDLL:
    """dlopen libg3.so (built by paper_1708_08619_b200.build).  Fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1708_08619_b200.build` "
                           "(needs nvcc). There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, i64, i32, f64 = C.c_void_p, C.c_int64, C.c_int32, C.c_double
    lib.g3_plan_create.argtypes = [C.POINTER(vp), i64, f64, f64, g3_bins]
    lib.g3_plan_set_option.argtypes = [vp, i32, i64]
    lib.g3_plan_get_info.argtypes = [vp, i32, C.POINTER(i64)]
    lib.g3_plan_clear_timing.argtypes = [vp]
    lib.g3_accumulate_frame.argtypes = [vp, vp, vp]
    lib.g3_accumulate_frames.argtypes = [vp, vp, i64, i64, vp]
    lib.g3_accumulate_frames_host.argtypes = [vp, vp, i64, i64, vp]
    lib.g3_finalize.argtypes = [vp, vp, vp, vp, vp]
    lib.g3_finalize_host.argtypes = [vp, vp, vp, vp, vp]
    lib.g3_finalize_g2.argtypes = [vp, vp, vp, vp]
    lib.g3_finalize_qtet.argtypes = [vp, vp, vp, vp]
    lib.g3_normalize.argtypes = [vp, vp, C.c_uint64, vp, vp]
    lib.g3_bin_volumes.argtypes = [vp, vp]
    lib.g3_msd.argtypes = [vp, i64, i64, i64, f64, i64, vp, vp, vp]
    lib.g3_msd_static.argtypes = [vp, i64, i64, i64, f64, i64, vp, vp, vp]
    lib.g3_plan_reset.argtypes = [vp, vp]
    lib.g3_plan_destroy.argtypes = [vp]
    lib.g3_plan_destroy.restype = None
    lib.g3_strerror.argtypes = [C.c_int]
    lib.g3_strerror.restype = C.c_char_p
    for name in EXPORTS:
        if name not in ("g3_plan_destroy", "g3_strerror"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def strerror(code: int) -> str:
    return load().g3_strerror(int(code)).decode()


def _check(code: int, what: str, allow=()):
    if code != G3_OK and code not in allow:
        raise G3Error(code, what)
    return code


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


BENCH_LIB_PATH = os.path.join(_HERE, "libg3bench.so")
BENCH_EXPORTS = ["g3_microbench"]
_bench_lib: Optional[C.CDLL] = None


def load_bench() -> C.CDLL:
    """dlopen libg3bench.so (include/g3_bench.h): bench.py's measurement aid, not the product."""
    global _bench_lib
    if _bench_lib is None:
        if not os.path.exists(BENCH_LIB_PATH):
            raise RuntimeError(f"{BENCH_LIB_PATH} is missing: run `python -m paper_1708_08619_b200.build`")
        lib = C.CDLL(BENCH_LIB_PATH)
        lib.g3_microbench.argtypes = [C.c_int32, C.c_int64, C.c_int64, C.POINTER(C.c_double), C.c_void_p]
        lib.g3_microbench.restype = C.c_int
        _bench_lib = lib
    return _bench_lib


def microbench(which: int, slots: int = 50776, iters: int = 1 << 14, stream=None) -> float:
    """g3_microbench: 0 = shared-atomic increments/s (random slots), 1 = FP32 thread instr/s."""
    rate = C.c_double()
    _check(load_bench().g3_microbench(int(which), int(slots), int(iters), C.byref(rate), _stream_ptr(stream)),
           "g3_microbench")
    return float(rate.value)


def msd(d_pos, box: float, max_lag: Optional[int] = None, stream=None):
    """g3_msd of an unwrapped fp64 cuda trajectory [F, n, 3]: (sums int64-viewed-as-uint64
    [max_lag+1, 2] = (low, high) words, msd fp64 [max_lag+1]) device tensors."""
    import torch
    if d_pos.dtype != torch.float64 or d_pos.device.type != "cuda" or not d_pos.is_contiguous() or \
            d_pos.dim() != 3 or d_pos.shape[2] != 3:
        raise ValueError("positions must be a contiguous float64 cuda tensor [F, n, 3]")
    F, n = int(d_pos.shape[0]), int(d_pos.shape[1])
    L = F - 1 if max_lag is None else int(max_lag)
    sums = torch.empty((L + 1, 2), dtype=torch.int64, device="cuda")
    out = torch.empty(L + 1, dtype=torch.float64, device="cuda")
    _check(load().g3_msd(d_pos.data_ptr(), F, n, 3 * n, float(box), L, sums.data_ptr(), out.data_ptr(),
                         _stream_ptr(stream)), "g3_msd")
    return sums, out


G3_MSD_STATIC_MAX_PARTIALS = 524288           # include/g3.h


def msd_static(d_pos, box: float, max_lag: Optional[int] = None, stream=None, sums=None, out=None):
    """g3_msd_static: msd() for programs that must not allocate device memory (see include/g3.h:
    their own allocator owns the GPU's memory, or they run under a fixed memory limit).  The
    library's scratch is a fixed built-in array, so the C call allocates nothing; pass `sums`
    (int64 cuda [max_lag+1, 2]) and `out` (float64 cuda [max_lag+1]) tensors created beforehand and
    this wrapper allocates nothing either.  Raises G3Error with code G3_ELIMIT when
    ceil(n/32) * (max_lag+1) > G3_MSD_STATIC_MAX_PARTIALS or the run has more than ~580 frames.
    Calls on one GPU share the array: do not let two of them overlap on the device."""
    import torch
    if d_pos.dtype != torch.float64 or d_pos.device.type != "cuda" or not d_pos.is_contiguous() or \
            d_pos.dim() != 3 or d_pos.shape[2] != 3:
        raise ValueError("positions must be a contiguous float64 cuda tensor [F, n, 3]")
    F, n = int(d_pos.shape[0]), int(d_pos.shape[1])
    L = F - 1 if max_lag is None else int(max_lag)
    if sums is None:
        sums = torch.empty((L + 1, 2), dtype=torch.int64, device="cuda")
    if out is None:
        out = torch.empty(L + 1, dtype=torch.float64, device="cuda")
    if sums.dtype != torch.int64 or out.dtype != torch.float64 or sums.device.type != "cuda" or \
            out.device.type != "cuda" or not sums.is_contiguous() or not out.is_contiguous() or \
            sums.numel() < 2 * (L + 1) or out.numel() < L + 1:
        raise ValueError("sums must be int64 cuda [max_lag+1, 2] and out float64 cuda [max_lag+1], contiguous")
    _check(load().g3_msd_static(d_pos.data_ptr(), F, n, 3 * n, float(box), L, sums.data_ptr(), out.data_ptr(),
                                _stream_ptr(stream)), "g3_msd_static")
    return sums, out


class Plan:
    """g3_plan with the same calls as the C ABI: accumulate_frame(s), finalize, reset."""

    def __init__(self, n: int, box: float, r_max: float, n_r: int, n_t: Optional[int] = None, *,
                 batch_frames: Optional[int] = None, kernel: Optional[int] = None,
                 max_neighbours: Optional[int] = None, timing: bool = False,
                 triplet_warps: Optional[int] = None, qtet_bins: Optional[int] = None, g2_wide: bool = False):
        self._lib = load()
        self.n, self.box, self.r_max = int(n), float(box), float(r_max)
        self.n_r, self.n_t = int(n_r), int(n_r if n_t is None else n_t)
        self._h = C.c_void_p()
        _check(self._lib.g3_plan_create(C.byref(self._h), self.n, self.box, self.r_max,
                                        g3_bins(self.n_r, self.n_t)), "g3_plan_create")
        if batch_frames is not None:
            self.set_option(G3_OPT_BATCH_FRAMES, batch_frames)
        if kernel is not None:
            self.set_option(G3_OPT_KERNEL, kernel)
        if max_neighbours is not None:
            self.set_option(G3_OPT_MAX_NEIGHBOURS, max_neighbours)
        if timing:
            self.set_option(G3_OPT_TIMING, 1)
        if triplet_warps is not None:
            self.set_option(G3_OPT_TRIPLET_WARPS, triplet_warps)
        if g2_wide:
            self.set_option(G3_OPT_G2_WIDE, 1)
        self.g2_shells = 2 * self.n_r if g2_wide else self.n_r
        self.qtet_bins = int(qtet_bins or 0)
        if self.qtet_bins:
            self.set_option(G3_OPT_QTET_BINS, self.qtet_bins)

    # -- options / info -------------------------------------------------------------------
    def set_option(self, option: int, value: int) -> None:
        _check(self._lib.g3_plan_set_option(self._h, option, int(value)), "g3_plan_set_option")

    def info(self, key: int) -> int:
        v = C.c_int64()
        _check(self._lib.g3_plan_get_info(self._h, key, C.byref(v)), "g3_plan_get_info")
        return int(v.value)

    def clear_timing(self) -> None:
        _check(self._lib.g3_plan_clear_timing(self._h), "g3_plan_clear_timing")

    @property
    def shape(self) -> Tuple[int, int, int]:
        return (self.n_r, self.n_r, self.n_t)

    # -- accumulation ---------------------------------------------------------------------
    def _check_pos(self, pos, device_type: str, frames: bool):
        import torch
        if pos.dtype != torch.float64 or pos.device.type != device_type or not pos.is_contiguous():
            raise ValueError(f"positions must be a contiguous float64 {device_type} tensor")
        want = (self.n, 3)
        if tuple(pos.shape[-2:]) != want or pos.dim() != (3 if frames else 2):
            raise ValueError(f"positions must have shape {'[F,' if frames else '['}{self.n},3]")

    def accumulate_frame(self, d_pos, stream=None) -> None:
        self._check_pos(d_pos, "cuda", False)
        _check(self._lib.g3_accumulate_frame(self._h, d_pos.data_ptr(), _stream_ptr(stream)),
               "g3_accumulate_frame")

    def accumulate_frames(self, d_pos, stream=None) -> None:
        self._check_pos(d_pos, "cuda", True)
        _check(self._lib.g3_accumulate_frames(self._h, d_pos.data_ptr(), d_pos.shape[0], 3 * self.n,
                                              _stream_ptr(stream)), "g3_accumulate_frames")

    def accumulate_frames_host(self, h_pos, stream=None) -> None:
        self._check_pos(h_pos, "cpu", True)
        _check(self._lib.g3_accumulate_frames_host(self._h, h_pos.data_ptr(), h_pos.shape[0],
                                                   3 * self.n, _stream_ptr(stream)),
               "g3_accumulate_frames_host")

    # -- results --------------------------------------------------------------------------
    def finalize(self, want_g3: bool = True, stream=None):
        """(counts int64-viewed-as-uint64 device tensor, g3 device tensor or None, stats list)."""
        import torch
        counts = torch.empty(self.shape, dtype=torch.int64, device="cuda")   # bit pattern of uint64
        g3 = torch.empty(self.shape, dtype=torch.float64, device="cuda") if want_g3 else None
        stats = (C.c_uint64 * 3)()
        _check(self._lib.g3_finalize(self._h, counts.data_ptr(), g3.data_ptr() if want_g3 else None,
                                     stats, _stream_ptr(stream)), "g3_finalize")
        return counts, g3, [int(v) for v in stats]

    def finalize_host(self, want_g3: bool = True, stream=None):
        import torch
        counts = torch.empty(self.shape, dtype=torch.int64).pin_memory()
        g3 = torch.empty(self.shape, dtype=torch.float64).pin_memory() if want_g3 else None
        stats = (C.c_uint64 * 3)()
        _check(self._lib.g3_finalize_host(self._h, counts.data_ptr(), g3.data_ptr() if want_g3 else None,
                                          stats, _stream_ptr(stream)), "g3_finalize_host")
        return counts, g3, [int(v) for v in stats]

    def finalize_g2(self, stream=None):
        """(counts2 int64-viewed-as-uint64 [S], g2 fp64 [S]) device tensors, S = n_r, or 2 n_r with
        g2_wide; stream-ordered."""
        import torch
        counts2 = torch.empty(self.g2_shells, dtype=torch.int64, device="cuda")
        g2 = torch.empty(self.g2_shells, dtype=torch.float64, device="cuda")
        _check(self._lib.g3_finalize_g2(self._h, counts2.data_ptr(), g2.data_ptr(), _stream_ptr(stream)),
               "g3_finalize_g2")
        return counts2, g2

    def finalize_qtet(self, stream=None):
        """(q_tet histogram int64-viewed-as-uint64 [qtet_bins] device tensor, [binned, skipped])."""
        import torch
        hist = torch.empty(self.qtet_bins, dtype=torch.int64, device="cuda")
        stats = (C.c_uint64 * 2)()
        _check(self._lib.g3_finalize_qtet(self._h, hist.data_ptr(), stats, _stream_ptr(stream)),
               "g3_finalize_qtet")
        return hist, [int(v) for v in stats]

    def normalize(self, d_counts, frames: int, stream=None):
        import torch
        if d_counts.dtype != torch.int64 or d_counts.device.type != "cuda" or not d_counts.is_contiguous():
            raise ValueError("counts must be a contiguous int64 cuda tensor")
        g3 = torch.empty(self.shape, dtype=torch.float64, device="cuda")
        _check(self._lib.g3_normalize(self._h, d_counts.data_ptr(), int(frames), g3.data_ptr(),
                                      _stream_ptr(stream)), "g3_normalize")
        return g3

    def bin_volumes(self):
        import numpy as np
        V = np.empty(self.shape, dtype=np.float64)
        _check(self._lib.g3_bin_volumes(self._h, V.ctypes.data_as(C.c_void_p)), "g3_bin_volumes")
        return V

    def reset(self, stream=None) -> None:
        _check(self._lib.g3_plan_reset(self._h, _stream_ptr(stream)), "g3_plan_reset")

    def close(self) -> None:
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.g3_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
