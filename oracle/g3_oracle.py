"""ctypes binding of oracle/g3_oracle.c (argument marshalling only).

TEST INFRASTRUCTURE: see the header of g3_oracle.c for who may import this.
`build()` compiles the C file with gcc into oracle/libg3oracle.so; nothing here
touches CUDA or the product package."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "g3_oracle.c")
_LIB = os.path.join(_HERE, "libg3oracle.so")
_lib: Optional[C.CDLL] = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -ffp-contract=off (no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
               "-Wall", "-Wextra", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        u64p, i32p, f64p = (C.POINTER(C.c_uint64), C.POINTER(C.c_int32), C.POINTER(C.c_double))
        _lib.g3o_thresholds.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_int32, u64p, u64p]
        _lib.g3o_quantise.argtypes = [f64p, C.c_int64, C.c_double, i32p]
        for fn in (_lib.g3o_frame_allpairs, _lib.g3o_frame_cells):
            fn.argtypes = [i32p, C.c_int64, u64p, C.c_int32, u64p, C.c_int32, u64p, u64p]
            fn.restype = None
        _lib.g3o_accumulate.argtypes = [f64p, C.c_int64, C.c_int64, C.c_double, C.c_double,
                                        C.c_int32, C.c_int32, C.c_int32, u64p, u64p]
        _lib.g3o_volumes.argtypes = [C.c_double, C.c_int32, C.c_int32, f64p]
        _lib.g3o_normalise.argtypes = [u64p, f64p, C.c_int64, C.c_int64, C.c_int64, C.c_double, f64p]
        _lib.g3o_g2_frame.argtypes = [i32p, C.c_int64, u64p, C.c_int32, u64p]
        _lib.g3o_g2_frame.restype = None
        _lib.g3o_g2_normalise.argtypes = [u64p, C.c_int32, C.c_double, C.c_int64, C.c_int64, C.c_double, f64p]
        _lib.g3o_g2_normalise.restype = None
        _lib.g3o_qtet_frame.argtypes = [i32p, C.c_int64, C.c_int32, u64p, u64p, f64p]
        _lib.g3o_qtet_frame.restype = None
        _lib.g3o_msd.argtypes = [f64p, C.c_int64, C.c_int64, C.c_double, C.c_int64, u64p, f64p]
        _lib.g3o_msd.restype = C.c_int64
        _lib.g3o_num_threads.restype = C.c_int32
        _lib.g3o_set_num_threads.argtypes = [C.c_int32]
        _lib.g3o_set_num_threads.restype = None
        for fn in (_lib.g3o_thresholds, _lib.g3o_quantise, _lib.g3o_accumulate, _lib.g3o_volumes,
                   _lib.g3o_normalise):
            fn.restype = None
    return _lib


def _p(a: np.ndarray, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def num_threads() -> int:
    return int(_load().g3o_num_threads())


def set_num_threads(n: int) -> None:
    """OpenMP threads of the following calls (results do not depend on it)."""
    _load().g3o_set_num_threads(int(n))


def thresholds(box: float, r_max: float, n_r: int, n_t: int) -> Tuple[np.ndarray, np.ndarray]:
    T_r = np.zeros(n_r + 1, dtype=np.uint64)
    T_t = np.zeros(n_t + 1, dtype=np.uint64)
    _load().g3o_thresholds(box, r_max, n_r, n_t, _p(T_r, C.c_uint64), _p(T_t, C.c_uint64))
    return T_r, T_t


def quantise(pos: np.ndarray, box: float) -> np.ndarray:
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    assert pos.ndim == 2 and pos.shape[1] == 3
    m = np.zeros(pos.shape, dtype=np.int32)
    _load().g3o_quantise(_p(pos, C.c_double), pos.shape[0], box, _p(m, C.c_int32))
    return m


def _frame(fn, m, T_r, T_t, H, stats):
    m = np.ascontiguousarray(m, dtype=np.int32)
    n_r, n_t = len(T_r) - 1, len(T_t) - 1
    if H is None:
        H = np.zeros((n_r, n_r, n_t), dtype=np.uint64)
    if stats is None:
        stats = np.zeros(3, dtype=np.uint64)
    assert H.shape == (n_r, n_r, n_t) and H.dtype == np.uint64 and H.flags.c_contiguous
    fn(_p(m, C.c_int32), m.shape[0], _p(T_r, C.c_uint64), n_r, _p(T_t, C.c_uint64), n_t,
       _p(H, C.c_uint64), _p(stats, C.c_uint64))
    return H, stats


def frame_allpairs(m, T_r, T_t, H=None, stats=None):
    """Add one frame of int32 grid coordinates [n,3] to (H, stats); reference routine."""
    return _frame(_load().g3o_frame_allpairs, m, T_r, T_t, H, stats)


def frame_cells(m, T_r, T_t, H=None, stats=None):
    """Same with the cell-grid candidate pre-filter."""
    return _frame(_load().g3o_frame_cells, m, T_r, T_t, H, stats)


def accumulate(pos: np.ndarray, box: float, r_max: float, n_r: int, n_t: int, mode: str = "allpairs",
               H: Optional[np.ndarray] = None, stats: Optional[np.ndarray] = None):
    """Quantise fp64 positions [F,n,3] and accumulate all F frames. Returns (H, stats)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    if pos.ndim == 2:
        pos = pos[None]
    F, n, three = pos.shape
    assert three == 3
    if H is None:
        H = np.zeros((n_r, n_r, n_t), dtype=np.uint64)
    if stats is None:
        stats = np.zeros(3, dtype=np.uint64)
    _load().g3o_accumulate(_p(pos, C.c_double), F, n, box, r_max, n_r, n_t,
                           {"allpairs": 0, "cells": 1}[mode], _p(H, C.c_uint64), _p(stats, C.c_uint64))
    return H, stats


def volumes(r_max: float, n_r: int, n_t: int) -> np.ndarray:
    V = np.zeros((n_r, n_r, n_t), dtype=np.float64)
    _load().g3o_volumes(r_max, n_r, n_t, _p(V, C.c_double))
    return V


def normalise(H: np.ndarray, V: np.ndarray, n_frames: int, n: int, box: float) -> np.ndarray:
    H = np.ascontiguousarray(H, dtype=np.uint64)
    V = np.ascontiguousarray(V, dtype=np.float64)
    g3 = np.zeros(H.shape, dtype=np.float64)
    _load().g3o_normalise(_p(H, C.c_uint64), _p(V, C.c_double), H.size, n_frames, n, box,
                          _p(g3, C.c_double))
    return g3


def g2_frame(m: np.ndarray, T_r: np.ndarray, H2: Optional[np.ndarray] = None) -> np.ndarray:
    """Add one frame's ordered-pair counts per r_ij shell to H2 [n_r] (g3o_g2_frame)."""
    m = np.ascontiguousarray(m, dtype=np.int32)
    T_r = np.ascontiguousarray(T_r, dtype=np.uint64)
    n_r = T_r.size - 1
    if H2 is None:
        H2 = np.zeros(n_r, dtype=np.uint64)
    _load().g3o_g2_frame(_p(m, C.c_int32), m.shape[0], _p(T_r, C.c_uint64), n_r, _p(H2, C.c_uint64))
    return H2


def g2_normalise(H2: np.ndarray, r_max: float, n_frames: int, n: int, box: float) -> np.ndarray:
    H2 = np.ascontiguousarray(H2, dtype=np.uint64)
    g2 = np.zeros(H2.size, dtype=np.float64)
    _load().g3o_g2_normalise(_p(H2, C.c_uint64), H2.size, r_max, n_frames, n, box, _p(g2, C.c_double))
    return g2


def qtet_frame(m: np.ndarray, n_q: int, H: Optional[np.ndarray] = None,
               stats: Optional[np.ndarray] = None, q_out: Optional[np.ndarray] = None):
    """Add one frame's q_tet histogram (n_q bins on [-3, 1]) to H; stats = [binned, skipped];
    q_out (fp64 [n], optional) receives the per-atom values (NaN where skipped)."""
    m = np.ascontiguousarray(m, dtype=np.int32)
    if H is None:
        H = np.zeros(n_q, dtype=np.uint64)
    if stats is None:
        stats = np.zeros(2, dtype=np.uint64)
    qp = _p(q_out, C.c_double) if q_out is not None else None
    _load().g3o_qtet_frame(_p(m, C.c_int32), m.shape[0], n_q, _p(H, C.c_uint64), _p(stats, C.c_uint64), qp)
    return H, stats


def msd(pos: np.ndarray, box: float, max_lag: Optional[int] = None):
    """(sums uint64 [max_lag+1, 2] = (lo, hi) of the exact 128-bit sums of squared grid
    displacements, msd fp64 [max_lag+1]) of an UNWRAPPED trajectory pos [F, n, 3] (g3o_msd)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    F, n, three = pos.shape
    assert three == 3
    L = F - 1 if max_lag is None else int(max_lag)
    assert 0 <= L <= F - 1
    sums = np.zeros((L + 1, 2), dtype=np.uint64)
    out = np.zeros(L + 1, dtype=np.float64)
    bad = _load().g3o_msd(_p(pos, C.c_double), F, n, box, L, _p(sums, C.c_uint64), _p(out, C.c_double))
    if bad:
        raise ValueError(f"{bad} coordinates outside +-2^30 grid units")
    return sums, out


class Oracle:
    """Plan-like convenience wrapper used by the parity tests."""

    def __init__(self, n: int, box: float, r_max: float, n_r: int, n_t: int, mode: str = "allpairs"):
        self.n, self.box, self.r_max, self.n_r, self.n_t, self.mode = n, box, r_max, n_r, n_t, mode
        self.H = np.zeros((n_r, n_r, n_t), dtype=np.uint64)
        self.stats = np.zeros(3, dtype=np.uint64)
        self._V: Optional[np.ndarray] = None

    def accumulate(self, pos: np.ndarray) -> None:
        accumulate(pos, self.box, self.r_max, self.n_r, self.n_t, self.mode, self.H, self.stats)

    def finalize(self):
        if self._V is None:
            self._V = volumes(self.r_max, self.n_r, self.n_t)
        g3 = normalise(self.H, self._V, int(self.stats[0]), self.n, self.box)
        return self.H.copy(), g3, self.stats.copy()
