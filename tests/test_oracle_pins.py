"""Pins for the CPU oracle's histogram (S1-S4): things fixed by the paper and by mathematics,
none of which call back into the oracle for their expected values.

Citations: PAPER.md:407-409 (three pair distances, cut-offs), Algorithm 6,
Algorithm 7; readings Q1-Q16 of SURVEY.md 8(c) / DESIGN.md.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

from workloads import GRID, WORKLOADS, frames, grid_to_pos, uniform_frame

HALF = GRID // 2
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------------------------
# independent helpers (exact Python integers; no oracle code)
def py_wrap(d):
    return ((d + HALF) % GRID) - HALF


def py_bin(T, q):
    """largest b with T[b] <= q, by plain linear scan"""
    b = 0
    for idx in range(len(T)):
        if int(T[idx]) <= q:
            b = idx
    return b


def py_thresholds(box, r_max, n_r, n_t):
    """SURVEY.md 8(c) S1 evaluated in Python floats (IEEE fp64, one rounding per operation)."""
    inv_g = 1048576.0 / box
    w = (r_max / n_r) * inv_g
    wt = ((2.0 * r_max) / n_t) * inv_g
    T_r = [int(math.ceil((b * w) * (b * w))) for b in range(n_r + 1)]
    T_t = [int(math.ceil((c * wt) * (c * wt))) for c in range(n_t + 1)]
    return T_r, T_t


def brute_force(m, T_r, T_t):
    """O(N^3): every ordered triple (i, j, k) of distinct particles, no neighbour list, no cells.
    i is the centre; r_ij, r_ik by minimum image; r_jk from the two minimum-image vectors."""
    n = len(m)
    n_r, n_t = len(T_r) - 1, len(T_t) - 1
    H = np.zeros((n_r, n_r, n_t), dtype=np.uint64)
    overflow = 0
    mm = [[int(v) for v in row] for row in m]
    for i in range(n):
        for j in range(n):
            if j == i:
                continue
            dj = [py_wrap(mm[j][x] - mm[i][x]) for x in range(3)]
            d2j = sum(v * v for v in dj)
            if d2j >= T_r[n_r]:
                continue
            aj = py_bin(T_r, d2j)
            for k in range(n):
                if k == i or k == j:
                    continue
                dk = [py_wrap(mm[k][x] - mm[i][x]) for x in range(3)]
                d2k = sum(v * v for v in dk)
                if d2k >= T_r[n_r]:
                    continue
                ak = py_bin(T_r, d2k)
                t2 = sum((dk[x] - dj[x]) ** 2 for x in range(3))
                c = py_bin(T_t, t2)
                if c < n_t:
                    H[aj, ak, c] += 1
                else:
                    overflow += 1
    return H, overflow


def neighbour_counts(m, T_r):
    """k_i [n] and per-shell neighbour counts n_i(a) [n, n_r] by an independent numpy all-pairs scan."""
    mm = m.astype(np.int64)
    n, n_r = len(mm), len(T_r) - 1
    edges = np.array(T_r, dtype=np.int64)
    n_ia = np.zeros((n, n_r), dtype=np.int64)
    for lo in range(0, n, 256):
        d = mm[None, :, :] - mm[lo:lo + 256, None, :]
        d = ((d + HALF) % GRID) - HALF
        d2 = (d * d).sum(-1)
        rows = np.arange(d2.shape[0])
        d2[rows, lo + rows] = np.iinfo(np.int64).max          # j != i
        r, c = np.nonzero(d2 < edges[-1])
        shell = np.searchsorted(edges, d2[r, c], side="right") - 1
        np.add.at(n_ia, (lo + r, shell), 1)
    return n_ia.sum(1), n_ia


# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,box,r_max,n_r,n_t,seed,clump", [
    (24, 6.0, 2.5, 8, 8, 1, 0),        # r_max > box/4: the no-re-wrap reading Q3 matters
    (40, 6.0, 1.4, 6, 12, 2, 0),       # n_t = 2 n_r (equal widths)
    (48, 4.0, 1.0, 5, 7, 3, 1),        # clumped: many neighbours, odd bin counts
    (30, 10.0, 4.9, 16, 16, 4, 0),     # r_max just under box/2
])
def test_brute_force_small(oracle_lib, n, box, r_max, n_r, n_t, seed, clump):
    rng = np.random.default_rng(seed)
    if clump:
        m = (rng.integers(0, GRID // 3, size=(n, 3)) + GRID - GRID // 6) % GRID   # straddles the boundary
        m[1] = m[0]                                                               # coincident pair (Q10)
    else:
        m = rng.integers(0, GRID, size=(n, 3))
    m = m.astype(np.int32)
    T_r, T_t = py_thresholds(box, r_max, n_r, n_t)
    H_ref, ov_ref = brute_force(m, T_r, T_t)
    for mode in ("allpairs", "cells"):
        H, st = oracle_lib.accumulate(grid_to_pos(m, box), box, r_max, n_r, n_t, mode)
        assert np.array_equal(H, H_ref), mode
        assert int(st[2]) == ov_ref and int(st[0]) == 1
        assert int(st[1]) == int(H_ref.sum()) + ov_ref
    assert H_ref.sum() > 0


def test_lattice_worked_example(oracle_lib):
    """tests/golden/lattice_4x4x4.txt (SURVEY.md 8(c) worked example)."""
    idx = np.arange(4) * (1 << 18)
    m = np.stack(np.meshgrid(idx, idx, idx, indexing="ij"), -1).reshape(-1, 3).astype(np.int32)
    H, st = oracle_lib.accumulate(grid_to_pos(m, 4.0), 4.0, 1.3, 4, 4)
    expect = np.zeros((4, 4, 4), dtype=np.uint64)
    for line in open(os.path.join(GOLDEN, "lattice_4x4x4.txt")):
        if line.strip() and not line.startswith("#"):
            a, b, c, v = (int(x) for x in line.split())
            expect[a, b, c] = v
    assert np.array_equal(H, expect)
    assert list(st) == [1, 1920, 0]


def test_hand_three_in_a_line(oracle_lib):
    """particles at 0, d, 2d on the x axis, box 8, r_max 1.0, 10 r-bins (w = 0.1), 10 t-bins (0.2).
    d = 45875 grid units = 0.349998, 2d = 0.699997: shells 3 and 6, away from every bin edge.
    centre = middle: neighbours at -d, +d, r_jk = 2d -> t-bin 3.
    centres = ends: neighbours at d and 2d on the same side, r_jk = d -> t-bin 1."""
    box, d = 8.0, 0.35
    g = round(d * GRID / box)                    # 45875.2 -> 45875 grid units; distances stay inside the bins
    m = np.array([[100, 5, 7], [100 + g, 5, 7], [100 + 2 * g, 5, 7]], dtype=np.int32)
    H, st = oracle_lib.accumulate(grid_to_pos(m, box), box, 1.0, 10, 10)
    expect = np.zeros((10, 10, 10), dtype=np.uint64)
    expect[3, 3, 3] = 2          # centre 1: (j,k) = (0,2), (2,0)
    expect[3, 6, 1] += 2         # centres 0 and 2: (near, far)   0.6999 -> shell 6
    expect[6, 3, 1] += 2         # and (far, near)
    assert np.array_equal(H, expect)
    assert list(st) == [1, 6, 0]


def test_hand_equilateral_and_boundary(oracle_lib):
    """(s,s,0), (s,0,s), (0,s,s): all three distances s*sqrt(2). Shifted so the triangle straddles the
    periodic boundary on every axis: the result must not change (minimum image)."""
    box, r_max, n_r, n_t = 5.0, 1.2, 6, 6          # w = 0.2, wt = 0.4
    s = 150000                                      # s*sqrt(2)*box/2^20 = 1.01153 -> shell 5, t-bin 2
    tri = np.array([[s, s, 0], [s, 0, s], [0, s, s]], dtype=np.int64)
    expect = np.zeros((n_r, n_r, n_t), dtype=np.uint64)
    expect[5, 5, 2] = 6
    for shift in (0, GRID - s // 2, GRID - 1):
        m = ((tri + shift) % GRID).astype(np.int32)
        H, st = oracle_lib.accumulate(grid_to_pos(m, box), box, r_max, n_r, n_t)
        assert np.array_equal(H, expect), shift
        assert list(st) == [1, 6, 0]


def test_no_rewrap_of_rjk(oracle_lib):
    """Q3: j and k on opposite sides of the centre, each within r_max, with r_max > box/4.
    The stored-vector difference is 2*0.45*box = 0.9 box; re-wrapping would give 0.1 box."""
    box, r_max, n_r, n_t = 1.0, 0.48, 4, 8          # wt = 0.12
    a = int(0.45 * GRID)
    m = np.array([[HALF, 9, 9], [HALF + a, 9, 9], [HALF - a, 9, 9]], dtype=np.int32)
    H, st = oracle_lib.accumulate(grid_to_pos(m, box), box, r_max, n_r, n_t)
    # centre 0: neighbours at +a and -a, shell floor(0.45/0.12)=3, t = 0.9 -> t-bin floor(0.9/0.12) = 7
    assert H[3, 3, 7] == 2
    # centres 1 and 2 see 0 at distance 0.45 and each other at min-image distance 0.1 (shell 0);
    # their j-k vector difference has length 0.55 or 0.35?  (centre 1: to 0 is -a, to 2 is wrap(-2a) = +0.1 box)
    # |(-0.45) - (+0.1)| = 0.55 -> t-bin 4, shells (3, 0) and (0, 3)
    assert H[3, 0, 4] == 2 and H[0, 3, 4] == 2
    assert H.sum() == 6 and list(st) == [1, 6, 0]


@pytest.mark.parametrize("widx,nf", [(1, 2), (2, 1), (3, 1)])
def test_invariants_on_workloads(oracle_lib, widx, nf):
    """count invariant, r12<->r13 symmetry, shell marginal, triangle-inequality support."""
    w = WORKLOADS[widx]
    m, pos = frames(w, nf)
    if widx == 3:
        m, pos = m[:, :2048], pos[:, :2048]       # a quarter of the chains: keeps the numpy N^2 check small
    T_r, T_t = py_thresholds(w.box, w.r_max, w.n_r, w.n_t)
    H, st = oracle_lib.accumulate(pos, w.box, w.r_max, w.n_r, w.n_t)
    Hi = H.astype(object)
    total_pairs = 0
    marg = np.zeros(w.n_r, dtype=object)
    for f in range(nf):
        k, n_ia = neighbour_counts(m[f], T_r)
        total_pairs += int((k * (k - 1)).sum())
        for a in range(w.n_r):
            marg[a] += int((n_ia[:, a] * (k - 1)).sum())
    assert int(st[1]) == total_pairs                       # sum_i k_i (k_i - 1)
    assert int(H.sum()) + int(st[2]) == total_pairs
    assert int(st[2]) == 0                                 # Q12: expected 0
    assert np.array_equal(H, H.transpose(1, 0, 2))         # exact symmetry (Q4)
    assert all(int(Hi[a].sum()) == marg[a] for a in range(w.n_r))
    # support: bin (a,b,c) can hold counts only if some (r,s,t) in it obeys |r-s| <= t <= r+s
    wr, wt = w.r_max / w.n_r, 2 * w.r_max / w.n_t
    a = np.arange(w.n_r)[:, None, None]
    b = np.arange(w.n_r)[None, :, None]
    c = np.arange(w.n_t)[None, None, :]
    slack = 2e-5 * wr                                      # thresholds are rounded to grid^2 units
    reachable = ((c + 1) * wt > np.maximum(np.abs(a - b) - 1, 0) * wr - slack) & (c * wt < (a + b + 2) * wr + slack)
    assert not H[~reachable].any()


def test_metamorphic(oracle_lib):
    """bit-identical H under grid translations, relabelling, axis permutation/reflection;
    a duplicated frame doubles H."""
    w = WORKLOADS[1]
    m, _ = frames(w, 1)
    m = m[0].astype(np.int64)
    args = (w.box, w.r_max, w.n_r, w.n_t)
    H0, st0 = oracle_lib.accumulate(grid_to_pos(m, w.box), *args)
    rng = np.random.default_rng(7)
    variants = {
        "translate": (m + rng.integers(0, GRID, size=3)) % GRID,
        "relabel": m[rng.permutation(len(m))],
        "axes": m[:, [2, 0, 1]],
        "reflect": (-m) % GRID,
    }
    for name, mv in variants.items():
        H, st = oracle_lib.accumulate(grid_to_pos(mv.astype(np.int32), w.box), *args)
        assert np.array_equal(H, H0), name
        assert np.array_equal(st, st0), name
    two = np.stack([m, m]).astype(np.int32)
    H2, st2 = oracle_lib.accumulate(grid_to_pos(two, w.box), *args)
    assert np.array_equal(H2, 2 * H0) and int(st2[0]) == 2 and int(st2[1]) == 2 * int(st0[1])


def test_quantise_snaps_and_wraps(oracle_lib):
    box = 9.93652
    mgrid = np.array([[0, 1, GRID - 1], [HALF, 12345, 777777]], dtype=np.int32)
    pos = grid_to_pos(mgrid, box)
    assert np.array_equal(oracle_lib.quantise(pos, box), mgrid)
    # any real value is wrapped into the box (8(b) "Units"); off-grid values snap to the nearest point
    shifted = pos + np.array([box, -box, 3 * box])
    assert np.array_equal(oracle_lib.quantise(shifted, box), mgrid)
    off = pos + 0.3 * box / GRID
    assert np.array_equal(oracle_lib.quantise(off, box), mgrid)


@pytest.mark.parametrize("widx", [1, 2, 3, 4, 5])
def test_thresholds_against_exact_rationals(oracle_lib, widx):
    """T[b] must be ceil of the fp64 expression as written (S1), and that expression must be the
    squared bin edge: compare with exact rational arithmetic on the (exactly rational) doubles."""
    w = WORKLOADS[widx]
    T_r, T_t = oracle_lib.thresholds(w.box, w.r_max, w.n_r, w.n_t)
    P_r, P_t = py_thresholds(w.box, w.r_max, w.n_r, w.n_t)
    assert [int(v) for v in T_r] == P_r and [int(v) for v in T_t] == P_t
    L, R = Fraction(w.box), Fraction(w.r_max)
    differ = 0
    for T, nb, span in ((T_r, w.n_r, R), (T_t, w.n_t, 2 * R)):
        assert int(T[0]) == 0 and all(int(T[i]) < int(T[i + 1]) for i in range(nb))
        for b in range(nb + 1):
            edge = Fraction(b, nb) * span * GRID / L           # exact real edge in grid units
            exact = math.ceil(edge * edge)
            assert abs(int(T[b]) - exact) <= 1
            differ += int(T[b]) != exact
    assert differ <= 2        # informational bound: fp64 rounding may move an edge that is ~integer


def test_cells_equals_allpairs_on_config4_frame(oracle_lib):
    w = WORKLOADS[4]
    m, pos = frames(w, 1)
    sub = pos[:, :8192]          # 8192 of the sites in the full box: sparse cells, some empty
    Ha, sa = oracle_lib.accumulate(sub, w.box, w.r_max, w.n_r, w.n_t, "allpairs")
    Hc, sc = oracle_lib.accumulate(sub, w.box, w.r_max, w.n_r, w.n_t, "cells")
    assert np.array_equal(Ha, Hc) and np.array_equal(sa, sc)
    assert Ha.sum() > 0
