"""Pins for the oracle's normalisation (S5): bin volumes V_abc and g3 = H / (F N rho^2 V_abc).

The paper gives only Eq. 3 and defers the rest to its refs; the
formula is reading Q8/Q9 of SURVEY.md 8(c).  Every expected value here comes from a closed form,
a textbook result or an independent quadrature, never from the oracle.
"""
import math

import numpy as np
import pytest
from scipy import integrate

from workloads import GRID, grid_to_pos, uniform_frame

CASES = [(0.7, 16, 16), (1.0, 12, 24), (2.5, 8, 8), (0.6, 9, 7)]


@pytest.mark.parametrize("r_max,n_r,n_t", CASES)
def test_row_sums_total_symmetry(oracle_lib, r_max, n_r, n_t):
    V = oracle_lib.volumes(r_max, n_r, n_t)
    w = r_max / n_r
    e3 = (np.arange(1, n_r + 1) * w) ** 3 - (np.arange(n_r) * w) ** 3
    rows = (4 * math.pi / 3) ** 2 * e3[:, None] * e3[None, :]      # both shells, any r_jk
    assert np.allclose(V.sum(-1), rows, rtol=2e-14, atol=0)
    assert math.isclose(V.sum(), (4 * math.pi * r_max ** 3 / 3) ** 2, rel_tol=1e-14)
    assert np.allclose(V, V.transpose(1, 0, 2), rtol=1e-13, atol=0)
    assert (V >= 0).all()


@pytest.mark.parametrize("r_max,n_r,n_t", CASES)
def test_interior_closed_form_and_support(oracle_lib, r_max, n_r, n_t):
    """bins wholly inside |r-s| <= t <= r+s have V = pi^2 D(r^2) D(s^2) D(t^2);
    bins wholly outside have V = 0."""
    V = oracle_lib.volumes(r_max, n_r, n_t)
    w, wt = r_max / n_r, 2 * r_max / n_t
    n_in = n_out = 0
    for a in range(n_r):
        for b in range(n_r):
            for c in range(n_t):
                r0, r1, s0, s1, t0, t1 = a * w, (a + 1) * w, b * w, (b + 1) * w, c * wt, (c + 1) * wt
                dmax = max(r1 - s0, s1 - r0)                    # max |r-s| over the cell
                dmin = max(r0 - s1, s0 - r1, 0.0)               # min |r-s|
                if t0 >= dmax and t1 <= r0 + s0:
                    exact = math.pi ** 2 * (r1 ** 2 - r0 ** 2) * (s1 ** 2 - s0 ** 2) * (t1 ** 2 - t0 ** 2)
                    assert math.isclose(V[a, b, c], exact, rel_tol=1e-13)
                    n_in += 1
                if t1 <= dmin * (1 - 1e-12) or t0 >= (r1 + s1) * (1 + 1e-12):
                    assert V[a, b, c] == 0.0
                    n_out += 1
    assert n_in > 0 and n_out > 0


def lens(d, S, T):
    """textbook volume of the intersection of spheres of radii S and T whose centres are d apart"""
    if d >= S + T:
        return 0.0
    if d <= abs(S - T):
        return 4 * math.pi / 3 * min(S, T) ** 3
    return math.pi * (S + T - d) ** 2 * (d * d + 2 * d * (S + T) - 3 * (S - T) ** 2) / (12 * d)


@pytest.mark.parametrize("r_max,n_r,n_t", [(0.7, 8, 8), (1.0, 6, 12)])
def test_cumulative_against_sphere_lens(oracle_lib, r_max, n_r, n_t):
    """sum_{b<B, c<C} V[a,b,c] = int_{shell a} 4 pi r^2 lens(r; S=B w, T=C wt) dr :
    k lies within S of the centre and within T of j, j on a shell of radius r."""
    V = oracle_lib.volumes(r_max, n_r, n_t)
    w, wt = r_max / n_r, 2 * r_max / n_t
    cum = V.cumsum(1).cumsum(2)
    for a in range(n_r):
        for B in range(1, n_r + 1):
            for C in range(1, n_t + 1):
                S, T = B * w, C * wt
                pts = sorted(p for p in {abs(S - T), S + T} if a * w < p < (a + 1) * w)
                val, _ = integrate.quad(lambda r: 4 * math.pi * r * r * lens(r, S, T), a * w, (a + 1) * w,
                                        points=pts or None, epsabs=0, epsrel=1e-13, limit=200)
                assert math.isclose(cum[a, B - 1, C - 1], val, rel_tol=2e-11, abs_tol=1e-15 * r_max ** 6)


def test_boundary_bins_against_adaptive_quadrature(oracle_lib):
    """a few bins cut by t = r+s or t = |r-s|: nested adaptive quadrature of 8 pi^2 r s t."""
    r_max, n_r, n_t = 1.0, 5, 5
    V = oracle_lib.volumes(r_max, n_r, n_t)
    w, wt = r_max / n_r, 2 * r_max / n_t

    def direct(a, b, c):
        t0, t1 = c * wt, (c + 1) * wt

        def inner(s, r):
            lo, hi = max(t0, abs(r - s)), min(t1, r + s)
            return 0.0 if hi <= lo else 8 * math.pi ** 2 * r * s * 0.5 * (hi * hi - lo * lo)
        val, _ = integrate.dblquad(inner, a * w, (a + 1) * w, b * w, (b + 1) * w, epsabs=1e-13, epsrel=1e-10)
        return val
    for (a, b, c) in [(0, 0, 0), (1, 0, 0), (2, 2, 0), (4, 0, 1), (4, 4, 4), (3, 1, 2), (0, 3, 1), (2, 4, 3)]:
        assert math.isclose(V[a, b, c], direct(a, b, c), rel_tol=1e-7, abs_tol=1e-12), (a, b, c)


def test_normalise_formula(oracle_lib):
    """g3 = H / (F N rho^2 V) with rho = N / L^3; 0 where V = 0 (Eq. 3's rho^3 convention, Q9)."""
    H = np.array([[[5, 0], [7, 3]], [[7, 3], [11, 2]]], dtype=np.uint64)
    V = np.array([[[0.5, 0.0], [0.25, 2.0]], [[0.25, 2.0], [1.0, 4.0]]])
    F, N, L = 3, 10, 2.0
    g3 = oracle_lib.normalise(H, V, F, N, L)
    rho = N / L ** 3
    with np.errstate(divide="ignore", invalid="ignore"):
        expect = np.where(V > 0, H / (F * N * rho * rho * V), 0.0)
    assert np.allclose(g3, expect, rtol=1e-15, atol=0)
    assert g3[0, 0, 1] == 0.0


@pytest.mark.parametrize("n,box,r_max,n_r,n_t,n_frames", [
    (1000, 10.0, 2.0, 8, 8, 40),        # r_max < L/4
    (40, 6.0, 2.5, 4, 4, 400),          # r_max > L/4: holds only with the no-re-wrap reading (Q3)
])
def test_ideal_gas_is_flat(oracle_lib, n, box, r_max, n_r, n_t, n_frames):
    """uniform random positions: every bin has g3 = (1 - 1/N)(1 - 2/N) within statistical error.
    Per-bin mean and standard error across independent frames; |z| < 6 on bins with >= 100 counts."""
    V = oracle_lib.volumes(r_max, n_r, n_t)
    per_frame = []
    total = np.zeros((n_r, n_r, n_t), dtype=np.uint64)
    for f in range(n_frames):
        m = uniform_frame(n, seed=9000 + f)
        H, _ = oracle_lib.accumulate(grid_to_pos(m, box), box, r_max, n_r, n_t, "cells")
        total += H
        per_frame.append(oracle_lib.normalise(H, V, 1, n, box))
    g = np.stack(per_frame)
    expected = (1 - 1 / n) * (1 - 2 / n)
    sel = (total >= 100) & (V > 0)
    assert sel.sum() >= 0.25 * n_r * n_r * n_t
    mean = g.mean(0)[sel]
    sem = g.std(0, ddof=1)[sel] / math.sqrt(n_frames)
    z = (mean - expected) / sem
    assert np.abs(z).max() < 6.0, float(np.abs(z).max())
    # pooled: the count-weighted average must sit on the expected value far more tightly
    pooled = oracle_lib.normalise(total, V, n_frames, n, box)
    wts = V[sel]
    assert abs(np.average(pooled[sel], weights=wts) - expected) < 5e-3 * expected
