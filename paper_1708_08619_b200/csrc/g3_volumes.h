// g3_volumes.h -- exact bin volumes V_abc for the normalisation (host code, plan creation).
//
// g(3) is the triplet density divided by its ideal-gas value (Eq. 3).
// For an ideal gas of density rho, the expected number of ordered neighbour pairs (j,k) of
// one centre with (r_ij, r_ik, r_jk) in a bin is rho^2 V_abc with
//     V_abc = integral over the bin of  8 pi^2 r s t  [ |r-s| <= t <= r+s ]  dr ds dt
// (DESIGN.md section 2.5).  The bin edges are rational multiples of r_max, so on a common
// lattice of spacing u all edges are integers and V_abc / (pi^2 u^6 / 18) is an INTEGER,
// evaluated here without rounding in 128-bit arithmetic:
//     [ |r-s| <= t <= r+s ] = 1 - [t > r+s] - [r > s+t] - [s > r+t]      (almost everywhere)
//     int_box r s t            = D(r^2) D(s^2) D(t^2) / 8
//     int_box x y z [z > x+y]  = sum over the 8 corners (+-) Q(X,Y,Z),
//     Q(X,Y,Z) = int_0^X int_0^Y x y (Z^2 - (x+y)^2)/2 [x+y < Z] dy dx, which after clipping
//     X,Y to Z is a polynomial:  144 Q = 18 X^2 Y^2 Z^2 - 9 X^4 Y^2 - 16 X^3 Y^3 - 9 X^2 Y^4
//     if X+Y <= Z, and 144 Q = -phi(X,Z) - phi(Y,Z) - Z^6 otherwise, with
//     phi(X,Z) = X^6 - 9 X^4 Z^2 + 16 X^3 Z^3 - 9 X^2 Z^4.
#pragma once

#include <stdint.h>

#include <cmath>
#include <vector>

namespace g3 {

typedef __int128 i128;

inline i128 vol_phi(i128 X, i128 Z) {
    i128 X2 = X * X, Z2 = Z * Z;
    return X2 * (X2 * X2 - 9 * X2 * Z2 + 16 * X * Z2 * Z - 9 * Z2 * Z2);
}

inline i128 vol_Q144(i128 X, i128 Y, i128 Z) {
    if (X <= 0 || Y <= 0 || Z <= 0) return 0;
    if (X > Z) X = Z;
    if (Y > Z) Y = Z;
    i128 X2 = X * X, Y2 = Y * Y, Z2 = Z * Z;
    if (X + Y <= Z) return X2 * Y2 * (18 * Z2 - 9 * X2 - 16 * X * Y - 9 * Y2);
    return -vol_phi(X, Z) - vol_phi(Y, Z) - Z2 * Z2 * Z2;
}

// 144 * integral over [x0,x1] x [y0,y1] x [z0,z1] of x y z [z > x+y]
inline i128 vol_P144(int64_t x0, int64_t x1, int64_t y0, int64_t y1, int64_t z0, int64_t z1) {
    const int64_t xs[2] = {x0, x1}, ys[2] = {y0, y1}, zs[2] = {z0, z1};
    i128 s = 0;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j)
            for (int k = 0; k < 2; ++k) {
                i128 q = vol_Q144(xs[i], ys[j], zs[k]);
                s += ((i + j + k) & 1) ? q : -q;      // sign (-1)^(3 - i - j - k)
            }
    return s;
}

inline int64_t vol_gcd(int64_t a, int64_t b) { while (b) { int64_t t = a % b; a = b; b = t; } return a; }

// Fills V [n_r][n_r][n_t] (c fastest) in (unit of r_max)^6.  Returns false if the lattice
// would overflow 128-bit arithmetic (coprime bin counts near the 1024 limit).
inline bool bin_volumes(double r_max, int32_t n_r, int32_t n_t, std::vector<double>& V) {
    const int64_t g = vol_gcd(n_t, 2ll * n_r);
    const int64_t p = n_t / g;            // r and s edges: a * p lattice units
    const int64_t q = 2ll * n_r / g;      // t edges:       c * q lattice units
    const long double top = (long double)(n_t * q > n_r * p ? n_t * q : n_r * p);
    if (6.0L * std::log2(top) + 12.0L > 126.0L) return false;
    const double u = (r_max / (double)n_r) / (double)p;
    const double pi = 3.14159265358979323846;
    const double scale = pi * pi / 18.0 * (u * u * u) * (u * u * u);
    V.assign((size_t)n_r * n_r * n_t, 0.0);
    for (int32_t a = 0; a < n_r; ++a)
        for (int32_t b = a; b < n_r; ++b)
            for (int32_t c = 0; c < n_t; ++c) {
                const int64_t r0 = a * p, r1 = (a + 1) * p, s0 = b * p, s1 = (b + 1) * p;
                const int64_t t0 = c * q, t1 = (c + 1) * q;
                i128 N = (i128)18 * (r1 * r1 - r0 * r0) * (s1 * s1 - s0 * s0) * (i128)(t1 * t1 - t0 * t0)
                         - vol_P144(r0, r1, s0, s1, t0, t1)     // t > r + s
                         - vol_P144(s0, s1, t0, t1, r0, r1)     // r > s + t
                         - vol_P144(r0, r1, t0, t1, s0, s1);    // s > r + t
                const double v = (double)N * scale;
                V[((size_t)a * n_r + b) * n_t + c] = v;
                V[((size_t)b * n_r + a) * n_t + c] = v;          // V_abc = V_bac
            }
    return true;
}

}  // namespace g3
