// g3_msd.cuh -- mean square displacement over all time origins: Eq. 5
// (PAPER.md:638), Algorithm 11 CUDA_msd: "dt and atom index is obtained from
// thread-id", loop over the origins t, "Accumulate local MSD data", "Update global MSD array".
//
// Here: a CTA owns 32 atoms (lane = atom) and each of its warps a set of lags dt (strided, so the
// (F - dt) origins per lag balance out).  The unwrapped positions are snapped to the box/2^20 grid
// once (m = llrint(x 2^20 / box), no wrap: DESIGN.md reading M1) and every squared displacement
// is an exact integer, accumulated in 128 bits (M2).
//   msd_kernel          the 32 trajectories of the CTA are staged in shared memory as int32
//                       [F][32][3] (lane stride 3 words: conflict-free), so HBM is read once:
//                       F x 400 B must fit shared memory (F <= ~580); squares through a prefix
//                       table, cross terms with four adjacent lags per warp (see the kernel);
//   msd_direct_kernel   longer trajectories: the direct loops (four strided lags per warp share
//                       the origin loads) over a snapped int32 copy in global memory ([F][n][3],
//                       written by msd_snap_kernel).
// A warp sums its 32 atoms with shuffles and writes one 128-bit partial per (CTA, lag);
// msd_reduce_kernel adds the partials of a lag and evaluates msd[dt] in fp64 (M3).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace g3 {

constexpr int kMsdWarps = 16;
constexpr int kMsdAtoms = 32;
constexpr int kMsdLags = 8;                    // adjacent lags a warp of msd_kernel takes together

struct MsdParams {
    const double* pos;                    // [F][stride] fp64, atom-major rows of 3
    long long stride;                     // doubles between frames
    int32_t n, n_frames, max_lag;
    double inv_g;
    int32_t* snapped;                     // [F][n][3] (global path only)
    ulonglong2* partial;                  // [n_blocks][max_lag + 1] (lo, hi)
    unsigned long long* bad;              // coordinates outside +-2^30 grid units
};

__device__ __forceinline__ int32_t msd_snap(double x, double inv_g, unsigned long long& bad) {
    const double s = __dmul_rn(x, inv_g);
    const long long m = __double2ll_rn(s);                 // saturates; NaN fails the range test below
    if (!(s == s) || m >= (1ll << 30) || m <= -(1ll << 30)) { bad += 1; return 0; }
    return (int32_t)m;
}

__global__ void __launch_bounds__(256)
msd_snap_kernel(MsdParams mp) {
    const long long per_frame = 3ll * mp.n, total = per_frame * mp.n_frames;
    unsigned long long bad = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < total;
         q += (long long)gridDim.x * blockDim.x) {
        const long long f = q / per_frame, r = q - f * per_frame;
        mp.snapped[q] = msd_snap(mp.pos[f * mp.stride + r], mp.inv_g, bad);
    }
    if (bad) atomicAdd(mp.bad, bad);
}

// 128-bit helpers on (lo, hi) pairs, arithmetic mod 2^128
__device__ __forceinline__ void u128_add(unsigned long long& lo, unsigned long long& hi, unsigned long long alo,
                                         unsigned long long ahi) {
    lo += alo;
    hi += ahi + (lo < alo ? 1ull : 0ull);
}

__device__ __forceinline__ void u128_sub(unsigned long long& lo, unsigned long long& hi, unsigned long long alo,
                                         unsigned long long ahi) {
    const unsigned long long borrow = lo < alo ? 1ull : 0ull;
    lo -= alo;
    hi -= ahi + borrow;
}

// add the sign-extended 64-bit value s
__device__ __forceinline__ void u128_add_s64(unsigned long long& lo, unsigned long long& hi, long long s) {
    u128_add(lo, hi, (unsigned long long)s, (unsigned long long)(s >> 63));
}

// msd_kernel: trajectories of 32 atoms staged in shared memory (F x 384 B + the prefix table).
//   sum_t |r(t+dt) - r(t)|^2 = sum_t |r(t+dt)|^2 + sum_t |r(t)|^2 - 2 sum_t r(t+dt).r(t)
// The first two sums are differences of ONE prefix table P[t] = sum_{u<t} sum_atoms |r(u)|^2 per
// CTA (O(F) work); only the cross term needs all (origin, lag) pairs: three multiply-adds per
// displacement.  |m| < 2^30, so a dot product is below 3 * 2^60 and two of them fit a signed
// 64-bit word before they are folded into a 128-bit sum; every quantity is an exact integer and
// the result is the same 128-bit sum as the direct evaluation (reading M2).
// A warp takes kMsdLags ADJACENT lags: moving the origin by one frame shifts their windows by one
// frame, so each step loads one new origin and one new end point (6 LDS for kMsdLags displacements).
__global__ void __launch_bounds__(kMsdWarps * 32)
msd_kernel(MsdParams mp) {
    extern __shared__ __align__(16) int32_t msd_traj[];    // [F][32][3], then ulonglong2 P[F + 1]
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t atom = blockIdx.x * kMsdAtoms + lane;
    const bool valid = atom < mp.n;
    const int32_t F = mp.n_frames;
    ulonglong2* P = reinterpret_cast<ulonglong2*>(msd_traj + (size_t)F * kMsdAtoms * 3);
    __shared__ unsigned int range_s;                      // OR of |m| over the CTA's coordinates
    if (threadIdx.x == 0) range_s = 0;
    __syncthreads();
    {
        unsigned long long bad = 0;
        unsigned int range = 0;
        for (int32_t t0 = wid; t0 < F; t0 += 4 * kMsdWarps) {
            double x[4][3];                                // four frames per pass: their loads are in flight together
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int32_t tu = min(t0 + u * kMsdWarps, F - 1);
                const double* row = mp.pos + (long long)tu * mp.stride + 3ll * atom;
#pragma unroll
                for (int c = 0; c < 3; ++c) x[u][c] = valid ? row[c] : 0.0;
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
            const int32_t t = t0 + u * kMsdWarps;
            if (t >= F) break;                             // uniform over the warp
            int32_t m[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                m[c] = valid ? msd_snap(x[u][c], mp.inv_g, bad) : 0;
                msd_traj[(t * kMsdAtoms + lane) * 3 + c] = m[c];
                range |= (unsigned int)abs(m[c]);
            }
            // sum over the CTA's atoms of |r(t)|^2 (< 32 * 3 * 2^60): 32-bit halves summed in 64 bits
            const unsigned long long q = (unsigned long long)((long long)m[0] * m[0]) + (unsigned long long)((long long)m[1] * m[1]) +
                                         (unsigned long long)((long long)m[2] * m[2]);
            unsigned long long ql = q & 0xFFFFFFFFull, qh = q >> 32;
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                ql += __shfl_xor_sync(0xffffffffu, ql, d);
                qh += __shfl_xor_sync(0xffffffffu, qh, d);
            }
            if (lane == 0) {
                unsigned long long lo = ql, hi = 0;
                u128_add(lo, hi, qh << 32, qh >> 32);
                P[t + 1] = make_ulonglong2(lo, hi);
            }
            }
        }
        if (bad) atomicAdd(mp.bad, bad);
        range = __reduce_or_sync(0xffffffffu, range);
        if (lane == 0) atomicOr(&range_s, range);
    }
    __syncthreads();
    // |m| < 2^28 for every coordinate of this CTA: a dot product is below 3 * 2^56 and 32 of them
    // fit a signed 64-bit word, so the 128-bit fold runs once per 32 origins instead of once per 2
    const bool narrow = range_s < (1u << 28);
    if (threadIdx.x == 0) {                               // exclusive prefix over the frames
        unsigned long long lo = 0, hi = 0;
        P[0] = make_ulonglong2(0ull, 0ull);
        for (int32_t t = 1; t <= F; ++t) {
            const ulonglong2 v = P[t];
            u128_add(lo, hi, v.x, v.y);
            P[t] = make_ulonglong2(lo, hi);
        }
    }
    __syncthreads();

    const int32_t* base = msd_traj + lane * 3;             // element (t, this atom, c) = base[t * 96 + c]
    constexpr int32_t TS = kMsdAtoms * 3;
    constexpr int L = kMsdLags;                             // adjacent lags per warp pass (a power of two)
    const int32_t n_groups = (mp.max_lag + L) / L;
    for (int32_t grp = wid; grp < n_groups; grp += kMsdWarps) {
        const int32_t d0 = grp * L;
        unsigned long long lo[L], hi[L];
#pragma unroll
        for (int jj = 0; jj < L; ++jj) { lo[jj] = 0; hi[jj] = 0; }
        const int32_t n_full = F - d0 - (L - 1);           // origins for which all L lags exist
        int32_t t = 0;
        if (n_full >= L) {
            int32_t bx[L], by[L], bz[L];                   // b[x & (L-1)] = r(t + d0 + x) for the L lags of a step
#pragma unroll
            for (int x = 0; x < L - 1; ++x) {
                const int32_t* b = base + (d0 + x) * TS;
                bx[x] = b[0]; by[x] = b[1]; bz[x] = b[2];
            }
            long long acc[L];
#pragma unroll
            for (int jj = 0; jj < L; ++jj) acc[jj] = 0;
            const int32_t* a = base;
            const int32_t* e = base + (d0 + L - 1) * TS;
            // one origin: load r(t + i) and the new end point r(t + i + d0 + L - 1), L dot products
            auto step = [&](int i) {
                const int32_t ax = a[i * TS], ay = a[i * TS + 1], az = a[i * TS + 2];
                bx[(i + L - 1) & (L - 1)] = e[i * TS]; by[(i + L - 1) & (L - 1)] = e[i * TS + 1]; bz[(i + L - 1) & (L - 1)] = e[i * TS + 2];
#pragma unroll
                for (int jj = 0; jj < L; ++jj)
                    acc[jj] += (long long)ax * bx[(i + jj) & (L - 1)] + (long long)ay * by[(i + jj) & (L - 1)] +
                               (long long)az * bz[(i + jj) & (L - 1)];
            };
            auto fold = [&]() {
#pragma unroll
                for (int jj = 0; jj < L; ++jj) { u128_add_s64(lo[jj], hi[jj], acc[jj]); acc[jj] = 0; }
            };
            if (narrow) {                                   // 32 origins per fold
                for (; t + 32 <= n_full; t += 32) {
#pragma unroll 1
                    for (int u = 0; u < 32 / L; ++u) {
#pragma unroll
                        for (int i = 0; i < L; ++i) step(i);
                        a += L * TS; e += L * TS;
                    }
                    fold();
                }
            }
            for (; t + L <= n_full; t += L) {               // two origins per fold
#pragma unroll
                for (int i = 0; i < L; i += 2) { step(i); step(i + 1); fold(); }
                a += L * TS; e += L * TS;
            }
        }
        // the remaining origins (fewer than L, plus those that exist only for the shorter lags)
        for (; t < F - d0; ++t) {
            const int32_t* a = base + t * TS;
            const int32_t ax = a[0], ay = a[1], az = a[2];
#pragma unroll
            for (int jj = 0; jj < L; ++jj) {
                if (t + d0 + jj < F) {
                    const int32_t* b = a + (d0 + jj) * TS;
                    u128_add_s64(lo[jj], hi[jj], (long long)ax * b[0] + (long long)ay * b[1] + (long long)az * b[2]);
                }
            }
        }
#pragma unroll
        for (int jj = 0; jj < L; ++jj) {
            const int32_t dt = d0 + jj;
            if (dt > mp.max_lag) break;                    // uniform over the warp
            unsigned long long l = lo[jj], h = hi[jj];     // cross term of this lane's atom
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                const unsigned long long olo = __shfl_xor_sync(0xffffffffu, l, d);
                const unsigned long long ohi = __shfl_xor_sync(0xffffffffu, h, d);
                l += olo;
                h += ohi + (l < olo ? 1ull : 0ull);
            }
            if (lane == 0) {
                // S = P[F - dt] + (P[F] - P[dt]) - 2 C
                const ulonglong2 p1 = P[F - dt], p2 = P[F], p3 = P[dt];
                unsigned long long slo = p1.x, shi = p1.y;
                u128_add(slo, shi, p2.x, p2.y);
                u128_sub(slo, shi, p3.x, p3.y);
                u128_sub(slo, shi, l, h);
                u128_sub(slo, shi, l, h);
                mp.partial[(size_t)blockIdx.x * (mp.max_lag + 1) + dt] = make_ulonglong2(slo, shi);
            }
        }
    }
}

__global__ void __launch_bounds__(kMsdWarps * 32)
msd_direct_kernel(MsdParams mp) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t atom = blockIdx.x * kMsdAtoms + lane;
    const bool valid = atom < mp.n;
    const int32_t F = mp.n_frames;
    // element (t, this atom, c) of the snapped copy: global [t][atom][c]
    const int32_t* base = mp.snapped + 3ll * (valid ? atom : 0);
    const long long tstride = 3ll * mp.n;
    // Four lags per pass share the loads of the origin r(t): lags dt, dt + W, dt + 2W, dt + 3W.
    // |m| < 2^30, so a displacement component fits int32 and its square is one 32 x 32 -> 64 multiply.
    auto sq = [](int32_t dx, int32_t dy, int32_t dz) {
        return (unsigned long long)((long long)dx * dx) + (unsigned long long)((long long)dy * dy) +
               (unsigned long long)((long long)dz * dz);
    };
    for (int32_t dt0 = wid; dt0 <= mp.max_lag; dt0 += 4 * kMsdWarps) {
        unsigned long long lo[4] = {0, 0, 0, 0}, hi[4] = {0, 0, 0, 0};
        int32_t cnt[4];                                     // origins of each of the four lags
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int32_t dt = dt0 + j * kMsdWarps;
            cnt[j] = dt <= mp.max_lag ? F - dt : 0;
        }
        const int32_t* a = base;
        int32_t t = 0;
        for (; t < cnt[3]; ++t) {                          // all four lags have this origin
            const int32_t ax = a[0], ay = a[1], az = a[2];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int32_t* b = a + (long long)(dt0 + j * kMsdWarps) * tstride;
                const unsigned long long s = sq(b[0] - ax, b[1] - ay, b[2] - az);
                lo[j] += s;
                hi[j] += lo[j] < s ? 1ull : 0ull;
            }
            a += tstride;
        }
        for (; t < cnt[0]; ++t) {                          // tails: fewer origins for the longer lags
            const int32_t ax = a[0], ay = a[1], az = a[2];
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                if (t < cnt[j]) {
                    const int32_t* b = a + (long long)(dt0 + j * kMsdWarps) * tstride;
                    const unsigned long long s = sq(b[0] - ax, b[1] - ay, b[2] - az);
                    lo[j] += s;
                    hi[j] += lo[j] < s ? 1ull : 0ull;
                }
            }
            a += tstride;
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int32_t dt = dt0 + j * kMsdWarps;
            if (dt > mp.max_lag) break;                    // uniform over the warp
            unsigned long long l = valid ? lo[j] : 0ull, h = valid ? hi[j] : 0ull;
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                const unsigned long long olo = __shfl_xor_sync(0xffffffffu, l, d);
                const unsigned long long ohi = __shfl_xor_sync(0xffffffffu, h, d);
                l += olo;
                h += ohi + (l < olo ? 1ull : 0ull);
            }
            if (lane == 0) mp.partial[(size_t)blockIdx.x * (mp.max_lag + 1) + dt] = make_ulonglong2(l, h);
        }
    }
}

// A block per 32 lags, 32 x 8 threads: thread (x, y) adds the per-CTA partials (128-bit) y, y + 8, ..
// of lag 32 blockIdx + x (coalesced over x), the eight slices are added through shared memory,
// and row 0 writes (lo, hi) and msd[dt] (reading M3).
__global__ void __launch_bounds__(256)
msd_reduce_kernel(const ulonglong2* __restrict__ partial, int32_t n_blocks, int32_t max_lag, int32_t n,
                  int32_t n_frames, double gg, unsigned long long* __restrict__ sums, double* __restrict__ msd) {
    __shared__ ulonglong2 slice[8][32];
    const int x = threadIdx.x & 31, y = threadIdx.x >> 5;
    const int32_t dt = blockIdx.x * 32 + x;
    unsigned long long lo = 0, hi = 0;
    if (dt <= max_lag)
        for (int32_t b = y; b < n_blocks; b += 8) {
            const ulonglong2 p = partial[(size_t)b * (max_lag + 1) + dt];
            lo += p.x;
            hi += p.y + (lo < p.x ? 1ull : 0ull);
        }
    slice[y][x] = make_ulonglong2(lo, hi);
    __syncthreads();
    if (y != 0 || dt > max_lag) return;
    for (int r = 1; r < 8; ++r) {
        const ulonglong2 p = slice[r][x];
        lo += p.x;
        hi += p.y + (lo < p.x ? 1ull : 0ull);
    }
    if (sums) { sums[2 * dt] = lo; sums[2 * dt + 1] = hi; }
    if (msd) {
        const double s = __dadd_rn(__dmul_rn((double)hi, 18446744073709551616.0), (double)lo);
        const double num = __dmul_rn(s, gg);
        const double den = __dmul_rn((double)n, (double)(n_frames - dt));
        msd[dt] = __ddiv_rn(num, den);
    }
}

}  // namespace g3
