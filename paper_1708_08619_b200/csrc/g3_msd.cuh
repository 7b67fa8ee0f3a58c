// g3_msd.cuh -- mean square displacement over all time origins: Eq. 5
// (PAPER.md:638), Algorithm 11 CUDA_msd: "dt and atom index is obtained from
// thread-id", loop over the origins t, "Accumulate local MSD data", "Update global MSD array".
//
// Here: a CTA owns 32 atoms (lane = atom) and each of its warps a set of lags dt (strided, so the
// (F - dt) origins per lag balance out).  The unwrapped positions are snapped to the box/2^20 grid
// once (m = llrint(x 2^20 / box), no wrap: DESIGN.md reading M1) and every squared displacement
// is an exact integer, accumulated in 128 bits (M2).
//   msd_kernel<true>   the 32 trajectories of the CTA are staged in shared memory as int32
//                      [F][32][3] (lane stride 3 words: conflict-free), so HBM is read once:
//                      F x 384 B must fit shared memory (F <= ~590);
//   msd_kernel<false>  longer trajectories: the same loops over a snapped int32 copy in global
//                      memory ([F][n][3], written by msd_snap_kernel).
// A warp sums its 32 atoms with shuffles and writes one 128-bit partial per (CTA, lag);
// msd_reduce_kernel adds the partials of a lag and evaluates msd[dt] in fp64 (M3).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace g3 {

constexpr int kMsdWarps = 16;
constexpr int kMsdAtoms = 32;

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

template <bool kSmem>
__global__ void __launch_bounds__(kMsdWarps * 32)
msd_kernel(MsdParams mp) {
    extern __shared__ int32_t msd_traj[];                  // [F][32][3] (kSmem)
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t atom = blockIdx.x * kMsdAtoms + lane;
    const bool valid = atom < mp.n;
    const int32_t F = mp.n_frames;
    if (kSmem) {
        unsigned long long bad = 0;
        for (int32_t t = wid; t < F; t += kMsdWarps) {
            const double* row = mp.pos + (long long)t * mp.stride + 3ll * atom;
#pragma unroll
            for (int c = 0; c < 3; ++c)
                msd_traj[(t * kMsdAtoms + lane) * 3 + c] = valid ? msd_snap(row[c], mp.inv_g, bad) : 0;
        }
        if (bad) atomicAdd(mp.bad, bad);
        __syncthreads();
    }
    // element (t, this atom, c): shared [t][lane][c] or global [t][atom][c]
    const int32_t* base = kSmem ? msd_traj + lane * 3 : mp.snapped + 3ll * (valid ? atom : 0);
    const long long tstride = kSmem ? kMsdAtoms * 3 : 3ll * mp.n;
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

// One thread per lag: add the per-CTA partials (128-bit), write (lo, hi) and msd[dt] (reading M3).
__global__ void __launch_bounds__(128)
msd_reduce_kernel(const ulonglong2* __restrict__ partial, int32_t n_blocks, int32_t max_lag, int32_t n,
                  int32_t n_frames, double gg, unsigned long long* __restrict__ sums, double* __restrict__ msd) {
    const int32_t dt = blockIdx.x * blockDim.x + threadIdx.x;
    if (dt > max_lag) return;
    unsigned long long lo = 0, hi = 0;
    for (int32_t b = 0; b < n_blocks; ++b) {
        const ulonglong2 p = partial[(size_t)b * (max_lag + 1) + dt];
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
