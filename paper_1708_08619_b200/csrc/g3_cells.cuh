// g3_cells.cuh -- per-frame cell list: quantise + count, exclusive scan, scatter.
//
// Step a1/a2 of DESIGN.md.  Not in the paper: its CUDA_g2 scans all N particles per
// centre.  The cell list is an integer counting sort keyed by
// cell id; the rank of a particle inside its cell is the value returned by the
// atomic that counts it, so no second pass over the keys is needed.  The order
// of particles inside a cell depends on the atomics' arrival order; the histogram
// does not (integer sums over an unordered set).
#pragma once

#include "g3_plan.h"

namespace g3 {

__device__ __forceinline__ int32_t quantise_coord(double x, double inv_g, bool& bad) {
    // m = llrint(x * 2^20/box) mod 2^20; one IEEE multiply, round-to-nearest-even conversion
    const double s = __dmul_rn(x, inv_g);
    // NaN, infinities and values the 64-bit conversion would saturate have no grid point
    if (!(fabs(s) < 4611686018427387904.0)) bad = true;
    long long q = __double2ll_rn(s);
    return (int32_t)(q & (kGrid - 1));
}

__device__ __forceinline__ int32_t cell_of(int32_t m, int32_t ncell) {
    return (int32_t)(((uint32_t)m * (uint32_t)ncell) >> kGridBits);   // m < 2^20, ncell <= 32
}

// One thread per (frame, particle).  Reads fp64 [n][3] rows; a warp reads 32 consecutive
// rows = 768 contiguous bytes.  Writes (x, y, z, cell) and the particle's rank in its cell.
__global__ void __launch_bounds__(256)
quantise_count_kernel(const double* __restrict__ pos, long long frame_stride, int32_t n,
                      int32_t n_frames, double inv_g, int32_t ncell,
                      int4* __restrict__ staged, int32_t* __restrict__ slot,
                      int32_t* __restrict__ cell_count, unsigned long long* __restrict__ bad_count) {
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= (long long)n_frames * n) return;
    int32_t f = (int32_t)(g / n);
    int32_t p = (int32_t)(g - (long long)f * n);
    const double* x = pos + (long long)f * frame_stride + 3ll * p;
    bool bad = false;
    int32_t mx = quantise_coord(__ldg(x + 0), inv_g, bad);
    int32_t my = quantise_coord(__ldg(x + 1), inv_g, bad);
    int32_t mz = quantise_coord(__ldg(x + 2), inv_g, bad);
    if (bad) atomicAdd(bad_count, 1ull);               // sticky: g3_finalize returns G3_EINVAL
    int32_t cell = (cell_of(mx, ncell) * ncell + cell_of(my, ncell)) * ncell + cell_of(mz, ncell);
    int32_t ncell3 = ncell * ncell * ncell;
    int32_t s = atomicAdd(cell_count + (long long)f * ncell3 + cell, 1);
    staged[g] = make_int4(mx, my, mz, cell);
    slot[g] = s;
}

// One block per frame: exclusive scan of the cell counts into cell_start[f][0..ncell3].
__global__ void __launch_bounds__(1024)
cell_scan_kernel(const int32_t* __restrict__ cell_count, int32_t* __restrict__ cell_start,
                 int32_t ncell3) {
    __shared__ int32_t warp_sums[32];
    __shared__ int32_t carry_s;
    const int32_t* cnt = cell_count + (long long)blockIdx.x * ncell3;
    int32_t* start = cell_start + (long long)blockIdx.x * (ncell3 + 1);
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int32_t base = 0; base < ncell3; base += blockDim.x) {
        int32_t i = base + threadIdx.x;
        int32_t v = i < ncell3 ? cnt[i] : 0;
        int32_t incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int32_t t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        if (lane == 31) warp_sums[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            int32_t ws = warp_sums[lane];
            int32_t wincl = ws;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                int32_t t = __shfl_up_sync(0xffffffffu, wincl, d);
                if (lane >= d) wincl += t;
            }
            warp_sums[lane] = wincl - ws;     // exclusive prefix of the warp sums
        }
        __syncthreads();
        int32_t carry = carry_s;
        if (i < ncell3) start[i] = carry + warp_sums[wid] + incl - v;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry_s = carry + warp_sums[wid] + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) start[ncell3] = carry_s;
}

// One thread per (frame, particle): counting-sort scatter; also clears the counts for the next batch.
__global__ void __launch_bounds__(256)
cell_scatter_kernel(const int4* __restrict__ staged, const int32_t* __restrict__ slot,
                    const int32_t* __restrict__ cell_start, int32_t n, int32_t n_frames,
                    int32_t ncell3, int4* __restrict__ sorted, float4* __restrict__ sortedf) {
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= (long long)n_frames * n) return;
    int32_t f = (int32_t)(g / n);
    int4 v = staged[g];
    int32_t dst = cell_start[(long long)f * (ncell3 + 1) + v.w] + slot[g];
    sorted[(long long)f * n + dst] = v;
    sortedf[(long long)f * n + dst] = make_float4((float)v.x, (float)v.y, (float)v.z, 0.f);
}

}  // namespace g3
