// g3_generic.cuh -- generic exact triplet kernel (kernel 1).
//
// Works for every plan (any bin counts, any r_max < box/2, any neighbour count up to
// the plan's capacity: the per-warp neighbour list lives in shared memory when it fits and in a
// global-memory slice of the warp otherwise).  All arithmetic that decides a bin is 64-bit integer; bins
// are found by binary search in the squared-edge tables; the histogram is updated
// with 64-bit global atomics.  It is the slow, always-available path; the tiled
// kernel (g3_tiled.cuh) is the fast one.
//
// One warp per central particle i (steps a3 + a4 of DESIGN.md):
//   a3  walk the 27 cells around i (or all particles when the grid is degenerate),
//       keep j != i with |d_j|^2 < T_r[n_r], store (d_j, a_j) in shared memory
//       -- Algorithm 7 CUDA_g2 "store minimum image neighbour vectors";
//   a4  lane = neighbour j, loop over all k != j, t2 = |d_k - d_j|^2 from the stored
//       vectors, update counts[a_j][a_k][bin(t2)] -- Algorithm 7 CUDA_g3.
#pragma once

#include "g3_plan.h"

namespace g3 {

__device__ __forceinline__ int32_t wrap_component(int32_t d) {
    // ((d + 2^19) mod 2^20) - 2^19 for |d| < 2^20: keep the low 20 bits, sign-extend bit 19
    return (int32_t)((uint32_t)d << (32 - kGridBits)) >> (32 - kGridBits);
}

__device__ __forceinline__ int32_t bin_search(const unsigned long long* T, int32_t n,
                                              unsigned long long q) {
    int32_t lo = 0, hi = n;                 // largest b in [0, n] with T[b] <= q
    while (lo < hi) {
        int32_t mid = lo + ((hi - lo + 1) >> 1);
        if (T[mid] <= q) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// Enumerates the candidate ranges [begin, end) in the sorted frame for a centre in `cell`.
// ncell == 1: one range, the whole frame.  Otherwise 9 columns (x,y offsets); the three
// z-adjacent cells of a column are contiguous in the cell-major order unless they wrap.
struct CandidateRanges {
    int32_t n_ranges;
    __device__ __forceinline__ static int32_t count(int32_t ncell) { return ncell == 1 ? 1 : 18; }
    __device__ __forceinline__ static void get(int32_t r, int32_t cell, int32_t ncell, int32_t n,
                                               const int32_t* __restrict__ start,
                                               int32_t& begin, int32_t& end) {
        if (ncell == 1) { begin = 0; end = n; return; }
        int32_t cz = cell % ncell, cy = (cell / ncell) % ncell, cx = cell / (ncell * ncell);
        int32_t col = r >> 1, part = r & 1;
        int32_t ox = col / 3 - 1, oy = col % 3 - 1;
        int32_t x = cx + ox; x += x < 0 ? ncell : 0; x -= x >= ncell ? ncell : 0;
        int32_t y = cy + oy; y += y < 0 ? ncell : 0; y -= y >= ncell ? ncell : 0;
        int32_t base = (x * ncell + y) * ncell;
        int32_t z0 = cz - 1, z1 = cz + 1;          // inclusive
        if (z0 >= 0 && z1 < ncell) {               // no wrap: one range, second part empty
            if (part == 0) { begin = start[base + z0]; end = start[base + z1 + 1]; }
            else { begin = 0; end = 0; }
        } else if (z0 < 0) {                       // cells ncell-1 | 0, 1
            if (part == 0) { begin = start[base + 0]; end = start[base + 2]; }
            else { begin = start[base + ncell - 1]; end = start[base + ncell]; }
        } else {                                   // cells ncell-2, ncell-1 | 0
            if (part == 0) { begin = start[base + ncell - 2]; end = start[base + ncell]; }
            else { begin = start[base + 0]; end = start[base + 1]; }
        }
    }
};

template <int kWarps>
__global__ void __launch_bounds__(kWarps * 32)
generic_triplet_kernel(FrameBatch fb, BinSpec bs, int32_t max_nb, int4* nb_global,
                       unsigned long long* __restrict__ counts,
                       unsigned long long* __restrict__ counts2,
                       unsigned long long* __restrict__ stats) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned long long* sT_r = reinterpret_cast<unsigned long long*>(smem_raw);
    unsigned long long* sT_t = sT_r + (bs.n_r + 1);
    size_t off = ((size_t)(bs.n_r + bs.n_t + 2) * 8 + 15) & ~size_t(15);
    int4* nb_all = reinterpret_cast<int4*>(smem_raw + off);

    for (int32_t i = threadIdx.x; i <= bs.n_r; i += blockDim.x) sT_r[i] = bs.T_r[i];
    for (int32_t i = threadIdx.x; i <= bs.n_t; i += blockDim.x) sT_t[i] = bs.T_t[i];
    __syncthreads();

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    // this warp's neighbour list: shared memory, or its slice of nb_global [grid][kWarps][max_nb]
    int4* nb = nb_global ? nb_global + ((size_t)blockIdx.x * kWarps + wid) * max_nb : nb_all + (size_t)wid * max_nb;
    const long long total = (long long)fb.n_frames * fb.n;
    unsigned long long my_overflow = 0, my_pairs = 0, my_cap = 0;

    for (long long g = (long long)blockIdx.x * kWarps + wid; g < total;
         g += (long long)gridDim.x * kWarps) {
        const int32_t f = (int32_t)(g / fb.n);
        const int32_t s = (int32_t)(g - (long long)f * fb.n);
        const int4* __restrict__ sorted = fb.sorted + (long long)f * fb.n;
        const int32_t* __restrict__ start = fb.cell_start + (long long)f * (fb.ncell3 + 1);
        const int4 me = sorted[s];

        // a3: neighbours of the centre
        int32_t count = 0;
        const int32_t n_ranges = CandidateRanges::count(fb.ncell);
        for (int32_t r = 0; r < n_ranges; ++r) {
            int32_t begin, end;
            CandidateRanges::get(r, me.w, fb.ncell, fb.n, start, begin, end);
            for (int32_t p0 = begin; p0 < end; p0 += 32) {
                int32_t p = p0 + lane;
                bool ok = p < end && p != s;
                int4 c = ok ? sorted[p] : me;
                long long dx = wrap_component(c.x - me.x);
                long long dy = wrap_component(c.y - me.y);
                long long dz = wrap_component(c.z - me.z);
                unsigned long long d2 = (unsigned long long)(dx * dx + dy * dy + dz * dz);
                ok = ok && d2 < bs.cut2;
                unsigned mask = __ballot_sync(0xffffffffu, ok);
                if (ok) {
                    int32_t pos = count + __popc(mask & ((1u << lane) - 1u));
                    if (pos < max_nb)
                        nb[pos] = make_int4((int32_t)dx, (int32_t)dy, (int32_t)dz,
                                            bin_search(sT_r, bs.n_r, d2));
                }
                count += __popc(mask);
            }
        }
        if (count > max_nb) { if (lane == 0) my_cap += 1; count = max_nb; }
        __syncwarp();
        if (lane == 0) my_pairs += (unsigned long long)count * (unsigned long long)(count - 1);

        // a4: ordered pairs (j, k), j != k; g2: one count per neighbour in its shell
        for (int32_t j = lane; j < count; j += 32) {
            const int4 vj = nb[j];
            atomicAdd(counts2 + vj.w, 1ull);
            unsigned long long* row = counts + (size_t)vj.w * bs.n_r * bs.n_t;
            for (int32_t k = 0; k < count; ++k) {
                if (k == j) continue;
                const int4 vk = nb[k];
                long long ex = (long long)vk.x - vj.x, ey = (long long)vk.y - vj.y,
                          ez = (long long)vk.z - vj.z;
                unsigned long long t2 = (unsigned long long)(ex * ex + ey * ey + ez * ez);
                int32_t c = bin_search(sT_t, bs.n_t, t2);
                if (c < bs.n_t) atomicAdd(row + (size_t)vk.w * bs.n_t + c, 1ull);
                else my_overflow += 1;
            }
        }
        __syncwarp();
    }
    if (my_pairs) atomicAdd(stats + 0, my_pairs);
    if (my_overflow) atomicAdd(stats + 1, my_overflow);
    if (my_cap) atomicAdd(stats + 2, my_cap);
}

// shared memory of the kernel: the edge tables, plus the lists unless they live in global memory
inline size_t generic_smem_bytes(int32_t n_r, int32_t n_t, int32_t max_nb, int warps, bool lists_in_smem = true) {
    size_t off = ((size_t)(n_r + n_t + 2) * 8 + 15) & ~size_t(15);
    return off + (lists_in_smem ? (size_t)warps * max_nb * sizeof(int4) : 0);
}

}  // namespace g3
