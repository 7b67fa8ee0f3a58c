// g3_qtet.cuh -- the tetrahedral order parameter q_tet on the same cell list (SURVEY.md 8(f)
// NEXT-3): Eq. 1, Algorithm 3 CUDA_qtet, which runs loops 3-5
// of Algorithm 2 for one atom per thread and updates the histogram with atomicAdd.
//
// Three kernels.
//  qtet_cell_kernel, the fast one: a CTA stages the 27 cells once in shared memory as fp32
//   coordinates relative to the cell centre (exact integers, as in g3_neighbour.cuh) and a warp per
//   atom (1) scans them in fp32, each lane keeping its four smallest d2 as bit patterns tagged with
//   the scan iteration (a min/max insertion network, no divergence), (2) takes the warp's fourth
//   smallest value tau with four REDUX.MIN rounds, (3) fetches again the kept candidates with
//   d2 <= tau (1 + 2^-16) -- a superset of the true four nearest, because the tagged fp32 d2 is
//   within 2^-18 + 2^-22 of the exact integer -- and writes their exact 64-bit keys
//       key = (d2, dx, dy, dz)  in lexicographic order            (reading T1)
//   to a per-warp list, (4) ranks those few by the exact key.  Every particle outside the 27 cells
//   is more than one cell width away, so the result is exact when the fourth distance is below
//   that width.  One THREAD per atom of the cell then evaluates Eq. 1 in fp64 with one rounding
//   per operation in the fixed order of reading T2, so the bin of q is decided by IEEE
//   fp64 arithmetic alone.
//  qtet_redo_kernel: the atoms the fast kernel hands over (fourth neighbour not provably inside
//   the 27 cells, a lane that may have dropped a fifth candidate inside the tolerance, crowded
//   stage, more than 64 atoms in the cell), a whole CTA per atom against all particles.
//  qtet_kernel: the plain exact routine (64-bit keys straight from global memory, warp per atom)
//   for degenerate cell grids.
#pragma once

#include "g3_generic.cuh"
#include "g3_neighbour.cuh"
#include "g3_plan.h"
#include "g3_qtet_eq.cuh"

namespace g3 {

__device__ __forceinline__ void qt_insert(QtKey (&top)[4], const QtKey k) {
    if (!qt_lt(k, top[3])) return;
    top[3] = k;
#pragma unroll
    for (int t = 3; t > 0; --t)
        if (qt_lt(top[t], top[t - 1])) { const QtKey x = top[t]; top[t] = top[t - 1]; top[t - 1] = x; }
}

__device__ __forceinline__ void qt_scan(const int4* __restrict__ sorted, int32_t begin, int32_t end,
                                        int32_t self, const int4 me, int lane, QtKey (&top)[4]) {
    for (int32_t p = begin + lane; p < end; p += 32) {
        if (p == self) continue;
        const int4 c = sorted[p];
        const long long dx = wrap_component(c.x - me.x), dy = wrap_component(c.y - me.y),
                        dz = wrap_component(c.z - me.z);
        QtKey k;
        k.hi = (unsigned long long)(dx * dx + dy * dy + dz * dz);
        k.lo = ((unsigned long long)(dx + 524288) << 40) | ((unsigned long long)(dy + 524288) << 20) |
               (unsigned long long)(dz + 524288);
        qt_insert(top, k);
    }
}

// The four smallest keys of the warp, in order, known to every lane.
__device__ __forceinline__ void qt_merge(QtKey (&top)[4], int lane, QtKey (&best)[4]) {
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        QtKey m = top[0];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            QtKey o;
            o.hi = __shfl_xor_sync(0xffffffffu, m.hi, d);
            o.lo = __shfl_xor_sync(0xffffffffu, m.lo, d);
            if (qt_lt(o, m)) m = o;
        }
        best[t] = m;
        // the lowest lane whose head equals the minimum pops it (identical keys: coincident particles)
        const unsigned who = __ballot_sync(0xffffffffu, top[0].hi == m.hi && top[0].lo == m.lo);
        if (lane == __ffs(who) - 1) {
            top[0] = top[1]; top[1] = top[2]; top[2] = top[3];
            top[3].hi = ~0ull; top[3].lo = ~0ull;
        }
    }
}

__device__ __forceinline__ void qt_flush(const QtParams& qp, const unsigned int* hist_s,
                                         unsigned long long binned, unsigned long long skipped) {
    __syncthreads();
    for (int32_t i = threadIdx.x; i < qp.n_q; i += blockDim.x) {
        const unsigned int v = hist_s[i];
        if (v) atomicAdd(qp.hist + i, (unsigned long long)v);
    }
    if (binned) atomicAdd(qp.stats + 0, binned);
    if (skipped) atomicAdd(qp.stats + 1, skipped);
}

// Plain exact routine: 64-bit keys straight from global memory, warp per atom.  use_redo = 0:
// every atom of the batch (27 cells first, all particles if the fourth neighbour is not provably
// inside them); use_redo = 1: only the atoms listed by qtet_cell_kernel, against all particles.
template <int kWarps>
__global__ void __launch_bounds__(kWarps * 32)
qtet_kernel(FrameBatch fb, QtParams qp) {
    extern __shared__ unsigned int qt_hist[];
    for (int32_t i = threadIdx.x; i < qp.n_q; i += blockDim.x) qt_hist[i] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long long total = qp.use_redo ? (long long)qp.redo[0] : (long long)fb.n_frames * fb.n;
    unsigned long long binned = 0, skipped = 0;
    for (long long it = (long long)blockIdx.x * kWarps + wid; it < total; it += (long long)gridDim.x * kWarps) {
        const long long g = qp.use_redo ? (long long)qp.redo[1 + it] : it;
        const int32_t f = (int32_t)(g / fb.n);
        const int32_t s = (int32_t)(g - (long long)f * fb.n);
        const int4* __restrict__ sorted = fb.sorted + (long long)f * fb.n;
        const int32_t* __restrict__ start = fb.cell_start + (long long)f * (fb.ncell3 + 1);
        const int4 me = sorted[s];
        QtKey top[4], best[4];
        bool exact = false;
        if (!qp.use_redo) {
#pragma unroll
            for (int t = 0; t < 4; ++t) { top[t].hi = ~0ull; top[t].lo = ~0ull; }
            const int32_t n_ranges = CandidateRanges::count(fb.ncell);
            for (int32_t r = 0; r < n_ranges; ++r) {
                int32_t begin, end;
                CandidateRanges::get(r, me.w, fb.ncell, fb.n, start, begin, end);
                qt_scan(sorted, begin, end, s, me, lane, top);
            }
            qt_merge(top, lane, best);
            exact = fb.ncell == 1 || best[3].hi < qp.guarantee2;
        }
        if (!exact) {                                            // all particles of the frame
#pragma unroll
            for (int t = 0; t < 4; ++t) { top[t].hi = ~0ull; top[t].lo = ~0ull; }
            qt_scan(sorted, 0, fb.n, s, me, lane, top);
            qt_merge(top, lane, best);
        }
        if (lane == 0) qt_finish(best, qp, qt_hist, binned, skipped);
    }
    qt_flush(qp, qt_hist, binned, skipped);
}

// The atoms qtet_cell_kernel could not decide, against ALL particles of their frame: a whole CTA
// per atom (the list is short, so one warp per atom would leave the GPU idle behind a few long
// scans).  Every warp scans a slice, the per-warp results are merged through shared memory.
template <int kWarps>
__global__ void __launch_bounds__(kWarps * 32)
qtet_redo_kernel(FrameBatch fb, QtParams qp) {
    extern __shared__ unsigned int qt_hist[];
    __shared__ ulonglong2 part[kWarps * 4];
    static_assert(kWarps * 4 <= 32, "one warp merges the partial results");
    for (int32_t i = threadIdx.x; i < qp.n_q; i += blockDim.x) qt_hist[i] = 0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t total = qp.redo[0];
    unsigned long long binned = 0, skipped = 0;
    for (int32_t it = blockIdx.x; it < total; it += gridDim.x) {
        const long long g = qp.redo[1 + it];
        const int32_t f = (int32_t)(g / fb.n);
        const int32_t s = (int32_t)(g - (long long)f * fb.n);
        const int4* __restrict__ sorted = fb.sorted + (long long)f * fb.n;
        const int4 me = sorted[s];
        QtKey top[4], best[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) { top[t].hi = ~0ull; top[t].lo = ~0ull; }
        for (int32_t p0 = wid * 32; p0 < fb.n; p0 += kWarps * 32)
            qt_scan(sorted, p0, min(p0 + 32, fb.n), s, me, lane, top);
        qt_merge(top, lane, best);
        __syncthreads();                                   // `part` of the previous atom is free
        if (lane == 0) {
#pragma unroll
            for (int t = 0; t < 4; ++t) part[wid * 4 + t] = make_ulonglong2(best[t].hi, best[t].lo);
        }
        __syncthreads();
        if (wid == 0) {
#pragma unroll
            for (int t = 0; t < 4; ++t) { top[t].hi = ~0ull; top[t].lo = ~0ull; }
            if (lane < kWarps * 4) { top[0].hi = part[lane].x; top[0].lo = part[lane].y; }
            qt_merge(top, lane, best);
            if (lane == 0) qt_finish(best, qp, qt_hist, binned, skipped);
        }
    }
    qt_flush(qp, qt_hist, binned, skipped);
}

// q_tet from the neighbour lists of the tiled g(3) path (g3_neighbour.cuh): nbv[atom][e] =
// (dx, dy, dz, .) exact minimum-image vectors of ALL particles inside r_max, sorted by shell of
// r_ij; nbj[atom][e] grows strictly with the shell.  With k >= 4 entries the four nearest
// neighbours are among the entries whose shell is not beyond the shell of the fourth entry (every
// entry of a lower shell is nearer than every entry of a higher one, and every particle outside
// the list is farther than all of them).  One THREAD per atom: exact keys of those few entries,
// top four by insertion, Eq. 1 in fp64 (reading T2).  Atoms with k < 4 go to qtet_redo_kernel.
__global__ void __launch_bounds__(256)
qtet_list_kernel(const float4* __restrict__ nbv, const uint32_t* __restrict__ nbj, const int32_t* __restrict__ nbcount,
                 long long total, int32_t max_nb, QtParams qp) {
    extern __shared__ unsigned int qt_hist[];
    for (int32_t i = threadIdx.x; i < qp.n_q; i += blockDim.x) qt_hist[i] = 0;
    __syncthreads();
    unsigned long long binned = 0, skipped = 0;
    for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (long long)gridDim.x * blockDim.x) {
        const int32_t k = nbcount[g];
        if (k < 4) {                                       // the fourth neighbour is beyond r_max: all particles
            const int32_t idx = atomicAdd(qp.redo, 1);
            qp.redo[1 + idx] = (int32_t)g;
            continue;
        }
        const float4* __restrict__ lv = nbv + g * max_nb;
        const uint32_t* __restrict__ lj = nbj + g * max_nb;
        const uint32_t shell4 = lj[3];
        QtKey top[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) { top[t].hi = ~0ull; top[t].lo = ~0ull; }
        for (int32_t e = 0; e < k; ++e) {
            if (e >= 4 && lj[e] > shell4) break;           // sorted by shell: nothing nearer follows
            const float4 v = lv[e];
            const long long X = (long long)v.x, Y = (long long)v.y, Z = (long long)v.z;
            QtKey key;
            key.hi = (unsigned long long)(X * X + Y * Y + Z * Z);
            key.lo = ((unsigned long long)(X + 524288) << 40) | ((unsigned long long)(Y + 524288) << 20) |
                     (unsigned long long)(Z + 524288);
            qt_insert(top, key);
        }
        qt_finish(top, qp, qt_hist, binned, skipped);
    }
    qt_flush(qp, qt_hist, binned, skipped);
}

constexpr int kQtCellWarps = 4;
constexpr int kQtSlots = 64;                    // atoms of one cell whose result is kept in shared memory

// sorted insertion of x into the ascending four a[0..3] (the largest of the five drops out)
__device__ __forceinline__ void qt_insert4(uint32_t (&a)[4], uint32_t x) {
    uint32_t lo;
    lo = min(a[0], x); x = max(a[0], x); a[0] = lo;
    lo = min(a[1], x); x = max(a[1], x); a[1] = lo;
    lo = min(a[2], x); x = max(a[2], x); a[2] = lo;
    a[3] = min(a[3], x);
}

// Fast path (see the file header).  Persistent: a CTA strides over (cell, frame) items.  The fp32
// d2 of a candidate is kept as its bit pattern (order-preserving for non-negative floats) with the
// scan iteration in the low 5 bits, so a lane can fetch its kept candidates again; the 2^-18
// perturbation this causes is covered by the 2^-16 tolerance of step (3).
__global__ void __launch_bounds__(kQtCellWarps * 32)
qtet_cell_kernel(FrameBatch fb, QtParams qp) {
    extern __shared__ __align__(16) unsigned char qt_smem[];
    float4* stage = reinterpret_cast<float4*>(qt_smem);
    ulonglong2* scratch_all = reinterpret_cast<ulonglong2*>(stage + qp.stage_cap);      // [warps][32] keys
    ulonglong2* best_s = scratch_all + kQtCellWarps * 32;                              // [kQtSlots][4]
    unsigned int* hist_s = reinterpret_cast<unsigned int*>(best_s + kQtSlots * 4);
    __shared__ int32_t range_begin[kMaxRanges], range_prefix[kMaxRanges + 1];
    __shared__ int32_t own_base_s, cell_range[2];
    __shared__ int32_t decided_s[kQtSlots];

    for (int32_t i = threadIdx.x; i < qp.n_q; i += blockDim.x) hist_s[i] = 0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    ulonglong2* scratch = scratch_all + wid * 32;
    const uint32_t lt_mask = (1u << lane) - 1u;
    constexpr uint32_t kInfBits = 0x7F000000u;             // 1.7e38 as fp32 bits
    unsigned long long binned = 0, skipped = 0;
    const long long n_items = (long long)fb.ncell3 * fb.n_frames;
    const int32_t n_ranges = CandidateRanges::count(fb.ncell);

    for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int32_t f = (int32_t)(item / fb.ncell3), cell = (int32_t)(item - (long long)f * fb.ncell3);
        const int4* __restrict__ sorted = fb.sorted + (long long)f * fb.n;
        const int32_t* __restrict__ start = fb.cell_start + (long long)f * (fb.ncell3 + 1);
        __syncthreads();                                   // the previous item's shared state is free
        if (wid == 0) {
            const int32_t c_begin = __ldg(start + cell), c_end = __ldg(start + cell + 1);
            int32_t b = 0, e = 0;
            if (lane < n_ranges) CandidateRanges::get(lane, cell, fb.ncell, fb.n, start, b, e);
            const int32_t len = e - b;
            int32_t incl = len;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int32_t t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            if (lane < n_ranges) { range_begin[lane] = b; range_prefix[lane] = incl - len; }
            if (lane == n_ranges - 1) range_prefix[n_ranges] = incl;
            if (lane < n_ranges && b <= c_begin && c_begin < e) own_base_s = incl - len + (c_begin - b);
            if (lane == 0) { cell_range[0] = c_begin; cell_range[1] = c_end; }
        }
        __syncthreads();
        const int32_t c_begin = cell_range[0], c_end = cell_range[1];
        if (c_begin == c_end) continue;                    // empty cell (uniform over the CTA)
        const int32_t n_stage = range_prefix[n_ranges];
        const int32_t n_pad = (n_stage + 31) & ~31;
        const bool staged = n_pad <= qp.stage_cap && n_pad <= 1024;      // iteration index fits 5 bits
        if (staged) {
            const int4 o = __ldg(qp.cell_origin + cell);
            for (int32_t r = wid; r < n_ranges; r += kQtCellWarps) {
                const int32_t b = range_begin[r], dst = range_prefix[r], len = range_prefix[r + 1] - dst;
                for (int32_t i = lane; i < len; i += 32) {
                    const int4 c = sorted[b + i];
                    stage[dst + i] = make_float4((float)wrap_component(c.x - o.x), (float)wrap_component(c.y - o.y),
                                                 (float)wrap_component(c.z - o.z), 0.f);
                }
            }
            for (int32_t i = n_stage + threadIdx.x; i < n_pad; i += blockDim.x)
                stage[i] = make_float4(kFarAway, 0.f, 0.f, 0.f);
        }
        __syncthreads();
        const int32_t own_base = own_base_s;
        for (int32_t s = c_begin + wid; s < c_end; s += kQtCellWarps) {
            const int32_t slot = s - c_begin;
            bool decided = false;
            if (staged && slot < kQtSlots) {
                const int32_t own = own_base + slot;
                const float4 p = stage[own];
                const int32_t own_it = own >> 5;
                const bool own_lane = lane == (own & 31);
                const float4* __restrict__ sp = stage + lane;
                // (1) per-lane four smallest fp32 d2 (bit patterns tagged with the iteration)
                uint32_t a[4] = {kInfBits, kInfBits, kInfBits, kInfBits};
                const int32_t n_it = n_pad >> 5;
#pragma unroll 2
                for (int32_t it = 0; it < n_it; ++it) {
                    const float4 c = sp[it << 5];
                    const float dx = c.x - p.x, dy = c.y - p.y, dz = c.z - p.z;
                    const float d2f = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    const uint32_t bits = (__float_as_uint(d2f) & ~31u) | (uint32_t)it;
                    qt_insert4(a, own_lane && it == own_it ? kInfBits : bits);
                }
                // (2) the warp's fourth smallest
                uint32_t h[4] = {a[0], a[1], a[2], a[3]};
                uint32_t tau_bits = 0;
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    tau_bits = __reduce_min_sync(0xffffffffu, h[0]);
                    const unsigned who = __ballot_sync(0xffffffffu, h[0] == tau_bits);
                    if (lane == __ffs(who) - 1) { h[0] = h[1]; h[1] = h[2]; h[2] = h[3]; h[3] = kInfBits; }
                }
                if (tau_bits < 0x60000000u) {              // at least four real candidates (sentinels: 9e36)
                    // (3) candidates within the fp32 tolerance of tau: exact 64-bit keys to scratch
                    const float cut = __fmul_ru(__uint_as_float(tau_bits | 31u), 1.0f + 1.52587890625e-5f);
                    const uint32_t cut_bits = __float_as_uint(cut) | 31u;
                    bool lost = a[3] <= cut_bits;          // a fifth candidate of this lane may have dropped out
                    int32_t count = 0;
#pragma unroll
                    for (int t = 0; t < 4; ++t) {
                        const bool acc = a[t] <= cut_bits;
                        const unsigned mask = __ballot_sync(0xffffffffu, acc);
                        const int32_t pos = count + __popc(mask & lt_mask);
                        if (acc && pos < 32) {
                            const float4 c = sp[(a[t] & 31u) << 5];
                            const long long X = (long long)(c.x - p.x), Y = (long long)(c.y - p.y),
                                            Z = (long long)(c.z - p.z);
                            scratch[pos] = make_ulonglong2(
                                (unsigned long long)(X * X + Y * Y + Z * Z),
                                ((unsigned long long)(X + 524288) << 40) | ((unsigned long long)(Y + 524288) << 20) |
                                    (unsigned long long)(Z + 524288));
                        }
                        count += __popc(mask);
                    }
                    lost = __any_sync(0xffffffffu, lost) || count > 32;
                    __syncwarp();
                    if (!lost) {
                        // (4) rank of every candidate by the exact key (ties by scratch position)
                        ulonglong2 my = make_ulonglong2(~0ull, ~0ull);
                        if (lane < count) my = scratch[lane];
                        int32_t rank = 0;
                        for (int32_t e = 0; e < count; ++e) {
                            const ulonglong2 k = scratch[e];
                            rank += (k.x < my.x || (k.x == my.x && (k.y < my.y || (k.y == my.y && e < lane)))) ? 1 : 0;
                        }
                        const bool mine = lane < count && rank < 4;
                        if (mine) best_s[slot * 4 + rank] = my;
                        decided = __any_sync(0xffffffffu, mine && rank == 3 && my.x < qp.guarantee2);
                    }
                    __syncwarp();
                }
            }
            if (lane == 0) {
                if (slot < kQtSlots) decided_s[slot] = decided ? 1 : 0;
                if (!decided) {                            // hand the atom to the exact routine
                    const int32_t idx = atomicAdd(qp.redo, 1);
                    qp.redo[1 + idx] = (int32_t)((long long)f * fb.n + s);
                }
            }
        }
        __syncthreads();
        // Eq. 1: one thread per decided atom of the cell
        if ((int32_t)threadIdx.x < min(c_end - c_begin, kQtSlots) && decided_s[threadIdx.x]) {
            QtKey best[4];
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const ulonglong2 k = best_s[threadIdx.x * 4 + t];
                best[t].hi = k.x; best[t].lo = k.y;
            }
            qt_finish(best, qp, hist_s, binned, skipped);
        }
    }
    qt_flush(qp, hist_s, binned, skipped);
}

inline size_t qtet_cell_smem_bytes(int32_t stage_cap, int32_t n_q) {
    return (size_t)stage_cap * 16 + (size_t)kQtCellWarps * 32 * 16 + (size_t)kQtSlots * 4 * 16 + (size_t)n_q * 4;
}

}  // namespace g3
