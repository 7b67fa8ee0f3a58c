// g3_qtet.cuh -- the tetrahedral order parameter q_tet on the same cell list (SURVEY.md 8(f)
// NEXT-3): Eq. 1, Algorithm 3 CUDA_qtet, which runs loops 3-5
// of Algorithm 2 for one atom per thread and updates the histogram with atomicAdd.
//
// Here: one warp per atom.  The lanes scan the 27 cells around the atom (or the whole frame when
// the cell grid is degenerate), each lane keeping its own four smallest keys
//     key = (d2, dx, dy, dz)  in lexicographic order            (reading T1)
// in registers; four rounds of a warp-wide minimum then give the four nearest neighbours.  Every
// particle outside the 27 cells is more than one cell width away, so the result is exact when the
// fourth distance is below that width; otherwise (sparse frames) the atom is redone against all
// particles.  Lane 0 evaluates Eq. 1 in fp64 with one rounding per operation in the fixed order
// of reading T2, so the bin of q is decided by IEEE fp64 arithmetic alone.
#pragma once

#include "g3_generic.cuh"
#include "g3_plan.h"

namespace g3 {

struct QtParams {
    int32_t n_q;                          // bins on [-3, 1]
    double scale;                         // n_q / 4
    unsigned long long guarantee2;        // (cell width)^2: below it the 27-cell search is exact
    unsigned long long* hist;             // [n_q]
    unsigned long long* stats;            // [2]: atoms binned, atoms skipped
};

struct QtKey {
    unsigned long long hi, lo;            // d2; (dx, dy, dz) + 2^19 packed 20 bits each
};

__device__ __forceinline__ bool qt_lt(const QtKey& a, const QtKey& b) {
    return a.hi < b.hi || (a.hi == b.hi && a.lo < b.lo);
}

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

template <int kWarps>
__global__ void __launch_bounds__(kWarps * 32)
qtet_kernel(FrameBatch fb, QtParams qp) {
    extern __shared__ unsigned int qt_hist[];
    for (int32_t i = threadIdx.x; i < qp.n_q; i += blockDim.x) qt_hist[i] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long long total = (long long)fb.n_frames * fb.n;
    unsigned long long binned = 0, skipped = 0;
    for (long long g = (long long)blockIdx.x * kWarps + wid; g < total; g += (long long)gridDim.x * kWarps) {
        const int32_t f = (int32_t)(g / fb.n);
        const int32_t s = (int32_t)(g - (long long)f * fb.n);
        const int4* __restrict__ sorted = fb.sorted + (long long)f * fb.n;
        const int32_t* __restrict__ start = fb.cell_start + (long long)f * (fb.ncell3 + 1);
        const int4 me = sorted[s];
        QtKey top[4], best[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) { top[t].hi = ~0ull; top[t].lo = ~0ull; }
        const int32_t n_ranges = CandidateRanges::count(fb.ncell);
        for (int32_t r = 0; r < n_ranges; ++r) {
            int32_t begin, end;
            CandidateRanges::get(r, me.w, fb.ncell, fb.n, start, begin, end);
            qt_scan(sorted, begin, end, s, me, lane, top);
        }
        qt_merge(top, lane, best);
        if (fb.ncell != 1 && best[3].hi >= qp.guarantee2) {      // sparse neighbourhood: all particles
#pragma unroll
            for (int t = 0; t < 4; ++t) { top[t].hi = ~0ull; top[t].lo = ~0ull; }
            qt_scan(sorted, 0, fb.n, s, me, lane, top);
            qt_merge(top, lane, best);
        }
        if (lane != 0) continue;
        // Eq. 1 in fp64, one rounding per operation, in the order of reading T2
        if (best[3].hi == ~0ull || best[0].hi == 0ull) { skipped += 1; continue; }   // T4
        double nrm[4];
        long long vx[4], vy[4], vz[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            nrm[j] = __dsqrt_rn((double)best[j].hi);
            vx[j] = (long long)(best[j].lo >> 40) - 524288;
            vy[j] = (long long)((best[j].lo >> 20) & 0xFFFFF) - 524288;
            vz[j] = (long long)(best[j].lo & 0xFFFFF) - 524288;
        }
        double acc = 0.0;
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int k = j + 1; k < 4; ++k) {
                const long long dot = vx[j] * vx[k] + vy[j] * vy[k] + vz[j] * vz[k];
                const double den = __dmul_rn(nrm[j], nrm[k]);
                const double c = __ddiv_rn((double)dot, den);
                const double t = __dadd_rn(c, 1.0 / 3.0);
                acc = __dadd_rn(acc, __dmul_rn(t, t));
            }
        const double q = __dsub_rn(1.0, __dmul_rn(0.375, acc));
        long long b = (long long)floor(__dmul_rn(__dadd_rn(q, 3.0), qp.scale));
        b = b < 0 ? 0 : (b > qp.n_q - 1 ? qp.n_q - 1 : b);
        atomicAdd(qt_hist + b, 1u);
        binned += 1;
    }
    __syncthreads();
    for (int32_t i = threadIdx.x; i < qp.n_q; i += blockDim.x) {
        const unsigned int v = qt_hist[i];
        if (v) atomicAdd(qp.hist + i, (unsigned long long)v);
    }
    if (binned) atomicAdd(qp.stats + 0, binned);
    if (skipped) atomicAdd(qp.stats + 1, skipped);
}

}  // namespace g3
