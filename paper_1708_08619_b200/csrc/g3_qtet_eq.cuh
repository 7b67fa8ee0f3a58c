// g3_qtet_eq.cuh -- the parts of the q_tet path (Eq. 1) that
// the q_tet kernels (g3_qtet.cuh) and the neighbour kernel (g3_neighbour.cuh, which takes the four
// nearest neighbours straight from its neighbour lists) share: the exact neighbour key of
// reading T1 and the fp64 evaluation of Eq. 1 in the fixed order of reading T2.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace g3 {

struct QtParams {
    int32_t n_q;                          // bins on [-3, 1]
    double scale;                         // n_q / 4
    unsigned long long guarantee2;        // (cell width)^2: below it the 27-cell search is exact
    unsigned long long* hist;             // [n_q]
    unsigned long long* stats;            // [2]: atoms binned, atoms skipped
    int32_t stage_cap;                    // qtet_cell_kernel: staged candidates per CTA
    const int4* cell_origin;              // [ncell3] grid coordinates of the cell centres
    int32_t* redo;                        // [frames * n + 1]: count, then atoms handed to qtet_kernel
    int32_t use_redo;                     // qtet_kernel: 1 = process the redo list, 0 = every atom
};

struct QtKey {
    unsigned long long hi, lo;            // d2; (dx, dy, dz) + 2^19 packed 20 bits each
};

__device__ __forceinline__ bool qt_lt(const QtKey& a, const QtKey& b) {
    return a.hi < b.hi || (a.hi == b.hi && a.lo < b.lo);
}

// Eq. 1 for one atom from its four nearest neighbours `best` (sorted by key), evaluated by one
// lane in fp64, one rounding per operation, in the order of reading T2; then the bin (T3, T4).
__device__ __forceinline__ void qt_finish(const QtKey (&best)[4], const QtParams& qp, unsigned int* hist_s,
                                          unsigned long long& binned, unsigned long long& skipped) {
    if (best[3].hi == ~0ull || best[0].hi == 0ull) { skipped += 1; return; }       // T4
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
    atomicAdd(hist_s + b, 1u);
    binned += 1;
}

}  // namespace g3
