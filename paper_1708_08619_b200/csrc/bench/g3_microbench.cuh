// g3_microbench.cuh -- the two ceilings SURVEY.md 8(d) asks to be MEASURED on the box for the
// triplet kernel's roofline: (0) the shared-memory atomic rate for pseudo-random slots of a
// tile as large as the triplet kernel's (bank conflicts included, full converged warps, the
// same red.shared.add.u32 with value 1 -> ATOMS.POPC.INC), and (1) the SM issue rate (FFMA
// chains, one warp instruction per scheduler per cycle).  One CTA per SM, 20 warps, like the
// triplet kernel.  These are measurement aids behind g3_microbench(); no result of the g(3)
// path depends on them.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace g3 {

constexpr int kMbThreads = 640;

__global__ void __launch_bounds__(kMbThreads, 1)
mb_shared_atomic_kernel(int32_t slots, int32_t iters, unsigned int* __restrict__ sink) {
    extern __shared__ __align__(16) unsigned char mb_smem[];
    uint32_t* tile = reinterpret_cast<uint32_t*>(mb_smem);
    for (int32_t i = threadIdx.x; i < slots; i += blockDim.x) tile[i] = 0;
    __syncthreads();
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(tile);
    // per-lane LCG (Numerical Recipes constants); slot = high bits scaled to [0, slots)
    uint32_t x = 1664525u * (blockIdx.x * blockDim.x + threadIdx.x + 1u) + 1013904223u;
#pragma unroll 1
    for (int32_t it = 0; it < iters; it += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            x = 1664525u * x + 1013904223u;
            const uint32_t slot = __umulhi(x, (uint32_t)slots);
            asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(base + (slot << 2)), "r"(1u) : "memory");
        }
    }
    __syncthreads();
    unsigned int s = 0;
    for (int32_t i = threadIdx.x; i < slots; i += blockDim.x) s += tile[i];
    if (s == 0xFFFFFFFFu) sink[0] = s;            // keeps the atomics observable
}

__global__ void __launch_bounds__(kMbThreads, 1)
mb_issue_kernel(int32_t iters, float seed, float* __restrict__ sink) {
    float a = seed + threadIdx.x, b = a + 1.f, c = a + 2.f, d = a + 3.f;
    float e = a + 4.f, f = a + 5.f, g = a + 6.f, h = a + 7.f;
    const float m = 0.999f, k = 0.001f;
#pragma unroll 1
    for (int32_t it = 0; it < iters; it += 128) {    // 128 FFMA (8 independent chains) per pass
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            a = fmaf(a, m, k); b = fmaf(b, m, k); c = fmaf(c, m, k); d = fmaf(d, m, k);
            e = fmaf(e, m, k); f = fmaf(f, m, k); g = fmaf(g, m, k); h = fmaf(h, m, k);
        }
    }
    const float s = a + b + c + d + e + f + g + h;
    if (s == 12345.678f) sink[0] = s;
}

}  // namespace g3
