// g3_microbench.cu -- libg3bench.so: the live measurement of the shared-atomic and issue ceilings
// (include/g3_bench.h).  A translation unit and a library of its own: bench.py loads it, the
// product library libg3.so does not contain it.
#include <cuda_runtime.h>

#include "../../../include/g3_bench.h"
#include "g3_microbench.cuh"

using namespace g3;

#define MB_CUDA(call)                                   \
    do {                                                \
        if ((call) != cudaSuccess) {                    \
            cudaGetLastError();                         \
            return 3;                                   \
        }                                               \
    } while (0)

extern "C" {

int g3_microbench(int32_t which, int64_t slots, int64_t iters, double* h_rate, void* stream) {
    if (!h_rate || iters < 8 || iters > (int64_t(1) << 30) || which < 0 || which > 1) return 1;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0;
    cudaDeviceProp prop;
    MB_CUDA(cudaGetDevice(&dev));
    MB_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major < 10) return 3;
    const int grid = prop.multiProcessorCount;
    const int32_t it = (int32_t)((iters + 127) / 128 * 128);
    unsigned int* d_sink = nullptr;
    MB_CUDA(cudaMalloc(&d_sink, 16));
    cudaEvent_t e0, e1;
    MB_CUDA(cudaEventCreate(&e0));
    MB_CUDA(cudaEventCreate(&e1));
    int rc = 0;
    float ms = 0.f;
    for (int rep = 0; rep < 2 && rc == 0; ++rep) {          // first pass warms up
        cudaEventRecord(e0, st);
        if (which == 0) {
            if (slots < 32 || slots * 4 > (int64_t)prop.sharedMemPerBlockOptin) { rc = 1; break; }
            cudaFuncSetAttribute(mb_shared_atomic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)(slots * 4));
            mb_shared_atomic_kernel<<<grid, kMbThreads, (size_t)slots * 4, st>>>((int32_t)slots, it, d_sink);
        } else {
            mb_issue_kernel<<<grid, kMbThreads, 0, st>>>(it, 1.0f, reinterpret_cast<float*>(d_sink));
        }
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = 3;
        else cudaEventElapsedTime(&ms, e0, e1);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_sink);
    if (rc != 0) return rc;
    // thread-level operations per second over the whole GPU (loop overhead not counted)
    *h_rate = (double)grid * kMbThreads * (double)it / ((double)ms * 1e-3);
    return 0;
}

}  // extern "C"
