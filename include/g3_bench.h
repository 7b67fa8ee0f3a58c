/* g3_bench.h -- measurement aid for bench.py, NOT part of the product ABI (include/g3.h).
 *
 * libg3bench.so (built from paper_1708_08619_b200/csrc/bench/) measures the two hardware
 * ceilings the triplet kernel's roofline is quoted against.  It
 * links nothing of libg3 and no result of the g(3) path depends on it; only bench.py loads it.
 */
#ifndef G3_BENCH_H_
#define G3_BENCH_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(_WIN32)
#define G3_BENCH_API __declspec(dllexport)
#else
#define G3_BENCH_API __attribute__((visibility("default")))
#endif

/* which = 0: shared-memory atomic increments per second over the whole GPU for pseudo-random
 * slots of a `slots`-word tile (bank conflicts included; one CTA of 20 full warps per SM, the
 * same red.shared.add.u32 the triplet kernel issues); which = 1: issued FP32 thread
 * instructions per second (slots ignored).  `iters` operations per thread.  Runs twice
 * (warm-up, then timed with CUDA events on `stream`, a cudaStream_t), synchronises, writes
 * *h_rate (host).  Returns 0 on success, 1 for invalid arguments, 3 for a CUDA error or a
 * device older than sm_100 (the status values of include/g3.h).                              */
G3_BENCH_API int g3_microbench(int32_t which, int64_t slots, int64_t iters, double *h_rate, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* G3_BENCH_H_ */
