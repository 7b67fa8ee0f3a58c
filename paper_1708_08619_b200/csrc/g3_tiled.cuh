// g3_tiled.cuh -- tiled fast triplet kernel (kernel 2).  Placeholder until the kernel lands:
// selection always answers "generic".
#pragma once

#include "g3_plan.h"

namespace g3 {

inline int32_t tiled_select(const g3_plan* p) { (void)p; return 1; }
inline int tiled_configure(g3_plan* p) { (void)p; return G3_EINVAL; }
inline int tiled_launch(g3_plan* p, const FrameBatch& fb, const BinSpec& bs, cudaStream_t st) {
    (void)p; (void)fb; (void)bs; (void)st;
    return G3_EINVAL;
}

}  // namespace g3
