// g3_neighbour.cuh -- step a3: minimum-image neighbour lists inside r_max, sorted by shell.
//
// Algorithm 7 CUDA_g2 "store minimum image neighbour vectors", done with a cell
// list instead of the paper's all-particle scan.
//
// One CTA (4 warps) per cell.  The particles of the 27 surrounding cells are staged once in
// shared memory as fp32 coordinates relative to the cell centre (exact: |value| < 2^20), so the
// minimum-image vector of a neighbour is a plain difference.  A warp per centre then runs
//   A  a tight scan of the stage: d2 < cut (fp32, widened by 2^-20) -> ballot-compacted list
//      of (dx, dy, dz, d2) in the warp's shared scratch;
//   B  per list entry: exact 64-bit test for entries within 2^-20 of the cut-off, shell
//      a = bin(T_r, d2) (fp32 twice with the scale lowered / raised by 2^-20; 64-bit search in
//      the exact edge table when the two disagree), rank inside the shell by a shared atomic;
//   C  exclusive scan of the shell counts and scatter to global memory in shell order:
//      nbv[centre][pos] = (dx, dy, dz, a).
// The order inside a shell depends on the atomics' arrival order; the histogram does not.
#pragma once

#include "g3_generic.cuh"
#include "g3_plan.h"

namespace g3 {

constexpr float kMagic = 12582912.0f;          // 1.5 * 2^23: fp32 integers with ulp 1 around it
constexpr uint32_t kMagicBits = 0x4B400000u;
constexpr int kNbWarps = 4;                    // warps per neighbour_kernel CTA
constexpr int kMaxRanges = 18;

struct NbParams {
    int32_t max_nb, stage_cap, n_r;
    float cut_lo, cut_hi;                 // fp32 window around T_r[n_r]
    unsigned long long cut2;
    float inv_w_lo, inv_w_hi;             // (1/w)(1 -+ 2^-20), w = shell width in grid units
    const unsigned long long* T_r;
    const int4* cell_origin;              // [ncell3] grid coordinates of the cell centres
    float4* nbv;                          // [frames][n][max_nb] (dx, dy, dz, shell as int bits)
    int32_t* nbcount;                     // [frames][n]
    unsigned long long* stats;
    // slab passes of the triplet kernel (n_slabs > 1): list position where each slab's shells start
    int32_t n_slabs;
    const int32_t* slab_shell;            // [n_slabs + 1] first shell of each slab; [n_slabs] = n_r
    int32_t* slabpos;                     // [frames][n][n_slabs + 1]
};

__device__ __forceinline__ float sqrt_approx(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

__device__ __forceinline__ unsigned long long exact_d2(float dx, float dy, float dz) {
    const long long X = (long long)dx, Y = (long long)dy, Z = (long long)dz;
    return (unsigned long long)(X * X + Y * Y + Z * Z);
}

__device__ __forceinline__ void sts128(uint32_t addr, float x, float y, float z, float w) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

constexpr float kFarAway = 3.0e18f;            // sentinel coordinate: its d2 is finite and beyond any cut-off

// Phase A for 32 candidates: `c` is this lane's candidate, `skip` = it is the centre itself.
// Accepted candidates are ballot-compacted into the warp's scratch list (shared address
// `scratch_s`, 16 B per entry) as (dx, dy, dz, d2).
template <bool kWrap>
__device__ __forceinline__ void nb_test(const float4 c, bool skip, float px, float py, float pz,
                                        float cut_hi, uint32_t lt_mask, int32_t max_nb,
                                        uint32_t scratch_s, int32_t& count) {
    float dx = c.x - px, dy = c.y - py, dz = c.z - pz;
    if (kWrap) {
        dx += dx < -524288.f ? 1048576.f : 0.f; dx -= dx >= 524288.f ? 1048576.f : 0.f;
        dy += dy < -524288.f ? 1048576.f : 0.f; dy -= dy >= 524288.f ? 1048576.f : 0.f;
        dz += dz < -524288.f ? 1048576.f : 0.f; dz -= dz >= 524288.f ? 1048576.f : 0.f;
    }
    const float d2f = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    const bool acc = d2f < cut_hi && !skip;
    const unsigned mask = __ballot_sync(0xffffffffu, acc);
    const int32_t pos = count + __popc(mask & lt_mask);
    if (acc && pos < max_nb) sts128(scratch_s + ((uint32_t)pos << 4), dx, dy, dz, d2f);
    count += __popc(mask);
}

// kWrap = the cell grid is degenerate (ncell == 1): the stage holds raw coordinates of the whole
// frame and every difference is wrapped; otherwise the stage is pre-shifted and no wrap is needed.
template <bool kWrap>
__global__ void __launch_bounds__(kNbWarps * 32)
neighbour_kernel(FrameBatch fb, NbParams np) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* stage = reinterpret_cast<float4*>(smem_raw);
    float4* scratch_all = stage + np.stage_cap;
    int32_t* hist_all = reinterpret_cast<int32_t*>(scratch_all + (size_t)kNbWarps * np.max_nb);
    __shared__ int32_t range_begin[kMaxRanges], range_prefix[kMaxRanges + 1];
    __shared__ int32_t own_base_s, cell_range[2];

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    // grid: x = cell (or slice of 64 centres when the cell grid is degenerate), y = frame
    const int32_t f = blockIdx.y, cell = kWrap ? 0 : blockIdx.x;
    const int4* __restrict__ sorted = fb.sorted + (long long)f * fb.n;
    const int32_t* __restrict__ start = fb.cell_start + (long long)f * (fb.ncell3 + 1);

    // ---- candidate ranges: one lane per range, all loads in flight together --------------------
    const int32_t n_ranges = CandidateRanges::count(fb.ncell);
    if (wid == 0) {
        const int32_t c_begin = kWrap ? 0 : __ldg(start + cell);
        const int32_t c_end = kWrap ? fb.n : __ldg(start + cell + 1);
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
    if (c_begin == c_end) return;                         // empty cell: no centres
    const int32_t n_stage = range_prefix[n_ranges];
    const int32_t n_pad = (n_stage + 31) & ~31;           // stage padded with far-away sentinels
    const bool staged = n_pad <= np.stage_cap;
    int32_t ox = 0, oy = 0, oz = 0;
    if (!kWrap) {
        const int4 o = __ldg(np.cell_origin + cell);
        ox = o.x; oy = o.y; oz = o.z;
    }
    auto relative = [&](int4 c) {
        if (kWrap) return make_float4((float)c.x, (float)c.y, (float)c.z, 0.f);
        return make_float4((float)wrap_component(c.x - ox), (float)wrap_component(c.y - oy),
                           (float)wrap_component(c.z - oz), 0.f);
    };
    if (staged) {                                         // a warp per range: straight copies
        for (int32_t r = wid; r < n_ranges; r += kNbWarps) {
            const int32_t b = range_begin[r], dst = range_prefix[r], len = range_prefix[r + 1] - dst;
            for (int32_t i = lane; i < len; i += 32) stage[dst + i] = relative(sorted[b + i]);
        }
        for (int32_t i = n_stage + threadIdx.x; i < n_pad; i += blockDim.x)
            stage[i] = make_float4(kFarAway, 0.f, 0.f, 0.f);
        __syncthreads();
    }

    // ---- one warp per centre -------------------------------------------------------------------
    float4* scratch = scratch_all + (size_t)wid * np.max_nb;
    int32_t* hist = hist_all + (size_t)wid * ((np.n_r + 3) & ~1);   // even stride: 8-byte aligned pairs
    const uint32_t scratch_s = (uint32_t)__cvta_generic_to_shared(scratch);
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int32_t own_base = own_base_s;
    const int32_t max_nb = np.max_nb, n_r = np.n_r;
    const float cut_hi = np.cut_hi;
    // degenerate grid: the centres are split over blockIdx.x in slices of 64
    const int32_t s_lo = kWrap ? min(c_end, (int32_t)blockIdx.x * 64) : c_begin;
    const int32_t s_hi = kWrap ? min(c_end, (int32_t)(blockIdx.x + 1) * 64) : c_end;
    unsigned long long my_pairs = 0, my_cap = 0;
    for (int32_t s = s_lo + wid; s < s_hi; s += kNbWarps) {
        int32_t count = 0;
        // phase A
        if (staged) {
            const int32_t own = own_base + (s - c_begin);
            const float4 p = stage[own];
            const int32_t own_q0 = own & ~31;
            const bool own_lane = lane == (own & 31);
            const float4* __restrict__ sp = stage + lane;
#pragma unroll 2
            for (int32_t q0 = 0; q0 < n_pad; q0 += 32)
                nb_test<kWrap>(sp[q0], own_lane && q0 == own_q0, p.x, p.y, p.z, cut_hi, lt_mask, max_nb,
                               scratch_s, count);
        } else {                                           // crowded neighbourhood: read from global
            const float4 p = relative(sorted[s]);
            for (int32_t r = 0; r < n_ranges; ++r) {
                const int32_t b = range_begin[r], e = b + (range_prefix[r + 1] - range_prefix[r]);
                for (int32_t q0 = b; q0 < e; q0 += 32) {
                    const int32_t q = q0 + lane;
                    const bool in = q < e && q != s;
                    const float4 c = in ? relative(sorted[q]) : p;
                    nb_test<kWrap>(c, !in, p.x, p.y, p.z, cut_hi, lt_mask, max_nb, scratch_s, count);
                }
            }
        }
        if (count > max_nb) { my_cap += 1; count = max_nb; }
        for (int32_t i = lane; i < n_r + 2; i += 32) hist[i] = 0;
        __syncwarp();

        // phase B: exact acceptance near the cut-off, shell, rank inside the shell
        for (int32_t e = lane; e < count; e += 32) {
            const float4 v = scratch[e];
            unsigned long long d2 = 0;
            bool have_exact = false, keep = true;
            if (v.w > np.cut_lo) {                         // too close to the cut-off for fp32
                d2 = exact_d2(v.x, v.y, v.z);
                have_exact = true;
                keep = d2 < np.cut2;
            }
            int32_t a = n_r;                               // n_r = rejected
            if (keep) {
                const float t = sqrt_approx(v.w);
                const uint32_t lo = __float_as_uint(__fmaf_rd(t, np.inv_w_lo, kMagic));
                const uint32_t hi = __float_as_uint(__fmaf_rd(t, np.inv_w_hi, kMagic));
                if (lo == hi) a = (int32_t)(lo - kMagicBits);
                else {
                    if (!have_exact) d2 = exact_d2(v.x, v.y, v.z);
                    a = bin_search(np.T_r, n_r, d2);
                }
            }
            const int32_t rank = atomicAdd(hist + a, 1);
            scratch[e].w = __int_as_float(a | (rank << 10));
        }
        __syncwarp();

        // phase C: exclusive scan of the shell counts (two shells per lane), scatter in shell order
        int32_t carry = 0;
        for (int32_t i0 = 0; i0 < n_r; i0 += 64) {
            const int32_t i = i0 + 2 * lane;
            int2 hv = make_int2(0, 0);                     // hist has >= n_r + 2 entries, i is even
            if (i < n_r) hv = *reinterpret_cast<const int2*>(hist + i);
            const int32_t v0 = i < n_r ? hv.x : 0, v1 = i + 1 < n_r ? hv.y : 0;
            const int32_t v = v0 + v1;
            int32_t incl = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int32_t t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            const int32_t total = __shfl_sync(0xffffffffu, incl, 31);
            __syncwarp();
            if (i < n_r) hist[i] = carry + incl - v;
            if (i + 1 < n_r) hist[i + 1] = carry + incl - v1;
            carry += total;
        }
        __syncwarp();
        const int32_t kept = carry;
        my_pairs += (unsigned long long)kept * (unsigned long long)(kept > 0 ? kept - 1 : 0);
        float4* __restrict__ dst = np.nbv + ((long long)f * fb.n + s) * max_nb;
        for (int32_t e = lane; e < count; e += 32) {
            const float4 v = scratch[e];
            const int32_t packed = __float_as_int(v.w);
            const int32_t a = packed & 1023, rank = packed >> 10;
            if (a < n_r) dst[hist[a] + rank] = make_float4(v.x, v.y, v.z, __int_as_float(a));
        }
        if (lane == 0) np.nbcount[(long long)f * fb.n + s] = kept;
        if (np.n_slabs > 1) {                     // hist[a] = list position of the first entry of shell a
            int32_t* sp = np.slabpos + ((long long)f * fb.n + s) * (np.n_slabs + 1);
            for (int32_t i = lane; i <= np.n_slabs; i += 32) {
                const int32_t a = np.slab_shell[i];
                sp[i] = a < n_r ? hist[a] : kept;
            }
        }
        __syncwarp();
    }
    if (lane == 0) {
        if (my_pairs) atomicAdd(np.stats + 0, my_pairs);
        if (my_cap) atomicAdd(np.stats + 2, my_cap);
    }
}

inline size_t nb_smem_bytes(int32_t stage_cap, int32_t max_nb, int32_t n_r) {
    return (size_t)stage_cap * 16 + (size_t)kNbWarps * max_nb * 16 + (size_t)kNbWarps * ((n_r + 3) & ~1) * 4;
}

}  // namespace g3
