// g3_neighbour.cuh -- step a3: minimum-image neighbour lists inside r_max, sorted by shell, and
// the pair histogram g2 over the same range.
//
// Algorithm 7 CUDA_g2 "store minimum image neighbour vectors" and "update the g2 histogram"
// (PAPER.md:518-520), done with a cell list instead of the paper's all-particle scan
// (PAPER.md:513-515).
//
// One CTA (4 warps) per cell and frame.  The particles of the 27 surrounding cells (up to 18
// contiguous ranges of the cell-major order, each with one constant periodic shift) are staged
// once in shared memory as fp32 coordinates relative to the cell centre (exact: |value| < 2^20),
// so the minimum-image vector of a neighbour is a plain difference.  A warp per centre then runs
//   A  a tight scan of the stage: d2 < cut (fp32, widened by 2^-20) -> ballot-compacted list
//      of (dx, dy, dz, d2) in the warp's shared scratch;
//   B  per list entry: exact 64-bit test for entries within 2^-20 of the cut-off, shell
//      a = bin(T_r, d2) (fp32 twice with the scale lowered / raised by 2^-20; 64-bit search in
//      the exact edge table when the two disagree), rank inside the shell by a shared atomic;
//   C  exclusive scan of the shell counts (which are also this centre's g2 counts) and scatter
//      to global memory in shell order, already in the form the triplet kernel's shared-memory
//      window wants: nbv[centre][pos] = (dx, dy, dz, addend(a)), nbj[centre][pos] = row offset(a).
// The order inside a shell depends on the atomics' arrival order; the histograms do not.
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
    const int4* cell_origin;              // [ncell3] (x, y, z) of the cell centre on the grid, w = cx | cy << 8 | cz << 16
    float4* nbv;                          // [frames][n][max_nb] (dx, dy, dz, addend of the shell): the k side of a pair
    uint32_t* nbj;                        // [frames][n][max_nb] tile byte offset of the shell's row: the j side
    const float* addend;                  // [n_r]  kMagic + BASE(b) - g(b) + 1  (g3_tiled.cuh)
    const int32_t* jconst;                // [n_r]  4 * (P(a) + h(a))
    int32_t* nbcount;                     // [frames][n]
    unsigned long long* stats;
    unsigned long long* counts2;          // [n_r] g2: ordered pairs (i, j) per shell of r_ij
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

__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr) : "memory");
    return v;
}

// per-warp shell histogram: n_r shells + "rejected" + "no entry", at least 66 slots, even
__host__ __device__ __forceinline__ int32_t nb_hist_stride(int32_t n_r) { return n_r < 64 ? 66 : (n_r + 3) & ~1; }

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

// Shell of one scratch entry v = (dx, dy, dz, fp32 d2): bin(T_r, d2) decided exactly, or n_r when
// the exact d2 is not below the cut-off.
__device__ __forceinline__ int32_t nb_shell(const float4 v, const NbParams& np) {
    unsigned long long d2 = 0;
    bool have_exact = false;
    if (v.w > np.cut_lo) {                         // too close to the cut-off for fp32
        d2 = exact_d2(v.x, v.y, v.z);
        have_exact = true;
        if (d2 >= np.cut2) return np.n_r;
    }
    const float t = sqrt_approx(v.w);
    const uint32_t lo = __float_as_uint(__fmaf_rd(t, np.inv_w_lo, kMagic));
    const uint32_t hi = __float_as_uint(__fmaf_rd(t, np.inv_w_hi, kMagic));
    if (lo == hi) return (int32_t)(lo - kMagicBits);
    if (!have_exact) d2 = exact_d2(v.x, v.y, v.z);
    return bin_search(np.T_r, np.n_r, d2);
}

// kWrap = the cell grid is degenerate (ncell == 1): the stage holds raw coordinates of the whole
// frame and every difference is wrapped; otherwise the stage is pre-shifted and no wrap is needed.
template <bool kWrap>
__global__ void __launch_bounds__(kNbWarps * 32)
neighbour_kernel(FrameBatch fb, NbParams np) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* stage = reinterpret_cast<float4*>(smem_raw);
    float4* scratch_all = stage + np.stage_cap;
    const int32_t hstride = nb_hist_stride(np.n_r);       // even stride: 8-byte aligned pairs
    int32_t* hist_all = reinterpret_cast<int32_t*>(scratch_all + (size_t)kNbWarps * np.max_nb);
    uint32_t* g2s = reinterpret_cast<uint32_t*>(hist_all + kNbWarps * hstride);   // [n_r] this CTA's g2 counts
    __shared__ int32_t range_begin[kMaxRanges], range_prefix[kMaxRanges + 1];
    __shared__ int4 range_shift[kMaxRanges];
    __shared__ int32_t own_base_s, cell_range[2];

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    // grid: x = cell (or slice of 64 centres when the cell grid is degenerate), y = frame
    const int32_t f = blockIdx.y, cell = kWrap ? 0 : blockIdx.x;
    const int4* __restrict__ sorted = fb.sorted + (long long)f * fb.n;
    const int32_t* __restrict__ start = fb.cell_start + (long long)f * (fb.ncell3 + 1);

    for (int32_t i = threadIdx.x; i < max(np.n_r, 64); i += blockDim.x) g2s[i] = 0;

    // ---- candidate ranges: one lane per range, all loads in flight together --------------------
    // 9 columns (x, y offsets) x 2 parts; the three z-adjacent cells of a column are contiguous in
    // the cell-major order unless they wrap.  Every range has one constant shift that turns grid
    // coordinates into minimum-image coordinates relative to the cell centre.
    const int32_t n_ranges = kWrap ? 1 : kMaxRanges;
    if (wid == 0) {
        const int32_t c_begin = kWrap ? 0 : __ldg(start + cell);
        const int32_t c_end = kWrap ? fb.n : __ldg(start + cell + 1);
        int32_t b = 0, e = 0;
        int4 sh = make_int4(0, 0, 0, 0);
        if (kWrap) { if (lane == 0) { b = 0; e = fb.n; } }
        else if (lane < kMaxRanges) {
            const int4 o = __ldg(np.cell_origin + cell);
            const int32_t nc = fb.ncell, cx = o.w & 255, cy = (o.w >> 8) & 255, cz = (o.w >> 16) & 255;
            const int32_t col = lane >> 1, part = lane & 1;
            const int32_t ox = (col * 11 >> 5) - 1, oy = col - 3 * (col * 11 >> 5) - 1;     // col / 3, col % 3 for col < 9
            int32_t x = cx + ox, y = cy + oy;
            sh.x = -o.x; sh.y = -o.y; sh.z = -o.z;
            if (x < 0) { x += nc; sh.x -= (int32_t)kGrid; } else if (x >= nc) { x -= nc; sh.x += (int32_t)kGrid; }
            if (y < 0) { y += nc; sh.y -= (int32_t)kGrid; } else if (y >= nc) { y -= nc; sh.y += (int32_t)kGrid; }
            const int32_t* __restrict__ colstart = start + (x * nc + y) * nc;
            int32_t zb, ze;                           // cells [zb, ze) of this part
            if (cz == 0) {
                if (part == 0) { zb = 0; ze = 2; } else { zb = nc - 1; ze = nc; sh.z -= (int32_t)kGrid; }
            } else if (cz == nc - 1) {
                if (part == 0) { zb = nc - 2; ze = nc; } else { zb = 0; ze = 1; sh.z += (int32_t)kGrid; }
            } else {
                zb = cz - 1; ze = part == 0 ? cz + 2 : cz - 1;
            }
            b = __ldg(colstart + zb); e = __ldg(colstart + ze);
        }
        const int32_t len = e - b;
        int32_t incl = len;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int32_t t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += t;
        }
        if (lane < n_ranges) { range_begin[lane] = b; range_prefix[lane] = incl - len; range_shift[lane] = sh; }
        if (lane == n_ranges - 1) range_prefix[n_ranges] = incl;
        if (lane < n_ranges && b <= c_begin && c_begin < e) own_base_s = incl - len + (c_begin - b);
        if (lane == 0) { cell_range[0] = c_begin; cell_range[1] = c_end; }
    }
    __syncthreads();
    const int32_t c_begin = cell_range[0], c_end = cell_range[1];
    if (c_begin == c_end) return;                         // empty cell: no centres
    const int32_t n_stage = range_prefix[n_ranges];
    const int32_t n_pad = (n_stage + 63) & ~63;           // stage padded with far-away sentinels
    const bool staged = n_pad <= np.stage_cap;
    if (staged) {                                         // a warp per range: straight copies
        for (int32_t r = wid; r < n_ranges; r += kNbWarps) {
            const int32_t b = range_begin[r], dst = range_prefix[r], len = range_prefix[r + 1] - dst;
            const int4 sh = range_shift[r];
            for (int32_t i = lane; i < len; i += 32) {
                const int4 c = sorted[b + i];
                stage[dst + i] = make_float4((float)(c.x + sh.x), (float)(c.y + sh.y), (float)(c.z + sh.z), 0.f);
            }
        }
        for (int32_t i = n_stage + threadIdx.x; i < n_pad; i += blockDim.x)
            stage[i] = make_float4(kFarAway, 0.f, 0.f, 0.f);
    }
    __syncthreads();

    // ---- one warp per centre -------------------------------------------------------------------
    float4* scratch = scratch_all + (size_t)wid * np.max_nb;
    int32_t* hist = hist_all + wid * hstride;
    const uint32_t stage_s = (uint32_t)__cvta_generic_to_shared(stage);
    const uint32_t scratch_s = (uint32_t)__cvta_generic_to_shared(scratch);
    const uint32_t hist_s = (uint32_t)__cvta_generic_to_shared(hist);
    const uint32_t g2_s = (uint32_t)__cvta_generic_to_shared(g2s);
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int32_t own_base = own_base_s;
    const int32_t max_nb = np.max_nb, n_r = np.n_r;
    const float cut_hi = np.cut_hi;
    // degenerate grid: the centres are split over blockIdx.x in slices of 64
    const int32_t s_lo = kWrap ? min(c_end, (int32_t)blockIdx.x * 64) : c_begin;
    const int32_t s_hi = kWrap ? min(c_end, (int32_t)(blockIdx.x + 1) * 64) : c_end;
    unsigned long long my_pairs = 0, my_cap = 0;
    const bool fast_bc = n_r <= 64;                     // one scan chunk: lists of <= 64 entries stay in registers
    for (int32_t s = s_lo + wid; s < s_hi; s += kNbWarps) {
        int32_t count = 0;
        // phase A
        if (staged) {
            const uint32_t own_s = stage_s + ((uint32_t)(own_base + (s - c_begin)) << 4);
            const float4 p = lds128(own_s);
            uint32_t sp = stage_s + ((uint32_t)lane << 4);
            const uint32_t sp_end = stage_s + ((uint32_t)n_pad << 4);
            if (kWrap) {
                for (; sp < sp_end; sp += 512)
                    nb_test<true>(lds128(sp), sp == own_s, p.x, p.y, p.z, cut_hi, lt_mask, max_nb, scratch_s, count);
            } else {
                // two rounds of 32 candidates per pass (n_pad is a multiple of 64); while 64 more
                // entries are sure to fit, the stores need no capacity test
                uint32_t wr = scratch_s;                       // write pointer of the compacted list
                const uint32_t wr_safe = scratch_s + ((uint32_t)max(max_nb - 64, 0) << 4);
                const uint32_t own_a = own_s, own_b = own_s - 512u;
                for (; sp < sp_end && wr <= wr_safe; sp += 1024) {
                    const float4 c0 = lds128(sp), c1 = lds128(sp + 512);
                    const float dx0 = c0.x - p.x, dy0 = c0.y - p.y, dz0 = c0.z - p.z;
                    const float dx1 = c1.x - p.x, dy1 = c1.y - p.y, dz1 = c1.z - p.z;
                    const float q0 = fmaf(dz0, dz0, fmaf(dy0, dy0, dx0 * dx0));
                    const float q1 = fmaf(dz1, dz1, fmaf(dy1, dy1, dx1 * dx1));
                    const bool a0 = q0 < cut_hi && sp != own_a, a1 = q1 < cut_hi && sp != own_b;
                    const unsigned m0 = __ballot_sync(0xffffffffu, a0), m1 = __ballot_sync(0xffffffffu, a1);
                    const int32_t n0 = __popc(m0);
                    if (a0) sts128(wr + ((uint32_t)__popc(m0 & lt_mask) << 4), dx0, dy0, dz0, q0);
                    if (a1) sts128(wr + ((uint32_t)(__popc(m1 & lt_mask) + n0) << 4), dx1, dy1, dz1, q1);
                    wr += (uint32_t)(n0 + __popc(m1)) << 4;
                }
                count = (int32_t)((wr - scratch_s) >> 4);
                for (; sp < sp_end; sp += 512)                 // list nearly full: tested stores
                    nb_test<false>(lds128(sp), sp == own_s, p.x, p.y, p.z, cut_hi, lt_mask, max_nb, scratch_s, count);
            }
        } else {                                           // crowded neighbourhood: read from global
            const int4 me = sorted[s];
            for (int32_t r = 0; r < n_ranges; ++r) {
                const int32_t b = range_begin[r], e = b + (range_prefix[r + 1] - range_prefix[r]);
                for (int32_t q0 = b; q0 < e; q0 += 32) {
                    const int32_t q = q0 + lane;
                    const bool in = q < e && q != s;
                    const int4 c = in ? sorted[q] : me;
                    const float4 rel = make_float4((float)wrap_component(c.x - me.x), (float)wrap_component(c.y - me.y),
                                                   (float)wrap_component(c.z - me.z), 0.f);
                    nb_test<false>(rel, !in, 0.f, 0.f, 0.f, cut_hi, lt_mask, max_nb, scratch_s, count);
                }
            }
        }
        if (count > max_nb) { my_cap += 1; count = max_nb; }
        const long long row = ((long long)f * fb.n + s) * max_nb;
        float4* __restrict__ dst = np.nbv + row;
        uint32_t* __restrict__ dstj = np.nbj + row;
        int32_t kept;
        if (fast_bc && count <= 64) {
            // ---- phases B + C with the list in registers (entries lane and lane + 32) ---------------
            // hist: shells 0..n_r-1, slot n_r = rejected by the exact cut-off test, slot n_r + 1 = no entry
            asm volatile("st.shared.v2.b32 [%0], {%1, %1};" ::"r"(hist_s + ((uint32_t)lane << 3)), "r"(0) : "memory");
            if (lane == 0) asm volatile("st.shared.v2.b32 [%0], {%1, %1};" ::"r"(hist_s + 256u), "r"(0) : "memory");
            __syncwarp();
            const bool val0 = lane < count, val1 = lane + 32 < count;
            float4 v0 = lds128(scratch_s + ((uint32_t)lane << 4)), v1 = lds128(scratch_s + 512u + ((uint32_t)lane << 4));
            if (!val0) v0.w = 1.f;
            if (!val1) v1.w = 1.f;
            int32_t a0 = nb_shell(v0, np), a1 = nb_shell(v1, np);
            a0 = val0 ? a0 : n_r + 1; a1 = val1 ? a1 : n_r + 1;
            const int32_t r0 = atomicAdd(hist + a0, 1);
            const int32_t r1 = atomicAdd(hist + a1, 1);
            __syncwarp();
            int2 hv = *reinterpret_cast<const int2*>(hist + 2 * lane);
            const int32_t c0 = 2 * lane < n_r ? hv.x : 0, c1 = 2 * lane + 1 < n_r ? hv.y : 0;
            const int32_t v = c0 + c1;
            int32_t incl = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int32_t t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            kept = __shfl_sync(0xffffffffu, incl, 31);
            __syncwarp();
            asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(hist_s + ((uint32_t)lane << 3)), "r"(incl - v), "r"(incl - c1) : "memory");
            // this centre's g2 counts; g2s has 64 slots
            asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(g2_s + ((uint32_t)lane << 3)), "r"(c0) : "memory");
            asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(g2_s + ((uint32_t)lane << 3) + 4u), "r"(c1) : "memory");
            __syncwarp();
            if (a0 < n_r) {
                const int32_t pos = hist[a0] + r0;
                dst[pos] = make_float4(v0.x, v0.y, v0.z, __ldg(np.addend + a0));
                dstj[pos] = (uint32_t)__ldg(np.jconst + a0);
            }
            if (a1 < n_r) {
                const int32_t pos = hist[a1] + r1;
                dst[pos] = make_float4(v1.x, v1.y, v1.z, __ldg(np.addend + a1));
                dstj[pos] = (uint32_t)__ldg(np.jconst + a1);
            }
        } else {
            for (int32_t i = 2 * lane; i < n_r + 2; i += 64) *reinterpret_cast<int2*>(hist + i) = make_int2(0, 0);
            __syncwarp();
            // phase B: exact acceptance near the cut-off, shell, rank inside the shell
            for (int32_t e = lane; e < count; e += 32) {
                const uint32_t es = scratch_s + ((uint32_t)e << 4);
                const float4 v = lds128(es);
                const int32_t a = nb_shell(v, np);             // n_r = rejected
                const int32_t rank = atomicAdd(hist + a, 1);
                asm volatile("st.shared.b32 [%0], %1;" ::"r"(es + 12), "r"(a | (rank << 10)) : "memory");
            }
            __syncwarp();
            // phase C: exclusive scan of the shell counts (two shells per lane); the counts are this
            // centre's g2 contribution; then scatter in shell order
            int32_t carry = 0;
            for (int32_t i0 = 0; i0 < n_r; i0 += 64) {
                const int32_t i = i0 + 2 * lane;
                int2 hv = make_int2(0, 0);                     // hist has >= n_r + 2 entries, i is even
                if (i < n_r) hv = *reinterpret_cast<const int2*>(hist + i);
                const int32_t v0 = hv.x, v1 = i + 1 < n_r ? hv.y : 0;
                const int32_t v = v0 + v1;
                int32_t incl = v;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const int32_t t = __shfl_up_sync(0xffffffffu, incl, d);
                    if (lane >= d) incl += t;
                }
                const int32_t total = __shfl_sync(0xffffffffu, incl, 31);
                if (i < n_r) {
                    *reinterpret_cast<int2*>(hist + i) = make_int2(carry + incl - v, carry + incl - v1);
                    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(g2_s + ((uint32_t)i << 2)), "r"(v0) : "memory");
                    if (i + 1 < n_r)
                        asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(g2_s + ((uint32_t)i << 2) + 4), "r"(v1) : "memory");
                }
                carry += total;
            }
            __syncwarp();
            kept = carry;
            for (int32_t e = lane; e < count; e += 32) {
                const float4 v = lds128(scratch_s + ((uint32_t)e << 4));
                const int32_t packed = __float_as_int(v.w);
                const int32_t a = packed & 1023, rank = packed >> 10;
                if (a < n_r) {
                    const int32_t pos = hist[a] + rank;
                    dst[pos] = make_float4(v.x, v.y, v.z, __ldg(np.addend + a));
                    dstj[pos] = (uint32_t)__ldg(np.jconst + a);
                }
            }
        }
        my_pairs += (unsigned long long)kept * (unsigned long long)(kept > 0 ? kept - 1 : 0);
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
    __syncthreads();
    for (int32_t i = threadIdx.x; i < n_r; i += blockDim.x) {
        const uint32_t v = g2s[i];
        if (v) atomicAdd(np.counts2 + i, (unsigned long long)v);
    }
}

inline size_t nb_smem_bytes(int32_t stage_cap, int32_t max_nb, int32_t n_r) {
    return (size_t)stage_cap * 16 + (size_t)kNbWarps * max_nb * 16 + (size_t)kNbWarps * nb_hist_stride(n_r) * 4 +
           (size_t)(n_r > 64 ? n_r : 64) * 4;
}

}  // namespace g3
