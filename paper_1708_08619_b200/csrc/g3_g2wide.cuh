// g3_g2wide.cuh -- the pair histogram beyond the neighbour range: shells n_r .. 2 n_r - 1 of
// width w = r_max / n_r, i.e. r_ij in [r_max, 2 r_max) (G3_OPT_G2_WIDE).
//
// PAPER.md:428-429 (Algorithm 6 "Update the g2 histogram") and 513-518 (Algorithm 7 CUDA_g2)
// count pairs beyond the cut-off of the neighbour vectors; SURVEY.md 8(f) NEXT-1 asks for g2 on
// the whole r_jk axis of g(3) (the Kirkwood-superposition denominator g2 g2 g2).  Shells below
// n_r come from the neighbour pass (g3_neighbour.cuh); this kernel adds the outer ones.
//
// The cells are at least r_max wide, so a 5 x 5 x 5 stencil covers 2 r_max.  Every unordered
// pair is visited ONCE (and counted twice): a centre looks only at the "forward" half of the
// stencil -- the 12 columns with (ox, oy) > (0, 0) over their five z cells, the two cells above
// its own in its own column, and the particles after itself in its own cell.
//   g2_wide_cell_kernel  (five or more cells per edge) has the structure of neighbour_cell_kernel:
//       a producer warp stages the forward half-stencil of a (cell, frame) item by TMA bulk
//       copies (up to 27 ranges, periodic shifts added in place), four consumer warps test it
//       against three centres per candidate load and bin the hits straight into a shared
//       histogram (no lists); ring of two stages, mbarriers only;
//   g2_wide_kernel       a warp per centre reading candidates from global memory: crowded cells
//       (more candidates than a stage holds) and grids with fewer than five cells per edge,
//       where the stencil would wrap onto itself and the centre scans all particles after itself.
// Exactness as in nb_shell: fp32 d2 decides unless it is within 2^-20 of an edge, then 64-bit.
#pragma once

#include "g3_neighbour.cuh"

namespace g3 {

constexpr int kG2wWarps = 8;

struct G2wParams {
    NbParams sh;                          // shell tables of the WIDE range: n_r = 2 n_r0, T_r = [2 n_r0 + 1] edges
    int32_t n_lo;                         // n_r0: shells below it are counted elsewhere
    unsigned long long* counts2;          // [2 n_r0] ordered pairs per shell
};

// 32 candidates: lane's candidate c (already shifted by the range's periodic offset) against centre p
__device__ __forceinline__ void g2w_count(const float4 c, bool in, float px, float py, float pz, const G2wParams& gp,
                                          uint32_t* hist) {
    float4 v;
    v.x = c.x - px; v.y = c.y - py; v.z = c.z - pz;
    v.w = fmaf(v.z, v.z, fmaf(v.y, v.y, v.x * v.x));
    const bool near = in && v.w < gp.sh.cut_hi;
    if (!near) v.w = 1.f;                              // nb_shell then takes the cheap path; result unused
    const int32_t a = nb_shell(v, gp.sh);             // 2 n_r0 = beyond the range
    if (near && a >= gp.n_lo && a < gp.sh.n_r) atomicAdd(hist + (a - gp.n_lo), 2u);      // (i, j) and (j, i)
}

// One centre (particle s of frame f) against the forward half-stencil, candidates read from global
// memory: the 40 candidate ranges (13 columns x 3 wrap parts + the rest of its own cell) are
// fetched at once, two per lane, then walked with two candidates per lane and step.
__device__ __forceinline__ void g2w_centre_global(const FrameBatch& fb, const G2wParams& gp, int32_t f, int32_t s, int lane,
                                                  uint32_t* g2w_hist) {
    const int32_t nc = fb.ncell;
    const float G = (float)kGrid;
    const float4* __restrict__ sf = fb.sortedf + (long long)f * fb.n;
    const float4 me = sf[s];
    const int32_t* __restrict__ start = fb.cell_start + (long long)f * (fb.ncell3 + 1);
    const int32_t cell = fb.sorted[(long long)f * fb.n + s].w;
    const int32_t cz = cell % nc, cy = (cell / nc) % nc, cx = cell / (nc * nc);
    // 13 forward columns x 3 z parts (cells below 0, inside, beyond nc - 1) and the rest of the
    // centre's own cell: 40 ranges, two per lane (slots lane and lane + 32), all fetched at once,
    // then walked one after the other.
    // columns 0..9 = ox in {1, 2} x oy in {-2..2}; 10, 11 = ox 0, oy in {1, 2}; 12 = own column
    int32_t begin[2] = {0, 0}, end[2] = {0, 0};
    float shx[2] = {0.f, 0.f}, shy[2] = {0.f, 0.f}, shz[2] = {0.f, 0.f};
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int slot = lane + 32 * h;
        if (slot < 39) {
            const int32_t col = slot / 3, part = slot - 3 * col;
            const int32_t ox = col < 10 ? 1 + col / 5 : 0;
            const int32_t oy = col < 10 ? col % 5 - 2 : (col < 12 ? col - 9 : 0);
            int32_t x = cx + ox, y = cy + oy;
            if (x >= nc) { x -= nc; shx[h] = G; }
            if (y < 0) { y += nc; shy[h] = -G; } else if (y >= nc) { y -= nc; shy[h] = G; }
            const int32_t* __restrict__ colstart = start + (x * nc + y) * nc;
            const int32_t z_lo = col < 12 ? cz - 2 : cz + 1, z_hi = cz + 2;      // inclusive, before wrapping
            int32_t za, zb;
            if (part == 0) { za = z_lo; zb = min(z_hi, -1); shz[h] = -G; za += nc; zb += nc; }
            else if (part == 1) { za = max(z_lo, 0); zb = min(z_hi, nc - 1); }
            else { za = max(z_lo, nc); zb = z_hi; shz[h] = G; za -= nc; zb -= nc; }
            if (za <= zb) { begin[h] = __ldg(colstart + za); end[h] = __ldg(colstart + zb + 1); }
        } else if (slot == 39) {                     // the particles after the centre in its own cell
            begin[h] = s + 1; end[h] = __ldg(start + cell + 1);
        }
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        unsigned todo = __ballot_sync(0xffffffffu, begin[h] < end[h]);
        while (todo) {
            const int src = __ffs(todo) - 1;
            todo &= todo - 1u;
            const int32_t rb = __shfl_sync(0xffffffffu, begin[h], src), re = __shfl_sync(0xffffffffu, end[h], src);
            const float px = me.x - __shfl_sync(0xffffffffu, shx[h], src), py = me.y - __shfl_sync(0xffffffffu, shy[h], src),
                        pz = me.z - __shfl_sync(0xffffffffu, shz[h], src);
            for (int32_t q0 = rb; q0 < re; q0 += 64) {       // two candidates per lane
                const int32_t qa = q0 + lane, qb = q0 + 32 + lane;
                const bool ina = qa < re, inb = qb < re;
                const float4 ca = ina ? sf[qa] : me, cb = inb ? sf[qb] : me;
                g2w_count(ca, ina, px, py, pz, gp, g2w_hist);
                g2w_count(cb, inb, px, py, pz, gp, g2w_hist);
            }
        }
    }
}

__global__ void __launch_bounds__(kG2wWarps * 32)
g2_wide_kernel(FrameBatch fb, G2wParams gp) {
    extern __shared__ uint32_t g2w_hist[];             // [n_r0] outer shells, this CTA
    const int32_t n_up = gp.sh.n_r - gp.n_lo;
    for (int32_t i = threadIdx.x; i < n_up; i += blockDim.x) g2w_hist[i] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long long total = (long long)fb.n_frames * fb.n;
    const int32_t nc = fb.ncell;
    const float G = (float)kGrid;
    // a u32 slot must not overflow: one centre adds at most 2 (n - 1), a round of the CTA 8 times that
    const long long flush_every = max(1ll, 0x7FFFFFFFll / ((long long)kG2wWarps * 2 * max(fb.n, 1)));
    long long since_flush = 0;
    auto flush = [&]() {
        __syncthreads();
        for (int32_t i = threadIdx.x; i < n_up; i += blockDim.x) {
            const uint32_t v = g2w_hist[i];
            if (v) { atomicAdd(gp.counts2 + gp.n_lo + i, (unsigned long long)v); g2w_hist[i] = 0; }
        }
        __syncthreads();
    };
    const long long per_round = (long long)gridDim.x * kG2wWarps;
    const long long rounds = (total + per_round - 1) / per_round;
    for (long long r = 0; r < rounds; ++r) {
        const long long g = r * per_round + (long long)blockIdx.x * kG2wWarps + wid;
        if (g < total) {
            const int32_t f = (int32_t)(g / fb.n), s = (int32_t)(g - (long long)f * fb.n);
            const float4* __restrict__ sf = fb.sortedf + (long long)f * fb.n;
            const float4 me = sf[s];
            if (nc < 5) {
                // all particles after the centre, minimum image by rounding to the nearest box length
                for (int32_t q0 = s + 1; q0 < fb.n; q0 += 32) {
                    const int32_t q = q0 + lane;
                    const bool in = q < fb.n;
                    float4 c = in ? sf[q] : me;
                    float dx = c.x - me.x, dy = c.y - me.y, dz = c.z - me.z;
                    dx -= G * rintf(dx * (1.0f / G)); dy -= G * rintf(dy * (1.0f / G)); dz -= G * rintf(dz * (1.0f / G));
                    if (dx >= 0.5f * G) dx -= G;       // the wrap convention of the path: [-2^19, 2^19)
                    if (dy >= 0.5f * G) dy -= G;
                    if (dz >= 0.5f * G) dz -= G;
                    g2w_count(make_float4(dx, dy, dz, 0.f), in, 0.f, 0.f, 0.f, gp, g2w_hist);
                }
            } else {
                g2w_centre_global(fb, gp, f, s, lane, g2w_hist);
            }
        }
        if (++since_flush >= flush_every) { flush(); since_flush = 0; }
    }
    flush();
}

// ---------------------------------------------------------------------------------------------
constexpr int kG2wRanges = 27;         // 12 columns x 2 parts, own column x 2 parts, the centre cell itself
constexpr int kG2wStages = 2;

struct G2wItem {
    int32_t range_prefix[kG2wRanges + 1]; // stage position of each range
    float4 range_shift[kG2wRanges];       // periodic shift of the range in grid units (w: non-zero flag)
    uint32_t shift_mask;
    int32_t c_begin, c_end;               // the cell's particles = the centres (staged last)
    int32_t staged;
    long long item;                       // -1 = no more work
};

__device__ __forceinline__ void g2w_prefetch(const FrameBatch& fb, int32_t stage_cap, long long item, long long n_items,
                                             G2wItem& it, float4* stage, uint32_t stage_s, uint32_t mbar, int lane) {
    int32_t f = 0, cell = 0, c_begin = 0, c_end = 0;
    const int32_t* __restrict__ start = nullptr;
    for (; item < n_items; item += gridDim.x) {
        f = (int32_t)(item / fb.ncell3);
        cell = (int32_t)(item - (long long)f * fb.ncell3);
        start = fb.cell_start + (long long)f * (fb.ncell3 + 1);
        c_begin = __ldg(start + cell);
        c_end = __ldg(start + cell + 1);
        if (c_begin != c_end) break;
    }
    if (item >= n_items) {
        if (lane == 0) it.item = -1;
        return;
    }
    const int32_t nc = fb.ncell;
    const float G = (float)kGrid;
    const int32_t cz = cell % nc, cy = (cell / nc) % nc, cx = cell / (nc * nc);
    int32_t b = 0, e = 0;
    float4 sh = make_float4(0.f, 0.f, 0.f, 0.f);
    if (lane < kG2wRanges - 1) {
        // columns 0..9 = ox in {1, 2} x oy in {-2..2}; 10, 11 = ox 0, oy in {1, 2}; 12 = own column (cells above)
        const int32_t col = lane >> 1, part = lane & 1;
        const int32_t ox = col < 10 ? 1 + col / 5 : 0;
        const int32_t oy = col < 10 ? col % 5 - 2 : (col < 12 ? col - 9 : 0);
        int32_t x = cx + ox, y = cy + oy;
        if (x >= nc) { x -= nc; sh.x = G; }
        if (y < 0) { y += nc; sh.y = -G; } else if (y >= nc) { y -= nc; sh.y = G; }
        const int32_t* __restrict__ colstart = start + (x * nc + y) * nc;
        const int32_t z_lo = col < 12 ? cz - 2 : cz + 1, z_hi = cz + 2;      // inclusive, before wrapping
        // part 0: the cells inside [0, nc); part 1: the wrapped ones (below 0 or beyond nc - 1, never both: nc >= 5)
        int32_t za, zb;
        if (part == 0) { za = max(z_lo, 0); zb = min(z_hi, nc - 1); }
        else if (z_lo < 0) { za = z_lo + nc; zb = min(z_hi, -1) + nc; sh.z = -G; }
        else { za = max(z_lo, nc) - nc; zb = z_hi - nc; sh.z = G; }
        if (za <= zb && za >= 0 && zb < nc) { b = __ldg(colstart + za); e = __ldg(colstart + zb + 1); }
        if (part == 1 && z_lo >= 0 && z_hi < nc) { b = 0; e = 0; }            // nothing wraps
    } else if (lane == kG2wRanges - 1) {
        b = c_begin; e = c_end;                            // the centres themselves, last in the stage
    }
    const int32_t len = e - b;
    int32_t incl = len;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int32_t t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
    }
    const int32_t n_stage = __shfl_sync(0xffffffffu, incl, kG2wRanges - 1);
    const int32_t n_pad = (n_stage + 31) & ~31;
    const bool staged = n_pad <= stage_cap;
    const bool shifted = len > 0 && (sh.x != 0.f || sh.y != 0.f || sh.z != 0.f);
    const unsigned smask = __ballot_sync(0xffffffffu, shifted);
    if (lane < kG2wRanges) { it.range_prefix[lane] = incl - len; it.range_shift[lane] = sh; }
    if (lane == kG2wRanges - 1) it.range_prefix[kG2wRanges] = incl;
    if (lane == 0) {
        it.c_begin = c_begin; it.c_end = c_end; it.item = item; it.staged = staged ? 1 : 0; it.shift_mask = smask;
        if (staged) mbar_expect_tx(mbar, (uint32_t)n_stage << 4);
    }
    __syncwarp();
    if (staged) {
        if (lane < kG2wRanges && len > 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            bulk_copy_g2s(stage_s + ((uint32_t)(incl - len) << 4), fb.sortedf + (long long)f * fb.n + b, (uint32_t)len << 4, mbar);
        }
        if (n_stage + lane < n_pad) stage[n_stage + lane] = make_float4(kFarAway, 0.f, 0.f, 0.f);
    }
}

// candidate c against centre p: bin the pair if its shell is in the outer range
__device__ __forceinline__ void g2w_test(const float4 c, const float4 p, bool ok, const G2wParams& gp, uint32_t* hist) {
    float4 v;
    v.x = c.x - p.x; v.y = c.y - p.y; v.z = c.z - p.z;
    v.w = fmaf(v.z, v.z, fmaf(v.y, v.y, v.x * v.x));
    const bool near = ok && v.w < gp.sh.cut_hi;
    if (!near) v.w = 1.f;
    const int32_t a = nb_shell(v, gp.sh);
    if (near && a >= gp.n_lo && a < gp.sh.n_r) atomicAdd(hist + (a - gp.n_lo), 2u);
}

__global__ void __launch_bounds__((kNbWarps + 1) * 32)
g2_wide_cell_kernel(FrameBatch fb, G2wParams gp, int32_t stage_cap) {
    extern __shared__ __align__(16) unsigned char g2w_smem[];
    float4* stage_all = reinterpret_cast<float4*>(g2w_smem);
    uint32_t* hist = reinterpret_cast<uint32_t*>(stage_all + (size_t)stage_cap * kG2wStages);   // [n_up]
    __shared__ G2wItem items[kG2wStages];
    __shared__ __align__(8) unsigned long long mbar_s[3 * kG2wStages];       // per stage: tma, full, empty
    const int32_t n_up = gp.sh.n_r - gp.n_lo;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int32_t i = threadIdx.x; i < n_up; i += blockDim.x) hist[i] = 0;
    const uint32_t mbar0 = (uint32_t)__cvta_generic_to_shared(&mbar_s[0]);
    if (threadIdx.x == 0) {
        for (int b = 0; b < kG2wStages; ++b) {
            mbar_init(mbar0 + 24u * b, 1);
            mbar_init(mbar0 + 24u * b + 8u, 1);
            mbar_init(mbar0 + 24u * b + 16u, kNbWarps);
        }
    }
    const uint32_t stage_s0 = (uint32_t)__cvta_generic_to_shared(stage_all);
    const uint32_t stage_bytes = (uint32_t)stage_cap << 4;
    const long long n_items = (long long)fb.ncell3 * fb.n_frames;
    __syncthreads();

    if (wid == kNbWarps) {
        // ---- producer warp (as in neighbour_cell_kernel) -------------------------------------------
        long long item = (long long)blockIdx.x;
        for (uint32_t iter = 0;; ++iter) {
            const uint32_t buf = iter % kG2wStages, round = iter / kG2wStages;
            const uint32_t mb = mbar0 + 24u * buf;
            mbar_wait(mb + 16u, (round & 1u) ^ 1u);
            G2wItem& it = items[buf];
            float4* stage = stage_all + (size_t)buf * stage_cap;
            g2w_prefetch(fb, stage_cap, item, n_items, it, stage, stage_s0 + buf * stage_bytes, mb, lane);
            __syncwarp();
            const long long found = it.item;
            if (found >= 0 && it.staged) {
                mbar_wait(mb, round & 1u);
                uint32_t sm = it.shift_mask;
                while (sm) {
                    const int r = __ffs(sm) - 1;
                    sm &= sm - 1u;
                    const float4 sh = it.range_shift[r];
                    const int32_t dst = it.range_prefix[r], len = it.range_prefix[r + 1] - dst;
                    for (int32_t i = lane; i < len; i += 32) {
                        float4 c = stage[dst + i];
                        c.x += sh.x; c.y += sh.y; c.z += sh.z;
                        stage[dst + i] = c;
                    }
                }
            } else if (lane == 0) {
                mbar_arrive(mb);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(mb + 8u);
            if (found < 0) break;
            item = found + gridDim.x;
        }
    } else {
        // ---- consumer warps: three centres per candidate load ---------------------------------------
        // u32 slots: a warp that has added up to 2^28 moves the CTA's counts to global memory (atomicExch,
        // safe beside the other warps' adds), so no slot can pass 4 x 2^28 + one item's adds
        unsigned long long added = 0;
        for (uint32_t iter = 0;; ++iter) {
            const uint32_t cur = iter % kG2wStages, round = iter / kG2wStages;
            const uint32_t mb = mbar0 + 24u * cur;
            mbar_wait(mb + 8u, round & 1u);
            const G2wItem& it = items[cur];
            const long long item = it.item;
            if (item < 0) break;
            const int32_t f = (int32_t)(item / fb.ncell3);
            const int32_t c_begin = it.c_begin, c_end = it.c_end, n_c = c_end - c_begin;
            if (it.staged) {
                const uint32_t stage_s = stage_s0 + cur * stage_bytes;
                const int32_t n_fwd = it.range_prefix[kG2wRanges - 1];       // the centres follow the forward candidates
                const int32_t n_g = (n_c + 2) / 3;
                for (int32_t gi = (wid + (int32_t)iter) & (kNbWarps - 1); gi < n_g; gi += kNbWarps) {
                    const int32_t o0 = 3 * gi, G = min(3, n_c - o0);
                    float4 p[3];
#pragma unroll
                    for (int g = 0; g < 3; ++g) p[g] = lds128(stage_s + ((uint32_t)(n_fwd + o0 + min(g, G - 1)) << 4));
                    // the forward half-stencil: every candidate counts for every centre of the group
                    for (int32_t q = lane; q < n_fwd; q += 32) {
                        const float4 c = lds128(stage_s + ((uint32_t)q << 4));
#pragma unroll
                        for (int g = 0; g < 3; ++g) g2w_test(c, p[g], g < G, gp, hist);
                    }
                    // the centre cell: the particles after each centre
                    for (int32_t q = o0 + 1 + lane; q < n_c; q += 32) {
                        const float4 c = lds128(stage_s + ((uint32_t)(n_fwd + q) << 4));
#pragma unroll
                        for (int g = 0; g < 3; ++g) g2w_test(c, p[g], g < G && q > o0 + g, gp, hist);
                    }
                }
            } else {
                for (int32_t s = c_begin + wid; s < c_end; s += kNbWarps) g2w_centre_global(fb, gp, f, s, lane, hist);
            }
            added += 2ull * 3ull * (unsigned long long)(it.range_prefix[kG2wRanges] + 64) * (unsigned long long)((n_c + 2) / 3);
            if (added >= (1ull << 28)) {
                for (int32_t i = lane; i < n_up; i += 32) {
                    const uint32_t v = atomicExch(hist + i, 0u);
                    if (v) atomicAdd(gp.counts2 + gp.n_lo + i, (unsigned long long)v);
                }
                added = 0;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(mb + 16u);
        }
        asm volatile("bar.sync 1, %0;" ::"r"(kNbWarps * 32) : "memory");     // the consumer warps only
        for (int32_t i = threadIdx.x; i < n_up; i += kNbWarps * 32) {
            const uint32_t v = hist[i];
            if (v) atomicAdd(gp.counts2 + gp.n_lo + i, (unsigned long long)v);
        }
    }
}

inline size_t g2w_cell_smem_bytes(int32_t stage_cap, int32_t n_up) {
    return (size_t)stage_cap * 16 * kG2wStages + (size_t)n_up * 4;
}

}  // namespace g3
