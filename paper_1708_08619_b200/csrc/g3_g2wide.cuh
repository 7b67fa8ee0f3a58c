// g3_g2wide.cuh -- the pair histogram beyond the neighbour range: shells n_r .. 2 n_r - 1 of
// width w = r_max / n_r, i.e. r_ij in [r_max, 2 r_max) (G3_OPT_G2_WIDE).
//
// PAPER.md:428-429 (Algorithm 6 "Update the g2 histogram") and 513-518 (Algorithm 7 CUDA_g2)
// count pairs beyond the cut-off of the neighbour vectors; SURVEY.md 8(f) NEXT-1 asks for g2 on
// the whole r_jk axis of g(3) (the Kirkwood-superposition denominator g2 g2 g2).  Shells below
// n_r come from the neighbour pass (g3_neighbour.cuh); this kernel adds the outer ones.
//
// A warp per centre.  The cells are at least r_max wide, so a 5 x 5 x 5 stencil covers 2 r_max.
// Every unordered pair is visited ONCE (and counted twice): the centre looks only at the
// "forward" half of the stencil -- the 12 columns with (ox, oy) > (0, 0) over their five z cells,
// the two cells above its own in its own column, and the particles after itself in its own cell.
// Each column part is one contiguous range of the cell-major fp32 copy of the frame with one
// periodic shift; lanes take candidates 32 at a time.  With fewer than five cells per edge the
// stencil would wrap onto itself: then the centre scans all particles after itself.
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
        }
        if (++since_flush >= flush_every) { flush(); since_flush = 0; }
    }
    flush();
}

}  // namespace g3
