// g3_tiled.cuh -- the fast path (kernel 2): neighbour-list kernel + tiled triplet kernel.
//
// neighbour_kernel (step a3, Algorithm 7 CUDA_g2 "store minimum image neighbour vectors",
// PAPER.md:520): one CTA per cell.  The particles of the 27 surrounding cells are staged once
// in shared memory as fp32 coordinates relative to the cell centre (exact: |value| < 2^20), so
// the minimum-image vector of a neighbour is a plain difference.  A warp per centre scans the
// stage, keeps |d|^2 < T_r[n_r], finds the shell a = bin(T_r, |d|^2), sorts the neighbours by
// shell with a shared-memory counting sort and writes the list to global memory.
//
// tiled_triplet_kernel (steps a4 + a5, Algorithm 7 CUDA_g3): persistent, one
// CTA per SM.  A warp per centre; lane = neighbour j (32 at a time), the partner k is broadcast
// from a 32-entry shared-memory window; every UNORDERED pair j < k is visited once (the lists
// are sorted by shell, so a_j <= a_k) and counted with one shared-memory atomic into a
// privatised histogram tile that holds only the bins the triangle inequality allows:
//     slot(a, b, c) = 1 + BASE(b) + P(a) + c - g(b) + h(a)          (a <= b)
// (DESIGN.md section 4.3).  The tile is added to a per-CTA global scratch tile when the kernel
// ends; merge_kernel mirrors the scratch tiles into the uint64 [a][b][c] histogram.
//
// Exactness.  Differences of neighbour vectors are exact in fp32 (integers below 2^21).  The
// squared distance, its square root and the bin index are computed in fp32 with a relative
// error below 2^-21; the bin is taken twice, with the scale factor lowered and raised by
// 2^-20.  If both agree, the exact integer rule bin(T_t, t2) gives the same bin (the exact
// quotient lies between the two); if they differ the pair is redone in 64-bit integers
// against the exact edge table and the histogram is corrected.  Same for the shells.
#pragma once

#include <cmath>
#include <vector>

#include "g3_generic.cuh"
#include "g3_plan.h"

namespace g3 {

constexpr float kMagic = 12582912.0f;          // 1.5 * 2^23: fp32 integers with ulp 1 around it
constexpr uint32_t kMagicBits = 0x4B400000u;
constexpr int kNbWarps = 4;                    // warps per neighbour_kernel CTA
constexpr int kItemCentres = 8;                // centres per work-queue fetch

struct TiledState {
    // histogram tile layout (host copies kept for tests/introspection)
    int64_t tile_bins = 0;                     // slots incl. 2 guards
    std::vector<int32_t> g, h, W, P, BASE;
    // device tables
    float* d_addend = nullptr;                 // [n_r]  kMagic + BASE(b) - g(b) + 1
    int32_t* d_jconst = nullptr;               // [n_r]  4 * (P(a) + h(a))
    uint32_t* d_slot_map = nullptr;            // [tile_bins] packed (a, b, c); 0xFFFFFFFF = unused
    uint32_t* d_scratch = nullptr;             // [grid][tile_bins] per-CTA partial tiles
    // neighbour lists of one batch
    float4* d_nbv = nullptr;                   // [batch][n][max_nb] (dx, dy, dz, addend(a))
    int32_t* d_nbj = nullptr;                  // [batch][n][max_nb] jconst(a)
    int32_t* d_nbcount = nullptr;              // [batch][n]
    unsigned int* d_work = nullptr;            // work-queue counter
    // launch configuration
    int tri_warps = 16;
    int grid = 0;
    size_t tri_smem = 0, nb_smem = 0;
    int32_t stage_cap = 0;
    int64_t frames_since_merge = 0, merge_every = 1;
};

// ---------------------------------------------------------------------------------------------
// host: histogram tile layout
inline int32_t host_bin(const std::vector<unsigned long long>& T, unsigned long long q) {
    int32_t lo = 0, hi = (int32_t)T.size() - 1;
    while (lo < hi) { int32_t mid = lo + ((hi - lo + 1) >> 1); if (T[mid] <= q) lo = mid; else hi = mid - 1; }
    return lo;
}

// Rigorous range of t-bins reachable for shells a <= b: r^2 in [T_r[a], T_r[a+1]-1],
// s^2 in [T_r[b], T_r[b+1]-1], and |s - r| <= t <= r + s for real vectors.
inline void reachable_c(const g3_plan* p, int32_t a, int32_t b, int32_t& c_lo, int32_t& c_hi) {
    const long double r_hi = std::sqrt((long double)(p->T_r[a + 1] - 1));
    const long double s_lo = std::sqrt((long double)p->T_r[b]);
    const long double s_hi = std::sqrt((long double)(p->T_r[b + 1] - 1));
    long double t_min = s_lo - r_hi;
    if (t_min < 0) t_min = 0;
    const long double t_max = r_hi + s_hi;
    long double lo2 = t_min * t_min * (1.0L - 1e-12L) - 1.0L;
    if (lo2 < 0) lo2 = 0;
    const long double hi2 = t_max * t_max * (1.0L + 1e-12L) + 1.0L;
    c_lo = host_bin(p->T_t, (unsigned long long)std::floor(lo2));
    c_hi = host_bin(p->T_t, (unsigned long long)std::ceil(hi2));   // may be n_t: the overflow bin
}

inline void build_layout(const g3_plan* p, TiledState& ts) {
    const int32_t n_r = p->bins.n_r;
    std::vector<int32_t> clo((size_t)n_r * n_r, 0), chi((size_t)n_r * n_r, 0);
    for (int32_t a = 0; a < n_r; ++a)
        for (int32_t b = a; b < n_r; ++b)
            reachable_c(p, a, b, clo[(size_t)a * n_r + b], chi[(size_t)a * n_r + b]);
    ts.g.assign(n_r, 0); ts.h.assign(n_r, 0); ts.W.assign(n_r, 0);
    ts.P.assign(n_r + 1, 0); ts.BASE.assign(n_r + 1, 0);
    for (int32_t b = 0; b < n_r; ++b) ts.g[b] = clo[b];                      // c_lo(0, b)
    for (int32_t a = 0; a < n_r; ++a) {
        int32_t hh = 0, top = 0;
        for (int32_t b = a; b < n_r; ++b) hh = std::max(hh, ts.g[b] - clo[(size_t)a * n_r + b]);
        for (int32_t b = a; b < n_r; ++b) top = std::max(top, chi[(size_t)a * n_r + b] - ts.g[b]);
        ts.h[a] = hh;
        ts.W[a] = top + hh + 1;
    }
    for (int32_t a = 0; a < n_r; ++a) ts.P[a + 1] = ts.P[a] + ts.W[a];
    int64_t base = 0;
    for (int32_t b = 0; b < n_r; ++b) { ts.BASE[b] = (int32_t)base; base += ts.P[b + 1]; }
    ts.BASE[n_r] = (int32_t)std::min<int64_t>(base, INT32_MAX);
    ts.tile_bins = base + 2;
}

// ---------------------------------------------------------------------------------------------
struct NbParams {
    int32_t max_nb, stage_cap, n_r;
    float cut_lo, cut_hi;                 // fp32 window around T_r[n_r]
    unsigned long long cut2;
    float inv_w_lo, inv_w_hi;             // (1/w)(1 -+ 2^-20), w = shell width in grid units
    const unsigned long long* T_r;
    const float* addend;
    const int32_t* jconst;
    float4* nbv;
    int32_t* nbj;
    int32_t* nbcount;
    unsigned long long* stats;
};

__device__ __forceinline__ float sqrt_approx(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// kWrap = the cell grid is degenerate (ncell == 1): the stage holds raw coordinates of the whole
// frame and every difference is wrapped; otherwise the stage is pre-shifted and no wrap is needed.
template <bool kWrap>
__global__ void __launch_bounds__(kNbWarps * 32)
neighbour_kernel(FrameBatch fb, NbParams np) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* sx = reinterpret_cast<float*>(smem_raw);
    float* sy = sx + np.stage_cap;
    float* sz = sy + np.stage_cap;
    float4* scratch_all = reinterpret_cast<float4*>(sz + np.stage_cap);
    int32_t* hist_all = reinterpret_cast<int32_t*>(scratch_all + (size_t)kNbWarps * np.max_nb);
    __shared__ int32_t range_begin[18], range_prefix[19];
    __shared__ int32_t own_base_s;

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t f = blockIdx.x / fb.ncell3, cell = blockIdx.x - f * fb.ncell3;
    const int4* __restrict__ sorted = fb.sorted + (long long)f * fb.n;
    const int32_t* __restrict__ start = fb.cell_start + (long long)f * (fb.ncell3 + 1);
    const int32_t c_begin = kWrap ? 0 : start[cell], c_end = kWrap ? fb.n : start[cell + 1];
    if (c_begin == c_end) return;                         // empty cell: no centres

    // ---- stage the candidates --------------------------------------------------------------
    const int32_t n_ranges = CandidateRanges::count(fb.ncell);
    if (threadIdx.x == 0) {
        int32_t acc = 0;
        for (int32_t r = 0; r < n_ranges; ++r) {
            int32_t b, e;
            CandidateRanges::get(r, cell, fb.ncell, fb.n, start, b, e);
            range_begin[r] = b;
            range_prefix[r] = acc;
            if (b <= c_begin && c_begin < e) own_base_s = acc + (c_begin - b);
            acc += e - b;
        }
        range_prefix[n_ranges] = acc;
    }
    __syncthreads();
    const int32_t n_stage = range_prefix[n_ranges];
    int32_t ox = 0, oy = 0, oz = 0;
    if (!kWrap) {
        const int32_t cz = cell % fb.ncell, cy = (cell / fb.ncell) % fb.ncell, cx = cell / (fb.ncell * fb.ncell);
        ox = (int32_t)(((long long)(2 * cx + 1) << (kGridBits - 1)) / fb.ncell);   // cell centre
        oy = (int32_t)(((long long)(2 * cy + 1) << (kGridBits - 1)) / fb.ncell);
        oz = (int32_t)(((long long)(2 * cz + 1) << (kGridBits - 1)) / fb.ncell);
    }
    if (n_stage > np.stage_cap) {                        // sticky capacity error; skip this cell
        if (threadIdx.x == 0) atomicAdd(np.stats + 2, 1ull);
        for (int32_t s = c_begin + threadIdx.x; s < c_end; s += blockDim.x)
            if (!kWrap || (s >= (int32_t)blockIdx.y * 64 && s < (int32_t)(blockIdx.y + 1) * 64))
                np.nbcount[(long long)f * fb.n + s] = 0;
        return;
    }
    for (int32_t r = 0; r < n_ranges; ++r) {
        const int32_t len = range_prefix[r + 1] - range_prefix[r];
        for (int32_t q = threadIdx.x; q < len; q += blockDim.x) {
            const int4 c = sorted[range_begin[r] + q];
            const int32_t d = range_prefix[r] + q;
            if (kWrap) { sx[d] = (float)c.x; sy[d] = (float)c.y; sz[d] = (float)c.z; }
            else {
                sx[d] = (float)wrap_component(c.x - ox);
                sy[d] = (float)wrap_component(c.y - oy);
                sz[d] = (float)wrap_component(c.z - oz);
            }
        }
    }
    __syncthreads();

    // ---- one warp per centre ---------------------------------------------------------------
    float4* scratch = scratch_all + (size_t)wid * np.max_nb;
    int32_t* hist = hist_all + (size_t)wid * np.n_r;
    const int32_t own_base = own_base_s;
    // degenerate grid: the centres are split over blockIdx.y in slices of 64
    const int32_t s_lo = kWrap ? min(c_end, (int32_t)blockIdx.y * 64) : c_begin;
    const int32_t s_hi = kWrap ? min(c_end, (int32_t)(blockIdx.y + 1) * 64) : c_end;
    unsigned long long my_pairs = 0, my_cap = 0;
    for (int32_t s = s_lo + wid; s < s_hi; s += kNbWarps) {
        const int32_t own = own_base + (s - c_begin);
        const float px = sx[own], py = sy[own], pz = sz[own];
        int32_t count = 0;
        for (int32_t q0 = 0; q0 < n_stage; q0 += 32) {
            const int32_t q = q0 + lane;
            const bool in = q < n_stage && q != own;
            float dx = (in ? sx[q] : px) - px, dy = (in ? sy[q] : py) - py, dz = (in ? sz[q] : pz) - pz;
            if (kWrap) {
                dx += dx < -524288.f ? 1048576.f : 0.f; dx -= dx >= 524288.f ? 1048576.f : 0.f;
                dy += dy < -524288.f ? 1048576.f : 0.f; dy -= dy >= 524288.f ? 1048576.f : 0.f;
                dz += dz < -524288.f ? 1048576.f : 0.f; dz -= dz >= 524288.f ? 1048576.f : 0.f;
            }
            const float d2f = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            bool acc = in && d2f < np.cut_hi;
            int32_t a = 0;
            if (acc) {
                unsigned long long d2 = 0;
                bool have_exact = false;
                if (d2f > np.cut_lo) {                    // too close to the cut-off for fp32
                    const long long X = (long long)dx, Y = (long long)dy, Z = (long long)dz;
                    d2 = (unsigned long long)(X * X + Y * Y + Z * Z);
                    have_exact = true;
                    acc = d2 < np.cut2;
                }
                if (acc) {
                    const float t = sqrt_approx(d2f);
                    const uint32_t lo = __float_as_uint(__fmaf_rd(t, np.inv_w_lo, kMagic));
                    const uint32_t hi = __float_as_uint(__fmaf_rd(t, np.inv_w_hi, kMagic));
                    if (lo == hi) a = (int32_t)(lo - kMagicBits);
                    else {
                        if (!have_exact) {
                            const long long X = (long long)dx, Y = (long long)dy, Z = (long long)dz;
                            d2 = (unsigned long long)(X * X + Y * Y + Z * Z);
                        }
                        a = bin_search(np.T_r, np.n_r, d2);
                    }
                }
            }
            const unsigned mask = __ballot_sync(0xffffffffu, acc);
            if (acc) {
                const int32_t pos = count + __popc(mask & ((1u << lane) - 1u));
                if (pos < np.max_nb) scratch[pos] = make_float4(dx, dy, dz, __int_as_float(a));
            }
            count += __popc(mask);
        }
        if (count > np.max_nb) { my_cap += 1; count = np.max_nb; }
        my_pairs += (unsigned long long)count * (unsigned long long)(count > 0 ? count - 1 : 0);

        // counting sort by shell: rank within shell, exclusive scan, scatter to global
        for (int32_t i = lane; i < np.n_r; i += 32) hist[i] = 0;
        __syncwarp();
        for (int32_t e = lane; e < count; e += 32) {
            const int32_t a = __float_as_int(scratch[e].w);
            const int32_t rank = atomicAdd(hist + a, 1);
            scratch[e].w = __int_as_float(a | (rank << 10));
        }
        __syncwarp();
        int32_t carry = 0;
        for (int32_t i0 = 0; i0 < np.n_r; i0 += 32) {
            const int32_t i = i0 + lane;
            const int32_t v = i < np.n_r ? hist[i] : 0;
            int32_t incl = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int32_t t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            if (i < np.n_r) hist[i] = carry + incl - v;
            carry += __shfl_sync(0xffffffffu, incl, 31);
        }
        __syncwarp();
        const long long gbase = ((long long)f * fb.n + s) * np.max_nb;
        for (int32_t e = lane; e < count; e += 32) {
            const float4 v = scratch[e];
            const int32_t packed = __float_as_int(v.w);
            const int32_t a = packed & 1023, rank = packed >> 10;
            const int32_t pos = hist[a] + rank;
            np.nbv[gbase + pos] = make_float4(v.x, v.y, v.z, __ldg(np.addend + a));
            np.nbj[gbase + pos] = __ldg(np.jconst + a);
        }
        if (lane == 0) np.nbcount[(long long)f * fb.n + s] = count;
        __syncwarp();
    }
    if (lane == 0) {
        if (my_pairs) atomicAdd(np.stats + 0, my_pairs);
        if (my_cap) atomicAdd(np.stats + 2, my_cap);
    }
}

// ---------------------------------------------------------------------------------------------
struct TriParams {
    long long total_centres;              // frames * n
    int32_t max_nb, n_t;
    int32_t tile_bins;
    float inv_lo, inv_hi;                 // (1/wt)(1 -+ 2^-20), wt = t-bin width in grid units
    const unsigned long long* T_t;
    const float4* nbv;
    const int32_t* nbj;
    const int32_t* nbcount;
    unsigned int* work;
    uint32_t* scratch;                    // [grid][tile_bins]
};

__device__ __forceinline__ void red_shared_add(uint32_t addr, uint32_t v) {
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// One pair: lane-resident j (jx,jy,jz,Jj), broadcast k = kv.  Returns the fp32 bin bits twice.
#define G3_PAIR_BITS(kv, lo, hi)                                          \
    do {                                                                  \
        const float ex_ = (kv).x - jx, ey_ = (kv).y - jy, ez_ = (kv).z - jz; \
        const float t2_ = fmaf(ez_, ez_, fmaf(ey_, ey_, ex_ * ex_));      \
        const float t_ = sqrt_approx(t2_);                                \
        lo = __float_as_uint(__fmaf_rd(t_, tp.inv_lo, (kv).w));           \
        hi = __float_as_uint(__fmaf_rd(t_, tp.inv_hi, (kv).w));           \
    } while (0)

// Redo one pair exactly (64-bit integers, exact edge table) and move its count if the fp32 bin
// was wrong.  Called only for pairs whose two fp32 bins differ.
__device__ __noinline__ void fix_pair(float4 kv, float jx, float jy, float jz, uint32_t lo,
                                      uint32_t Jj, const unsigned long long* __restrict__ T_t,
                                      int32_t n_t) {
    const long long X = (long long)(kv.x - jx), Y = (long long)(kv.y - jy), Z = (long long)(kv.z - jz);
    const unsigned long long t2 = (unsigned long long)(X * X + Y * Y + Z * Z);
    const int32_t c_exact = bin_search(T_t, n_t, t2);
    const int32_t kk1 = (int32_t)(kv.w - kMagic);                 // BASE(b) - g(b) + 1, exact
    const int32_t c_fast = (int32_t)(lo - kMagicBits) - kk1;
    if (c_exact != c_fast) {
        const uint32_t addr = Jj + (lo << 2);
        red_shared_add(addr, 0xFFFFFFFFu);
        red_shared_add(addr + 4u * (uint32_t)(c_exact - c_fast), 1u);
    }
}

template <int kWarps>
__global__ void __launch_bounds__(kWarps * 32, 1)
tiled_triplet_kernel(TriParams tp) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t* tile = reinterpret_cast<uint32_t*>(smem_raw);
    const size_t tile_bytes = ((size_t)tp.tile_bins * 4 + 15) & ~size_t(15);
    float4* win_all = reinterpret_cast<float4*>(smem_raw + tile_bytes);

    for (int32_t i = threadIdx.x; i < tp.tile_bins; i += blockDim.x) tile[i] = 0;
    __syncthreads();

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    float4* win = win_all + wid * 32;
    // shared-window byte address of slot 0 minus the magic bits (mod 2^32), see file header
    const uint32_t cbase = (uint32_t)__cvta_generic_to_shared(tile) - (kMagicBits << 2);

    while (true) {
        unsigned int item = 0;
        if (lane == 0) item = atomicAdd(tp.work, 1u);
        item = __shfl_sync(0xffffffffu, item, 0);
        const long long c0 = (long long)item * kItemCentres;
        if (c0 >= tp.total_centres) break;
        const long long c1 = min(c0 + (long long)kItemCentres, tp.total_centres);
        for (long long c = c0; c < c1; ++c) {
            const int32_t K = min(tp.nbcount[c], tp.max_nb);
            if (K < 2) continue;
            const float4* __restrict__ lv = tp.nbv + c * tp.max_nb;
            const int32_t* __restrict__ lj = tp.nbj + c * tp.max_nb;
            const int32_t nchunks = (K + 31) >> 5;
            for (int32_t r = 0; r < nchunks; ++r) {
                const int32_t jidx = (r << 5) + lane;
                float4 jv = make_float4(0.f, 0.f, 0.f, kMagic);
                uint32_t Jj = cbase;
                if (jidx < K) { jv = lv[jidx]; Jj = cbase + (uint32_t)lj[jidx]; }
                const float jx = jv.x, jy = jv.y, jz = jv.z;
                // prefetch the first rectangular window while the triangle runs
                float4 nextv = make_float4(0.f, 0.f, 0.f, kMagic);
                if (r + 1 < nchunks && ((r + 1) << 5) + lane < K) nextv = lv[((r + 1) << 5) + lane];

                // ---- triangle: k in the same 32-block as j, k > j ----------------------------
                __syncwarp();
                win[lane] = jv;
                __syncwarp();
                const int32_t kt = min(32, K - (r << 5));
                for (int32_t kk = 1; kk < kt; ++kk) {
                    const float4 kv = win[kk];
                    uint32_t lo, hi;
                    G3_PAIR_BITS(kv, lo, hi);
                    if (lane < kk) {
                        red_shared_add(Jj + (lo << 2), 1u);
                        if (lo != hi) fix_pair(kv, jx, jy, jz, lo, Jj, tp.T_t, tp.n_t);
                    }
                }
                // ---- rectangles: k in later 32-blocks, every lane valid ----------------------
                for (int32_t q = r + 1; q < nchunks; ++q) {
                    __syncwarp();
                    win[lane] = nextv;
                    __syncwarp();
                    nextv = make_float4(0.f, 0.f, 0.f, kMagic);
                    if (q + 1 < nchunks && ((q + 1) << 5) + lane < K) nextv = lv[((q + 1) << 5) + lane];
                    const int32_t kc = min(32, K - (q << 5));
                    int32_t kk = 0;
                    for (; kk + 4 <= kc; kk += 4) {
                        const float4 k0 = win[kk], k1 = win[kk + 1], k2 = win[kk + 2], k3 = win[kk + 3];
                        uint32_t l0, h0, l1, h1, l2, h2, l3, h3;
                        G3_PAIR_BITS(k0, l0, h0);
                        G3_PAIR_BITS(k1, l1, h1);
                        G3_PAIR_BITS(k2, l2, h2);
                        G3_PAIR_BITS(k3, l3, h3);
                        red_shared_add(Jj + (l0 << 2), 1u);
                        red_shared_add(Jj + (l1 << 2), 1u);
                        red_shared_add(Jj + (l2 << 2), 1u);
                        red_shared_add(Jj + (l3 << 2), 1u);
                        if (((l0 ^ h0) | (l1 ^ h1) | (l2 ^ h2) | (l3 ^ h3)) != 0u) {
                            if (l0 != h0) fix_pair(k0, jx, jy, jz, l0, Jj, tp.T_t, tp.n_t);
                            if (l1 != h1) fix_pair(k1, jx, jy, jz, l1, Jj, tp.T_t, tp.n_t);
                            if (l2 != h2) fix_pair(k2, jx, jy, jz, l2, Jj, tp.T_t, tp.n_t);
                            if (l3 != h3) fix_pair(k3, jx, jy, jz, l3, Jj, tp.T_t, tp.n_t);
                        }
                    }
                    for (; kk < kc; ++kk) {
                        const float4 kv = win[kk];
                        uint32_t lo, hi;
                        G3_PAIR_BITS(kv, lo, hi);
                        red_shared_add(Jj + (lo << 2), 1u);
                        if (lo != hi) fix_pair(kv, jx, jy, jz, lo, Jj, tp.T_t, tp.n_t);
                    }
                }
            }
        }
    }
    __syncthreads();
    uint32_t* out = tp.scratch + (size_t)blockIdx.x * tp.tile_bins;
    for (int32_t i = threadIdx.x; i < tp.tile_bins; i += blockDim.x) {
        const uint32_t v = tile[i];
        if (v) out[i] += v;
    }
}

// Mirror the per-CTA partial tiles into the uint64 histogram (step a5) and clear them.
// One thread per slot; each slot maps to a unique (a, b, c), so no atomics are needed.
__global__ void __launch_bounds__(256)
merge_kernel(uint32_t* __restrict__ scratch, const uint32_t* __restrict__ slot_map,
             int32_t tile_bins, int32_t grid, int32_t n_r, int32_t n_t,
             unsigned long long* __restrict__ counts, unsigned long long* __restrict__ stats) {
    const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= tile_bins) return;
    unsigned long long v = 0;
    for (int32_t gidx = 0; gidx < grid; ++gidx) {
        uint32_t* p = scratch + (size_t)gidx * tile_bins + i;
        const uint32_t x = *p;
        if (x) { v += x; *p = 0; }
    }
    if (v == 0) return;
    const uint32_t m = slot_map[i];
    if (m == 0xFFFFFFFFu) { atomicAdd(stats + 3, v); return; }      // must never happen
    const int32_t a = (int32_t)(m >> 21), b = (int32_t)((m >> 11) & 1023), c = (int32_t)(m & 2047);
    if (c >= n_t) { atomicAdd(stats + 1, 2ull * v); return; }       // beyond 2 r_max: overflow
    if (a == b) counts[((size_t)a * n_r + a) * n_t + c] += 2ull * v;
    else {
        counts[((size_t)a * n_r + b) * n_t + c] += v;
        counts[((size_t)b * n_r + a) * n_t + c] += v;
    }
}

// ---------------------------------------------------------------------------------------------
// host side
inline size_t nb_smem_bytes(int32_t stage_cap, int32_t max_nb, int32_t n_r) {
    return (size_t)stage_cap * 12 + (size_t)kNbWarps * max_nb * 16 + (size_t)kNbWarps * n_r * 4;
}
inline size_t tri_smem_bytes(int64_t tile_bins, int warps) {
    return (((size_t)tile_bins * 4 + 15) & ~size_t(15)) + (size_t)warps * 32 * 16;
}

inline int32_t tiled_stage_cap(const g3_plan* p) {
    if (p->ncell == 1) return (int32_t)((p->n + 31) / 32 * 32);
    // twice the mean occupancy of 27 cells, and never less than min(n, 2048): clumped inputs
    // put far more than the mean into one neighbourhood
    const double per27 = 27.0 * (double)p->n / ((double)p->ncell * p->ncell * p->ncell);
    int64_t cap = (int64_t)(2.0 * per27) + 96;
    cap = std::max<int64_t>(cap, std::min<int64_t>(p->n, 2048));
    return (int32_t)((cap + 31) / 32 * 32);
}

// 2 if the tiled path can serve this plan, else 1 (generic).
inline int32_t tiled_select(g3_plan* p) {
    if (p->kernel_opt == 1) return 1;
    if (p->bins.n_r > 1023 || p->bins.n_t > 2046) return 1;
    if (p->max_nb > (1 << 20)) return 1;
    TiledState ts;
    build_layout(p, ts);
    if (ts.tile_bins > (1 << 22)) return 1;                        // addend must stay below 2^24
    if (tri_smem_bytes(ts.tile_bins, 8) > (size_t)p->smem_optin) return 1;   // TODO slabs
    if (nb_smem_bytes(tiled_stage_cap(p), p->max_nb, p->bins.n_r) > (size_t)p->smem_optin) return 1;
    if (p->ncell == 1 && p->n > 8192) return 1;
    // u32 tile counters: one launch must not be able to overflow a slot
    const long double per_frame = (long double)p->n * p->max_nb * (p->max_nb - 1) / 2;
    if (per_frame > 4.0e9L) return 1;
    return 2;
}

inline void tiled_free(g3_plan* p) {
    TiledState* ts = p->tiled;
    if (!ts) return;
    cudaFree(ts->d_addend); cudaFree(ts->d_jconst); cudaFree(ts->d_slot_map); cudaFree(ts->d_scratch);
    cudaFree(ts->d_nbv); cudaFree(ts->d_nbj); cudaFree(ts->d_nbcount); cudaFree(ts->d_work);
    delete ts;
    p->tiled = nullptr;
}

#define G3T_CUDA(call)                                                        \
    do {                                                                      \
        cudaError_t e__ = (call);                                             \
        if (e__ != cudaSuccess) {                                             \
            cudaGetLastError();                                               \
            return e__ == cudaErrorMemoryAllocation ? G3_ENOMEM : G3_ECUDA;   \
        }                                                                     \
    } while (0)

template <int kWarps>
inline int tiled_set_attr(size_t smem) {
    G3T_CUDA(cudaFuncSetAttribute(tiled_triplet_kernel<kWarps>,
                                  cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    return G3_OK;
}

inline int tiled_configure(g3_plan* p) {
    tiled_free(p);
    TiledState* ts = new (std::nothrow) TiledState;
    if (!ts) return G3_ENOMEM;
    p->tiled = ts;
    build_layout(p, *ts);
    p->tile_bins = ts->tile_bins;
    const int32_t n_r = p->bins.n_r, n_t = p->bins.n_t;

    // one launch (= one batch) must not be able to overflow a u32 slot, whatever the input
    const long double per_frame = (long double)p->n * p->max_nb * (p->max_nb - 1) / 2;
    ts->merge_every = (int64_t)std::max<long double>(1.0L, std::floor(4.0e9L / per_frame));
    if (p->batch_frames > ts->merge_every) p->batch_frames = (int32_t)ts->merge_every;

    ts->tri_warps = 32;
    while (ts->tri_warps > 8 && tri_smem_bytes(ts->tile_bins, ts->tri_warps) > (size_t)p->smem_optin)
        ts->tri_warps -= 8;
    ts->tri_smem = tri_smem_bytes(ts->tile_bins, ts->tri_warps);
    ts->grid = p->sm_count;
    ts->stage_cap = tiled_stage_cap(p);
    ts->nb_smem = nb_smem_bytes(ts->stage_cap, p->max_nb, n_r);

    std::vector<float> addend(n_r);
    std::vector<int32_t> jconst(n_r);
    for (int32_t b = 0; b < n_r; ++b) {
        addend[b] = kMagic + (float)(ts->BASE[b] - ts->g[b] + 1);
        jconst[b] = 4 * (ts->P[b] + ts->h[b]);
    }
    std::vector<uint32_t> slot_map((size_t)ts->tile_bins, 0xFFFFFFFFu);
    {
        std::vector<int32_t> clo(1), chi(1);
        for (int32_t a = 0; a < n_r; ++a)
            for (int32_t b = a; b < n_r; ++b) {
                int32_t lo, hi;
                reachable_c(p, a, b, lo, hi);
                for (int32_t c = lo; c <= hi; ++c) {
                    const int64_t slot = 1 + (int64_t)ts->BASE[b] + ts->P[a] + c - ts->g[b] + ts->h[a];
                    if (slot < 1 || slot >= ts->tile_bins - 1 || slot_map[slot] != 0xFFFFFFFFu) return G3_EINVAL;
                    slot_map[slot] = ((uint32_t)a << 21) | ((uint32_t)b << 11) | (uint32_t)c;
                }
            }
    }
    const size_t per_frame_entries = (size_t)p->n * p->max_nb;
    const size_t B = (size_t)p->batch_frames;
    G3T_CUDA(cudaMalloc(&ts->d_addend, sizeof(float) * n_r));
    G3T_CUDA(cudaMalloc(&ts->d_jconst, sizeof(int32_t) * n_r));
    G3T_CUDA(cudaMalloc(&ts->d_slot_map, sizeof(uint32_t) * ts->tile_bins));
    G3T_CUDA(cudaMalloc(&ts->d_scratch, sizeof(uint32_t) * ts->tile_bins * ts->grid));
    G3T_CUDA(cudaMalloc(&ts->d_nbv, sizeof(float4) * per_frame_entries * B));
    G3T_CUDA(cudaMalloc(&ts->d_nbj, sizeof(int32_t) * per_frame_entries * B));
    G3T_CUDA(cudaMalloc(&ts->d_nbcount, sizeof(int32_t) * (size_t)p->n * B));
    G3T_CUDA(cudaMalloc(&ts->d_work, sizeof(unsigned int)));
    G3T_CUDA(cudaMemcpy(ts->d_addend, addend.data(), sizeof(float) * n_r, cudaMemcpyHostToDevice));
    G3T_CUDA(cudaMemcpy(ts->d_jconst, jconst.data(), sizeof(int32_t) * n_r, cudaMemcpyHostToDevice));
    G3T_CUDA(cudaMemcpy(ts->d_slot_map, slot_map.data(), sizeof(uint32_t) * ts->tile_bins, cudaMemcpyHostToDevice));
    G3T_CUDA(cudaMemset(ts->d_scratch, 0, sizeof(uint32_t) * ts->tile_bins * ts->grid));
    G3T_CUDA(cudaFuncSetAttribute(neighbour_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ts->nb_smem));
    G3T_CUDA(cudaFuncSetAttribute(neighbour_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ts->nb_smem));
    int rc = G3_OK;
    switch (ts->tri_warps) {
        case 32: rc = tiled_set_attr<32>(ts->tri_smem); break;
        case 24: rc = tiled_set_attr<24>(ts->tri_smem); break;
        case 16: rc = tiled_set_attr<16>(ts->tri_smem); break;
        default: rc = tiled_set_attr<8>(ts->tri_smem); break;
    }
    (void)n_t;
    return rc;
}

inline int tiled_merge(g3_plan* p, cudaStream_t st) {
    TiledState* ts = p->tiled;
    if (!ts || ts->frames_since_merge == 0) return G3_OK;
    merge_kernel<<<(unsigned)((ts->tile_bins + 255) / 256), 256, 0, st>>>(
        ts->d_scratch, ts->d_slot_map, (int32_t)ts->tile_bins, ts->grid, p->bins.n_r, p->bins.n_t,
        p->d_counts, p->d_stats);
    p->launches += 1;
    ts->frames_since_merge = 0;
    G3T_CUDA(cudaGetLastError());
    return G3_OK;
}

inline int tiled_launch(g3_plan* p, const FrameBatch& fb, const BinSpec& bs, cudaStream_t st) {
    TiledState* ts = p->tiled;
    if (!ts) return G3_ESTATE;
    // scratch slots are u32 too: merge before their worst case could overflow
    if (ts->frames_since_merge + fb.n_frames > ts->merge_every) {
        int rc = tiled_merge(p, st);
        if (rc != G3_OK) return rc;
    }
    const double w = (p->r_max / (double)bs.n_r) * p->inv_g;
    const double wt = ((2.0 * p->r_max) / (double)bs.n_t) * p->inv_g;
    const double eps = 1.0 / 1048576.0;
    NbParams np;
    np.max_nb = p->max_nb; np.stage_cap = ts->stage_cap; np.n_r = bs.n_r;
    np.cut2 = bs.cut2;
    np.cut_lo = (float)((double)bs.cut2 * (1.0 - eps));
    np.cut_hi = (float)((double)bs.cut2 * (1.0 + eps));
    np.inv_w_lo = (float)((1.0 / w) * (1.0 - eps));
    np.inv_w_hi = (float)((1.0 / w) * (1.0 + eps));
    np.T_r = bs.T_r; np.addend = ts->d_addend; np.jconst = ts->d_jconst;
    np.nbv = ts->d_nbv; np.nbj = ts->d_nbj; np.nbcount = ts->d_nbcount; np.stats = p->d_stats;
    G3T_CUDA(cudaMemsetAsync(ts->d_work, 0, sizeof(unsigned int), st));
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    if (p->timing) {
        for (int i = 0; i < 3; ++i) {
            if (p->ev_used == p->ev_pool.size()) {
                cudaEvent_t e;
                G3T_CUDA(cudaEventCreate(&e));
                p->ev_pool.push_back(e);
            }
            ev[i] = p->ev_pool[p->ev_used++];
        }
        G3T_CUDA(cudaEventRecord(ev[0], st));
    }
    if (fb.ncell == 1) {
        dim3 grid((unsigned)fb.n_frames, (unsigned)((fb.n + 63) / 64));
        neighbour_kernel<true><<<grid, kNbWarps * 32, ts->nb_smem, st>>>(fb, np);
    } else {
        dim3 grid((unsigned)((long long)fb.n_frames * fb.ncell3), 1);
        neighbour_kernel<false><<<grid, kNbWarps * 32, ts->nb_smem, st>>>(fb, np);
    }
    if (p->timing) G3T_CUDA(cudaEventRecord(ev[1], st));
    TriParams tp;
    tp.total_centres = (long long)fb.n_frames * fb.n;
    tp.max_nb = p->max_nb; tp.n_t = bs.n_t; tp.tile_bins = (int32_t)ts->tile_bins;
    tp.inv_lo = (float)((1.0 / wt) * (1.0 - eps));
    tp.inv_hi = (float)((1.0 / wt) * (1.0 + eps));
    tp.T_t = bs.T_t; tp.nbv = ts->d_nbv; tp.nbj = ts->d_nbj; tp.nbcount = ts->d_nbcount;
    tp.work = ts->d_work; tp.scratch = ts->d_scratch;
    switch (ts->tri_warps) {
        case 32: tiled_triplet_kernel<32><<<ts->grid, 32 * 32, ts->tri_smem, st>>>(tp); break;
        case 24: tiled_triplet_kernel<24><<<ts->grid, 24 * 32, ts->tri_smem, st>>>(tp); break;
        case 16: tiled_triplet_kernel<16><<<ts->grid, 16 * 32, ts->tri_smem, st>>>(tp); break;
        default: tiled_triplet_kernel<8><<<ts->grid, 8 * 32, ts->tri_smem, st>>>(tp); break;
    }
    if (p->timing) G3T_CUDA(cudaEventRecord(ev[2], st));
    p->launches += 2;
    ts->frames_since_merge += fb.n_frames;
    G3T_CUDA(cudaGetLastError());
    return G3_OK;
}

}  // namespace g3
