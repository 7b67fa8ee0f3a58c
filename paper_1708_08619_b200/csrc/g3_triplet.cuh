// g3_triplet.cuh -- steps a4 + a5: the triplet kernel (Algorithm 7 CUDA_g3)
// and the merge of its per-CTA partial histograms.
//
// tiled_triplet_kernel: persistent, one CTA per SM, a warp per centre.  The centre's neighbour
// list (sorted by shell, so a_j <= a_k for j < k; written by the neighbour kernels already in window
// form) is staged in a per-warp shared-memory window; every UNORDERED pair j < k is visited once
// and counted with one shared-memory atomic into a privatised histogram tile that holds only the
// bins the triangle inequality allows:
//     slot(a, b, c) = 1 + BASE(b) + P(a) + c - g(b) + h(a)          (a <= b)
// (DESIGN.md section 5.3).  The k side of a pair comes from the window as (x, y, z, addend(b)),
// the j side is held in registers as (x, y, z, row offset(a)): four j entries per lane
// (g, g + 8, g + 16, g + 24 of a 32-block, g = lane & 7), so that one quarter-warp broadcast load
// of a k entry serves four pairs.  Slot 0 is a guard: lanes without a pair in an iteration add
// to it, so every shared atomic is issued by a full, converged warp (measured on B200: a
// full-warp ATOMS.POPC.INC retires in 2.3-2.8 SM cycles whatever the bank conflicts, a partially
// predicated one in 4.1).  The list of the NEXT centre is loaded into registers while the current
// one is processed.  When the kernel ends each CTA adds its tile to its own uint64 partial tile
// in global memory; merge_kernel mirrors the partial tiles into the [a][b][c] histogram.
//
// Exactness.  Differences of neighbour vectors are exact in fp32 (integers below 2^21).  The
// squared distance, its square root and the bin index are computed in fp32 with a relative
// error below 2^-21; the bin is taken twice, with the scale factor lowered and raised by
// 2^-20.  If both agree, the exact integer rule bin(T_t, t2) gives the same bin (the exact
// quotient lies between the two); if they differ the pair is redone in 64-bit integers
// against the exact edge table and the histogram is corrected.
#pragma once

#include "g3_neighbour.cuh"

namespace g3 {

constexpr int kItemCentres = 8;                // centres per work-queue fetch
constexpr int kWinEntries = 64;                // entries of a warp's window
constexpr int kWinBytes = kWinEntries * 20;    // (x, y, z, addend) + row offset per entry

struct TriParams {
    long long total_centres;              // frames * n
    int32_t max_nb, n_t, n_r;
    int32_t tile_bins;
    uint32_t cta_item_cap;                // items one CTA may take (u32 tile slots cannot overflow)
    float inv_lo, inv_hi;                 // (1/wt)(1 -+ 2^-20), wt = t-bin width in grid units
    const unsigned long long* T_t;
    const float4* nbv;                    // [centres][max_nb] (dx, dy, dz, addend(shell))
    const uint32_t* nbj;                  // [centres][max_nb] 4 * (P(shell) + h(shell))
    const int32_t* nbcount;
    unsigned int* work;
    unsigned long long* scratch;          // [grid][scratch_stride], already offset by slot_base
    // slab passes (kSlab kernels): this launch counts only pairs whose outer member k lies in
    // the shell range of slab `slab`; its tile holds the slots slot_base+1 .. slot_base+tile_bins-2
    long long scratch_stride;             // slots of one CTA's partial tile: the whole layout
    int32_t slot_base;                    // BASE(first shell of the slab)
    int32_t n_slabs, slab;
    const int32_t* slabpos;               // [centres][n_slabs + 1] list position where each slab starts
};

__device__ __forceinline__ void red_shared_add(uint32_t addr, uint32_t v) {
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// One pair: j = (jx, jy, jz), k = kv (x, y, z, addend of k's shell).  Returns the fp32 slot bits
// twice, with the scale lowered and raised by 2^-20.
__device__ __forceinline__ void pair_bits(const float4 kv, float jx, float jy, float jz,
                                          float inv_lo, float inv_hi, uint32_t& lo, uint32_t& hi) {
    const float ex = kv.x - jx, ey = kv.y - jy, ez = kv.z - jz;
    const float t2 = fmaf(ez, ez, fmaf(ey, ey, ex * ex));
    const float t = sqrt_approx(t2);
    lo = __float_as_uint(__fmaf_rd(t, inv_lo, kv.w));
    hi = __float_as_uint(__fmaf_rd(t, inv_hi, kv.w));
}

// Redo one pair exactly (64-bit integers, exact edge table) and move its count if the fp32 bin
// was wrong.  Called only for pairs whose two fp32 bins differ.
__device__ __noinline__ void fix_pair(float4 kv, float jx, float jy, float jz, uint32_t lo,
                                      uint32_t Jj, const unsigned long long* __restrict__ T_t,
                                      int32_t n_t) {
    const unsigned long long t2 = exact_d2(kv.x - jx, kv.y - jy, kv.z - jz);
    const int32_t c_exact = bin_search(T_t, n_t, t2);
    const int32_t kk1 = (int32_t)(kv.w - kMagic);                 // BASE(b) - g(b) + 1, exact
    const int32_t c_fast = (int32_t)(lo - kMagicBits) - kk1;
    if (c_exact != c_fast) {
        const uint32_t addr = Jj + (lo << 2);
        red_shared_add(addr, 0xFFFFFFFFu);
        red_shared_add(addr + 4u * (uint32_t)(c_exact - c_fast), 1u);
    }
}

// The j side of a pair: vector and the tile byte address of its shell row (window base folded in).
struct JSide {
    float x, y, z;
    uint32_t J;
};

__device__ __forceinline__ JSide load_jside(const float4* __restrict__ win, const uint32_t* __restrict__ winJ, int idx) {
    const float4 v = win[idx];
    JSide r;
    r.x = v.x; r.y = v.y; r.z = v.z; r.J = winJ[idx];
    return r;
}

// Four independent pairs (j0,k0) .. (j3,k3) of this lane.  pN = the lane really has pair N; a
// lane without one adds to the guard slot, so every shared atomic is issued by the full warp.
// kPred = false: all four exist on every lane (the predicates are ignored).
template <bool kPred>
__device__ __forceinline__ void four_pairs(const TriParams& tp, uint32_t guard,
                                           const float4 k0, const float4 k1, const float4 k2, const float4 k3,
                                           const JSide& j0, const JSide& j1, const JSide& j2, const JSide& j3,
                                           bool p0, bool p1, bool p2, bool p3) {
    if (!kPred) p0 = p1 = p2 = p3 = true;
    uint32_t l0, h0, l1, h1, l2, h2, l3, h3;
    pair_bits(k0, j0.x, j0.y, j0.z, tp.inv_lo, tp.inv_hi, l0, h0);
    pair_bits(k1, j1.x, j1.y, j1.z, tp.inv_lo, tp.inv_hi, l1, h1);
    pair_bits(k2, j2.x, j2.y, j2.z, tp.inv_lo, tp.inv_hi, l2, h2);
    pair_bits(k3, j3.x, j3.y, j3.z, tp.inv_lo, tp.inv_hi, l3, h3);
    red_shared_add(p0 ? j0.J + (l0 << 2) : guard, 1u);
    red_shared_add(p1 ? j1.J + (l1 << 2) : guard, 1u);
    red_shared_add(p2 ? j2.J + (l2 << 2) : guard, 1u);
    red_shared_add(p3 ? j3.J + (l3 << 2) : guard, 1u);
    if (((l0 ^ h0) | (l1 ^ h1) | (l2 ^ h2) | (l3 ^ h3)) != 0u) {
        if (p0 && l0 != h0) fix_pair(k0, j0.x, j0.y, j0.z, l0, j0.J, tp.T_t, tp.n_t);
        if (p1 && l1 != h1) fix_pair(k1, j1.x, j1.y, j1.z, l1, j1.J, tp.T_t, tp.n_t);
        if (p2 && l2 != h2) fix_pair(k2, j2.x, j2.y, j2.z, l2, j2.J, tp.T_t, tp.n_t);
        if (p3 && l3 != h3) fix_pair(k3, j3.x, j3.y, j3.z, l3, j3.J, tp.T_t, tp.n_t);
    }
}

// The four j entries a lane holds of the 32-block at `win`: g, g + 8, g + 16, g + 24 (g = lane & 7).
struct JQuad {
    JSide j[4];
};

__device__ __forceinline__ JQuad load_jquad(const float4* __restrict__ win, const uint32_t* __restrict__ winJ, int lane) {
    JQuad q;
    const int g = lane & 7;
#pragma unroll
    for (int m = 0; m < 4; ++m) q.j[m] = load_jside(win, winJ, g + 8 * m);
    return q;
}

// All unordered pairs inside one 32-block of a neighbour list whose entries 0..kt-1 are valid
// (16 < kt <= 32) and staged in `win` (vectors + addends) and `winJ` (row offsets); `q` = the
// block's j entries this lane holds.  Recursive halving: at level H (16, 8, 4, 2, 1) the block
// splits into aligned sub-blocks of 2H entries and every pair whose members first differ in bit H
// is visited, j from the lower half (so j < k and a_j <= a_k), k from the upper half.  Each level
// is an H x H rectangle per sub-block.  Levels 16 and 8 take their j side from `q`; their k side
// is one address per quarter-warp.  A full block takes 16 pair slots per lane for its 496 pairs
// (97 % of the lane slots used); a lane-vs-broadcast triangle would take 31 (50 %).
template <bool kFull>
__device__ __forceinline__ void triangle32(const TriParams& tp, const float4* __restrict__ win,
                                           const uint32_t* __restrict__ winJ, uint32_t guard,
                                           int lane, int32_t kt, const JQuad& q) {
    const int kq = lane >> 3;
    {   // H = 16: j = {g, g + 8}, k = 16 + kq + 4 it, it = 0..3
        const int kidx = 16 + kq;
        {
            const float4 k0 = win[kidx], k1 = win[kidx + 4];
            four_pairs<!kFull>(tp, guard, k0, k0, k1, k1, q.j[0], q.j[1], q.j[0], q.j[1],
                               kidx < kt, kidx < kt, kidx + 4 < kt, kidx + 4 < kt);
        }
        if (kFull || kt > 24) {
            const float4 k0 = win[kidx + 8], k1 = win[kidx + 12];
            four_pairs<!kFull>(tp, guard, k0, k0, k1, k1, q.j[0], q.j[1], q.j[0], q.j[1],
                               kidx + 8 < kt, kidx + 8 < kt, kidx + 12 < kt, kidx + 12 < kt);
        }
    }
    {   // H = 8: j = g with k = 8 + 2 kq + {0, 1}; j = g + 16 with k = 24 + 2 kq + {0, 1}
        const int ka = 8 + 2 * kq, kb = 24 + 2 * kq;
        const float4 k0 = win[ka], k1 = win[ka + 1], k2 = win[kb], k3 = win[kb + 1];
        four_pairs<!kFull>(tp, guard, k0, k1, k2, k3, q.j[0], q.j[0], q.j[2], q.j[2],
                           true, true, kb < kt, kb + 1 < kt);
    }
    {   // H = 4 (j = {b + g, b + g + 2}, k = b + 4 + kg), H = 2 and H = 1 (one pair each)
        const int b8 = lane & 24, g = lane & 1, k4 = b8 + 4 + ((lane >> 1) & 3);
        const JSide ja = load_jside(win, winJ, b8 + g), jb = load_jside(win, winJ, b8 + g + 2);
        const int b4 = lane & 28, k2 = b4 + 2 + ((lane >> 1) & 1);
        const JSide jc = load_jside(win, winJ, b4 + g);
        const JSide own = load_jside(win, winJ, lane);
        const int k1 = lane | 1;
        const float4 kA = win[k4], kB = win[k2], kC = win[k1];
        four_pairs<true>(tp, guard, kA, kA, kB, kC, ja, jb, jc, own,
                         kFull || k4 < kt, kFull || k4 < kt, kFull || k2 < kt, g == 0 && (kFull || k1 < kt));
    }
}

// Same for a block with 2 <= kt <= 16 valid entries: the 8 x 8, 4 x 4, 2 x 2 and 1 x 1
// rectangles are spread over all 32 lanes, four pair slots per lane for up to 120 pairs.
__device__ __forceinline__ void triangle16(const TriParams& tp, const float4* __restrict__ win,
                                           const uint32_t* __restrict__ winJ, uint32_t guard,
                                           int lane, int32_t kt) {
    // H = 8: j = lane & 7, k = 8 + kg + 4 it (it = 0..1)
    const int kidx = 8 + (lane >> 3);
    const JSide ja = load_jside(win, winJ, lane & 7);
    // H = 4, two sub-blocks: j = b + (lane & 3), k = b + 4 + kg
    const int b = (lane >> 4) << 3, k4 = b + 4 + ((lane >> 2) & 3);
    const JSide jb = load_jside(win, winJ, b + (lane & 3));
    // H = 2 on lanes 0..15 (four sub-blocks), H = 1 on lanes 16..23 (eight pairs)
    const bool low = lane < 16;
    const int b4 = (lane >> 2) << 2;
    const int jl = low ? b4 + (lane & 1) : 2 * (lane & 7);
    const int kl = low ? b4 + 2 + ((lane >> 1) & 1) : 2 * (lane & 7) + 1;
    const JSide jc = load_jside(win, winJ, jl);
    const float4 k0 = win[kidx], k1 = win[kidx + 4], kB = win[k4], kC = win[kl];
    four_pairs<true>(tp, guard, k0, k1, kB, kC, ja, ja, jb, jc,
                     kidx < kt, kidx + 4 < kt, k4 < kt, lane < 24 && kl < kt);
}

// Rectangle between the 32-block whose j entries are in `q` and the window entries
// kwin[klo .. kc): k = 4 i + kq per quarter-warp, four pairs (one per held j) per lane.
__device__ __forceinline__ void rect32(const TriParams& tp, const float4* __restrict__ kwin, uint32_t guard,
                                       int lane, int32_t klo, int32_t kc, const JQuad& q) {
    const int kq = lane >> 3;
    int32_t k0 = klo & ~3;
    if (k0 < klo) {                                       // slab passes: first group bounded below
        const int32_t kidx = k0 + kq;
        const float4 kv = kwin[kidx];
        const bool p = kidx >= klo && kidx < kc;
        four_pairs<true>(tp, guard, kv, kv, kv, kv, q.j[0], q.j[1], q.j[2], q.j[3], p, p, p, p);
        k0 += 4;
    }
    for (; k0 + 4 <= kc; k0 += 4) {
        const float4 kv = kwin[k0 + kq];
        four_pairs<false>(tp, guard, kv, kv, kv, kv, q.j[0], q.j[1], q.j[2], q.j[3], true, true, true, true);
    }
    if (k0 < kc) {
        const float4 kv = kwin[k0 + kq];
        const bool p = k0 + kq < kc;
        four_pairs<true>(tp, guard, kv, kv, kv, kv, q.j[0], q.j[1], q.j[2], q.j[3], p, p, p, p);
    }
}

// Rectangle between the 16 entries jwin[0..16) (all valid) and kwin[0..m), 1 <= m <= 16:
// j = {g, g + 8}, k = 4 i + kq.
__device__ __forceinline__ void rect16(const TriParams& tp, const float4* __restrict__ jwin,
                                       const uint32_t* __restrict__ jwinJ, const float4* __restrict__ kwin,
                                       uint32_t guard, int lane, int32_t m) {
    const int kq = lane >> 3, g = lane & 7;
    const JSide ja = load_jside(jwin, jwinJ, g), jb = load_jside(jwin, jwinJ, g + 8);
    for (int32_t i0 = 0; i0 < m; i0 += 8) {
        const float4 k0 = kwin[i0 + kq], k1 = kwin[i0 + 4 + kq];
        const bool p0 = i0 + kq < m, p1 = i0 + 4 + kq < m;
        four_pairs<true>(tp, guard, k0, k0, k1, k1, ja, jb, ja, jb, p0, p0, p1, p1);
    }
}

// Triangle of a 32-block whose k members are bounded below (slab passes): lane = j, the k
// members klo <= k < kt are broadcast four at a time.  Runs at most once per centre and slab.
__device__ __forceinline__ void triangle_from(const TriParams& tp, const float4* __restrict__ win,
                                              uint32_t guard, int lane, int32_t klo, int32_t kt,
                                              const JSide& own) {
    for (int32_t k0 = klo; k0 < kt; k0 += 4) {
        const float4 ka = win[k0], kb = win[min(k0 + 1, 31)], kc = win[min(k0 + 2, 31)], kd = win[min(k0 + 3, 31)];
        four_pairs<true>(tp, guard, ka, kb, kc, kd, own, own, own, own,
                         lane < k0, lane < k0 + 1 && k0 + 1 < kt, lane < k0 + 2 && k0 + 2 < kt,
                         lane < k0 + 3 && k0 + 3 < kt);
    }
}

// All pairs inside a block of 2 <= kt <= 32 entries at `win`.
__device__ __forceinline__ void block_pairs(const TriParams& tp, const float4* __restrict__ win,
                                            const uint32_t* __restrict__ winJ, uint32_t guard,
                                            int lane, int32_t kt, const JQuad& q) {
    if (kt == 32) triangle32<true>(tp, win, winJ, guard, lane, kt, q);
    else if (kt > 16) triangle32<false>(tp, win, winJ, guard, lane, kt, q);
    else if (kt >= 2) triangle16(tp, win, winJ, guard, lane, kt);
}

template <int kWarps, bool kSlab>
__global__ void __launch_bounds__(kWarps * 32, 1)
tiled_triplet_kernel(TriParams tp) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t* tile = reinterpret_cast<uint32_t*>(smem_raw);
    const size_t tile_bytes = ((size_t)tp.tile_bins * 4 + 15) & ~size_t(15);
    __shared__ unsigned int cta_items;

    for (int32_t i = threadIdx.x; i < tp.tile_bins; i += blockDim.x) tile[i] = 0;
    if (threadIdx.x == 0) cta_items = 0;
    __syncthreads();

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    float4* win = reinterpret_cast<float4*>(smem_raw + tile_bytes + (size_t)wid * kWinBytes);   // [64] k side
    uint32_t* winJ = reinterpret_cast<uint32_t*>(win + kWinEntries);                             // [64] row addresses
    const uint32_t guard = (uint32_t)__cvta_generic_to_shared(tile);      // slot 0
    // shared-window byte address of slot 0 minus the magic bits (mod 2^32), see file header
    const uint32_t cbase = guard - (kMagicBits << 2) - (kSlab ? ((uint32_t)tp.slot_base << 2) : 0u);
    const long long n_items = (tp.total_centres + kItemCentres - 1) / kItemCentres;

    // work queue: a CTA first takes one of its own `cta_item_cap` tickets, then a global item
    auto fetch_item = [&]() -> long long {
        unsigned int it = 0xFFFFFFFFu;
        if (lane == 0 && atomicAdd(&cta_items, 1u) < tp.cta_item_cap) it = atomicAdd(tp.work, 1u);
        it = __shfl_sync(0xffffffffu, it, 0);
        return it < n_items ? (long long)it : -1;
    };

    long long item = fetch_item();
    if (item >= 0) {
        long long item_next = fetch_item();
        long long c = item * kItemCentres;
        long long c_end = min(c + (long long)kItemCentres, tp.total_centres);
        int32_t Kn = tp.nbcount[c], ksn = 0;
        if (kSlab) {
            const int32_t* sp = tp.slabpos + c * (tp.n_slabs + 1) + tp.slab;
            ksn = sp[0]; Kn = sp[1];              // entries at or beyond the slab's end are not needed
        }
        float4 v0n = tp.nbv[c * tp.max_nb + lane], v1n = tp.nbv[c * tp.max_nb + 32 + lane];
        uint32_t j0n = tp.nbj[c * tp.max_nb + lane], j1n = tp.nbj[c * tp.max_nb + 32 + lane];
        bool more = true;
        while (more) {
            const int32_t K = Kn, ks = ksn;
            const float4 v0 = v0n, v1 = v1n;
            const uint32_t j0 = j0n, j1 = j1n;
            const float4* __restrict__ lv = tp.nbv + c * tp.max_nb;
            const uint32_t* __restrict__ lj = tp.nbj + c * tp.max_nb;
            // ---- advance and prefetch the next centre ------------------------------------------
            ++c;
            if (c >= c_end) {
                if (item_next >= 0) {
                    c = item_next * kItemCentres;
                    c_end = min(c + (long long)kItemCentres, tp.total_centres);
                    item_next = fetch_item();
                } else more = false;
            }
            if (more) {
                if (kSlab) {
                    const int32_t* sp = tp.slabpos + c * (tp.n_slabs + 1) + tp.slab;
                    ksn = sp[0]; Kn = sp[1];
                } else Kn = tp.nbcount[c];
                v0n = tp.nbv[c * tp.max_nb + lane];
                v1n = tp.nbv[c * tp.max_nb + 32 + lane];
                j0n = tp.nbj[c * tp.max_nb + lane];
                j1n = tp.nbj[c * tp.max_nb + 32 + lane];
            }
            if (K < 2 || (kSlab && ks >= K)) continue;

            if (!kSlab && K <= kWinEntries) {
                // ---- the whole list fits the window: entries 0..31 = block A, 32..K-1 = block B ----
                __syncwarp();
                win[lane] = v0; win[32 + lane] = v1;
                winJ[lane] = cbase + j0; winJ[32 + lane] = cbase + j1;
                __syncwarp();
                const JQuad qa = load_jquad(win, winJ, lane);
                block_pairs(tp, win, winJ, guard, lane, min(K, 32), qa);
                const int32_t kb = K - 32;
                if (kb > 0) {
                    rect32(tp, win + 32, guard, lane, 0, kb, qa);
                    if (kb <= 16) {
                        if (kb >= 2) triangle16(tp, win + 32, winJ + 32, guard, lane, kb);
                    } else {                               // B = 16 + m entries
                        triangle16(tp, win + 32, winJ + 32, guard, lane, 16);
                        rect16(tp, win + 32, winJ + 32, win + 48, guard, lane, kb - 16);
                        if (kb >= 18) triangle16(tp, win + 48, winJ + 48, guard, lane, kb - 16);
                    }
                }
                continue;
            }

            // ---- long lists and slab passes: a 32-block of j entries against all later k ----------
            float4* winB = win + 32;
            const int32_t nchunks = (K + 31) >> 5;
            for (int32_t r = 0; r < nchunks; ++r) {
                const int32_t jidx = (r << 5) + lane;
                float4 jraw = r == 0 ? v0 : v1;
                uint32_t jj = r == 0 ? j0 : j1;
                if (r >= 2 && jidx < K) { jraw = lv[jidx]; jj = lj[jidx]; }
                // prefetch the first rectangular window while the triangle runs
                // (slab passes: the first k block is the one that holds list position ks)
                const int32_t q_first = kSlab ? max(r + 1, ks >> 5) : r + 1;
                float4 nextv = v1;
                if (q_first >= 2 && q_first < nchunks && (q_first << 5) + lane < K) nextv = lv[(q_first << 5) + lane];

                // ---- triangle: both members in this 32-block -------------------------------------
                __syncwarp();
                win[lane] = jraw;
                winJ[lane] = cbase + jj;
                __syncwarp();
                const int32_t kt = min(32, K - (r << 5));
                const JQuad qa = load_jquad(win, winJ, lane);
                if (kSlab && ks > (r << 5)) {          // k members bounded below inside this block
                    if (ks < (r << 5) + kt) {
                        JSide own;
                        own.x = jraw.x; own.y = jraw.y; own.z = jraw.z; own.J = cbase + jj;
                        triangle_from(tp, win, guard, lane, ks - (r << 5), kt, own);
                    }
                } else block_pairs(tp, win, winJ, guard, lane, kt, qa);
                if (r + 1 == nchunks) break;

                // ---- rectangles: k in later 32-blocks; this block is full ---------------------------
                for (int32_t q = q_first; q < nchunks; ++q) {
                    __syncwarp();
                    winB[lane] = nextv;
                    __syncwarp();
                    if (q + 1 < nchunks && ((q + 1) << 5) + lane < K) nextv = lv[((q + 1) << 5) + lane];
                    const int32_t kc = min(32, K - (q << 5));
                    const int32_t klo = kSlab ? max(0, ks - (q << 5)) : 0;
                    rect32(tp, winB, guard, lane, klo, kc, qa);
                }
            }
        }
    }
    __syncthreads();
    unsigned long long* out = tp.scratch + (size_t)blockIdx.x * (size_t)tp.scratch_stride;
    for (int32_t i = 1 + threadIdx.x; i < tp.tile_bins - 1; i += blockDim.x) {
        const uint32_t v = tile[i];
        if (v) out[i] += v;
    }
    // the two guard slots hold only the dummy adds of lanes without a pair; the top one must stay
    // empty: anything there is reported through the unmapped slot 0 of the partial tile (stats[3])
    if (threadIdx.x == 0 && tile[tp.tile_bins - 1] != 0) out[kSlab ? -(long long)tp.slot_base : 0] += tile[tp.tile_bins - 1];
}

// Mirror the per-CTA partial tiles into the uint64 histogram (step a5) and clear them.
// One thread per slot; each slot maps to a unique (a, b, c), so no atomics are needed.
// stats[3] counts what must never happen: counts in a slot no (a, b, c) maps to, or in a
// top guard slot (slot 0 of a CTA's partial tile, see above).
__global__ void __launch_bounds__(256)
merge_kernel(unsigned long long* __restrict__ scratch, const uint32_t* __restrict__ slot_map,
             int32_t tile_bins, int32_t grid, int32_t n_r, int32_t n_t,
             unsigned long long* __restrict__ counts, unsigned long long* __restrict__ stats) {
    const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= tile_bins) return;
    unsigned long long v = 0;
    for (int32_t gidx = 0; gidx < grid; ++gidx) {
        unsigned long long* p = scratch + (size_t)gidx * tile_bins + i;
        const unsigned long long x = *p;
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

inline size_t tri_smem_bytes(int64_t tile_bins, int warps, int32_t n_r) {
    (void)n_r;
    return (((size_t)tile_bins * 4 + 15) & ~size_t(15)) + (size_t)warps * kWinBytes;
}

}  // namespace g3
