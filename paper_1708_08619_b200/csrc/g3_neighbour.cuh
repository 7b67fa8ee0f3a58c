// g3_neighbour.cuh -- step a3: minimum-image neighbour lists inside r_max, sorted by shell, and
// the pair histogram g2 over the same range.
//
// Algorithm 7 CUDA_g2 "store minimum image neighbour vectors" and "update the g2 histogram"
// (PAPER.md:518-520), done with a cell list instead of the paper's all-particle scan
// (PAPER.md:513-515).
//
// Two kernels (descriptions at their definitions): neighbour_cell_kernel for cell grids -- a
// producer warp stages the 27 surrounding cells of a (cell, frame) item by TMA, consumer warps scan
// them for three centres at a time, keep hits as stage indices, decide acceptance and shell
// exactly, sort by shell with a shared-memory counting sort and write the lists in the triplet
// kernel's window form: nbv[centre][pos] = (dx, dy, dz, addend(a)), nbj[centre][pos] = row offset(a);
// neighbour_all_kernel for the degenerate grid (the whole frame staged per CTA).  The shell counts
// are also the g2 histogram.  The order inside a shell depends on the atomics' arrival order; the
// histograms do not.
#pragma once

#include "g3_generic.cuh"
#include "g3_plan.h"

namespace g3 {

constexpr float kMagic = 12582912.0f;          // 1.5 * 2^23: fp32 integers with ulp 1 around it
constexpr uint32_t kMagicBits = 0x4B400000u;
constexpr int kNbWarps = 4;                    // (consumer) warps per neighbour kernel CTA
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
    float4* crowd_scratch;                // [grid][kNbWarps][max_nb] lists of the crowded path (neighbour_cell_kernel)
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

// Phase A of the degenerate-grid kernel for 32 candidates: `c` is this lane's candidate in raw grid
// coordinates, `skip` = it is the centre itself; the difference is wrapped to the minimum image.
// Accepted candidates are ballot-compacted into the warp's list (shared address `scratch_s`,
// 16 B per entry) as (dx, dy, dz, d2).
__device__ __forceinline__ void nb_test_wrap(const float4 c, bool skip, float px, float py, float pz,
                                             float cut_hi, uint32_t lt_mask, int32_t max_nb,
                                             uint32_t scratch_s, int32_t& count) {
    float dx = c.x - px, dy = c.y - py, dz = c.z - pz;
    dx += dx < -524288.f ? 1048576.f : 0.f; dx -= dx >= 524288.f ? 1048576.f : 0.f;
    dy += dy < -524288.f ? 1048576.f : 0.f; dy -= dy >= 524288.f ? 1048576.f : 0.f;
    dz += dz < -524288.f ? 1048576.f : 0.f; dz -= dz >= 524288.f ? 1048576.f : 0.f;
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

// ---------------------------------------------------------------------------------------------
// neighbour_cell_kernel: the cell-grid path (ncell > 1).
//
// Persistent CTAs (4 warps) stride over (cell, frame) items.  Per item:
//   stage  the particles of the 27 surrounding cells (up to 18 contiguous ranges of the cell-major
//          fp32 copy of the frame) are copied into shared memory by the TMA engine
//          (cp.async.bulk + mbarrier: no LSU instructions); ranges that wrap around the box get
//          their periodic shift (+-2^20, exact in fp32) added in place, so the minimum-image
//          vector of a neighbour is a plain difference of staged coordinates;
//   A      a warp scans the stage for up to three of its centres at once (one LDS.128 per 32
//          candidates serves three distance tests) and keeps the stage INDEX of every candidate
//          with fp32 d2 < cut (widened by 2^-20) in a per-centre u16 list; the centre itself
//          passes the test and is dropped in phase B by its index;
//   B, C   per centre: the list entries (two per lane) are fetched again, the exact acceptance
//          test / shell are taken as in nb_shell, entries are ranked inside their shell by a
//          shared atomic, the shell counts are scanned and the entries written to global memory
//          in shell order in the triplet kernel's window format.
// The order inside a shell depends on the atomics' arrival order; the histograms do not.
constexpr int kNbMaxG = 3;                       // centres scanned together by one warp
constexpr int kNbStages = 2;                     // ring of candidate stages per CTA

__device__ __forceinline__ uint32_t lds_u16(uint32_t addr) {
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr) : "memory");
    return v;
}

__device__ __forceinline__ void sts_u16(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v) : "memory");
}

__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive(uint32_t mbar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}

// global -> shared bulk copy by the TMA engine; dst, src and bytes are multiples of 16
__device__ __forceinline__ void bulk_copy_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t mbar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "NB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra NB_DONE;\n"
        "bra NB_WAIT;\n"
        "NB_DONE:\n"
        "}" ::"r"(mbar), "r"(parity) : "memory");
}

// Phase A of the crowded path for 32 candidates read from global memory: rel = minimum-image
// vector of this lane's candidate; accepted ones are ballot-compacted into `list` as (dx, dy, dz, d2).
__device__ __forceinline__ void nb_test_global(const float4 rel, bool skip, float cut_hi, uint32_t lt_mask,
                                               int32_t max_nb, float4* list, int32_t& count) {
    const float d2f = fmaf(rel.z, rel.z, fmaf(rel.y, rel.y, rel.x * rel.x));
    const bool acc = d2f < cut_hi && !skip;
    const unsigned mask = __ballot_sync(0xffffffffu, acc);
    const int32_t pos = count + __popc(mask & lt_mask);
    if (acc && pos < max_nb) list[pos] = make_float4(rel.x, rel.y, rel.z, d2f);
    count += __popc(mask);
}

// u16 list entries of one centre (incl. the centre itself), at least 64 so that phase B may read
// entries lane and lane + 32 unconditionally
__host__ __device__ __forceinline__ int32_t nb_list_stride(int32_t max_nb) { return (max_nb + 1 + 63) & ~63; }

// Phase A for G centres of one warp: p[g] = staged coordinates of centre g.  Every staged
// candidate with fp32 d2 < cut_hi (the centre itself included) gets its stage index appended to
// list g (shared address list_s + g * list_bytes); cnt[g] counts all of them, stored or not.
template <int G>
__device__ __forceinline__ void nb_scan_group(uint32_t stage_s, int32_t n_pad, int lane, uint32_t lt_mask,
                                              float cut_hi, const float4 (&p)[G], uint32_t list_s,
                                              uint32_t list_bytes, int32_t cap, int32_t (&cnt)[G]) {
    uint32_t sp = stage_s + ((uint32_t)lane << 4);
    const uint32_t sp_end = stage_s + ((uint32_t)n_pad << 4);
    uint32_t q = (uint32_t)lane;
#pragma unroll
    for (int g = 0; g < G; ++g) cnt[g] = 0;
    const int32_t safe = cap - 32;                      // while 32 more entries fit, stores need no test
    for (; sp < sp_end; sp += 512, q += 32) {
        int32_t mx = cnt[0];
        if (G > 1) mx = max(mx, cnt[1]);
        if (G > 2) mx = max(mx, cnt[2]);
        if (mx > safe) break;
        const float4 c = lds128(sp);
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const float dx = c.x - p[g].x, dy = c.y - p[g].y, dz = c.z - p[g].z;
            const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            const bool hit = d2 < cut_hi;
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (hit) sts_u16(list_s + (uint32_t)g * list_bytes + ((uint32_t)(cnt[g] + __popc(m & lt_mask)) << 1), q);
            cnt[g] += __popc(m);
        }
    }
    for (; sp < sp_end; sp += 512, q += 32) {           // a list is nearly full: tested stores
        const float4 c = lds128(sp);
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const float dx = c.x - p[g].x, dy = c.y - p[g].y, dz = c.z - p[g].z;
            const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            const bool hit = d2 < cut_hi;
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            const int32_t pos = cnt[g] + __popc(m & lt_mask);
            if (hit && pos < cap) sts_u16(list_s + (uint32_t)g * list_bytes + ((uint32_t)pos << 1), q);
            cnt[g] += __popc(m);
        }
    }
}

// (dx, dy, dz, fp32 d2) of staged candidate `idx` seen from the centre at p: the same arithmetic as phase A
__device__ __forceinline__ float4 nb_rel(uint32_t stage_s, uint32_t idx, const float4 p) {
    const float4 c = lds128(stage_s + (idx << 4));
    float4 v;
    v.x = c.x - p.x; v.y = c.y - p.y; v.z = c.z - p.z;
    v.w = fmaf(v.z, v.z, fmaf(v.y, v.y, v.x * v.x));
    return v;
}

struct NbWarpCtx {
    int lane;
    int32_t n_r, hstride;
    int32_t* hist;                 // this warp's shell histogram
    uint32_t hist_s, g2_s;
    uint32_t* aux;                 // this warp's [max_nb + 1] scratch words (long lists)
    const float* addend_s;         // shared copies of np.addend / np.jconst
    const uint32_t* jconst_s;
};

// Phases B + C for a list of any length: fetch(e) returns entry e as (dx, dy, dz, fp32 d2) and
// whether it is the centre itself.  Returns the number of entries kept.
template <class Fetch>
__device__ __forceinline__ int32_t nb_emit_long(const NbWarpCtx& w, const NbParams& np, int32_t count, Fetch fetch,
                                                float4* __restrict__ dst, uint32_t* __restrict__ dstj) {
    const int lane = w.lane;
    const int32_t n_r = w.n_r;
    int32_t* hist = w.hist;
    for (int32_t i = 2 * lane; i < n_r + 2; i += 64) *reinterpret_cast<int2*>(hist + i) = make_int2(0, 0);
    __syncwarp();
    // phase B: exact acceptance near the cut-off, shell, rank inside the shell
    for (int32_t e = lane; e < count; e += 32) {
        bool self;
        const float4 v = fetch(e, self);
        const int32_t a = self ? n_r : nb_shell(v, np);    // n_r = rejected
        const int32_t rank = atomicAdd(hist + a, 1);
        w.aux[e] = (uint32_t)a | ((uint32_t)rank << 10);
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
            asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(w.g2_s + ((uint32_t)i << 2)), "r"(v0) : "memory");
            if (i + 1 < n_r)
                asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(w.g2_s + ((uint32_t)i << 2) + 4), "r"(v1) : "memory");
        }
        carry += total;
    }
    __syncwarp();
    for (int32_t e = lane; e < count; e += 32) {
        const uint32_t packed = w.aux[e];
        const int32_t a = (int32_t)(packed & 1023u), rank = (int32_t)(packed >> 10);
        if (a < n_r) {
            bool self;
            const float4 v = fetch(e, self);
            const int32_t pos = hist[a] + rank;
            dst[pos] = make_float4(v.x, v.y, v.z, w.addend_s[a]);
            dstj[pos] = w.jconst_s[a];
        }
    }
    return carry;
}

// neighbour_all_kernel: the degenerate cell grid (ncell == 1: 27 cells would cover the box).  A CTA
// stages the WHOLE frame (raw grid coordinates as fp32) and takes a slice of 64 centres; a warp per
// centre scans all particles with the minimum image taken per difference (nb_test_wrap) and
// emits its list through the general routine nb_emit_long.  Small or dense frames only (config 1).
__global__ void __launch_bounds__(kNbWarps * 32)
neighbour_all_kernel(FrameBatch fb, NbParams np) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* stage = reinterpret_cast<float4*>(smem_raw);                   // [stage_cap >= n, padded to 32]
    float4* scratch_all = stage + np.stage_cap;                            // [kNbWarps][max_nb] (dx, dy, dz, d2)
    uint32_t* aux_all = reinterpret_cast<uint32_t*>(scratch_all + (size_t)kNbWarps * np.max_nb);
    const int32_t aux_stride = (np.max_nb + 1 + 3) & ~3;
    const int32_t hstride = nb_hist_stride(np.n_r);
    int32_t* hist_all = reinterpret_cast<int32_t*>(aux_all + (size_t)kNbWarps * aux_stride);
    float* addend_s = reinterpret_cast<float*>(hist_all + kNbWarps * hstride);
    uint32_t* jconst_s = reinterpret_cast<uint32_t*>(addend_s + np.n_r);
    uint32_t* g2s = jconst_s + np.n_r;                                     // [n_r] this CTA's g2 counts

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t f = blockIdx.y, n = fb.n, n_r = np.n_r, max_nb = np.max_nb;
    const float4* __restrict__ sortedf = fb.sortedf + (long long)f * n;
    for (int32_t i = threadIdx.x; i < n_r; i += blockDim.x) {
        g2s[i] = 0;
        addend_s[i] = __ldg(np.addend + i);
        jconst_s[i] = (uint32_t)__ldg(np.jconst + i);
    }
    const int32_t n_pad = (n + 31) & ~31;
    for (int32_t i = threadIdx.x; i < n_pad; i += blockDim.x)
        stage[i] = i < n ? sortedf[i] : make_float4(kFarAway, 0.f, 0.f, 0.f);
    __syncthreads();

    NbWarpCtx w;
    w.lane = lane; w.n_r = n_r; w.hstride = hstride;
    w.hist = hist_all + wid * hstride;
    w.hist_s = (uint32_t)__cvta_generic_to_shared(w.hist);
    w.g2_s = (uint32_t)__cvta_generic_to_shared(g2s);
    w.aux = aux_all + (size_t)wid * aux_stride;
    w.addend_s = addend_s; w.jconst_s = jconst_s;
    float4* scratch = scratch_all + (size_t)wid * max_nb;
    const uint32_t stage_s = (uint32_t)__cvta_generic_to_shared(stage);
    const uint32_t scratch_s = (uint32_t)__cvta_generic_to_shared(scratch);
    const uint32_t lt_mask = (1u << lane) - 1u;
    unsigned long long my_pairs = 0, my_cap = 0;
    const int32_t s_lo = min(n, (int32_t)blockIdx.x * 64), s_hi = min(n, (int32_t)(blockIdx.x + 1) * 64);
    for (int32_t s = s_lo + wid; s < s_hi; s += kNbWarps) {
        const uint32_t own_s = stage_s + ((uint32_t)s << 4);
        const float4 p = lds128(own_s);
        int32_t count = 0;
        for (uint32_t sp = stage_s + ((uint32_t)lane << 4); sp < stage_s + ((uint32_t)n_pad << 4); sp += 512)
            nb_test_wrap(lds128(sp), sp == own_s, p.x, p.y, p.z, np.cut_hi, lt_mask, max_nb, scratch_s, count);
        if (count > max_nb) { my_cap += 1; count = max_nb; }
        __syncwarp();
        const long long row = ((long long)f * n + s) * max_nb;
        const int32_t kept = nb_emit_long(w, np, count, [&](int32_t e, bool& self) {
            self = false;
            return scratch[e];
        }, np.nbv + row, np.nbj + row);
        my_pairs += (unsigned long long)kept * (unsigned long long)(kept > 0 ? kept - 1 : 0);
        if (lane == 0) np.nbcount[(long long)f * n + s] = kept;
        if (np.n_slabs > 1) {                     // hist[a] = list position of the first entry of shell a
            int32_t* sp = np.slabpos + ((long long)f * n + s) * (np.n_slabs + 1);
            for (int32_t i = lane; i <= np.n_slabs; i += 32) {
                const int32_t a = np.slab_shell[i];
                sp[i] = a < n_r ? w.hist[a] : kept;
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

inline size_t nb_all_smem_bytes(int32_t stage_cap, int32_t max_nb, int32_t n_r) {
    return (size_t)stage_cap * 16 + (size_t)kNbWarps * max_nb * 16 + (size_t)kNbWarps * ((max_nb + 1 + 3) & ~3) * 4 +
           (size_t)kNbWarps * nb_hist_stride(n_r) * 4 + (size_t)n_r * 12;
}

// Everything a CTA needs to know about one (cell, frame) item; written by the producer warp.
struct NbItem {
    int32_t range_begin[kMaxRanges];      // first particle of each candidate range in the cell-major order
    int32_t range_prefix[kMaxRanges + 1]; // stage position of each range
    int4 range_shift[kMaxRanges];         // periodic shift of the range in grid units
    uint32_t shift_mask;                  // ranges with a non-zero shift
    int32_t own_base;                     // stage position of the first centre of the cell
    int32_t c_begin, c_end;               // the cell's particles = the centres
    int32_t staged;                       // 1 = candidates fit the stage (TMA issued), 0 = crowded path
    long long item;                       // item index, -1 = no more work
};

// One warp: find the next non-empty item at or after `item` (stride gridDim.x), describe it in
// `it`, and start the TMA copies of its candidates into the stage at shared address stage_s.
__device__ __forceinline__ void nb_prefetch(const FrameBatch& fb, const NbParams& np, long long item, long long n_items,
                                            NbItem& it, float4* stage, uint32_t stage_s, uint32_t mbar, int lane) {
    int32_t f = 0, cell = 0, c_begin = 0, c_end = 0;
    const int32_t* __restrict__ start = nullptr;
    for (; item < n_items; item += gridDim.x) {
        f = (int32_t)(item / fb.ncell3);
        cell = (int32_t)(item - (long long)f * fb.ncell3);
        start = fb.cell_start + (long long)f * (fb.ncell3 + 1);
        c_begin = __ldg(start + cell);
        c_end = __ldg(start + cell + 1);
        if (c_begin != c_end) break;                    // empty cells have no centres
    }
    if (item >= n_items) {
        if (lane == 0) it.item = -1;
        return;
    }
    // 9 columns (x, y offsets) x 2 parts; the three z-adjacent cells of a column are contiguous in
    // the cell-major order unless they wrap.  Every range has one constant periodic shift.
    int32_t b = 0, e = 0;
    int4 sh = make_int4(0, 0, 0, 0);
    if (lane < kMaxRanges) {
        const int4 o = __ldg(np.cell_origin + cell);
        const int32_t nc = fb.ncell, cx = o.w & 255, cy = (o.w >> 8) & 255, cz = (o.w >> 16) & 255;
        const int32_t col = lane >> 1, part = lane & 1;
        const int32_t ox = (col * 11 >> 5) - 1, oy = col - 3 * (col * 11 >> 5) - 1;     // col / 3, col % 3 for col < 9
        int32_t x = cx + ox, y = cy + oy;
        if (x < 0) { x += nc; sh.x = -(int32_t)kGrid; } else if (x >= nc) { x -= nc; sh.x = (int32_t)kGrid; }
        if (y < 0) { y += nc; sh.y = -(int32_t)kGrid; } else if (y >= nc) { y -= nc; sh.y = (int32_t)kGrid; }
        const int32_t* __restrict__ colstart = start + (x * nc + y) * nc;
        int32_t zb, ze;                                   // cells [zb, ze) of this part
        if (cz == 0) {
            if (part == 0) { zb = 0; ze = 2; } else { zb = nc - 1; ze = nc; sh.z = -(int32_t)kGrid; }
        } else if (cz == nc - 1) {
            if (part == 0) { zb = nc - 2; ze = nc; } else { zb = 0; ze = 1; sh.z = (int32_t)kGrid; }
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
    const int32_t n_stage = __shfl_sync(0xffffffffu, incl, kMaxRanges - 1);
    const int32_t n_pad = (n_stage + 31) & ~31;           // stage padded with far-away sentinels
    const bool staged = n_pad <= np.stage_cap;
    const unsigned shifted = __ballot_sync(0xffffffffu, len > 0 && (sh.x | sh.y | sh.z) != 0);
    if (lane < kMaxRanges) { it.range_begin[lane] = b; it.range_prefix[lane] = incl - len; it.range_shift[lane] = sh; }
    if (lane == kMaxRanges - 1) it.range_prefix[kMaxRanges] = incl;
    if (lane < kMaxRanges && b <= c_begin && c_begin < e) it.own_base = incl - len + (c_begin - b);
    if (lane == 0) {
        it.c_begin = c_begin; it.c_end = c_end; it.item = item; it.staged = staged ? 1 : 0; it.shift_mask = shifted;
        if (staged) mbar_expect_tx(mbar, (uint32_t)n_stage << 4);
    }
    __syncwarp();
    if (staged) {
        if (lane < kMaxRanges && len > 0) {
            // the stage was read and written through the generic proxy by an earlier item
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            bulk_copy_g2s(stage_s + ((uint32_t)(incl - len) << 4), fb.sortedf + (long long)f * fb.n + b, (uint32_t)len << 4, mbar);
        }
        if (n_stage + lane < n_pad) stage[n_stage + lane] = make_float4(kFarAway, 0.f, 0.f, 0.f);
    }
}

// A CTA = four consumer warps + one producer warp, coupled only by mbarriers over a ring of
// kStages candidate stages:
//   producer  waits until a stage is empty, describes the next non-empty (cell, frame) item,
//             starts the TMA copies, waits for them, adds the periodic shifts, signals "full";
//   consumers wait for "full", scan / sort / write the lists of their groups of centres, and
//             signal "empty" (one arrival per warp).
// No __syncthreads in the item loop: a warp that finishes its groups early runs on into the
// next item, so the uneven number of centres per cell averages out over the ring.
template <int kStages>
__global__ void __launch_bounds__((kNbWarps + 1) * 32)
neighbour_cell_kernel(FrameBatch fb, NbParams np) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* stage_all = reinterpret_cast<float4*>(smem_raw);               // kStages stages of stage_cap entries
    const int32_t list_stride = nb_list_stride(np.max_nb);
    unsigned char* lists_raw = smem_raw + (size_t)np.stage_cap * 16 * kStages;
    uint32_t* aux_all = reinterpret_cast<uint32_t*>(lists_raw + (size_t)kNbWarps * kNbMaxG * list_stride * 2);
    const int32_t aux_stride = (np.max_nb + 1 + 3) & ~3;
    const int32_t hstride = nb_hist_stride(np.n_r);       // even stride: 8-byte aligned pairs
    int32_t* hist_all = reinterpret_cast<int32_t*>(aux_all + (size_t)kNbWarps * aux_stride);
    float* addend_s = reinterpret_cast<float*>(hist_all + kNbWarps * hstride);
    uint32_t* jconst_s = reinterpret_cast<uint32_t*>(addend_s + np.n_r);
    uint32_t* g2s = jconst_s + np.n_r;                     // [max(n_r, 64)] this CTA's g2 counts
    __shared__ NbItem items[kStages];
    __shared__ __align__(8) unsigned long long mbar_s[3 * kStages];       // per stage: tma, full, empty

    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int32_t n_r = np.n_r, max_nb = np.max_nb;
    for (int32_t i = threadIdx.x; i < max(n_r, 64); i += blockDim.x) g2s[i] = 0;
    for (int32_t i = threadIdx.x; i < n_r; i += blockDim.x) {
        addend_s[i] = __ldg(np.addend + i);
        jconst_s[i] = (uint32_t)__ldg(np.jconst + i);
    }
    const uint32_t mbar0 = (uint32_t)__cvta_generic_to_shared(&mbar_s[0]);
    if (threadIdx.x == 0) {
        for (int b = 0; b < kStages; ++b) {
            mbar_init(mbar0 + 24u * b, 1);                 // tma: the producer's expect_tx arrival + the bytes
            mbar_init(mbar0 + 24u * b + 8u, 1);            // full: the producer
            mbar_init(mbar0 + 24u * b + 16u, kNbWarps);    // empty: one arrival per consumer warp
        }
    }
    const uint32_t stage_s0 = (uint32_t)__cvta_generic_to_shared(stage_all);
    const uint32_t stage_bytes = (uint32_t)np.stage_cap << 4;
    const long long n_items = (long long)fb.ncell3 * fb.n_frames;
    __syncthreads();                                     // barriers initialised, tables loaded

    if (wid == kNbWarps) {
        // ---- producer warp ---------------------------------------------------------------------
        long long item = (long long)blockIdx.x;
        for (uint32_t iter = 0;; ++iter) {
            const uint32_t buf = iter % kStages, round = iter / kStages;
            const uint32_t mb = mbar0 + 24u * buf;
            mbar_wait(mb + 16u, (round & 1u) ^ 1u);        // stage empty (passes at once the first time round)
            NbItem& it = items[buf];
            float4* stage = stage_all + (size_t)buf * np.stage_cap;
            nb_prefetch(fb, np, item, n_items, it, stage, stage_s0 + buf * stage_bytes, mb, lane);
            __syncwarp();
            const long long found = it.item;
            if (found >= 0) {
                if (it.staged) {
                    mbar_wait(mb, round & 1u);             // candidates have landed
                    uint32_t sm = it.shift_mask;           // periodic shifts of wrapped ranges
                    while (sm) {
                        const int r = __ffs(sm) - 1;
                        sm &= sm - 1u;
                        const int4 sh = it.range_shift[r];
                        const int32_t dst = it.range_prefix[r], len = it.range_prefix[r + 1] - dst;
                        const float sx = (float)sh.x, sy = (float)sh.y, sz = (float)sh.z;
                        for (int32_t i = lane; i < len; i += 32) {
                            float4 c = stage[dst + i];
                            c.x += sx; c.y += sy; c.z += sz;
                            stage[dst + i] = c;
                        }
                    }
                } else if (lane == 0) {
                    mbar_arrive(mb);                       // keep the tma barrier's phase in step
                }
            } else if (lane == 0) {
                mbar_arrive(mb);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(mb + 8u);           // full (release: the description and the shifts are visible)
            if (found < 0) break;
            item = found + gridDim.x;
        }
        return;
    }

    // ---- consumer warps ----------------------------------------------------------------------------
    const uint32_t list_bytes = (uint32_t)list_stride * 2u;
    const uint32_t list_s = (uint32_t)__cvta_generic_to_shared(lists_raw) + (uint32_t)(wid * kNbMaxG) * list_bytes;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const float cut_hi = np.cut_hi;
    const int32_t cap = max_nb + 1;                     // list capacity: the neighbours and the centre itself
    const bool fast_bc = n_r <= 64;
    NbWarpCtx w;
    w.lane = lane; w.n_r = n_r; w.hstride = hstride;
    w.hist = hist_all + wid * hstride;
    w.hist_s = (uint32_t)__cvta_generic_to_shared(w.hist);
    w.g2_s = (uint32_t)__cvta_generic_to_shared(g2s);
    w.aux = aux_all + (size_t)wid * aux_stride;
    w.addend_s = addend_s; w.jconst_s = jconst_s;
    unsigned long long my_pairs = 0, my_cap = 0;
    uint32_t g2a0 = 0, g2a1 = 0;                         // this lane's g2 counts of shells 2 lane, 2 lane + 1

    for (uint32_t iter = 0;; ++iter) {
        const uint32_t cur = iter % kStages, round = iter / kStages;
        const uint32_t mb = mbar0 + 24u * cur;
        mbar_wait(mb + 8u, round & 1u);                    // full
        const NbItem& it = items[cur];
        const long long item = it.item;
        if (item < 0) break;
        const uint32_t stage_s = stage_s0 + cur * stage_bytes;
        const int32_t f = (int32_t)(item / fb.ncell3);
        const int4* __restrict__ sorted = fb.sorted + (long long)f * fb.n;
        const int32_t c_begin = it.c_begin, c_end = it.c_end;
        const int32_t n_stage = it.range_prefix[kMaxRanges];
        const int32_t n_pad = (n_stage + 31) & ~31;
        const bool staged = it.staged != 0;
        const int32_t own_base = it.own_base;
        if (staged) {
            // groups of three consecutive centres; the warp that takes an extra group rotates
            const int32_t n_c = c_end - c_begin, n_g = (n_c + kNbMaxG - 1) / kNbMaxG;
            const int32_t first = (wid + (int32_t)iter) & (kNbWarps - 1);
            for (int32_t gi = first; gi < n_g; gi += kNbWarps) {
                const int32_t s0 = c_begin + gi * kNbMaxG;
                const int32_t G = min(kNbMaxG, c_end - s0);
                int32_t cnt[kNbMaxG] = {0, 0, 0};
                float4 p[kNbMaxG];
#pragma unroll
                for (int g = 0; g < kNbMaxG; ++g)
                    p[g] = lds128(stage_s + ((uint32_t)(own_base + (s0 - c_begin) + min(g, G - 1)) << 4));
                __syncwarp();                                  // lists of the previous group are consumed
                if (G == 3) {
                    nb_scan_group<3>(stage_s, n_pad, lane, lt_mask, cut_hi, p, list_s, list_bytes, cap, cnt);
                } else if (G == 2) {
                    const float4 p2[2] = {p[0], p[1]};
                    int32_t c2[2];
                    nb_scan_group<2>(stage_s, n_pad, lane, lt_mask, cut_hi, p2, list_s, list_bytes, cap, c2);
                    cnt[0] = c2[0]; cnt[1] = c2[1];
                } else {
                    const float4 p1[1] = {p[0]};
                    int32_t c1[1];
                    nb_scan_group<1>(stage_s, n_pad, lane, lt_mask, cut_hi, p1, list_s, list_bytes, cap, c1);
                    cnt[0] = c1[0];
                }
                __syncwarp();
#pragma unroll
                for (int g = 0; g < kNbMaxG; ++g) {
                    if (g >= G) break;
                    const int32_t s = s0 + g;
                    const uint32_t own_q = (uint32_t)(own_base + (s - c_begin));
                    const uint32_t lst = list_s + (uint32_t)g * list_bytes;
                    const float4 pc = p[g];
                    int32_t count = cnt[g];
                    // overflow: the centre itself may be among the dropped hits, so that all cap kept
                    // entries could be neighbours; max_nb of them at most fit this centre's row
                    if (count > cap) { my_cap += 1; count = max_nb; }
                    const long long row = ((long long)f * fb.n + s) * max_nb;
                    float4* __restrict__ dst = np.nbv + row;
                    uint32_t* __restrict__ dstj = np.nbj + row;
                    int32_t kept;
                    if (fast_bc && count <= 64) {
                        // ---- phases B + C with the list in registers (entries lane and lane + 32) -------
                        // hist: shells 0..n_r-1, slot n_r = rejected by the exact cut-off test, n_r + 1 = no entry
                        asm volatile("st.shared.v2.b32 [%0], {%1, %1};" ::"r"(w.hist_s + ((uint32_t)lane << 3)), "r"(0) : "memory");
                        if (lane == 0) asm volatile("st.shared.v2.b32 [%0], {%1, %1};" ::"r"(w.hist_s + 256u), "r"(0) : "memory");
                        const uint32_t l0 = lds_u16(lst + ((uint32_t)lane << 1)), l1 = lds_u16(lst + 64u + ((uint32_t)lane << 1));
                        const bool val0 = lane < count && l0 != own_q, val1 = lane + 32 < count && l1 != own_q;
                        float4 v0 = nb_rel(stage_s, val0 ? l0 : own_q, pc), v1 = nb_rel(stage_s, val1 ? l1 : own_q, pc);
                        if (!val0) v0.w = 1.f;
                        if (!val1) v1.w = 1.f;
                        int32_t a0 = nb_shell(v0, np), a1 = nb_shell(v1, np);
                        a0 = val0 ? a0 : n_r + 1; a1 = val1 ? a1 : n_r + 1;
                        __syncwarp();
                        const int32_t r0 = atomicAdd(w.hist + a0, 1);
                        const int32_t r1 = atomicAdd(w.hist + a1, 1);
                        __syncwarp();
                        const int2 hv = *reinterpret_cast<const int2*>(w.hist + 2 * lane);
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
                        asm volatile("st.shared.v2.b32 [%0], {%1, %2};" ::"r"(w.hist_s + ((uint32_t)lane << 3)), "r"(incl - v), "r"(incl - c1) : "memory");
                        g2a0 += (uint32_t)c0; g2a1 += (uint32_t)c1;      // this centre's g2 counts
                        __syncwarp();
                        if (a0 < n_r) {
                            const int32_t pos = w.hist[a0] + r0;
                            dst[pos] = make_float4(v0.x, v0.y, v0.z, addend_s[a0]);
                            dstj[pos] = jconst_s[a0];
                        }
                        if (a1 < n_r) {
                            const int32_t pos = w.hist[a1] + r1;
                            dst[pos] = make_float4(v1.x, v1.y, v1.z, addend_s[a1]);
                            dstj[pos] = jconst_s[a1];
                        }
                    } else {
                        kept = nb_emit_long(w, np, count, [&](int32_t e, bool& self) {
                            const uint32_t idx = lds_u16(lst + ((uint32_t)e << 1));
                            self = idx == own_q;
                            return nb_rel(stage_s, idx, pc);
                        }, dst, dstj);
                    }
                    my_pairs += (unsigned long long)kept * (unsigned long long)(kept > 0 ? kept - 1 : 0);
                    if (lane == 0) np.nbcount[(long long)f * fb.n + s] = kept;
                    if (np.n_slabs > 1) {                     // hist[a] = list position of the first entry of shell a
                        int32_t* sp = np.slabpos + ((long long)f * fb.n + s) * (np.n_slabs + 1);
                        for (int32_t i = lane; i <= np.n_slabs; i += 32) {
                            const int32_t a = np.slab_shell[i];
                            sp[i] = a < n_r ? w.hist[a] : kept;
                        }
                    }
                    __syncwarp();
                }
            }
        } else {
            // crowded neighbourhood: candidates straight from global memory, one centre at a time;
            // the (dx, dy, dz, d2) list of the centre lives in this warp's slice of a global scratch
            float4* scratch = np.crowd_scratch + ((size_t)blockIdx.x * kNbWarps + wid) * max_nb;
            for (int32_t s = c_begin + wid; s < c_end; s += kNbWarps) {
                int32_t count = 0;
                const int4 me = sorted[s];
                for (int32_t r = 0; r < kMaxRanges; ++r) {
                    const int32_t b = it.range_begin[r], e = b + (it.range_prefix[r + 1] - it.range_prefix[r]);
                    for (int32_t q0 = b; q0 < e; q0 += 32) {
                        const int32_t q = q0 + lane;
                        const bool in = q < e && q != s;
                        const int4 c = in ? sorted[q] : me;
                        const float4 rel = make_float4((float)wrap_component(c.x - me.x), (float)wrap_component(c.y - me.y),
                                                       (float)wrap_component(c.z - me.z), 0.f);
                        nb_test_global(rel, !in, cut_hi, lt_mask, max_nb, scratch, count);
                    }
                }
                if (count > max_nb) { my_cap += 1; count = max_nb; }
                __syncwarp();
                const long long row = ((long long)f * fb.n + s) * max_nb;
                const int32_t kept = nb_emit_long(w, np, count, [&](int32_t e, bool& self) {
                    self = false;
                    return scratch[e];
                }, np.nbv + row, np.nbj + row);
                my_pairs += (unsigned long long)kept * (unsigned long long)(kept > 0 ? kept - 1 : 0);
                if (lane == 0) np.nbcount[(long long)f * fb.n + s] = kept;
                if (np.n_slabs > 1) {
                    int32_t* sp = np.slabpos + ((long long)f * fb.n + s) * (np.n_slabs + 1);
                    for (int32_t i = lane; i <= np.n_slabs; i += 32) {
                        const int32_t a = np.slab_shell[i];
                        sp[i] = a < n_r ? w.hist[a] : kept;
                    }
                }
                __syncwarp();
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(mb + 16u);              // this warp is done with the stage
    }
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(w.g2_s + ((uint32_t)lane << 3)), "r"(g2a0) : "memory");
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(w.g2_s + ((uint32_t)lane << 3) + 4u), "r"(g2a1) : "memory");
    if (lane == 0) {
        if (my_pairs) atomicAdd(np.stats + 0, my_pairs);
        if (my_cap) atomicAdd(np.stats + 2, my_cap);
    }
    asm volatile("bar.sync 1, %0;" ::"r"(kNbWarps * 32) : "memory");     // the consumer warps only
    for (int32_t i = threadIdx.x; i < n_r; i += kNbWarps * 32) {
        const uint32_t v = g2s[i];
        if (v) atomicAdd(np.counts2 + i, (unsigned long long)v);
    }
}

// the ring of candidate stages, the u16 lists, the
// long-list scratch words, the per-warp shell histograms, the shell tables and the g2 counts
inline size_t nb_cell_smem_bytes(int32_t stage_cap, int32_t max_nb, int32_t n_r, int stages) {
    return (size_t)stage_cap * 16 * stages + (size_t)kNbWarps * kNbMaxG * nb_list_stride(max_nb) * 2 +
           (size_t)kNbWarps * ((max_nb + 1 + 3) & ~3) * 4 + (size_t)kNbWarps * nb_hist_stride(n_r) * 4 +
           (size_t)n_r * 8 + (size_t)(n_r > 64 ? n_r : 64) * 4;
}


}  // namespace g3
