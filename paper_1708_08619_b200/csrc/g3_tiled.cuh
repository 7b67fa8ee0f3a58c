// g3_tiled.cuh -- the fast path (kernel 2): histogram tile layout and host-side orchestration of
// the neighbour kernels (g3_neighbour.cuh) and tiled_triplet_kernel / merge_kernel (g3_triplet.cuh).
//
// Tile layout.  Only bins with a <= b that the triangle inequality
// allows get a slot:  slot(a, b, c) = 1 + BASE(b) + P(a) + c - g(b) + h(a), with
//   g(b)  = lowest reachable c for shells (0, b),
//   h(a)  = max_b (g(b) - c_lo(a, b))   (how far below g(b) row a can reach),
//   W(a)  = row width that covers c_lo(a,b)..c_hi(a,b) for every b >= a,  P = prefix sum of W,
//   BASE(b) = sum_{b' < b} P(b' + 1)   (rows 0..b' of column block b').
// The slot is a sum of a term that depends on k only (folded into the fp32 magic addend), a term
// that depends on j only (a byte offset) and the bin c, so the kernel needs no multiplication.
#pragma once

#include <cmath>
#include <vector>

#include "g3_generic.cuh"
#include "g3_neighbour.cuh"
#include "g3_plan.h"
#include "g3_triplet.cuh"

namespace g3 {


struct TiledState {
    // histogram tile layout (host copies kept for tests/introspection)
    int64_t tile_bins = 0;                     // slots incl. 2 guards
    std::vector<int32_t> g, h, W, P, BASE;
    // device tables
    float* d_addend = nullptr;                 // [n_r]  kMagic + BASE(b) - g(b) + 1
    int32_t* d_jconst = nullptr;               // [n_r]  4 * (P(a) + h(a))
    uint32_t* d_slot_map = nullptr;            // [tile_bins] packed (a, b, c); 0xFFFFFFFF = unused
    unsigned long long* d_scratch = nullptr;   // [grid][tile_bins] per-CTA partial tiles
    // neighbour lists of one batch
    float4* d_nbv = nullptr;                   // [batch][n][max_nb] (dx, dy, dz, addend(shell))
    uint32_t* d_nbj = nullptr;                 // [batch][n][max_nb] row offset of the shell
    int32_t* d_nbcount = nullptr;              // [batch][n]
    unsigned int* d_work = nullptr;            // work-queue counter
    int4* d_cell_origin = nullptr;             // [ncell3] cell centres on the grid
    float4* d_crowd = nullptr;                 // [nb_grid][kNbWarps][max_nb] lists of the neighbour kernel's crowded path
    // launch configuration
    int tri_warps = 16;
    int grid = 0;
    int nb_grid = 0;                           // persistent CTAs of neighbour_cell_kernel
    size_t tri_smem = 0, nb_smem = 0;
    int32_t stage_cap = 0;
    uint32_t cta_item_cap = 0;                 // work items one CTA may take per launch
    int64_t max_batch_frames = 1;              // frames per launch the item cap allows
    bool dirty = false;                        // partial tiles hold counts not yet merged
    // slab passes: when the whole tile does not fit shared memory the outer shell b is split
    // into n_slabs ranges [slab_shell[s], slab_shell[s+1]); one triplet launch per slab
    int32_t n_slabs = 1;
    std::vector<int32_t> slab_shell;           // [n_slabs + 1]
    int64_t slab_bins_max = 0;                 // slots (incl. 2 guards) of the largest slab
    int32_t* d_slab_shell = nullptr;
    int32_t* d_slabpos = nullptr;              // [batch][n][n_slabs + 1]
};

// Split the outer shell range so that every slab's slots fit `cap_slots`.  False if one
// column block alone is too large.
inline bool build_slabs(TiledState& ts, int32_t n_r, int64_t cap_slots) {
    ts.slab_shell.assign(1, 0);
    ts.slab_bins_max = 0;
    int32_t b0 = 0;
    while (b0 < n_r) {
        int32_t b1 = b0;
        while (b1 < n_r && (int64_t)ts.BASE[b1 + 1] - ts.BASE[b0] + 2 <= cap_slots) ++b1;
        if (b1 == b0) return false;
        ts.slab_bins_max = std::max<int64_t>(ts.slab_bins_max, (int64_t)ts.BASE[b1] - ts.BASE[b0] + 2);
        ts.slab_shell.push_back(b1);
        b0 = b1;
    }
    ts.n_slabs = (int32_t)ts.slab_shell.size() - 1;
    return true;
}

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
// host side
inline int32_t tiled_stage_cap(const g3_plan* p) {
    if (p->ncell == 1) return (int32_t)((p->n + 63) / 64 * 64);
    // 1.5 x the mean occupancy of 27 cells; more crowded neighbourhoods are read from global
    const double per27 = 27.0 * (double)p->n / ((double)p->ncell * p->ncell * p->ncell);
    const int64_t cap = (int64_t)(1.5 * per27) + 96;
    return (int32_t)((cap + 63) / 64 * 64);
}

inline int tiled_warps(const g3_plan* p, int64_t tile_bins) {
    int w = p->tri_warps_opt ? p->tri_warps_opt : 16;   // 16 warps x 128 registers: no spills (measured best)
    while (w > 8 && tri_smem_bytes(tile_bins, w, p->bins.n_r) > (size_t)p->smem_optin) w -= 4;
    return w;
}

// Slots a tile may hold beside the windows of `warps` warps and the shell tables.
inline int64_t tiled_cap_slots(const g3_plan* p, int warps) {
    const int64_t fixed = (int64_t)tri_smem_bytes(0, warps, p->bins.n_r) + 64;   // + static shared
    return ((int64_t)p->smem_optin - fixed) / 4;
}

// Layout + slabs for this plan; false if the tiled path cannot serve it.
inline bool tiled_plan_slabs(const g3_plan* p, TiledState& ts) {
    build_layout(p, ts);
    if (ts.tile_bins > (1 << 22)) return false;                    // addend must stay below 2^24
    if (tri_smem_bytes(ts.tile_bins, 8, p->bins.n_r) <= (size_t)p->smem_optin) {
        ts.n_slabs = 1;
        ts.slab_shell = {0, p->bins.n_r};
        ts.slab_bins_max = ts.tile_bins;
        return true;
    }
    const int warps = p->tri_warps_opt ? p->tri_warps_opt : 16;
    return build_slabs(ts, p->bins.n_r, tiled_cap_slots(p, warps)) && ts.n_slabs <= 64;
}

// 2 if the tiled path can serve this plan, else 1 (generic).
inline int32_t tiled_select(g3_plan* p) {
    if (p->kernel_opt == 1) return 1;
    if (p->bins.n_r > 1022 || p->bins.n_t > 2046) return 1;
    if (p->max_nb > (1 << 16)) return 1;
    TiledState ts;
    if (!tiled_plan_slabs(p, ts)) return 1;
    if ((p->ncell == 1 ? nb_all_smem_bytes(tiled_stage_cap(p), p->max_nb, p->bins.n_r)
                       : nb_cell_smem_bytes(tiled_stage_cap(p), p->max_nb, p->bins.n_r, kNbStages)) + 1024 > (size_t)p->smem_optin) return 1;   // + static shared
    if (p->ncell == 1 && p->n > 8192) return 1;
    return 2;
}

inline void tiled_free(g3_plan* p) {
    TiledState* ts = p->tiled;
    if (!ts) return;
    cudaFree(ts->d_addend); cudaFree(ts->d_jconst); cudaFree(ts->d_slot_map); cudaFree(ts->d_scratch);
    cudaFree(ts->d_nbv); cudaFree(ts->d_nbj); cudaFree(ts->d_nbcount); cudaFree(ts->d_work); cudaFree(ts->d_cell_origin);
    cudaFree(ts->d_slab_shell); cudaFree(ts->d_slabpos); cudaFree(ts->d_crowd);
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
inline int tiled_set_attr(int smem_optin) {
    G3T_CUDA(allow_max_dynamic_smem(tiled_triplet_kernel<kWarps, false>, smem_optin));
    G3T_CUDA(allow_max_dynamic_smem(tiled_triplet_kernel<kWarps, true>, smem_optin));
    return G3_OK;
}

template <int kWarps>
inline void tiled_launch_triplet(const TiledState* ts, const TriParams& tp, cudaStream_t st) {
    if (ts->n_slabs > 1)
        tiled_triplet_kernel<kWarps, true><<<ts->grid, kWarps * 32, ts->tri_smem, st>>>(tp);
    else
        tiled_triplet_kernel<kWarps, false><<<ts->grid, kWarps * 32, ts->tri_smem, st>>>(tp);
}

inline int tiled_configure(g3_plan* p) {
    tiled_free(p);
    TiledState* ts = new (std::nothrow) TiledState;
    if (!ts) return G3_ENOMEM;
    p->tiled = ts;
    if (!tiled_plan_slabs(p, *ts)) return G3_EINVAL;
    p->tile_bins = ts->tile_bins;
    const int32_t n_r = p->bins.n_r;

    // A tile slot is a u32 and belongs to one CTA: a CTA takes at most cta_item_cap work items
    // per launch, each worth at most kItemCentres * C(max_nb, 2) pairs, so no slot can overflow
    // whatever the input.  The queue always drains if grid * cap covers the launch's items.
    ts->grid = p->sm_count;
    const long double per_item = (long double)kItemCentres * p->max_nb * (p->max_nb - 1) / 2;
    ts->cta_item_cap = (uint32_t)std::min<long double>(4.0e9L / per_item, 1.0e9L);
    if (ts->cta_item_cap < 1) return G3_EINVAL;
    ts->max_batch_frames = (int64_t)((long double)ts->grid * ts->cta_item_cap * kItemCentres / (long double)p->n);
    if (ts->max_batch_frames < 1) return G3_EINVAL;
    if (p->batch_frames > ts->max_batch_frames) p->batch_frames = (int32_t)ts->max_batch_frames;
    // neighbour lists of one batch: keep them below ~16 GiB, and, when the batch size is the
    // library's own choice, below a quarter of the memory that is free right now (an empty B200
    // leaves the 16 GiB standing; next to a simulation or other plans the plan shrinks instead of
    // failing).  configure() halves the batch further if an allocation fails all the same.
    size_t list_budget = size_t(16) << 30;
    if (p->batch_auto) {
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) list_budget = std::min(list_budget, free_b / 4);
        else cudaGetLastError();
    }
    const size_t frame_bytes = (size_t)p->n * p->max_nb * (sizeof(float4) + sizeof(uint32_t));
    const int64_t mem_frames = std::max<int64_t>(1, (int64_t)(list_budget / frame_bytes));
    if (p->batch_frames > mem_frames) p->batch_frames = (int32_t)mem_frames;

    ts->tri_warps = tiled_warps(p, ts->slab_bins_max);
    ts->tri_smem = tri_smem_bytes(ts->slab_bins_max, ts->tri_warps, n_r);
    ts->stage_cap = tiled_stage_cap(p);
    ts->nb_smem = p->ncell == 1 ? nb_all_smem_bytes(ts->stage_cap, p->max_nb, n_r)
                                : nb_cell_smem_bytes(ts->stage_cap, p->max_nb, n_r, kNbStages);

    std::vector<float> addend(n_r);
    std::vector<int32_t> jconst(n_r);
    for (int32_t b = 0; b < n_r; ++b) {
        addend[b] = kMagic + (float)(ts->BASE[b] - ts->g[b] + 1);
        jconst[b] = 4 * (ts->P[b] + ts->h[b]);
    }
    std::vector<uint32_t> slot_map((size_t)ts->tile_bins, 0xFFFFFFFFu);
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
    const size_t per_frame_entries = (size_t)p->n * p->max_nb;
    const size_t B = (size_t)p->batch_frames;
    G3T_CUDA(cudaMalloc(&ts->d_addend, sizeof(float) * n_r));
    G3T_CUDA(cudaMalloc(&ts->d_jconst, sizeof(int32_t) * n_r));
    G3T_CUDA(cudaMalloc(&ts->d_slot_map, sizeof(uint32_t) * ts->tile_bins));
    G3T_CUDA(cudaMalloc(&ts->d_scratch, sizeof(unsigned long long) * ts->tile_bins * ts->grid));
    G3T_CUDA(cudaMalloc(&ts->d_nbv, sizeof(float4) * (per_frame_entries * B + 64)));   // +64: prefetch overrun
    G3T_CUDA(cudaMalloc(&ts->d_nbj, sizeof(uint32_t) * (per_frame_entries * B + 64)));
    G3T_CUDA(cudaMemset(ts->d_nbj, 0, sizeof(uint32_t) * (per_frame_entries * B + 64)));
    G3T_CUDA(cudaMalloc(&ts->d_nbcount, sizeof(int32_t) * (size_t)p->n * B));
    G3T_CUDA(cudaMalloc(&ts->d_work, sizeof(unsigned int)));
    if (ts->n_slabs > 1) {
        G3T_CUDA(cudaMalloc(&ts->d_slab_shell, sizeof(int32_t) * (ts->n_slabs + 1)));
        G3T_CUDA(cudaMemcpy(ts->d_slab_shell, ts->slab_shell.data(), sizeof(int32_t) * (ts->n_slabs + 1),
                            cudaMemcpyHostToDevice));
        G3T_CUDA(cudaMalloc(&ts->d_slabpos, sizeof(int32_t) * (size_t)p->n * B * (ts->n_slabs + 1)));
    }
    {
        const int32_t nc = p->ncell;
        std::vector<int4> origin((size_t)nc * nc * nc);
        for (int32_t cx = 0; cx < nc; ++cx)
            for (int32_t cy = 0; cy < nc; ++cy)
                for (int32_t cz = 0; cz < nc; ++cz)
                    origin[((size_t)cx * nc + cy) * nc + cz] =
                        make_int4((int32_t)(((int64_t)(2 * cx + 1) << (kGridBits - 1)) / nc),
                                  (int32_t)(((int64_t)(2 * cy + 1) << (kGridBits - 1)) / nc),
                                  (int32_t)(((int64_t)(2 * cz + 1) << (kGridBits - 1)) / nc),
                                  cx | (cy << 8) | (cz << 16));
        G3T_CUDA(cudaMalloc(&ts->d_cell_origin, sizeof(int4) * origin.size()));
        G3T_CUDA(cudaMemcpy(ts->d_cell_origin, origin.data(), sizeof(int4) * origin.size(), cudaMemcpyHostToDevice));
    }
    G3T_CUDA(cudaMemcpy(ts->d_addend, addend.data(), sizeof(float) * n_r, cudaMemcpyHostToDevice));
    G3T_CUDA(cudaMemcpy(ts->d_jconst, jconst.data(), sizeof(int32_t) * n_r, cudaMemcpyHostToDevice));
    G3T_CUDA(cudaMemcpy(ts->d_slot_map, slot_map.data(), sizeof(uint32_t) * ts->tile_bins, cudaMemcpyHostToDevice));
    G3T_CUDA(cudaMemset(ts->d_scratch, 0, sizeof(unsigned long long) * ts->tile_bins * ts->grid));
    G3T_CUDA(cudaMemset(ts->d_nbv, 0, sizeof(float4) * (per_frame_entries * B + 64)));
    if (p->ncell == 1) {
        G3T_CUDA(allow_max_dynamic_smem(neighbour_all_kernel, p->smem_optin));
    } else {
        auto kern = neighbour_cell_kernel<kNbStages>;
        G3T_CUDA(allow_max_dynamic_smem(kern, p->smem_optin));
        int per_sm = 0;      // persistent: exactly the CTAs that are resident together
        G3T_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, (kNbWarps + 1) * 32, ts->nb_smem));
        ts->nb_grid = p->sm_count * std::max(per_sm, 1);
        G3T_CUDA(cudaMalloc(&ts->d_crowd, sizeof(float4) * (size_t)ts->nb_grid * kNbWarps * p->max_nb));
    }
    switch (ts->tri_warps) {
        case 24: return tiled_set_attr<24>(p->smem_optin);
        case 20: return tiled_set_attr<20>(p->smem_optin);
        case 12: return tiled_set_attr<12>(p->smem_optin);
        case 16: return tiled_set_attr<16>(p->smem_optin);
        default: return tiled_set_attr<8>(p->smem_optin);
    }
}

inline int tiled_merge(g3_plan* p, cudaStream_t st) {
    TiledState* ts = p->tiled;
    if (!ts || !ts->dirty) return G3_OK;
    merge_kernel<<<(unsigned)((ts->tile_bins + 255) / 256), 256, 0, st>>>(
        ts->d_scratch, ts->d_slot_map, (int32_t)ts->tile_bins, ts->grid, p->bins.n_r, p->bins.n_t,
        p->d_counts, p->d_stats);
    p->launches += 1;
    ts->dirty = false;
    G3T_CUDA(cudaGetLastError());
    return G3_OK;
}

inline int tiled_launch(g3_plan* p, const FrameBatch& fb, const BinSpec& bs, cudaStream_t st) {
    TiledState* ts = p->tiled;
    if (!ts) return G3_ESTATE;
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
    np.T_r = bs.T_r;
    np.cell_origin = ts->d_cell_origin;
    np.nbv = ts->d_nbv; np.nbj = ts->d_nbj; np.addend = ts->d_addend; np.jconst = ts->d_jconst; np.nbcount = ts->d_nbcount; np.stats = p->d_stats; np.counts2 = p->d_counts2;
    np.n_slabs = ts->n_slabs; np.slab_shell = ts->d_slab_shell; np.slabpos = ts->d_slabpos; np.crowd_scratch = ts->d_crowd;
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
        dim3 grid((unsigned)((fb.n + 63) / 64), (unsigned)fb.n_frames);
        neighbour_all_kernel<<<grid, kNbWarps * 32, ts->nb_smem, st>>>(fb, np);
    } else {
        const long long items = (long long)fb.ncell3 * fb.n_frames;
        auto kern = neighbour_cell_kernel<kNbStages>;
        kern<<<(unsigned)std::min<long long>(items, ts->nb_grid), (kNbWarps + 1) * 32, ts->nb_smem, st>>>(fb, np);
    }
    if (p->timing) G3T_CUDA(cudaEventRecord(ev[1], st));
    TriParams tp;
    tp.total_centres = (long long)fb.n_frames * fb.n;
    tp.max_nb = p->max_nb; tp.n_t = bs.n_t; tp.n_r = bs.n_r; tp.tile_bins = (int32_t)ts->tile_bins;
    tp.cta_item_cap = ts->cta_item_cap;
    tp.inv_lo = (float)((1.0 / wt) * (1.0 - eps));
    tp.inv_hi = (float)((1.0 / wt) * (1.0 + eps));
    tp.T_t = bs.T_t; tp.nbv = ts->d_nbv; tp.nbj = ts->d_nbj; tp.nbcount = ts->d_nbcount;
    tp.work = ts->d_work;
    tp.scratch_stride = ts->tile_bins;
    tp.n_slabs = ts->n_slabs; tp.slabpos = ts->d_slabpos;
    for (int32_t s = 0; s < ts->n_slabs; ++s) {
        const int32_t b0 = ts->slab_shell[s], b1 = ts->slab_shell[s + 1];
        tp.slab = s;
        tp.slot_base = ts->BASE[b0];
        tp.tile_bins = ts->n_slabs > 1 ? ts->BASE[b1] - ts->BASE[b0] + 2 : (int32_t)ts->tile_bins;
        tp.scratch = ts->d_scratch + tp.slot_base;
        if (s > 0) G3T_CUDA(cudaMemsetAsync(ts->d_work, 0, sizeof(unsigned int), st));
        switch (ts->tri_warps) {
            case 24: tiled_launch_triplet<24>(ts, tp, st); break;
            case 20: tiled_launch_triplet<20>(ts, tp, st); break;
            case 12: tiled_launch_triplet<12>(ts, tp, st); break;
            case 16: tiled_launch_triplet<16>(ts, tp, st); break;
            default: tiled_launch_triplet<8>(ts, tp, st); break;
        }
    }
    if (p->timing) G3T_CUDA(cudaEventRecord(ev[2], st));
    p->launches += 1 + (uint64_t)ts->n_slabs;
    ts->dirty = true;
    G3T_CUDA(cudaGetLastError());
    return G3_OK;
}

}  // namespace g3
