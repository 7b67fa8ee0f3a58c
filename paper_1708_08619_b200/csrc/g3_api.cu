// g3_api.cu -- the C ABI of libg3 (include/g3.h): plan management and launch orchestration.
//
// Per batch of staged frames, all stream-ordered and without host synchronisation:
//   quantise_count_kernel   a1 + a2  snap to the 2^20 grid, cell id, rank within cell
//   cell_scan_kernel        a2       exclusive scan of cell counts (one block per frame)
//   cell_scatter_kernel     a2       counting-sort scatter into cell-major order (int4 + fp32 copies)
//   neighbour kernel        a3       shell-sorted minimum-image lists, g2 counts (tiled path)
//   triplet kernel          a4, a5   pairs, histogram tile (tiled path); the generic kernel does a3..a5
//   optional: g2_wide_(cell_)kernel (g2 to 2 r_max), qtet_list_kernel / qtet_cell_kernel (+ redo)
// and at g3_finalize:  merge_kernel (a5), normalise_kernel (a6).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "g3_cells.cuh"
#include "g3_g2wide.cuh"
#include "g3_generic.cuh"
#include "g3_msd.cuh"
#include "g3_plan.h"
#include "g3_qtet.cuh"
#include "g3_tiled.cuh"
#include "g3_volumes.h"

using namespace g3;

#define G3_CUDA(call)                                   \
    do {                                                \
        cudaError_t e__ = (call);                       \
        if (e__ != cudaSuccess) {                       \
            if (e__ == cudaErrorMemoryAllocation) {     \
                cudaGetLastError();                     \
                return G3_ENOMEM;                       \
            }                                           \
            return G3_ECUDA;                            \
        }                                               \
    } while (0)

namespace {

constexpr int kGenericWarps = 8;
constexpr int kQtetWarps = 8;

__global__ void __launch_bounds__(256)
normalise_kernel(const unsigned long long* __restrict__ counts, const double* __restrict__ volumes,
                 long long nbins, double inv_ideal, double* __restrict__ g3out) {
    long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nbins) return;
    double v = volumes[b];
    // g3 = H / (F N rho^2 V_abc); 0 where V_abc = 0.  inv_ideal = 1 / (F N rho^2).
    g3out[b] = v > 0.0 ? __ddiv_rn(__dmul_rn((double)counts[b], inv_ideal), v) : 0.0;
}

__global__ void __launch_bounds__(256)
normalise_g2_kernel(const unsigned long long* __restrict__ counts2, const double* __restrict__ shell_volumes,
                    int32_t n_r, double inv_ideal, double* __restrict__ g2out) {
    int32_t a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= n_r) return;
    // g2 = H2 / (F N rho V_a); inv_ideal = 1 / (F N rho)
    g2out[a] = __ddiv_rn(__dmul_rn((double)counts2[a], inv_ideal), shell_volumes[a]);
}

void free_buffers(g3_plan* p) {
    cudaFree(p->d_staged); p->d_staged = nullptr;
    cudaFree(p->d_slot); p->d_slot = nullptr;
    cudaFree(p->d_cell_count); p->d_cell_count = nullptr;
    cudaFree(p->d_cell_start); p->d_cell_start = nullptr;
    cudaFree(p->d_sorted); p->d_sorted = nullptr;
    cudaFree(p->d_sortedf); p->d_sortedf = nullptr;
    cudaFree(p->d_generic_nb); p->d_generic_nb = nullptr;
    cudaFree(p->d_h2d); p->d_h2d = nullptr;
    cudaFree(p->d_qtet); p->d_qtet = nullptr;
    cudaFree(p->d_qtet_stats); p->d_qtet_stats = nullptr;
    cudaFree(p->d_qtet_redo); p->d_qtet_redo = nullptr;
    cudaFree(p->d_qtet_origin); p->d_qtet_origin = nullptr;
    tiled_free(p);
    p->configured = false;
}

// Fold the recorded event triples into the running sums (waits for the last event).
int fold_timing(g3_plan* p) {
    for (size_t i = 0; i + 2 < p->ev_used; i += 3) {
        float nb = 0.f, tri = 0.f;
        G3_CUDA(cudaEventSynchronize(p->ev_pool[i + 2]));
        G3_CUDA(cudaEventElapsedTime(&nb, p->ev_pool[i], p->ev_pool[i + 1]));
        G3_CUDA(cudaEventElapsedTime(&tri, p->ev_pool[i + 1], p->ev_pool[i + 2]));
        p->neighbour_ms += nb;
        p->triplet_ms += tri;
        p->timed_launches += 1;
    }
    p->ev_used = 0;
    return G3_OK;
}

// Choose the cell grid, the neighbour capacity and the kernel; allocate batch buffers.
int configure_once(g3_plan* p) {
    const double cut = std::sqrt((double)p->T_r.back());
    const int64_t reach = (int64_t)std::ceil(cut) + 1;     // > any neighbour |component|
    int64_t ncell = kGrid / reach;                         // cell width >= reach
    ncell = std::min<int64_t>(ncell, kMaxCellsPerEdge);
    // do not build cells far finer than the particle spacing
    while (ncell > 4 && ncell * ncell * ncell > 4 * p->n) --ncell;
    if (ncell < 4) ncell = 1;     // degenerate grid (27 cells would cover the box): all particles
    p->ncell = (int32_t)ncell;

    const double frac = p->r_max / p->box;
    const double mean_k = (double)p->n * 4.18879020478639 * frac * frac * frac;
    int64_t cap = p->max_nb_opt > 0 ? p->max_nb_opt : (int64_t)(3.0 * mean_k) + 64;
    cap = std::min<int64_t>(cap, p->n - 1);
    cap = std::max<int64_t>((cap + 31) / 32 * 32, 64);   // >= 64: the triplet kernel prefetches two chunks
    p->max_nb = (int32_t)cap;

    if (p->batch_auto) {
        // every triplet launch zeroes and flushes a whole histogram tile per CTA (~75 us at 64^3
        // bins): stage enough frames for ~2^22 centres per launch sequence
        const int64_t want = ((int64_t(1) << 22) + p->n - 1) / p->n;
        p->batch_frames = (int32_t)std::min<int64_t>(std::max<int64_t>(want, 16), 256);
    }
    p->batch_frames = std::min(p->batch_frames, p->batch_limit);
    p->kernel = tiled_select(p);                           // 1 = generic, 2 = tiled
    // q_tet straight from the shell-sorted neighbour lists of the tiled path (qtet_list_kernel);
    // plans served by the generic kernel have no lists and use the 27-cell scan of g3_qtet.cuh
    p->qtet_lists = p->qtet_bins > 0 && p->kernel == 2 && (int64_t)p->batch_frames * p->n < (int64_t(1) << 31);
    if (p->kernel == 1) {
        G3_CUDA(allow_max_dynamic_smem(generic_triplet_kernel<kGenericWarps>, p->smem_optin));
        p->generic_blocks = std::min<int64_t>(((int64_t)p->batch_frames * p->n + kGenericWarps - 1) / kGenericWarps,
                                              (int64_t)p->sm_count * 32);
        if (generic_smem_bytes(p->bins.n_r, p->bins.n_t, p->max_nb, kGenericWarps) > (size_t)p->smem_optin) {
            // neighbour lists too long for shared memory: one global slice per warp
            if (generic_smem_bytes(p->bins.n_r, p->bins.n_t, 0, kGenericWarps, false) > (size_t)p->smem_optin) return G3_EINVAL;
            p->generic_blocks = std::min<int64_t>(p->generic_blocks, (int64_t)p->sm_count * 8);
            // max_nb may be as large as n - 1 or 2^20: the pool of slices stays below 2 GiB (the
            // kernel walks the centres with a grid stride, so fewer blocks only run longer)
            const int64_t block_bytes = (int64_t)sizeof(int4) * kGenericWarps * p->max_nb;
            p->generic_blocks = std::max<int64_t>(1, std::min<int64_t>(p->generic_blocks, (int64_t(2) << 30) / block_bytes));
            G3_CUDA(cudaMalloc(&p->d_generic_nb, sizeof(int4) * (size_t)p->generic_blocks * kGenericWarps * p->max_nb));
        }
    } else {
        int rc = tiled_configure(p);
        if (rc != G3_OK) return rc;
    }

    const int64_t B = p->batch_frames, n = p->n, nc3 = (int64_t)p->ncell * p->ncell * p->ncell;
    G3_CUDA(cudaMalloc(&p->d_staged, sizeof(int4) * B * n));
    G3_CUDA(cudaMalloc(&p->d_slot, sizeof(int32_t) * B * n));
    G3_CUDA(cudaMalloc(&p->d_cell_count, sizeof(int32_t) * B * nc3));
    G3_CUDA(cudaMalloc(&p->d_cell_start, sizeof(int32_t) * B * (nc3 + 1)));
    G3_CUDA(cudaMalloc(&p->d_sorted, sizeof(int4) * B * n));
    G3_CUDA(cudaMalloc(&p->d_sortedf, sizeof(float4) * B * n));
    G3_CUDA(cudaMemset(p->d_cell_count, 0, sizeof(int32_t) * B * nc3));
    if (p->qtet_bins > 0) {
        G3_CUDA(cudaMalloc(&p->d_qtet, sizeof(unsigned long long) * p->qtet_bins));
        G3_CUDA(cudaMalloc(&p->d_qtet_stats, sizeof(unsigned long long) * 2));
        G3_CUDA(cudaMemset(p->d_qtet, 0, sizeof(unsigned long long) * p->qtet_bins));
        G3_CUDA(cudaMemset(p->d_qtet_stats, 0, sizeof(unsigned long long) * 2));
        G3_CUDA(allow_max_dynamic_smem(qtet_kernel<kQtetWarps>, p->smem_optin));
        G3_CUDA(allow_max_dynamic_smem(qtet_redo_kernel<kQtetWarps>, p->smem_optin));
        G3_CUDA(allow_max_dynamic_smem(qtet_list_kernel, p->smem_optin));
        if (p->qtet_lists) {                                // only the list of undecided atoms is needed
            G3_CUDA(cudaMalloc(&p->d_qtet_redo, sizeof(int32_t) * (size_t)(B * n + 1)));
        } else if (p->ncell > 1 && B * n < (int64_t(1) << 31)) {   // fast path: 27 cells staged per CTA
            p->qtet_stage_cap = tiled_stage_cap(p);
            const size_t smem = qtet_cell_smem_bytes(p->qtet_stage_cap, p->qtet_bins);
            if (smem <= (size_t)p->smem_optin) {
                G3_CUDA(allow_max_dynamic_smem(qtet_cell_kernel, p->smem_optin));
                G3_CUDA(cudaMalloc(&p->d_qtet_redo, sizeof(int32_t) * (size_t)(B * n + 1)));
                const int32_t nc = p->ncell;
                std::vector<int4> origin((size_t)nc3);
                for (int32_t cx = 0; cx < nc; ++cx)
                    for (int32_t cy = 0; cy < nc; ++cy)
                        for (int32_t cz = 0; cz < nc; ++cz)
                            origin[((size_t)cx * nc + cy) * nc + cz] =
                                make_int4((int32_t)(((int64_t)(2 * cx + 1) << (kGridBits - 1)) / nc),
                                          (int32_t)(((int64_t)(2 * cy + 1) << (kGridBits - 1)) / nc),
                                          (int32_t)(((int64_t)(2 * cz + 1) << (kGridBits - 1)) / nc), 0);
                G3_CUDA(cudaMalloc(&p->d_qtet_origin, sizeof(int4) * origin.size()));
                G3_CUDA(cudaMemcpy(p->d_qtet_origin, origin.data(), sizeof(int4) * origin.size(), cudaMemcpyHostToDevice));
            }
        }
    }
    if (p->g2_wide) {
        // staged half-stencil: 64 of the 125 cells around a centre cell (1.5 x their mean occupancy)
        p->g2w_cap = (int32_t)(((int64_t)(1.5 * 64.0 * (double)p->n / (double)nc3) + 96 + 63) / 64 * 64);
        p->g2w_smem = g2w_cell_smem_bytes(p->g2w_cap, p->bins.n_r);
        p->g2w_grid = 0;
        if (p->ncell >= 5 && p->g2w_smem + 2048 <= (size_t)p->smem_optin) {
            G3_CUDA(allow_max_dynamic_smem(g2_wide_cell_kernel, p->smem_optin));
            int per_sm = 0;      // persistent: exactly the CTAs that are resident together
            G3_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, g2_wide_cell_kernel, (kNbWarps + 1) * 32, p->g2w_smem));
            p->g2w_grid = p->sm_count * std::max(per_sm, 1);
        }
    }
    p->configured = true;
    return G3_OK;
}

// The batch size changes no result, only how many frames share one launch sequence: when device
// memory is short (another plan, a co-resident simulation) the batch is halved until the buffers fit.
int configure(g3_plan* p) {
    if (p->configured) return G3_OK;
    p->batch_limit = INT32_MAX;
    for (;;) {
        const int rc = configure_once(p);
        if (rc == G3_OK) return rc;
        free_buffers(p);
        if (rc != G3_ENOMEM || p->batch_frames <= 1) return rc;
        p->batch_limit = std::max(1, p->batch_frames / 2);
    }
}

// Reduce the staged frames into the histogram.
int flush(g3_plan* p, cudaStream_t st) {
    if (p->pending == 0) return G3_OK;
    const int32_t F = p->pending, n = (int32_t)p->n;
    const int32_t nc3 = p->ncell * p->ncell * p->ncell;
    const long long total = (long long)F * n;
    cell_scan_kernel<<<F, 1024, 0, st>>>(p->d_cell_count, p->d_cell_start, nc3);
    cell_scatter_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(
        p->d_staged, p->d_slot, p->d_cell_start, n, F, nc3, p->d_sorted, p->d_sortedf);
    p->launches += 2;
    G3_CUDA(cudaMemsetAsync(p->d_cell_count, 0, sizeof(int32_t) * (size_t)F * nc3, st));

    FrameBatch fb{n, F, p->ncell, nc3, p->d_sorted, p->d_sortedf, p->d_cell_start};
    BinSpec bs{p->bins.n_r, p->bins.n_t, p->d_T_r, p->d_T_t, p->T_r.back()};
    if (p->kernel == 1) {
        size_t smem = generic_smem_bytes(bs.n_r, bs.n_t, p->max_nb, kGenericWarps, p->d_generic_nb == nullptr);
        long long blocks = std::min<long long>((total + kGenericWarps - 1) / kGenericWarps, (long long)p->generic_blocks);
        generic_triplet_kernel<kGenericWarps><<<(unsigned)blocks, kGenericWarps * 32, smem, st>>>(
            fb, bs, p->max_nb, p->d_generic_nb, p->d_counts, p->d_counts2, p->d_stats);
        p->launches += 1;
    } else {
        int rc = tiled_launch(p, fb, bs, st);
        if (rc != G3_OK) return rc;
    }
    G3_CUDA(cudaGetLastError());
    if (p->g2_wide) {                                      // pair histogram of the shells n_r .. 2 n_r - 1
        const double w = (p->r_max / (double)bs.n_r) * p->inv_g, eps = 1.0 / 1048576.0;
        G2wParams gp{};
        gp.sh.n_r = 2 * bs.n_r; gp.sh.T_r = p->d_T2; gp.sh.cut2 = p->T2.back();
        gp.sh.cut_lo = (float)((double)p->T2.back() * (1.0 - eps));
        gp.sh.cut_hi = (float)((double)p->T2.back() * (1.0 + eps));
        gp.sh.inv_w_lo = (float)((1.0 / w) * (1.0 - eps));
        gp.sh.inv_w_hi = (float)((1.0 / w) * (1.0 + eps));
        gp.n_lo = bs.n_r; gp.counts2 = p->d_counts2;
        if (p->g2w_grid > 0) {                             // stage capacity, shared memory and grid: see configure_once
            const long long items = (long long)nc3 * F;
            g2_wide_cell_kernel<<<(unsigned)std::min<long long>(items, (long long)p->g2w_grid),
                                  (kNbWarps + 1) * 32, p->g2w_smem, st>>>(fb, gp, p->g2w_cap);
        } else {
            const long long blocks = std::min<long long>((total + kG2wWarps - 1) / kG2wWarps, (long long)p->sm_count * 8);
            g2_wide_kernel<<<(unsigned)blocks, kG2wWarps * 32, sizeof(uint32_t) * bs.n_r, st>>>(fb, gp);
        }
        p->launches += 1;
        G3_CUDA(cudaGetLastError());
    }
    if (p->qtet_bins > 0) {                                // q_tet on the same cell list (Eq. 1)
        const unsigned long long cw = (unsigned long long)(kGrid / p->ncell);
        QtParams qp{p->qtet_bins, (double)p->qtet_bins / 4.0, cw * cw, p->d_qtet, p->d_qtet_stats,
                    p->qtet_stage_cap, p->d_qtet_origin, p->d_qtet_redo, 0};
        const size_t hist_smem = sizeof(unsigned int) * p->qtet_bins;
        if (p->qtet_lists) {
            // the four nearest neighbours sit at the head of the shell-sorted lists this batch's
            // neighbour kernel has just written; atoms with fewer than four go to the exact routine
            G3_CUDA(cudaMemsetAsync(p->d_qtet_redo, 0, sizeof(int32_t), st));
            const g3::TiledState* ts = p->tiled;
            qtet_list_kernel<<<(unsigned)std::min<long long>((total + 255) / 256, (long long)p->sm_count * 8), 256,
                               hist_smem, st>>>(ts->d_nbv, ts->d_nbj, ts->d_nbcount, total, p->max_nb, qp);
            qp.use_redo = 1;
            qtet_redo_kernel<kQtetWarps><<<(unsigned)p->sm_count * 2, kQtetWarps * 32, hist_smem, st>>>(fb, qp);
            p->launches += 2;
        } else if (p->d_qtet_redo) {
            G3_CUDA(cudaMemsetAsync(p->d_qtet_redo, 0, sizeof(int32_t), st));
            const long long items = (long long)nc3 * F;
            // persistent: exactly the CTAs that are resident together (a larger grid would run a second wave)
            const size_t cell_smem = qtet_cell_smem_bytes(p->qtet_stage_cap, p->qtet_bins);
            int per_sm = 0;
            G3_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, qtet_cell_kernel, kQtCellWarps * 32, cell_smem));
            per_sm = std::max(per_sm, 1);
            qtet_cell_kernel<<<(unsigned)std::min<long long>(items, (long long)p->sm_count * per_sm), kQtCellWarps * 32,
                               cell_smem, st>>>(fb, qp);
            qp.use_redo = 1;                               // the few atoms the fast path could not decide
            qtet_redo_kernel<kQtetWarps><<<(unsigned)p->sm_count * 2, kQtetWarps * 32, hist_smem, st>>>(fb, qp);
            p->launches += 2;
        } else {
            long long blocks = std::min<long long>((total + kQtetWarps - 1) / kQtetWarps, (long long)p->sm_count * 8);
            qtet_kernel<kQtetWarps><<<(unsigned)blocks, kQtetWarps * 32, hist_smem, st>>>(fb, qp);
            p->launches += 1;
        }
        G3_CUDA(cudaGetLastError());
    }
    p->pending = 0;
    return G3_OK;
}

int accumulate_device(g3_plan* p, const double* d_pos, int64_t n_frames, int64_t stride,
                      cudaStream_t st) {
    int rc = configure(p);
    if (rc != G3_OK) return rc;
    int64_t done = 0;
    while (done < n_frames) {
        const int64_t room = p->batch_frames - p->pending;
        const int64_t take = std::min(room, n_frames - done);
        const long long total = (long long)take * p->n;
        const int32_t nc3 = p->ncell * p->ncell * p->ncell;
        quantise_count_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(
            d_pos + done * stride, stride, (int32_t)p->n, (int32_t)take, p->inv_g, p->ncell,
            p->d_staged + (size_t)p->pending * p->n, p->d_slot + (size_t)p->pending * p->n,
            p->d_cell_count + (size_t)p->pending * nc3, p->d_stats + 4);
        p->launches += 1;
        G3_CUDA(cudaGetLastError());
        p->pending += (int32_t)take;
        p->frames += (uint64_t)take;
        done += take;
        if (p->pending == p->batch_frames) {
            rc = flush(p, st);
            if (rc != G3_OK) return rc;
        }
    }
    return G3_OK;
}

}  // namespace

extern "C" {

const char* g3_strerror(int code) {
    switch (code) {
        case G3_OK: return "ok";
        case G3_EINVAL: return "invalid argument";
        case G3_ENOMEM: return "out of memory";
        case G3_ECUDA: return "CUDA error or no usable sm_100 device";
        case G3_ECAPACITY: return "neighbour capacity exceeded";
        case G3_ESTATE: return "call not valid in this plan state";
        case G3_EINTERNAL: return "internal invariant violated (histogram tile)";
        case G3_ELIMIT: return "problem exceeds the built-in scratch of a no-allocation entry point";
        default: return "unknown status";
    }
}

int g3_plan_create(g3_plan** out, int64_t n, double box, double r_max, g3_bins bins) {
    if (!out) return G3_EINVAL;
    *out = nullptr;
    if (n < 3 || n > (int64_t(1) << 30) || !(box > 0.0) || !(r_max > 0.0) || !(r_max < 0.5 * box) ||
        !std::isfinite(box) || bins.n_r < 1 || bins.n_t < 1 || bins.n_r > 1024 || bins.n_t > 1024)
        return G3_EINVAL;
    int dev = -1, count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || count < 1) { cudaGetLastError(); return G3_ECUDA; }
    G3_CUDA(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    G3_CUDA(cudaGetDeviceProperties(&prop, dev));
    if (prop.major < 10) return G3_ECUDA;              // built for sm_100a only; no fallback

    g3_plan* p = new (std::nothrow) g3_plan;
    if (!p) return G3_ENOMEM;
    p->n = n; p->box = box; p->r_max = r_max; p->bins = bins;
    p->nbins = (int64_t)bins.n_r * bins.n_r * bins.n_t;
    p->device = dev;
    p->sm_count = prop.multiProcessorCount;
    p->smem_optin = (int)prop.sharedMemPerBlockOptin;

    // squared bin edges in grid units: fp64, one rounding per operation
    p->inv_g = 1048576.0 / box;
    {
        volatile double w = (r_max / (double)bins.n_r) * p->inv_g;
        volatile double wt = ((2.0 * r_max) / (double)bins.n_t) * p->inv_g;
        p->T_r.resize(bins.n_r + 1);
        p->T_t.resize(bins.n_t + 1);
        for (int32_t b = 0; b <= bins.n_r; ++b) {
            volatile double e = (double)b * w;
            volatile double e2 = e * e;
            p->T_r[b] = (unsigned long long)std::ceil(e2);
        }
        for (int32_t c = 0; c <= bins.n_t; ++c) {
            volatile double e = (double)c * wt;
            volatile double e2 = e * e;
            p->T_t[c] = (unsigned long long)std::ceil(e2);
        }
        p->T2.resize(2 * bins.n_r + 1);                       // the same shells carried on to 2 r_max (g2)
        for (int32_t b = 0; b <= 2 * bins.n_r; ++b) {
            volatile double e = (double)b * w;
            volatile double e2 = e * e;
            p->T2[b] = (unsigned long long)std::ceil(e2);
        }
    }
    // strictly increasing edges are required by bin(); they fail only for absurd bin counts
    for (size_t i = 0; i + 1 < p->T_r.size(); ++i)
        if (p->T_r[i] >= p->T_r[i + 1]) { delete p; return G3_EINVAL; }
    for (size_t i = 0; i + 1 < p->T_t.size(); ++i)
        if (p->T_t[i] >= p->T_t[i + 1]) { delete p; return G3_EINVAL; }
    if (!bin_volumes(r_max, bins.n_r, bins.n_t, p->volumes)) { delete p; return G3_EINVAL; }

    auto fail = [&](int code) { g3_plan_destroy(p); return code; };
#define G3_TRY(call)                                                           \
    do {                                                                       \
        cudaError_t e__ = (call);                                              \
        if (e__ != cudaSuccess) {                                              \
            cudaGetLastError();                                                \
            return fail(e__ == cudaErrorMemoryAllocation ? G3_ENOMEM : G3_ECUDA); \
        }                                                                      \
    } while (0)
    G3_TRY(cudaMalloc(&p->d_T_r, sizeof(unsigned long long) * p->T_r.size()));
    G3_TRY(cudaMalloc(&p->d_T_t, sizeof(unsigned long long) * p->T_t.size()));
    G3_TRY(cudaMalloc(&p->d_counts, sizeof(unsigned long long) * p->nbins));
    G3_TRY(cudaMalloc(&p->d_stats, sizeof(unsigned long long) * 8));
    G3_TRY(cudaMalloc(&p->d_counts2, sizeof(unsigned long long) * 2 * bins.n_r));
    G3_TRY(cudaMemset(p->d_counts2, 0, sizeof(unsigned long long) * 2 * bins.n_r));
    G3_TRY(cudaMalloc(&p->d_T2, sizeof(unsigned long long) * p->T2.size()));
    G3_TRY(cudaMemcpy(p->d_T2, p->T2.data(), sizeof(unsigned long long) * p->T2.size(), cudaMemcpyHostToDevice));
    {   // shell volumes V_a = (4 pi / 3)(r_{a+1}^3 - r_a^3) for g2, up to 2 r_max
        std::vector<double> v2(2 * bins.n_r);
        const double w = r_max / (double)bins.n_r;
        for (int32_t a = 0; a < 2 * bins.n_r; ++a) {
            const double r0 = a * w, r1 = (a + 1) * w;
            v2[a] = (4.0 * 3.14159265358979323846 / 3.0) * (r1 * r1 * r1 - r0 * r0 * r0);
        }
        G3_TRY(cudaMalloc(&p->d_volumes2, sizeof(double) * 2 * bins.n_r));
        G3_TRY(cudaMemcpy(p->d_volumes2, v2.data(), sizeof(double) * 2 * bins.n_r, cudaMemcpyHostToDevice));
    }
    G3_TRY(cudaMalloc(&p->d_volumes, sizeof(double) * p->nbins));
    G3_TRY(cudaMemcpy(p->d_T_r, p->T_r.data(), sizeof(unsigned long long) * p->T_r.size(), cudaMemcpyHostToDevice));
    G3_TRY(cudaMemcpy(p->d_T_t, p->T_t.data(), sizeof(unsigned long long) * p->T_t.size(), cudaMemcpyHostToDevice));
    G3_TRY(cudaMemcpy(p->d_volumes, p->volumes.data(), sizeof(double) * p->nbins, cudaMemcpyHostToDevice));
    G3_TRY(cudaMemset(p->d_counts, 0, sizeof(unsigned long long) * p->nbins));
    G3_TRY(cudaMemset(p->d_stats, 0, sizeof(unsigned long long) * 8));
#undef G3_TRY
    *out = p;
    return G3_OK;
}

int g3_plan_set_option(g3_plan* p, int32_t option, int64_t value) {
    if (!p) return G3_EINVAL;
    if (p->frames != 0) return G3_ESTATE;
    switch (option) {
        case G3_OPT_BATCH_FRAMES:
            if (value < 1 || value > 4096) return G3_EINVAL;
            p->batch_frames = (int32_t)value; p->batch_auto = false; break;
        case G3_OPT_KERNEL:
            if (value < 0 || value > 2) return G3_EINVAL;
            p->kernel_opt = (int32_t)value; break;
        case G3_OPT_MAX_NEIGHBOURS:
            if (value < 0 || value > (1 << 20)) return G3_EINVAL;
            p->max_nb_opt = (int32_t)value; break;
        case G3_OPT_TRIPLET_WARPS:
            if (value != 0 && (value < 8 || value > 24 || value % 4 != 0)) return G3_EINVAL;
            p->tri_warps_opt = (int32_t)value; break;
        case G3_OPT_G2_WIDE:
            if (value < 0 || value > 1) return G3_EINVAL;
            p->g2_wide = (int32_t)value; break;
        case G3_OPT_QTET_BINS:
            if (value < 0 || value > 8192 || (value > 0 && p->n < 5)) return G3_EINVAL;
            p->qtet_bins = (int32_t)value; break;
        case G3_OPT_TIMING:
            if (value < 0 || value > 1) return G3_EINVAL;
            p->timing = (int32_t)value; return G3_OK;
        default: return G3_EINVAL;
    }
    if (p->configured) free_buffers(p);
    return G3_OK;
}

int g3_plan_get_info(const g3_plan* cp, int32_t key, int64_t* value) {
    if (!cp || !value) return G3_EINVAL;
    g3_plan* p = const_cast<g3_plan*>(cp);
    if (key >= G3_INFO_TRIPLET_NS && key <= G3_INFO_TIMED_LAUNCHES) {
        int rc = fold_timing(p);
        if (rc != G3_OK) return rc;
        *value = key == G3_INFO_TRIPLET_NS ? (int64_t)llround(p->triplet_ms * 1e6)
               : key == G3_INFO_NEIGHBOUR_NS ? (int64_t)llround(p->neighbour_ms * 1e6)
               : p->timed_launches;
        return G3_OK;
    }
    if (key != G3_INFO_KERNEL_LAUNCHES && key != G3_INFO_FRAMES_PENDING && key != G3_INFO_SM_COUNT) {
        int rc = configure(p);
        if (rc != G3_OK) return rc;
    }
    switch (key) {
        case G3_INFO_KERNEL_LAUNCHES: *value = (int64_t)p->launches; break;
        case G3_INFO_BATCH_FRAMES: *value = p->batch_frames; break;
        case G3_INFO_KERNEL: *value = p->kernel; break;
        case G3_INFO_CELLS_PER_EDGE: *value = p->ncell; break;
        case G3_INFO_MAX_NEIGHBOURS: *value = p->max_nb; break;
        case G3_INFO_TILE_BINS: *value = p->tile_bins; break;
        case G3_INFO_SM_COUNT: *value = p->sm_count; break;
        case G3_INFO_FRAMES_PENDING: *value = p->pending; break;
        case G3_INFO_SLABS: *value = p->tiled ? p->tiled->n_slabs : 0; break;
        case G3_INFO_G2_SHELLS: *value = p->g2_wide ? 2 * p->bins.n_r : p->bins.n_r; break;
        default: return G3_EINVAL;
    }
    return G3_OK;
}

int g3_plan_clear_timing(g3_plan* p) {
    if (!p) return G3_EINVAL;
    int rc = fold_timing(p);
    p->triplet_ms = p->neighbour_ms = 0;
    p->timed_launches = 0;
    p->launches = 0;
    return rc;
}

int g3_accumulate_frames(g3_plan* p, const double* d_pos, int64_t n_frames, int64_t frame_stride,
                         void* stream) {
    if (!p || !d_pos || n_frames < 0 || frame_stride < 3 * p->n) return G3_EINVAL;
    return accumulate_device(p, d_pos, n_frames, frame_stride, (cudaStream_t)stream);
}

int g3_accumulate_frame(g3_plan* p, const double* d_pos, void* stream) {
    if (!p || !d_pos) return G3_EINVAL;
    return accumulate_device(p, d_pos, 1, 3 * p->n, (cudaStream_t)stream);
}

int g3_accumulate_frames_host(g3_plan* p, const double* h_pos, int64_t n_frames,
                              int64_t frame_stride, void* stream) {
    if (!p || !h_pos || n_frames < 0 || frame_stride < 3 * p->n) return G3_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = configure(p);
    if (rc != G3_OK) return rc;
    const int64_t chunk = p->batch_frames;
    const size_t frame_bytes = sizeof(double) * 3 * (size_t)p->n;
    if (!p->d_h2d) {
        G3_CUDA(cudaMalloc(&p->d_h2d, 2 * chunk * frame_bytes));
        p->h2d_chunk_frames = chunk;
        p->h2d_chunks = 0;
        if (!p->copy_stream) {
            G3_CUDA(cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
            for (int i = 0; i < 2; ++i) {
                G3_CUDA(cudaEventCreateWithFlags(&p->h2d_done[i], cudaEventDisableTiming));
                G3_CUDA(cudaEventCreateWithFlags(&p->h2d_free[i], cudaEventDisableTiming));
            }
        }
    }
    // Two device staging halves.  The copies run on the plan's own copy stream (copy engine), the
    // kernels on the caller's stream: the copy of chunk c+1 overlaps the neighbour/triplet
    // kernels of chunk c.  h2d_done[h] orders copy -> quantise kernel, h2d_free[h] orders the
    // kernels that read half h -> the next copy into it.  When the caller's stream has passed
    // this call every copy has completed, so the include/g3.h lifetime rule for h_pos holds.
    // A long call ramps up: its first two chunks are a quarter and a half of a batch and are reduced at
    // once, so that the GPU starts after a quarter of a batch's copy time and every later copy is hidden
    // behind the kernels of the chunk before it.
    const bool ramp = p->pending == 0 && n_frames >= 3 * chunk && chunk >= 8;
    int64_t done = 0;
    int n_chunk = 0;
    while (done < n_frames) {
        const bool head = ramp && n_chunk < 2;
        const int64_t take = head ? (n_chunk == 0 ? chunk / 4 : chunk / 2) : std::min(chunk, n_frames - done);
        ++n_chunk;
        const int h = (int)(p->h2d_chunks & 1);
        double* dst = p->d_h2d + (size_t)h * chunk * 3 * p->n;
        if (p->h2d_chunks >= 2) G3_CUDA(cudaStreamWaitEvent(p->copy_stream, p->h2d_free[h], 0));
        if (frame_stride == 3 * p->n) {
            G3_CUDA(cudaMemcpyAsync(dst, h_pos + done * frame_stride, take * frame_bytes,
                                    cudaMemcpyHostToDevice, p->copy_stream));
        } else {
            G3_CUDA(cudaMemcpy2DAsync(dst, frame_bytes, h_pos + done * frame_stride,
                                      sizeof(double) * frame_stride, frame_bytes, take,
                                      cudaMemcpyHostToDevice, p->copy_stream));
        }
        G3_CUDA(cudaEventRecord(p->h2d_done[h], p->copy_stream));
        G3_CUDA(cudaStreamWaitEvent(st, p->h2d_done[h], 0));
        rc = accumulate_device(p, dst, take, 3 * p->n, st);
        if (rc == G3_OK && head) rc = flush(p, st);
        if (rc != G3_OK) return rc;
        G3_CUDA(cudaEventRecord(p->h2d_free[h], st));
        p->h2d_chunks += 1;
        done += take;
    }
    return G3_OK;
}

int g3_normalize(g3_plan* p, const uint64_t* d_counts, uint64_t frames, double* d_g3, void* stream) {
    if (!p || !d_counts || !d_g3) return G3_EINVAL;
    const double rho = (double)p->n / (p->box * p->box * p->box);
    const double ideal = (double)frames * (double)p->n * rho * rho;
    const double inv_ideal = frames ? 1.0 / ideal : 0.0;
    normalise_kernel<<<(unsigned)((p->nbins + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        reinterpret_cast<const unsigned long long*>(d_counts), p->d_volumes, p->nbins, inv_ideal, d_g3);
    p->launches += 1;
    G3_CUDA(cudaGetLastError());
    return G3_OK;
}

int g3_finalize(g3_plan* p, uint64_t* d_counts, double* d_g3, uint64_t* h_stats, void* stream) {
    if (!p) return G3_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = configure(p);
    if (rc != G3_OK) return rc;
    rc = flush(p, st);
    if (rc != G3_OK) return rc;
    rc = tiled_merge(p, st);
    if (rc != G3_OK) return rc;
    if (d_counts)
        G3_CUDA(cudaMemcpyAsync(d_counts, p->d_counts, sizeof(uint64_t) * p->nbins,
                                cudaMemcpyDeviceToDevice, st));
    if (d_g3) {
        rc = g3_normalize(p, reinterpret_cast<const uint64_t*>(p->d_counts), p->frames, d_g3, stream);
        if (rc != G3_OK) return rc;
    }
    unsigned long long stats[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    G3_CUDA(cudaMemcpyAsync(stats, p->d_stats, sizeof(stats), cudaMemcpyDeviceToHost, st));
    G3_CUDA(cudaStreamSynchronize(st));
    if (h_stats) { h_stats[0] = p->frames; h_stats[1] = stats[0]; h_stats[2] = stats[1]; }
    if (stats[3]) return G3_EINTERNAL;      // counts outside the mapped tile slots: must never happen
    if (stats[4]) return G3_EINVAL;         // NaN, infinite or absurdly large coordinates were staged
    return stats[2] ? G3_ECAPACITY : G3_OK;
}

int g3_finalize_g2(g3_plan* p, uint64_t* d_counts2, double* d_g2, void* stream) {
    if (!p) return G3_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = configure(p);
    if (rc != G3_OK) return rc;
    rc = flush(p, st);
    if (rc != G3_OK) return rc;
    rc = tiled_merge(p, st);
    if (rc != G3_OK) return rc;
    const int32_t n_r = p->g2_wide ? 2 * p->bins.n_r : p->bins.n_r;       // shells returned
    if (d_counts2)
        G3_CUDA(cudaMemcpyAsync(d_counts2, p->d_counts2, sizeof(uint64_t) * n_r, cudaMemcpyDeviceToDevice, st));
    if (d_g2) {
        const double rho = (double)p->n / (p->box * p->box * p->box);
        const double ideal = (double)p->frames * (double)p->n * rho;
        normalise_g2_kernel<<<(unsigned)((n_r + 255) / 256), 256, 0, st>>>(
            p->d_counts2, p->d_volumes2, n_r, p->frames ? 1.0 / ideal : 0.0, d_g2);
        p->launches += 1;
        G3_CUDA(cudaGetLastError());
    }
    return G3_OK;
}

int g3_finalize_qtet(g3_plan* p, uint64_t* d_hist, uint64_t* h_stats, void* stream) {
    if (!p) return G3_EINVAL;
    if (p->qtet_bins <= 0) return G3_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = configure(p);
    if (rc != G3_OK) return rc;
    rc = flush(p, st);
    if (rc != G3_OK) return rc;
    if (d_hist)
        G3_CUDA(cudaMemcpyAsync(d_hist, p->d_qtet, sizeof(uint64_t) * p->qtet_bins, cudaMemcpyDeviceToDevice, st));
    unsigned long long stats[2] = {0, 0}, plan_stats[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    G3_CUDA(cudaMemcpyAsync(stats, p->d_qtet_stats, sizeof(stats), cudaMemcpyDeviceToHost, st));
    G3_CUDA(cudaMemcpyAsync(plan_stats, p->d_stats, sizeof(plan_stats), cudaMemcpyDeviceToHost, st));
    G3_CUDA(cudaStreamSynchronize(st));
    if (h_stats) { h_stats[0] = stats[0]; h_stats[1] = stats[1]; }
    if (plan_stats[4]) return G3_EINVAL;    // NaN, infinite or absurdly large coordinates were staged
    // q_tet read off the neighbour lists: a list cut at the capacity is cut in scan order, not by
    // distance, so the four nearest may be among the dropped entries
    if (plan_stats[2] && p->qtet_lists) return G3_ECAPACITY;
    return G3_OK;
}

int g3_finalize_host(g3_plan* p, uint64_t* h_counts, double* h_g3, uint64_t* h_stats, void* stream) {
    if (!p) return G3_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    double* d_g3 = nullptr;
    if (h_g3) G3_CUDA(cudaMallocAsync(&d_g3, sizeof(double) * p->nbins, st));
    int rc = g3_finalize(p, nullptr, d_g3, h_stats, stream);
    if (rc == G3_OK || rc == G3_ECAPACITY || rc == G3_EINVAL) {
        cudaError_t e = cudaSuccess;
        if (h_counts) e = cudaMemcpyAsync(h_counts, p->d_counts, sizeof(uint64_t) * p->nbins, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && h_g3) e = cudaMemcpyAsync(h_g3, d_g3, sizeof(double) * p->nbins, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) rc = G3_ECUDA;
    }
    if (d_g3) cudaFreeAsync(d_g3, st);
    return rc;
}

int g3_msd(const double* d_pos, int64_t n_frames, int64_t n, int64_t frame_stride, double box,
           int64_t max_lag, uint64_t* d_sums, double* d_msd, void* stream) {
    if (!d_pos || n_frames < 1 || n < 1 || n > (int64_t(1) << 30) || n_frames > (int64_t(1) << 24) ||
        frame_stride < 3 * n || !(box > 0.0) || !std::isfinite(box) || max_lag < 0 || max_lag > n_frames - 1)
        return G3_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, cc_major = 0, smem_optin = 0, sm_count = 0;    // (cudaGetDeviceProperties takes ms)
    G3_CUDA(cudaGetDevice(&dev));
    G3_CUDA(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev));
    G3_CUDA(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    G3_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
    if (cc_major < 10) return G3_ECUDA;
    const int32_t n_blocks = (int32_t)((n + kMsdAtoms - 1) / kMsdAtoms);
    // trajectories of 32 atoms + the prefix table of their squares
    const size_t traj_smem = (size_t)n_frames * kMsdAtoms * 3 * sizeof(int32_t) + (size_t)(n_frames + 1) * sizeof(ulonglong2);
    const bool smem_path = traj_smem <= (size_t)smem_optin;
    MsdParams mp;
    mp.pos = d_pos; mp.stride = frame_stride; mp.n = (int32_t)n; mp.n_frames = (int32_t)n_frames;
    mp.max_lag = (int32_t)max_lag; mp.inv_g = 1048576.0 / box; mp.snapped = nullptr;
    void* ws = nullptr;                   // partials | bad counter | snapped copy (global path)
    const size_t part_bytes = sizeof(ulonglong2) * (size_t)n_blocks * (size_t)(max_lag + 1);
    const size_t snap_bytes = smem_path ? 0 : sizeof(int32_t) * 3 * (size_t)n * (size_t)n_frames;
    G3_CUDA(cudaMallocAsync(&ws, part_bytes + 16 + snap_bytes, st));
    mp.partial = reinterpret_cast<ulonglong2*>(ws);
    mp.bad = reinterpret_cast<unsigned long long*>(reinterpret_cast<char*>(ws) + part_bytes);
    int rc = G3_OK;
    auto fail = [&](int code) { cudaFreeAsync(ws, st); cudaGetLastError(); return code; };
    if (cudaMemsetAsync(mp.bad, 0, 16, st) != cudaSuccess) return fail(G3_ECUDA);
    if (smem_path) {
        if (allow_max_dynamic_smem(msd_kernel, smem_optin) != cudaSuccess) return fail(G3_ECUDA);
        msd_kernel<<<n_blocks, kMsdWarps * 32, traj_smem, st>>>(mp);
    } else {
        mp.snapped = reinterpret_cast<int32_t*>(reinterpret_cast<char*>(ws) + part_bytes + 16);
        msd_snap_kernel<<<sm_count * 8, 256, 0, st>>>(mp);
        msd_direct_kernel<<<n_blocks, kMsdWarps * 32, 0, st>>>(mp);
    }
    const double g = box / 1048576.0;
    msd_reduce_kernel<<<(unsigned)((max_lag + 32) / 32), 256, 0, st>>>(
        mp.partial, n_blocks, (int32_t)max_lag, (int32_t)n, (int32_t)n_frames, g * g,
        reinterpret_cast<unsigned long long*>(d_sums), d_msd);
    if (cudaGetLastError() != cudaSuccess) return fail(G3_ECUDA);
    unsigned long long bad = 0;
    if (cudaMemcpyAsync(&bad, mp.bad, sizeof(bad), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) return fail(G3_ECUDA);
    cudaFreeAsync(ws, st);
    if (bad) rc = G3_EINVAL;              // coordinates outside +-2^30 grid units: results invalid
    return rc;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// g3_msd_static: g3_msd without any device allocation (include/g3.h says who needs that and why).
// The scratch of msd_kernel / msd_reduce_kernel -- the per-(CTA, lag) 128-bit partial sums and the
// bad-coordinate counter -- lives in the array below instead of in memory from the stream's pool.
// The kernels are the ones g3_msd launches, so the sums are the same integers.
//
// The array has static storage on the device: the driver creates one copy per GPU when this
// library's kernels are loaded there, and it stays until the process ends.  Layout: bytes [0, 8)
// the bad-coordinate counter, bytes [256, 256 + 16 * kMsdStaticPartials) the partial sums.
//
// NOTE for whoever edits this: in HOST code the name `g3_msd_static_scratch` is only a handle for
// the runtime's symbol table, not a device pointer.  Passing it (or its address) to a kernel
// compiles, and the kernel then faults or, on systems where the GPU can read host memory, quietly
// works on the wrong bytes.  Host code gets the real address from cudaGetSymbolAddress, once per
// device, with that device current (msd_static_scratch_ptr below).
constexpr size_t kMsdStaticHeader = 256;
constexpr size_t kMsdStaticPartials = G3_MSD_STATIC_MAX_PARTIALS;
static_assert(G3_MSD_STATIC_SCRATCH_BYTES == kMsdStaticHeader + sizeof(ulonglong2) * kMsdStaticPartials,
              "include/g3.h states the size of the built-in scratch");
static __device__ __align__(256) unsigned char g3_msd_static_scratch[G3_MSD_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMsdStaticMaxDevices = 64;
std::mutex g_msd_static_mutex;
unsigned char* g_msd_static_ptr[kMsdStaticMaxDevices] = {};     // device address of the array, per GPU

// One-time set-up per device; `dev` must be the current device (the symbol is resolved in the
// current device's context).  No allocation of ours: the array already exists once the module is
// loaded, and loading it is what the first lookup may trigger.
int msd_static_scratch_ptr(int dev, unsigned char** out) {
    if (dev < 0 || dev >= kMsdStaticMaxDevices) return G3_ECUDA;
    std::lock_guard<std::mutex> lock(g_msd_static_mutex);
    if (!g_msd_static_ptr[dev]) {
        unsigned char* ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g3_msd_static_scratch);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return G3_ECUDA;
        }
        g_msd_static_ptr[dev] = ptr;
    }
    *out = g_msd_static_ptr[dev];
    return G3_OK;
}

}  // namespace

extern "C" {

int g3_msd_static(const double* d_pos, int64_t n_frames, int64_t n, int64_t frame_stride, double box,
                  int64_t max_lag, uint64_t* d_sums, double* d_msd, void* stream) {
    if (!d_pos || n_frames < 1 || n < 1 || n > (int64_t(1) << 30) || n_frames > (int64_t(1) << 24) ||
        frame_stride < 3 * n || !(box > 0.0) || !std::isfinite(box) || max_lag < 0 || max_lag > n_frames - 1)
        return G3_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, cc_major = 0, smem_optin = 0;
    G3_CUDA(cudaGetDevice(&dev));
    G3_CUDA(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev));
    G3_CUDA(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    if (cc_major < 10) return G3_ECUDA;
    // the two limits of the built-in scratch, checked before anything is enqueued
    const int64_t n_blocks = (n + kMsdAtoms - 1) / kMsdAtoms;
    const size_t traj_smem = (size_t)n_frames * kMsdAtoms * 3 * sizeof(int32_t) + (size_t)(n_frames + 1) * sizeof(ulonglong2);
    if (traj_smem > (size_t)smem_optin) return G3_ELIMIT;                  // would need the global snapped copy
    if (n_blocks * (max_lag + 1) > (int64_t)kMsdStaticPartials) return G3_ELIMIT;
    unsigned char* ws = nullptr;
    int rc = msd_static_scratch_ptr(dev, &ws);
    if (rc != G3_OK) return rc;
    MsdParams mp;
    mp.pos = d_pos; mp.stride = frame_stride; mp.n = (int32_t)n; mp.n_frames = (int32_t)n_frames;
    mp.max_lag = (int32_t)max_lag; mp.inv_g = 1048576.0 / box; mp.snapped = nullptr;
    mp.bad = reinterpret_cast<unsigned long long*>(ws);
    mp.partial = reinterpret_cast<ulonglong2*>(ws + kMsdStaticHeader);
    // The array still holds the previous call's contents.  The counter is the only word that is
    // accumulated into, so it is cleared here; every partial sum the reduce kernel reads,
    // [n_blocks][max_lag + 1], is written by msd_kernel in this call (each CTA stores all its lags).
    G3_CUDA(cudaMemsetAsync(mp.bad, 0, sizeof(unsigned long long), st));
    G3_CUDA(allow_max_dynamic_smem(msd_kernel, smem_optin));
    msd_kernel<<<(unsigned)n_blocks, kMsdWarps * 32, traj_smem, st>>>(mp);
    const double g = box / 1048576.0;
    msd_reduce_kernel<<<(unsigned)((max_lag + 32) / 32), 256, 0, st>>>(
        mp.partial, (int32_t)n_blocks, (int32_t)max_lag, (int32_t)n, (int32_t)n_frames, g * g,
        reinterpret_cast<unsigned long long*>(d_sums), d_msd);
    G3_CUDA(cudaGetLastError());
    unsigned long long bad = 0;
    G3_CUDA(cudaMemcpyAsync(&bad, mp.bad, sizeof(bad), cudaMemcpyDeviceToHost, st));
    G3_CUDA(cudaStreamSynchronize(st));
    return bad ? G3_EINVAL : G3_OK;       // coordinates outside +-2^30 grid units: results invalid
}

int g3_bin_volumes(const g3_plan* p, double* h_volumes) {
    if (!p || !h_volumes) return G3_EINVAL;
    std::memcpy(h_volumes, p->volumes.data(), sizeof(double) * p->nbins);
    return G3_OK;
}

int g3_plan_reset(g3_plan* p, void* stream) {
    if (!p) return G3_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    G3_CUDA(cudaMemsetAsync(p->d_counts, 0, sizeof(unsigned long long) * p->nbins, st));
    G3_CUDA(cudaMemsetAsync(p->d_stats, 0, sizeof(unsigned long long) * 8, st));
    G3_CUDA(cudaMemsetAsync(p->d_counts2, 0, sizeof(unsigned long long) * 2 * p->bins.n_r, st));
    if (p->d_qtet) {
        G3_CUDA(cudaMemsetAsync(p->d_qtet, 0, sizeof(unsigned long long) * p->qtet_bins, st));
        G3_CUDA(cudaMemsetAsync(p->d_qtet_stats, 0, sizeof(unsigned long long) * 2, st));
    }
    if (p->configured && p->pending) {
        const size_t nc3 = (size_t)p->ncell * p->ncell * p->ncell;
        G3_CUDA(cudaMemsetAsync(p->d_cell_count, 0, sizeof(int32_t) * p->batch_frames * nc3, st));
    }
    if (p->tiled) {
        G3_CUDA(cudaMemsetAsync(p->tiled->d_scratch, 0,
                                sizeof(unsigned long long) * p->tiled->tile_bins * p->tiled->grid, st));
        p->tiled->dirty = false;
    }
    p->pending = 0;
    p->frames = 0;
    return G3_OK;
}

void g3_plan_destroy(g3_plan* p) {
    if (!p) return;
    cudaDeviceSynchronize();
    free_buffers(p);
    for (int i = 0; i < 2; ++i) {
        if (p->h2d_done[i]) cudaEventDestroy(p->h2d_done[i]);
        if (p->h2d_free[i]) cudaEventDestroy(p->h2d_free[i]);
    }
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    for (cudaEvent_t e : p->ev_pool) cudaEventDestroy(e);
    cudaFree(p->d_T_r); cudaFree(p->d_T_t); cudaFree(p->d_counts); cudaFree(p->d_stats);
    cudaFree(p->d_volumes); cudaFree(p->d_counts2); cudaFree(p->d_volumes2); cudaFree(p->d_T2);
    cudaGetLastError();
    delete p;
}

}  // extern "C"
