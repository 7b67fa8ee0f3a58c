// g3_plan.h -- internal plan state of libg3 (not part of the public ABI, see include/g3.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <climits>
#include <vector>

#include "../../include/g3.h"

namespace g3 {

constexpr int kGridBits = 20;                 // positions live on the box/2^20 grid
constexpr int64_t kGrid = int64_t(1) << kGridBits;
constexpr int kMaxCellsPerEdge = 32;          // cell ids fit 15 bits

// Device-visible description of one batch of staged frames.  Passed by value to kernels.
struct FrameBatch {
    int32_t n;                 // particles per frame
    int32_t n_frames;          // frames in this batch
    int32_t ncell;             // cells per edge (1 = no cell grid: every particle is a candidate)
    int32_t ncell3;
    const int4* sorted;        // [frames][n]  (x, y, z, cell id), cell-major order
    const float4* sortedf;     // [frames][n]  the same coordinates as fp32 (exact: < 2^20), w = 0
    const int32_t* cell_start; // [frames][ncell3 + 1]
};

struct BinSpec {
    int32_t n_r, n_t;
    const unsigned long long* T_r;  // device, [n_r + 1] squared edges in grid units
    const unsigned long long* T_t;  // device, [n_t + 1]
    unsigned long long cut2;        // T_r[n_r]
};

// The dynamic shared-memory limit of a kernel is state of the whole context, shared by every
// plan: it is always set to the device maximum (opt-in limit minus the kernel's static shared
// memory), never to one plan's own size, so plans of different shape cannot disturb each other.
template <class Kernel>
inline cudaError_t allow_max_dynamic_smem(Kernel kernel, int smem_optin) {
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, kernel);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                smem_optin - (int)fa.sharedSizeBytes);
}

}  // namespace g3

namespace g3 { struct TiledState; }

struct g3_plan {
    // problem
    int64_t n = 0;
    double box = 0, r_max = 0;
    g3_bins bins{0, 0};
    int64_t nbins = 0;
    double inv_g = 0;                        // 2^20 / box
    std::vector<unsigned long long> T_r, T_t; // host copies of the squared edges
    std::vector<double> volumes;             // V_abc in box length units^6 (host)

    // device
    int device = -1;
    int sm_count = 0;
    int smem_optin = 0;

    // options / derived
    int32_t batch_frames = 16;               // frames per launch sequence (see batch_auto)
    bool batch_auto = true;                  // derive batch_frames from n: ~2^22 centres per launch sequence
    int32_t batch_limit = INT32_MAX;         // configure(): upper bound after an allocation failed (halved per retry)
    int32_t kernel_opt = 0;                  // G3_OPT_KERNEL
    int32_t kernel = 1;                      // selected kernel
    int32_t ncell = 1;
    int32_t max_nb = 0;                      // neighbour capacity per centre
    int32_t max_nb_opt = 0;
    int32_t timing = 0;                      // G3_OPT_TIMING
    int32_t tri_warps_opt = 0;               // G3_OPT_TRIPLET_WARPS
    int64_t tile_bins = 0;

    // device buffers
    unsigned long long* d_T_r = nullptr;
    unsigned long long* d_T_t = nullptr;
    unsigned long long* d_counts = nullptr;  // [nbins] running histogram (ordered pairs)
    unsigned long long* d_counts2 = nullptr; // [2 n_r] g2: ordered pairs (i, j) per shell of r_ij (upper half: G3_OPT_G2_WIDE)
    unsigned long long* d_T2 = nullptr;      // [2 n_r + 1] squared shell edges b w up to 2 r_max
    std::vector<unsigned long long> T2;
    int32_t g2_wide = 0;                     // G3_OPT_G2_WIDE
    int32_t g2w_cap = 0;                     // g2_wide_cell_kernel: entries per staged half stencil,
    size_t g2w_smem = 0;                     //   its dynamic shared memory and its persistent grid
    int32_t g2w_grid = 0;                    //   (0 = the warp-per-centre g2_wide_kernel serves this plan)
    unsigned long long* d_stats = nullptr;   // [8]: pairs, overflow, capacity error, internal error, bad coordinates
    double* d_volumes = nullptr;             // [nbins]
    double* d_volumes2 = nullptr;            // [2 n_r] shell volumes for g2
    int32_t qtet_bins = 0;                   // G3_OPT_QTET_BINS: 0 = q_tet off
    unsigned long long* d_qtet = nullptr;    // [qtet_bins] histogram of q_tet on [-3, 1]
    unsigned long long* d_qtet_stats = nullptr; // [2]: atoms binned, atoms skipped
    int32_t* d_qtet_redo = nullptr;          // [1 + batch * n]: atoms handed to the exact routine
    int4* d_qtet_origin = nullptr;           // [ncell3] cell centres on the grid
    int32_t qtet_stage_cap = 0;
    bool qtet_lists = false;                 // q_tet taken from the shell-sorted neighbour lists (qtet_list_kernel)
    int4* d_staged = nullptr;                // [batch][n] quantised (x,y,z,cell) in input order
    int32_t* d_slot = nullptr;               // [batch][n] rank of the particle inside its cell
    int32_t* d_cell_count = nullptr;         // [batch][ncell3]
    int32_t* d_cell_start = nullptr;         // [batch][ncell3 + 1]
    int4* d_sorted = nullptr;                // [batch][n]
    int4* d_generic_nb = nullptr;            // generic kernel: [blocks][warps][max_nb] lists when shared memory is too small
    int64_t generic_blocks = 0;
    float4* d_sortedf = nullptr;             // [batch][n] fp32 copy of d_sorted (TMA source of the neighbour kernel)
    double* d_h2d = nullptr;                 // staging for g3_accumulate_frames_host, 2 x chunk
    cudaEvent_t h2d_done[2] = {nullptr, nullptr};   // copy of a staging half finished (copy stream)
    cudaEvent_t h2d_free[2] = {nullptr, nullptr};   // staging half consumed (caller's stream)
    cudaStream_t copy_stream = nullptr;             // host->device copies overlap the kernels
    int64_t h2d_chunk_frames = 0;
    uint64_t h2d_chunks = 0;                        // chunks copied so far (selects the half)
    // G3_OPT_TIMING: event triples (before neighbour, between, after triplet) per launch pair
    std::vector<cudaEvent_t> ev_pool;        // all events ever created (reused after a clear)
    size_t ev_used = 0;                      // events of ev_pool recorded since the last clear
    double triplet_ms = 0, neighbour_ms = 0; // sums already folded in
    int64_t timed_launches = 0;
    g3::TiledState* tiled = nullptr;         // owned by the tiled kernel path (g3_tiled.cuh)

    // state
    int32_t pending = 0;                     // frames staged, not yet reduced
    uint64_t frames = 0;                     // frames accumulated in total (staged included)
    uint64_t launches = 0;                   // kernels launched
    bool configured = false;                 // buffers allocated for the current options
};
