/*
 * g3.h -- C ABI of libg3: the triplet correlation function g(3) of a particle
 * trajectory on one NVIDIA B200 (sm_100a).
 *
 * Method: arxiv 1708.08619 section 3.2.  g(3) is defined by Eq. 3
 * (PAPER.md:403-405); it is computed as a "3D histogram binning of distances
 * with imposed conditions": for every central particle i
 * and every pair (j,k) of its neighbours inside the cut-off, the three pair
 * distances (r_ij, r_ik, r_jk) select one bin.  Algorithm 6
 * is the serial form, Algorithm 7 the GPU form the paper
 * used: CUDA_g2 stores each particle's minimum-image neighbour vectors,
 * CUDA_g3 bins the j-k distance computed from those stored vectors.  Where
 * the paper is silent, DESIGN.md ("Readings of the paper") fixes the reading.
 *
 * Exact definition implemented:
 *   grid      positions are snapped to the box/2^20 grid:
 *             m = llrint(x * (2^20/box)) mod 2^20 per coordinate;
 *   edges     T_r[b] = ceil((b*w)^2), w = (r_max/n_r)*(2^20/box), b = 0..n_r
 *             T_t[c] = ceil((c*wt)^2), wt = ((2*r_max)/n_t)*(2^20/box), c = 0..n_t
 *             (fp64, one rounding per operation); bin(T,q) = max{b : T[b] <= q};
 *   neighbour j != i with minimum-image vector d_j (components in [-2^19, 2^19))
 *             and |d_j|^2 < T_r[n_r]; shell a_j = bin(T_r, |d_j|^2);
 *   triplet   every ORDERED pair (j,k), j != k, of neighbours of i:
 *             t2 = |d_k - d_j|^2 (no second minimum image), c = bin(T_t, t2);
 *             c < n_t  ->  counts[a_j][a_k][c] += 1, else overflow += 1;
 *   g3        counts / (frames * n * rho^2 * V_abc), rho = n/box^3, V_abc the
 *             integral of 8 pi^2 r s t over the part of the bin that obeys
 *             |r-s| <= t <= r+s; 0 where V_abc = 0.
 * counts is symmetric in its first two axes; the number of DISTINCT triplets is
 * (sum(counts) + overflow) / 2 = sum_i C(k_i, 2).
 *
 * General rules
 *   - Every function returns a g3_status (int); nothing throws, aborts or prints.
 *   - "device" pointers are CUDA device pointers on the plan's GPU; "host"
 *     pointers are ordinary host memory.  `stream` is a cudaStream_t passed as
 *     void* (NULL = the legacy default stream).
 *   - The plan owns all scratch memory and the running histogram.  The caller
 *     owns every buffer it passes in.
 *   - A plan is not thread-safe; distinct plans are independent.  All calls on
 *     one plan must be issued on one stream, or be ordered by the caller.
 *   - The library never falls back to the CPU: if no CUDA device is usable,
 *     g3_plan_create fails with G3_ECUDA.
 */
#ifndef G3_H_
#define G3_H_

#include <stdint.h>

#if defined(__GNUC__)
#define G3_API __attribute__((visibility("default")))
#else
#define G3_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct g3_plan g3_plan; /* opaque; created by g3_plan_create, freed by g3_plan_destroy */

/* Bin specification.  r_ij and r_ik: n_r uniform bins on [0, r_max).
 * r_jk: n_t uniform bins on [0, 2*r_max).  1 <= n_r, n_t <= 1024, and the common lattice of the
 * r and t edges must stay below 2^19 units: 2 n_r n_t / gcd(n_t, 2 n_r) <= 524288 (the exact
 * 128-bit bin volumes need it; n_t = n_r and n_t = 2 n_r always qualify, two coprime counts
 * near 1024 do not: g3_plan_create then returns G3_EINVAL). */
typedef struct {
    int32_t n_r;
    int32_t n_t;
} g3_bins;

typedef enum {
    G3_OK = 0,
    G3_EINVAL = 1,    /* bad argument (see each function)                                   */
    G3_ENOMEM = 2,    /* host or device allocation failed                                   */
    G3_ECUDA = 3,     /* a CUDA runtime call failed, or no sm_100 device is present         */
    G3_ECAPACITY = 4, /* a central particle had more neighbours than the plan can hold      */
    G3_ESTATE = 5,    /* call not valid in the plan's current state                         */
    G3_EINTERNAL = 6, /* an internal invariant failed (counts outside the histogram tile): a bug   */
    G3_ELIMIT = 7     /* the problem needs more scratch than a no-allocation entry point owns (see
                         g3_msd_static); nothing was computed, the allocating call still serves it */
} g3_status;

/* Options for g3_plan_set_option (all optional; defaults are chosen for the B200). */
typedef enum {
    G3_OPT_BATCH_FRAMES = 1, /* frames staged before one batched launch sequence (>= 1); default:
                                max(16, 2^22 / n) capped at 256, and so that the neighbour lists of
                                a batch take at most 16 GiB and at most a quarter of the device
                                memory free when the first frame arrives.  Whether chosen or
                                default, the batch is halved until the plan's buffers can be
                                allocated: it changes no result (G3_INFO_BATCH_FRAMES = the value
                                in use)                                                         */
    G3_OPT_KERNEL = 2,       /* 0 = auto, 1 = generic exact kernel, 2 = tiled fast kernel    */
    G3_OPT_MAX_NEIGHBOURS = 3, /* per-centre neighbour capacity (0 = derive from density)    */
    G3_OPT_TRIPLET_WARPS = 5, /* warps per triplet-kernel CTA: 0 = auto, or 8, 12, .. 24  */
    G3_OPT_QTET_BINS = 6,    /* > 0: also histogram the tetrahedral order parameter q_tet (Eq. 1,
                                PAPER.md:201) of every atom into this many bins on [-3, 1] while
                                frames are accumulated; 0 (default) = off; needs n >= 5      */
    G3_OPT_G2_WIDE = 7,      /* 1 = the pair histogram g2 also covers [r_max, 2 r_max), the rest of the
                                r_jk axis of g(3), in n_r more shells of the same width (a second
                                pair search per frame over eight times the volume: it about
                                DOUBLES the time of a step, +26 ms on the 27.5 ms of config 4);
                                0 (default) = the neighbour range only                        */
    G3_OPT_TIMING = 4         /* 1 = bracket the neighbour and triplet kernels with CUDA events
                                 on the caller's stream (read back with g3_plan_get_info)     */
} g3_option;

/* Keys for g3_plan_get_info. */
typedef enum {
    G3_INFO_KERNEL_LAUNCHES = 1, /* kernels launched since creation / g3_plan_clear_timing    */
    G3_INFO_BATCH_FRAMES = 2,
    G3_INFO_KERNEL = 3,          /* kernel actually selected (1 or 2)                        */
    G3_INFO_CELLS_PER_EDGE = 4,
    G3_INFO_MAX_NEIGHBOURS = 5,
    G3_INFO_TILE_BINS = 6,       /* histogram bins privatised in shared memory per CTA       */
    G3_INFO_SM_COUNT = 7,
    G3_INFO_FRAMES_PENDING = 8,  /* staged frames not yet reduced into the histogram         */
    /* G3_OPT_TIMING = 1 only.  Reading any of the three waits for the recorded events; the
     * sums cover the launches since creation or the last g3_plan_clear_timing.             */
    G3_INFO_TRIPLET_NS = 9,      /* device time of the triplet kernel launches, nanoseconds  */
    G3_INFO_NEIGHBOUR_NS = 10,   /* device time of the neighbour kernel launches             */
    G3_INFO_TIMED_LAUNCHES = 11, /* launches of EACH of the two kernels covered by the sums
                                    (a triplet "launch" = all slab passes of one batch)      */
    G3_INFO_SLABS = 12,          /* tiled kernel: slab passes per batch (1 = the reachable bins
                                    fit one shared-memory tile; G3_INFO_TILE_BINS counts all
                                    reachable slots, over all slabs)                          */
    G3_INFO_G2_SHELLS = 13       /* shells g3_finalize_g2 writes: n_r, or 2 n_r with G3_OPT_G2_WIDE */
} g3_info;

/* Create a plan for frames of `n` particles in a cubic periodic box of edge `box`
 * (positions + box lengths; cubic because the paper's cut-offs
 * are fractions of one "Boxlength").
 *   n      >= 3
 *   box    > 0, same length unit as the positions
 *   r_max  cut-off on r_ij and r_ik (replaces the paper's Boxlength/4,
 *          PAPER.md:407); 0 < r_max < box/2 so that the minimum image is unique
 *   bins   see g3_bins
 * On success *out holds the plan and its histogram is zero.  Uses the CUDA device
 * current at the time of the call for the whole life of the plan.
 * Errors: G3_EINVAL (null out, bad n/box/r_max/bins), G3_ENOMEM, G3_ECUDA.          */
G3_API int g3_plan_create(g3_plan **out, int64_t n, double box, double r_max, g3_bins bins);

/* Tune a plan before the first frame.  G3_ESTATE after frames were accumulated
 * (until g3_plan_reset), G3_EINVAL for unknown keys or bad values.                  */
G3_API int g3_plan_set_option(g3_plan *p, int32_t option, int64_t value);
G3_API int g3_plan_get_info(const g3_plan *p, int32_t key, int64_t *value);

/* Forget the kernel times and the launch counter gathered so far (histogram untouched).  */
G3_API int g3_plan_clear_timing(g3_plan *p);

/* Add one frame (Algorithm 6/7's loop body).
 *   d_pos  device, fp64, [n][3] row-major (x,y,z of particle 0, then particle 1, ...).
 *          Any finite coordinate is accepted: it is snapped to the box/2^20 grid and
 *          wrapped into the box.  NaN, infinities and |x| >= 2^42 box lengths have no grid
 *          point: they set a sticky error that g3_finalize reports as G3_EINVAL.
 * Asynchronous and stream-ordered: never synchronises the host.  d_pos is fully
 * consumed by work enqueued during this call (it is quantised into plan-owned
 * staging), so it may be reused as soon as `stream` has passed this call.  The
 * triplet work itself may be deferred until G3_OPT_BATCH_FRAMES frames are staged
 * or g3_finalize is called; results are identical either way.
 * Errors: G3_EINVAL (null), G3_ECUDA.                                               */
G3_API int g3_accumulate_frame(g3_plan *p, const double *d_pos, void *stream);

/* Same as calling g3_accumulate_frame for f = 0..n_frames-1 on d_pos + f*frame_stride
 * (frame_stride in doubles, >= 3*n), with one batched launch sequence.              */
G3_API int g3_accumulate_frames(g3_plan *p, const double *d_pos, int64_t n_frames, int64_t frame_stride,
                         void *stream);

/* Same, from HOST memory (pinned memory gives asynchronous copies; pageable works).
 * Copies are issued on `stream` in chunks that overlap with compute.  h_pos must
 * stay valid until `stream` has passed this call.                                   */
G3_API int g3_accumulate_frames_host(g3_plan *p, const double *h_pos, int64_t n_frames,
                              int64_t frame_stride, void *stream);

/* Reduce all staged frames, then write the results and SYNCHRONISE `stream`.
 *   d_counts  device, uint64 [n_r][n_r][n_t], c (r_jk bin) fastest; may be NULL
 *   d_g3      device, fp64, same shape: counts / (frames n rho^2 V_abc); may be NULL
 *   h_stats   host, uint64[3] = { frames, sum_i k_i (k_i - 1), overflow }; may be NULL
 * Does not reset the plan: more frames may follow, and it may be called again.
 * Errors: G3_ECAPACITY if any centre exceeded the neighbour capacity (counts are
 * then incomplete), G3_EINVAL if a non-finite coordinate was accumulated since the last
 * reset (results meaningless), G3_EINTERNAL, G3_ECUDA.                              */
G3_API int g3_finalize(g3_plan *p, uint64_t *d_counts, double *d_g3, uint64_t *h_stats, void *stream);

/* Same with HOST output buffers (device-to-host copies included).                   */
G3_API int g3_finalize_host(g3_plan *p, uint64_t *h_counts, double *h_g3, uint64_t *h_stats, void *stream);

/* g2, the pair distribution function (Algorithm 6 "g2 histogram"; Algorithm 7
 * CUDA_g2; reading G1).  By default over the neighbour range
 * [0, r_max) with the n_r shells of r_ij, counted in the same neighbour pass; with
 * G3_OPT_G2_WIDE over [0, 2 r_max), the whole r_jk axis of g(3) (the Kirkwood denominator
 * g2 g2 g2), in S = 2 n_r shells of the same width (S = G3_INFO_G2_SHELLS).  Minimum-image
 * distances: shells beyond box/2 (possible only when r_max > box/4) are geometrically incomplete.
 * Reduces all staged frames like g3_finalize, then, asynchronously on `stream`:
 *   d_counts2  device, uint64 [S]: ordered pairs (i, j), j != i, per shell; may be NULL
 *   d_g2       device, fp64 [S]: counts2 / (frames n rho V_a), V_a = 4 pi/3 (r_{a+1}^3 - r_a^3),
 *              rho = n / box^3 (ideal gas -> (n-1)/n); may be NULL
 * Does not synchronise and does not reset.  sum(counts2[0 .. n_r)) = sum_i k_i.       */
G3_API int g3_finalize_g2(g3_plan *p, uint64_t *d_counts2, double *d_g2, void *stream);

/* q_tet, the tetrahedral order parameter (Eq. 1; Algorithms 2-3),
 * histogrammed on the same cell list when G3_OPT_QTET_BINS > 0 (readings T1-T4: four
 * nearest neighbours by (d^2, dx, dy, dz); fp64 in a fixed operation order; bins of width
 * 4/n_q on [-3, 1], q = 1 in the last bin; atoms with a coincident neighbour are skipped).
 * Reduces all staged frames, then copies the histogram and SYNCHRONISES `stream`.
 *   d_hist   device, uint64 [n_q]; may be NULL
 *   h_stats  host, uint64[2] = { atoms binned, atoms skipped }; may be NULL
 * Errors: G3_ESTATE if the option is off; G3_EINVAL if a non-finite coordinate was accumulated
 * since the last reset; G3_ECAPACITY if a centre exceeded the neighbour capacity on the tiled path
 * (kernel 2), where q_tet is read off the same capacity-limited neighbour lists: the four nearest
 * of such a centre may be missing and the histogram is not to be used (raise
 * G3_OPT_MAX_NEIGHBOURS).  Plans served by the generic kernel scan the cells for q_tet and do not
 * depend on the capacity.                                                                   */
G3_API int g3_finalize_qtet(g3_plan *p, uint64_t *d_hist, uint64_t *h_stats, void *stream);

/* Normalise externally merged counts (e.g. the sum over ranks of a frame-sharded
 * run; the paper's "split the trajectory, merge the results"):
 * d_g3 = d_counts / (frames n rho^2 V_abc).  Asynchronous on `stream`.              */
G3_API int g3_normalize(g3_plan *p, const uint64_t *d_counts, uint64_t frames, double *d_g3, void *stream);

/* Copy the plan's bin-volume table V_abc (fp64 [n_r][n_r][n_t], units of box^6
 * length) to host memory.                                                           */
G3_API int g3_bin_volumes(const g3_plan *p, double *h_volumes);

/* Mean square displacement over all time origins (Eq. 5; Algorithms 10-11,
 * PAPER.md:642-702) of an UNWRAPPED trajectory; no plan is needed.  DESIGN.md readings M1-M3:
 * positions are snapped to the box/2^20 grid without wrapping (|x| < 1024 box lengths), so
 *   S[dt] = sum_i sum_{t=0}^{F-dt-1} |m_i(t+dt) - m_i(t)|^2,  dt = 0 .. max_lag <= F - 1,
 * is an exact 128-bit integer, and msd[dt] = S[dt] (box/2^20)^2 / (n (F - dt)).
 *   d_pos    device, fp64 [n_frames][n][3], frame f at d_pos + f * frame_stride (>= 3 n doubles)
 *   d_sums   device, uint64 [max_lag + 1][2] = (low, high) words of S; may be NULL
 *   d_msd    device, fp64 [max_lag + 1], in the length unit of `box` squared; may be NULL
 * Stream-ordered work, then SYNCHRONISES `stream` (scratch comes from the stream's memory pool).
 * Errors: G3_EINVAL (arguments, or a coordinate outside the grid range: outputs are then
 * meaningless), G3_ENOMEM, G3_ECUDA.                                                       */
G3_API int g3_msd(const double *d_pos, int64_t n_frames, int64_t n, int64_t frame_stride, double box,
                  int64_t max_lag, uint64_t *d_sums, double *d_msd, void *stream);

/* g3_msd for callers that must not allocate device memory: same arguments, same outputs (the
 * sums are the same exact integers, bit for bit), but NO cudaMalloc / cudaMallocAsync / cudaFree or
 * any other allocating routine is called, on any call.
 *
 * Who needs it.  g3_msd takes its scratch (one 128-bit partial sum per (block of 32 atoms, lag) and
 * an error counter) from the stream's memory pool on every call.  That is a driver allocation
 * outside whatever allocator the host program runs, and some host programs cannot afford one:
 *   - an MD engine or a PyTorch job that analyses in situ and has already handed (nearly) all of
 *     HBM to its own pool or caching allocator: the driver then has nothing left to give, and
 *     g3_msd fails with G3_ENOMEM although the program itself still shows plenty of free memory;
 *   - a job that runs under a fixed per-process memory limit (MPS partition, batch-system quota)
 *     sized from its start-up footprint, where any later growth is a hard failure;
 *   - an analysis step between time steps that must cost the same on every call: a pool that has
 *     to grow goes to the driver for memory, which is slow and is one more thing that can fail.
 * Such callers pre-allocate d_pos / d_sums / d_msd themselves, once, and call this function.
 *
 * How.  The scratch is a fixed array compiled into libg3 (device memory with static storage:
 * G3_MSD_STATIC_SCRATCH_BYTES, about 8 MiB).  Every GPU on which libg3's kernels get loaded
 * holds that array from then until the process exits, whether or not this function is used.
 *
 * Limits (G3_ELIMIT beyond them, before any device work; g3_msd has neither limit):
 *   - ceil(n / 32) * (max_lag + 1) <= G3_MSD_STATIC_MAX_PARTIALS (the config-4 shape, n = 32768
 *     with 500 lags, fits: 512000);
 *   - the trajectories of 32 atoms must fit the shared memory of one SM: 400 n_frames + 16 bytes
 *     <= the device's opt-in limit (n_frames <= 580 on a B200).  Longer runs need the snapped
 *     global copy of g3_msd, which is far too large for a built-in array.
 *
 * First call on each device: looks up the device address of the built-in array, with that device
 * current, and caches it per device (thread-safe).  This may load libg3's kernels onto the GPU,
 * which is where the driver places the array.  Make this first call early, during set-up, and
 * before any stream capture is started.  Later calls on that device touch no set-up code.
 *
 * Sharing.  All calls in the process, from all threads and streams, use the ONE array of their
 * device, and it keeps whatever the previous call left in it.  Each call clears the error counter
 * itself and overwrites every partial sum before reading it, so calls that follow each other
 * are independent; two calls whose GPU work overlaps in time (different streams, or threads that
 * do not order their calls) race on the array and give wrong sums without any error.  The
 * caller serialises them.  g3_msd is not affected: it never touches the array.
 *
 * Stream-ordered work, then SYNCHRONISES `stream`, like g3_msd.
 * Errors: G3_EINVAL and G3_ECUDA as g3_msd; G3_ELIMIT (see above).                              */
#define G3_MSD_STATIC_MAX_PARTIALS 524288
#define G3_MSD_STATIC_SCRATCH_BYTES (256 + 16 * G3_MSD_STATIC_MAX_PARTIALS)
G3_API int g3_msd_static(const double *d_pos, int64_t n_frames, int64_t n, int64_t frame_stride, double box,
                         int64_t max_lag, uint64_t *d_sums, double *d_msd, void *stream);

/* Zero the histogram, frame count and error state; keep all buffers.                */
G3_API int g3_plan_reset(g3_plan *p, void *stream);

/* Free the plan (NULL is allowed).  Synchronises the device.                        */
G3_API void g3_plan_destroy(g3_plan *p);

/* Static description of a status code.                                              */
G3_API const char *g3_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* G3_H_ */
