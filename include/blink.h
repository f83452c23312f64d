/*
 * blink.h -- C ABI of libblink: the data-parallel hot path of the BLINK high-time-resolution
 * imager (arxiv 2405.13478; citations are /root/reference/PAPER.md line numbers), hand-written
 * for NVIDIA B200 (sm_100a).
 *
 *   for every (time step t, channel ch) snapshot:
 *     grid the complex visibilities of all baselines on an N x N uv grid (nearest cell, V and its
 *     Hermitian conjugate, per-cell weight count)            PAPER.md:348-370 (sec 5.2.1), :211
 *     -> natural / uniform weighting                           PAPER.md:209-213 (sec 4.4.2), :360
 *     -> 2-D inverse DFT, fftshift, normalise, real part       PAPER.md:160-176 (Eq. 4-6), :372-376
 *
 * Conventions
 *   - plain C linkage, no exceptions cross the boundary, no torch / C++ types in signatures;
 *   - every pointer argument says HOST or DEVICE; device pointers are raw CUDA device addresses
 *     on the current device; `stream` is a cudaStream_t passed as void* (NULL = legacy default);
 *   - all functions return 0 (BLINK_OK) or a negative blink_status; on error outputs are
 *     untouched unless stated;
 *   - complex64 = interleaved float (re, im) pairs, i.e. float2 / cufftComplex layout
 *     ("gpufftComplex");
 *   - there is NO CPU fallback: without a CUDA device every call except blink_version,
 *     blink_strerror returns BLINK_ECUDA.
 *
 * Baseline order (cross-correlations only):
 *   bl(i,j) = i (2 n_ant - i - 1) / 2 + (j - i - 1)  for 0 <= i < j < n_ant,  b_ij = r_j - r_i.
 *
 * Cell rule (bit-exact, identical to the oracle; DESIGN.md "Readings" c5-c7):
 *   sc = freq_hz / 299792458.0;  u = (E_j - E_i) * sc;  v = (N_j - N_i) * sc   (fp64, no FMA)
 *   G  = (double)n_pix * pixscale            (= 1/du, Eq. 9)
 *   kx = llround(u * G), ky = llround(v * G) (nearest, ties away from zero)
 *   kept iff |kx| <= N/2-1 and |ky| <= N/2-1, else the baseline AND its conjugate are dropped
 *   cell = (ky mod N) * N + (kx mod N)       (FFT-native order, DC at [0][0])
 *   conjugate cell = ((-ky) mod N) * N + ((-kx) mod N)
 */
#ifndef BLINK_H_
#define BLINK_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BLINK_VERSION 210 /* 0.2.1: + blink_image_static, BLINK_ECAPACITY, BLINK_Q_FUSED_NZ / _D; test hooks in libblink_testing.so */

typedef enum blink_status {
  BLINK_OK = 0,
  BLINK_EINVAL = -1, /* bad argument (NULL, odd / unsupported n_pix, n_ant < 2, ...) */
  BLINK_ENOMEM = -2, /* host or device allocation failed */
  BLINK_ECUDA = -3,  /* CUDA runtime error or no device (see blink_last_cuda_error) */
  BLINK_EUNSUPPORTED = -4, /* valid request outside what this build implements */
  BLINK_ERESERVE = -5, /* the plan's device scratch is too small for this n_t: call blink_plan_reserve(plan, n_t)
                          first (hot calls never allocate) */
  BLINK_ECAPACITY = -6 /* the request does not fit the fixed, built-in scratch of blink_image_static
                          (BLINK_STATIC_SCRATCH_BYTES); nothing was launched */
} blink_status;

typedef enum blink_weighting {
  BLINK_NATURAL = 0, /* plain sum per cell; image norm = sum of counts */
  BLINK_UNIFORM = 1  /* cell sum / cell count; image norm = occupied cells */
} blink_weighting;

/* `what` selectors of blink_plan_query.  [ch] forms take the channel in the low 16 bits of
 * `index`.  Device-pointer queries return pointers that stay valid until blink_plan_destroy. */
typedef enum blink_query {
  BLINK_Q_N_ANT = 0,      /* out: int32                                            */
  BLINK_Q_N_BL = 1,       /* out: int32   n_ant (n_ant-1)/2                        */
  BLINK_Q_N_CH = 2,       /* out: int32                                            */
  BLINK_Q_N_PIX = 3,      /* out: int32                                            */
  BLINK_Q_N_DROPPED = 4,  /* out: int64   [ch] baselines outside the grid          */
  BLINK_Q_WSUM = 5,       /* out: int64   [ch] sum of counts = 2 (n_bl - n_dropped) */
  BLINK_Q_N_OCC = 6,      /* out: int64   [ch] number of cells with count > 0      */
  BLINK_Q_BBOX = 7,       /* out: int32[2] [ch] kx_max, ky_max over kept baselines */
  BLINK_Q_NORM = 8,       /* out: double  [ch] image normalisation (WSUM or N_OCC) */
  BLINK_Q_CELL_IDX = 9,   /* out: const int32* DEVICE [n_ch][n_bl], cell of V, -1 = dropped */
  BLINK_Q_COUNTS = 10,    /* out: const uint32* DEVICE [n_ch][N][N] weight counts  */
  BLINK_Q_IMAGE_PATH = 11,/* out: int32   0 = shared-memory single pass, 1 = two-pass */
  BLINK_Q_SCRATCH_BYTES = 12, /* out: int64 device scratch currently held by the plan */
  BLINK_Q_IMAGE_CHUNK = 13, /* out: int32  snapshots per launch pair of the two-pass imaging path */
  BLINK_Q_FUSED_PATH = 14,  /* out: int32  route of blink_grid_image: 1 = shared memory, 2 = warp-per-transform, 0 = two kernels */
  BLINK_Q_FUSED_CHUNK = 15, /* out: int32  snapshots per chunk of the two-kernel route */
  BLINK_Q_CORR = 16,        /* out: const float2* DEVICE [n_ch][n_bl] correction factors (NULL until set) */
  BLINK_Q_CORR_FUSED = 17,  /* out: int32  1 = blink_grid / blink_grid_image apply the factors at load */
  BLINK_Q_TENSOR_ROUTE = 18,/* out: int32  1 = the shared-memory route runs its transforms on the tensor cores (k_fused_tc) */
  BLINK_Q_WARP_KERNEL = 19, /* out: int32  kernel behind BLINK_Q_FUSED_PATH 2: 2 = residue-class kernel (intermediate in shared
                               memory, k_img1024r), 1 = ring kernel (intermediate in an L2-sized ring, k_img1024), 3 = BLINK_Q_FUSED_PATH is 0
                               and the column pass of the two kernels is the residue-class kernel k_cols_res (N = 2048 / 4096,
                               sparse half-plane), 0 = none of these */
  BLINK_Q_FUSED_NZ = 20,    /* out: int32  which k_fused instance BLINK_Q_FUSED_PATH 1 runs in the plan's current state: its
                               first transform stage reads NZ of the 8 N/16-cell blocks on either side of DC (2, 3, 4 or 8;
                               8 = unpruned); 0 = not on that route, or on its tensor-core form.  For harnesses that must
                               know which compiled instance they exercised */
  BLINK_Q_FUSED_D = 21      /* out: int32  that route's polyphase factor: the image is D x D interleaved sub-images of
                               N / D (1, 2 or 4); 0 = not on that route */
} blink_query;

typedef struct blink_plan blink_plan; /* opaque */

/*
 * Optional arguments of blink_plan_create_opts.  Zero-initialise, set struct_size = sizeof(blink_options)
 * and change what is needed; every field's 0 means "let the plan decide".  The route fields exist so
 * that a harness can compare the library's alternative routes against each other and the oracle; the
 * library reads no environment variable.
 */
typedef struct blink_options {
  int32_t struct_size;        /* sizeof(blink_options) of the caller's header */
  int32_t fused_route;        /* blink_grid_image shared-memory route (BLINK_Q_FUSED_PATH 1): 0 auto, -1 never */
  int32_t polyphase;          /* its polyphase form for N = 512 / 1024: 0 auto, -1 never */
  int32_t warp_route;         /* warp-per-transform route at N = 1024 (BLINK_Q_FUSED_PATH 2): 0 auto, -1 never, 2 = its ring kernel */
  int32_t warp_ring;          /* snapshots of intermediate U kept in flight by that route: 0 auto (32 MB), else >= 2 */
  int32_t grid_ring;          /* blink_grid ring route: 0 auto, -1 never */
  int32_t grid_ring_min_snap; /* fewest snapshots per call that take it: 0 auto (one per SM), else >= 1 */
  int32_t image_chunk_mb;     /* scratch budget (MiB) of the two-kernel imaging routes: 0 auto (2048) */
  int32_t tune[8];            /* implementation tuning knobs, meaning private to this version (csrc/blink_internal.h) */
} blink_options;

int blink_version(void);
const char *blink_strerror(int status);
/* text of the last CUDA error seen by this thread's last failing call ("" if none) */
const char *blink_last_cuda_error(void);

/*
 * blink_plan_create -- step a0: uv-index precompute (the paper recomputes
 * frequency and wavelength per thread per launch; here the fixed array geometry
 * is exploited once).  Runs the fp64 index kernel on the device, builds the per-channel count grid
 * (PAPER.md:354), normalisation constants, bounding box and the cell-sorted gather tables used
 * by blink_grid.
 *   out         HOST  receives the plan; untouched on error
 *   ant_enu_m   HOST  [n_ant][3] East, North, Up in metres (Up ignored: coplanar)
 *   freq_hz     HOST  [n_ch] channel centre frequencies in Hz
 *   n_pix       grid = image side N; power of two, 32 <= N <= 4096 in this build
 *   pixscale    pixel size dx in direction-cosine units (all-sky: 2.0 / n_pix; small field:
 *               radians per pixel); du = 1 / (n_pix * pixscale), Eq. 9
 *   weighting   blink_weighting
 *   stream      cudaStream_t for the plan-time kernels / copies; the call synchronises it
 * Inputs are copied; the caller may free them on return.  The plan owns its device tables.
 */
int blink_plan_create(blink_plan **out, const double *ant_enu_m, int n_ant, const double *freq_hz,
                      int n_ch, int n_pix, double pixscale, int weighting, void *stream);

/* same, with options (NULL = defaults = blink_plan_create); BLINK_EINVAL on an unknown struct_size or value */
int blink_plan_create_opts(blink_plan **out, const double *ant_enu_m, int n_ant, const double *freq_hz,
                           int n_ch, int n_pix, double pixscale, int weighting, void *stream,
                           const blink_options *opts);

/*
 * Threads, streams, devices.  A plan belongs to the device that was current at blink_plan_create; every
 * call that takes it returns BLINK_EINVAL when another device is current.  Calls that use plan-owned
 * scratch (blink_image always; blink_grid_image when BLINK_Q_FUSED_PATH != 1) must not overlap in time
 * with each other on the same plan: issue them on one stream, or order the streams.  blink_grid,
 * blink_correct, blink_dynspec and blink_grid_image on the shared-memory route (BLINK_Q_FUSED_PATH == 1)
 * use no plan scratch and may run concurrently.  Plan-mutating calls (blink_plan_reserve,
 * blink_plan_set_corrections, blink_plan_refresh, blink_plan_destroy) must not run concurrently with
 * anything else on the same plan.
 */

/*
 * blink_plan_refresh -- step a0 again, for new antenna coordinates: the periodic plan refresh that
 * time-dependent (u,v) need (a tracking array's projected baselines move
 * with hour angle).  Same n_ant, frequencies, grid, weighting and options as at
 * creation; runs the fp64 index kernel on the device and rebuilds every table (host cores, one channel
 * per thread), then swaps them in, so afterwards the plan is indistinguishable from a new plan of the new
 * coordinates (bit-exact indices, counts and images), with scratch for the n_t reserved before and the
 * host staging kept.
 *   ant_enu_m  HOST [n_ant][3], the coordinates whose differences are the new baselines
 * Synchronises the device (work queued on the old tables finishes first).  Allocates: the new tables and
 * the new scratch exist beside the old ones until the swap.  On error (BLINK_ENOMEM included) the plan is
 * unchanged: nothing is swapped in unless everything, scratch included, could be built.
 * Corrections: the factor table depends on the geometry and is dropped.  If the plan was applying it at
 * load (blink_plan_apply_corrections on), blink_grid / blink_grid_image / blink_grid_image_host return
 * BLINK_EINVAL after the refresh -- they do not quietly grid uncorrected data -- until the caller calls
 * blink_plan_set_corrections + blink_plan_apply_corrections(plan, 1) again, or
 * blink_plan_apply_corrections(plan, 0) to say that uncorrected is what it wants.
 * Cost and cadence: the table packing runs on the host cores, about 0.13 s for the 256-antenna, 32-channel
 * station plan (0.17 s to create it) -- meant for a refresh every few seconds of data or slower (a tracking
 * array's cells move by a fraction of a cell per second), not once per batch: a 100-step station batch
 * images in 0.4 ms.
 */
int blink_plan_refresh(blink_plan *plan, const double *ant_enu_m, void *stream);

/* frees the plan and its device memory; NULL is a no-op */
int blink_plan_destroy(blink_plan *plan);

/* read-only view of plan facts; `out` HOST, sized per blink_query */
int blink_plan_query(const blink_plan *plan, int what, int index, void *out);

/*
 * blink_grid -- steps a1/a2: gridding.  For each snapshot s = t*n_ch + ch:
 *   uv_grid[s][cell(bl)] += vis[s][bl];  uv_grid[s][cell*(bl)] += conj(vis[s][bl])
 * over all kept baselines, every other cell = 0.  Unweighted sums regardless of the plan's
 * weighting.  The per-cell summation order is fixed by the plan (ascending baseline index; the
 * bulk-copy route adds them in pieces of up to four), so the result is bit-reproducible run to run for
 * the same plan, batch size and alignment -- the deterministic reduction the paper plans
 * (PAPER.md:370, :396).
 *   vis      DEVICE complex64 [n_t][n_ch][n_bl], baseline fastest; 8-byte aligned (a 16-byte aligned
 *            base lets the call take its bulk-copy route)
 *   uv_grid  DEVICE complex64 [n_t][n_ch][N][N] row-major [ky][kx], FFT-native order (DC at
 *            [0][0]); COMPLETELY overwritten, zeros included (no memset needed); 16-byte aligned
 *   n_t      number of time steps in this call (any >= 0; 0 is a no-op)
 * Asynchronous on `stream`; no allocation, no host synchronisation.  Caller owns both buffers.
 */
int blink_grid(const blink_plan *plan, const void *vis, int n_t, void *uv_grid, void *stream);

/*
 * blink_image -- steps a3-a5:
 *   G'  = uv_grid (natural) or uv_grid / count where count > 0 (uniform)
 *   img[s][y][x] = Re sum_{ky,kx} G'[ky][kx] exp(+2 pi i (kx (x-N/2) + ky (y-N/2)) / N) / norm[ch]
 * i.e. unnormalised inverse DFT, fftshift so pixel (N/2, N/2) is the phase centre
 * (l = (x-N/2) dx East, m = (y-N/2) dx North), 1/norm, real part.
 *   uv_grid  DEVICE complex64 [n_t][n_ch][N][N], const (never used as scratch).  CONTRACT: it is a
 *            grid OF THIS PLAN -- zero in every cell whose weight count (BLINK_Q_COUNTS) is zero and
 *            Hermitian, G[-k] = conj(G[k]); true of every blink_grid output.  A route may rely on
 *            either fact: the line kernels read the whole bounding box (BLINK_Q_BBOX) and form the
 *            real part exactly, i.e. symmetrise a non-Hermitian grid, (G[k] + conj(G[-k])) / 2; the
 *            warp-per-transform route (N = 1024, wide sparse half-planes: BLINK_Q_FUSED_PATH == 2)
 *            reads only the occupied cells with kx >= 0.  Cells outside the box are never read.
 *   images   DEVICE float32 [n_t][n_ch][N][N] row-major [y][x]; completely overwritten
 * Asynchronous on `stream`; no allocation, no host synchronisation: the intermediate of the two passes
 * lives in plan-owned scratch that blink_plan_reserve(plan, n_t) must have sized for this n_t (or a
 * larger one) beforehand, else BLINK_ERESERVE.
 */
int blink_image(const blink_plan *plan, const void *uv_grid, int n_t, void *images, void *stream);

/*
 * blink_image_static -- blink_image for callers that are not allowed to allocate device memory.
 *
 * Who that is.  blink_image keeps the intermediate U of its two passes in plan scratch, and that scratch
 * only exists after blink_plan_reserve, which calls cudaMalloc (and, when it has to grow, synchronises the
 * whole device and calls cudaFree).  Some users of an imager like this one cannot make that call at the
 * point where they need images: a real-time ingest loop behind a correlator, where a device-wide stall
 * from the allocator means dropped telescope data; a process that shares the GPU with a component (a
 * correlator ring buffer, a framework's caching pool) which has already claimed the memory, so a later
 * cudaMalloc may simply fail; code that runs under a "no driver allocation after start-up" rule.  For them
 * this call images with an intermediate that was never allocated at run time: it lives in an array
 * compiled into the library, BLINK_STATIC_SCRATCH_BYTES (32 MiB) of device memory that every GPU which
 * loads libblink's imaging module holds until the process exits, whether or not this call is ever used.
 *
 * What it computes.  Exactly blink_image: same arguments, same layouts, same input contract on uv_grid,
 * same arithmetic -- the two line kernels of blink_image (column pass, row pass) pointed at the built-in
 * array instead of plan scratch, whatever route the plan would pick for blink_image itself.  For a plan
 * whose blink_image runs the line kernels the images are bit-identical; for the other routes (N = 1024
 * residue-class / ring kernels, N >= 2048 residue-class column pass) they agree to fp32 rounding order
 * and both meet the oracle bar (1e-4 of the image peak).  The batch is cut into launch pairs of
 * floor(BLINK_STATIC_SCRATCH_BYTES / (8 N wu)) snapshots, wu = the plan's half-plane width (kx_max over
 * all channels + 1, rounded up to 16), so any n_t is accepted.
 *
 * The limit.  One snapshot's U (8 N wu bytes) must fit the array, else BLINK_ECAPACITY and nothing is
 * launched; blink_last_cuda_error() then holds a sentence with both numbers.  Every plan with N <= 2048
 * fits; at N = 4096 the half-plane may be at most 1024 columns wide (true of the MWA-shaped workloads).
 *
 * No allocation of any kind: no cudaMalloc / cudaFree / cudaMallocAsync, no host allocation, no library
 * call that allocates.  The plan (an input, created at start-up) needs no blink_plan_reserve for it.
 *
 * First call on a device.  It looks up the array's device address (cudaGetSymbolAddress, with that device
 * current -- the array's name is not a device pointer in host code) and raises the kernels' shared-memory
 * limit; both are remembered per device.  Make that first call during set-up, and before any stream
 * capture is begun; later calls only launch.
 *
 * Sharing.  There is ONE array per device, shared by every plan, thread and stream of the process, and it
 * keeps whatever the last call left in it.  Nothing in it has to start at zero (the column pass writes
 * every element of a chunk's U before the row pass reads it), so stale contents are harmless -- but two
 * blink_image_static calls that overlap in time on the same GPU (different streams, or different threads
 * on different streams) overwrite each other's intermediate and both results are garbage: issue all of
 * them on one stream, or order the streams yourself.  blink_image and the other calls never touch the
 * array and may overlap with it.
 *
 * Asynchronous on `stream`; no host synchronisation.  Errors as blink_image, plus BLINK_ECAPACITY.
 */
#define BLINK_STATIC_SCRATCH_BYTES (32u << 20)
int blink_image_static(const blink_plan *plan, const void *uv_grid, int n_t, void *images, void *stream);

/*
 * blink_plan_set_corrections -- the pre-gridding corrections of PAPER.md section 4.2 (:142-156):
 * (i) cable-length phase, (ii) calibration in phase and amplitude, (iii) geometric phase rotation of
 * the phase centre.  "In the presented software, most of these corrections are already implemented
 * as GPU kernels and are executed post-correlation"; the paper gives no formulas, the
 * readings are DESIGN.md c18-c20:
 *   antenna model   measured V_ij = a_i conj(a_j) V_ij(true),  a_i(nu) = g_i(nu) exp(-2 pi i nu L_i / c)
 *   correction      F[ch][bl(i,j)] = exp(+2 pi i (u l0 + v m0 + w (n0 - 1))) / (a_i conj(a_j)),
 *                   (u, v, w) = (r_j - r_i) nu / c un-snapped, n0 = sqrt(1 - l0^2 - m0^2)
 * A device kernel builds F once (fp64, stored complex64); geometry, gains, cables and pointing are
 * fixed across the snapshots of a plan, like the uv indices.
 *   gains        HOST double [n_ch][n_ant][2] (re, im) calibration solutions g_i, or NULL (all 1);
 *                every |g_i| must be > 0 and finite
 *   cable_len_m  HOST double [n_ant] electrical lengths L_i in metres, or NULL (all 0)
 *   l0, m0       direction cosines of the new phase centre, l0^2 + m0^2 < 1; (0, 0) = none
 * Copies its inputs; synchronises `stream`; replaces any earlier table.  BLINK_EINVAL on bad values.
 */
int blink_plan_set_corrections(blink_plan *plan, const double *gains, const double *cable_len_m,
                               double l0, double m0, void *stream);

/*
 * blink_plan_apply_corrections -- the corrections fused into the gridder's load (SURVEY.md section 8(f)
 * item f2).  on = 1: from now on blink_grid and blink_grid_image (and blink_grid_image_host) multiply
 * every visibility by the plan's factor F[ch][bl] as they read it, i.e. they grid blink_correct's output
 * without that pass existing: no extra kernel, and no extra HBM traffic beyond the 8-byte factors per
 * (channel, baseline), which are shared by all time steps and stay in L2.  on = 0 (the default): the
 * visibilities are gridded as given.  Needs a table (BLINK_EINVAL before blink_plan_set_corrections); a
 * later blink_plan_set_corrections replaces the factors and leaves the switch as it is.  The first call
 * with on = 1 builds the shared-memory table layouts that carry the factors (host work, synchronises
 * `stream`); BLINK_Q_FUSED_PATH may change with the switch (a plan whose snapshots fit the SM without
 * the factors but not with them falls back to the next route, which needs blink_plan_reserve).
 */
int blink_plan_apply_corrections(blink_plan *plan, int on, void *stream);

/*
 * blink_correct -- vis_out[t][ch][bl] = vis_in[t][ch][bl] * F[ch][bl] (complex64 product), the
 * table set by blink_plan_set_corrections (BLINK_EINVAL if none is set).
 *   vis_in, vis_out  DEVICE complex64 [n_t][n_ch][n_bl]; may be the same buffer (in place)
 * Asynchronous on `stream`; no allocation.  Algorithmic bytes: 16 per visibility.
 */
int blink_correct(const blink_plan *plan, const void *vis_in, int n_t, void *vis_out, void *stream);

/*
 * blink_dynspec -- the stage right after imaging: subtraction of a running reference image and
 * transposition of the image cube into per-pixel dynamic spectra (the paper
 * prints no formula, readings DESIGN.md c21-c23).  Per channel and pixel, for t = 0 .. n_t-1:
 *     D_t = I_t - R_t;   R_{t+1} = (1 - alpha) R_t + alpha I_t;   dynspec[y][x][ch][t] = D_t
 * alpha = 1: R_t is the preceding dirty image; alpha = 0: a fixed model / prepared image;
 * 0 < alpha < 1: an exponentially weighted average of the previous images.
 *   images     DEVICE float32 [n_t][n_ch][N][N] (a blink_image / blink_grid_image output), const
 *   alpha      in [0, 1] (BLINK_EINVAL otherwise)
 *   ref_state  DEVICE float32 [n_ch][N][N], in/out: R_0 on entry, R_{n_t} on return, so consecutive
 *              batches chain like one long batch; NULL = R_0 is zero and no state is kept
 *   dynspec    DEVICE float32 [N][N][n_ch][n_t], time fastest; completely overwritten; must not
 *              overlap `images`
 * Asynchronous on `stream`; no allocation.  Algorithmic bytes: 8 per voxel (+ 8 per (ch, pixel) of
 * state).  n_t == 0 is a no-op.
 */
int blink_dynspec(const blink_plan *plan, const void *images, int n_t, double alpha, void *ref_state,
                  void *dynspec, void *stream);

/*
 * blink_grid_image -- steps a1-a5 in one call: images straight from visibilities, with no uv grid
 * in HBM at all (the paper's aim of processing "fully inside GPU
 * memory" with minimal I/O).  Same result as blink_grid followed by blink_image
 * up to fp32 rounding order (both meet the oracle bars).  Three internal routes, chosen by the plan:
 *   - shared-memory route (BLINK_Q_FUSED_PATH == 1; small bounding box): one kernel; the gridded
 *     half-plane never leaves the SM.  N <= 256 directly; N = 512 / 1024 with a bounding box inside
 *     |k| < 128 (a compact array on a large image) as 2 x 2 / 4 x 4 interleaved 256^2 sub-images of
 *     the same cell sums (polyphase split of the inverse DFT: each sub-image is the 256^2 transform
 *     of the grid times a unit-modulus factor per cell);
 *   - residue-class route (BLINK_Q_FUSED_PATH == 2; N = 1024 with a wide, sparsely filled half-plane,
 *     e.g. MWA; BLINK_Q_WARP_KERNEL says which kernel): one kernel; the image rows are dealt by y mod 64,
 *     a class's 16 x 512 intermediate lives in shared memory between the warps that form it from the
 *     plan's occupied cells and the warps that run the row transforms -- no scratch.  Planes with more
 *     cells than fit the SM take the ring kernel instead: one cooperative launch, column-pass CTAs feeding
 *     row-pass CTAs through a 32 MB ring of plan-owned scratch that stays in L2;
 *   - two-kernel route (BLINK_Q_FUSED_PATH == 0): the column transforms are fed straight from the
 *     visibilities through the plan's cell-sorted tables (each occupied cell sums its own baselines in
 *     ascending order; at N = 2048 / 4096 with a sparse half-plane at most 1024 columns wide by residue
 *     class as above), the row transforms follow; only the half-plane intermediate U passes through
 *     plan-owned scratch, in chunks of BLINK_Q_FUSED_CHUNK snapshots (up to 2 GB).
 *   vis     DEVICE complex64 [n_t][n_ch][n_bl]; 16-byte aligned base (BLINK_EINVAL otherwise: the routes
 *           read it with bulk asynchronous copies)
 *   images  DEVICE float32   [n_t][n_ch][N][N]
 * Reproducibility: the residue-class and two-kernel routes return the same bits for the same plan and input, call
 * after call.  The shared-memory route does so for the first snapshot each of its persistent CTAs images; later
 * snapshots may differ between two calls in the last bit of the largest pixels (<= 2^-23 of the image peak; known
 * issue).
 * Asynchronous on `stream`; no allocation, no host synchronisation.  The shared-memory route and the
 * residue-class kernel need no scratch; the others need blink_plan_reserve(plan, n_t) beforehand
 * (BLINK_ERESERVE otherwise).
 */
int blink_grid_image(const blink_plan *plan, const void *vis, int n_t, void *images, void *stream);

/*
 * blink_grid_image_host -- blink_grid_image for data in HOST memory: the end-to-end call.  The batch is
 * cut into chunks of `chunk_t` time steps (set by blink_plan_reserve_host); the host-to-device copy of one
 * chunk, the imaging of the previous one and the device-to-host copy of the one before run concurrently on
 * three internal streams over a ring of plan-owned device buffers -- the interleaving of kernels and
 * transfers with pinned host memory that the paper lists as its next optimisation.
 * Results are those of blink_grid_image on the same visibilities (bit-identical on the routes that are
 * bit-reproducible; see the note on reproducibility at blink_grid_image).
 *   vis_host     HOST complex64 [n_t][n_ch][n_bl]; page-locked (cudaHostAlloc / cudaHostRegister) for the
 *                copies to overlap -- pageable memory works, but the copies then serialise with the host
 *   images_host  HOST float32   [n_t][n_ch][N][N]; same
 * Asynchronous: ordered after the work already in `stream`, and `stream` waits for its completion, so
 * the host buffers must stay valid (and images_host unread) until `stream` has been synchronised.  No
 * allocation: BLINK_ERESERVE until blink_plan_reserve_host has run.  Not concurrent with any other call
 * on the same plan.  The transfers bound it: 8 n_bl + 4 N^2 bytes per snapshot over the host link.
 */
int blink_grid_image_host(blink_plan *plan, const void *vis_host, int n_t, void *images_host, void *stream);

/* allocates the staging of blink_grid_image_host for chunks of chunk_t time steps (three buffers of
 * chunk_t x (8 n_ch n_bl + 4 n_ch N^2) bytes, streams, events) and blink_grid_image's own scratch for such a
 * chunk; synchronises the device when it has to grow; never shrinks.  chunk_t = 0: the plan picks the chunk
 * (about 32 MiB each way) unless one is reserved already */
int blink_plan_reserve_host(blink_plan *plan, int chunk_t);

/*
 * blink_plan_read -- copies one channel's slice of a plan table to HOST memory (synchronous):
 *   what = BLINK_Q_CELL_IDX -> int32 [n_bl];  what = BLINK_Q_COUNTS -> uint32 [N*N];
 *   what = BLINK_Q_CORR -> complex64 [n_bl] (BLINK_EINVAL until blink_plan_set_corrections).
 * `bytes` must equal the slice size.  This is how a harness checks indices and counts bit-exactly.
 */
int blink_plan_read(const blink_plan *plan, int what, int ch, void *dst_host, size_t bytes);

/*
 * blink_plan_reserve -- sizes the plan's device scratch for blink_image / blink_grid_image calls of up
 * to n_t time steps (BLINK_Q_SCRATCH_BYTES reports it).  The only place scratch is allocated: may
 * synchronise the device and free / allocate memory; never shrinks.  BLINK_ENOMEM if it does not fit.
 */
int blink_plan_reserve(blink_plan *plan, int n_t);

/*
 * blink_grid_validate -- checks blink_image's input contract on a uv grid: counts the cells that are
 * non-zero although the plan's weight count there is zero, plus the cells G[k] != conj(G[-k]) (bitwise).
 * 0 for every blink_grid output.  blink_image's result is defined by the transform of PAPER.md:372-376
 * only for grids that pass (a route may read just the plan's occupied cells); a harness that feeds it
 * grids from elsewhere calls this first.
 *   uv_grid       DEVICE complex64 [n_t][n_ch][N][N]
 *   n_violations  HOST   int64, out
 * Synchronous (waits for `stream`).
 */
int blink_grid_validate(const blink_plan *plan, const void *uv_grid, int n_t, int64_t *n_violations,
                        void *stream);

#ifdef __cplusplus
}
#endif
#endif /* BLINK_H_ */
