/*
 * blink_testing.h -- hooks of libblink exported for its test suite and its benchmark, NOT part of the
 * product ABI (include/blink.h); may change.  blink_host_*: host-only, run the plan's table builders and a
 * byte-for-byte model of the gridding phase on the CPU, so the host logic is testable without a GPU
 * (tests/test_host_logic.py).  blink_probe_fp32: the in-run fp32 peak probe bench.py times.
 */
#ifndef BLINK_TESTING_H_
#define BLINK_TESTING_H_

#include "blink.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Host-side table helper, exported so the host logic is testable without a GPU.
 * Builds the cell-sorted gather tables blink_grid uses from per-baseline cell indices of ONE
 * channel (as returned by BLINK_Q_CELL_IDX): every kept baseline contributes once to its
 * canonical cell (the member of {cell, cell*} in the half-plane ky > 0 or ky == 0, kx >= 0), as V
 * or as conj(V).  Entries are sorted by (canonical cell, baseline).
 *   cell        HOST int32 [n_bl], -1 = dropped
 *   n_can_out   HOST number of distinct canonical cells
 *   can_cell    HOST int32 [n_bl]   out: canonical cell index per segment (first n_can valid)
 *   seg_start   HOST int32 [n_bl+1] out: CSR offsets into src (first n_can+1 valid)
 *   src         HOST int32 [n_bl]   out: (baseline << 1) | conj_flag, n_kept entries
 * Returns the number of kept baselines or a negative blink_status.
 */
int blink_host_build_gather(const int32_t *cell, int n_bl, int n_pix, int32_t *n_can_out,
                            int32_t *can_cell, int32_t *seg_start, int32_t *src);

/*
 * Host emulation of the gridding phase of blink_grid_image's shared-memory route (steps a1/a2,
 * PAPER.md:348-370), exported so its plan tables are testable without a GPU.  For ONE channel it
 * builds the gather tables the kernel streams through shared memory -- cells owned by warps,
 * baselines taken in chunks of chunk_vis (even, <= 32766), groups of 32 lanes x at most 4 rows --
 * and walks them over a host model of shared memory exactly as a warp does.
 *   cell       HOST int32 [n_bl], -1 = dropped (BLINK_Q_CELL_IDX of the channel)
 *   vis        HOST complex64 [n_bl] (interleaved floats)
 *   sums       HOST complex64 [n_can] out: per canonical cell (blink_host_build_gather's order) the
 *              sum of V (or conj V) over its baselines, fp32, in the kernel's summation order
 *   stats      HOST int32 [3] out (may be NULL): n_can, groups, rows over all chunks
 * Returns 0 or a negative blink_status.
 */
int blink_host_fused_emulate(const int32_t *cell, int n_bl, int n_pix, int chunk_vis, const float *vis,
                             float *sums, int32_t *stats);

/*
 * Host model of the residue-class kernels (csrc/blink_image_r.cu; steps a1-a5) for ONE channel
 * and ONE snapshot, exported so their plan tables and index algebra are testable without a GPU: builds the
 * tables as the plan does (bins of the occupied half-plane cells dealt to the lanes of 16 warps; at N = 2048 /
 * 4096 also the columns dealt to the warps) and walks them as the kernels do -- cell values, bins of a unit,
 * column transforms, row transforms -- in fp64 with direct DFT sums in place of the butterflies.
 *   n_pix = 1024: k_img1024r, a unit r in 0..63 = image rows 64 p + r (p = 0..7) and those + 512
 *   n_pix = 2048 / 4096: k_cols_res, a unit r in 0..N/8-1 = image rows (N / 8) y' + r, y' = 0..7
 *   cell       HOST int32 [n_bl], -1 = dropped (cells of an n_pix x n_pix grid)
 *   weighting  BLINK_NATURAL / BLINK_UNIFORM
 *   vis        HOST complex64 [n_bl] (interleaved floats)
 *   units      HOST int32 [n_units]
 *   rows       HOST float32 [n_units][16 or 8][n_pix] out: the unit's image rows in the order given above
 *   stats      HOST int32 [3] out (may be NULL): list positions, longest lane list, canonical cells
 * Returns 0, BLINK_EUNSUPPORTED when the cells do not fit the route, or a negative blink_status.
 */
int blink_host_residue_emulate(const int32_t *cell, int n_bl, int n_pix, int weighting, const float *vis, int n_units,
                               const int32_t *units, float *rows, int32_t *stats);

/*
 * Measurement hook for bench.py (the fp32 peak is measured in-run): launches a
 * register-only kernel of out_floats / 256 blocks x 256 threads, each thread running `iters` x 64
 * instructions of one kind in eight independent chains: op 0 = add.f32, 1 = fma.rn.f32,
 * 2 = add.rn.f32x2, 3 = fma.rn.f32x2.  Asynchronous on `stream`; the caller times it.
 *   out_dev   DEVICE float [out_floats] (written, values meaningless)
 *   flops     HOST   out: floating-point operations of the launch (an FMA counts 2)
 */
int blink_probe_fp32(int op, int iters, void *out_dev, size_t out_floats, int64_t *flops, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* BLINK_TESTING_H_ */
