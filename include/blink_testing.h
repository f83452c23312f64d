/*
 * blink_testing.h -- host-only hooks of libblink exported for its test suite (tests/test_host_logic.py):
 * they run the plan's table builders and a byte-for-byte model of the gridding phase on the CPU, so the
 * host logic is testable without a GPU.  NOT part of the product ABI (include/blink.h); may change.
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

#ifdef __cplusplus
}
#endif
#endif /* BLINK_TESTING_H_ */
