// sphase.cuh -- phase S of the gridder, shared by blink_grid (k_grid) and blink_grid_image
// (k_fused): table-driven sort of one pass of visibilities into a rank-major shared-memory stage,
// then per-cell sums in ascending baseline order (steps a1/a2; deterministic
// reduction per PAPER.md:370, :396).  Also the bulk-copy (TMA) helpers.
#pragma once

#include "blink_internal.h"

namespace blink {

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void bulk_store(void *gdst, const void *ssrc, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst),
               "r"(smem_u32(ssrc)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() {
  asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// registers of one pass: PF visibilities per thread and their stage slots
template <int PF> struct PassRegs {
  float2 v[PF];
  uint16_t sc[PF];
};

template <int THREADS, int PF>
__device__ __forceinline__ void pass_load(PassRegs<PF> &r, const float2 *__restrict__ vis,
                                          const uint16_t *__restrict__ scat, int b0, int cnt, int tid) {
#pragma unroll
  for (int q = 0; q < PF; ++q) {
    const int i = q * THREADS + tid;
    r.sc[q] = kScatDropped;
    if (i < cnt) {
      r.sc[q] = scat[b0 + i];
      r.v[q] = __ldcs(vis + b0 + i);               // streamed once: evict-first
    }
  }
}

template <int PF> __device__ __forceinline__ void pass_scatter(const PassRegs<PF> &r, float2 *stage) {
#pragma unroll
  for (int q = 0; q < PF; ++q) {
    const uint32_t sc = r.sc[q];
    if (sc != kScatDropped)
      stage[sc & 0x7FFFu] = make_float2(r.v[q].x, (sc & 0x8000u) ? -r.v[q].y : r.v[q].y);
  }
}

// Per-cell sums of one pass.  Cells are ordered by descending length: rank r is held by the first
// n_r cells, so every thread runs the same r loop and its CPT accumulators are independent (ILP,
// no divergence); consecutive threads read consecutive stage slots (no bank conflicts).
template <int THREADS>
__device__ __forceinline__ void sphase_sums(const uint32_t *__restrict__ cellrec,
                                            const uint16_t *__restrict__ roff, int n_act,
                                            const float2 *stage, float2 *S, int tid) {
  constexpr int CPT = kGridCellsPerThread;
  for (int k0 = 0; k0 < n_act; k0 += CPT * THREADS) {
    uint32_t rec[CPT];
    float2 acc[CPT];
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      const int k = k0 + c * THREADS + tid;
      rec[c] = k < n_act ? cellrec[k] : 0u;
      acc[c] = make_float2(0.f, 0.f);
    }
    const int maxlen = (int)(cellrec[k0] >> 16);
    int off = roff[0];
    for (int r = 0; r < maxlen; ++r) {
      const int off1 = roff[r + 1];
      const int n_r = off1 - off;            // cells (from position 0) that have a rank-r entry
#pragma unroll
      for (int c = 0; c < CPT; ++c) {
        const int k = k0 + c * THREADS + tid;
        if (k < n_r) {
          const float2 v = stage[off + k];
          acc[c].x += v.x;
          acc[c].y += v.y;
        }
      }
      off = off1;
    }
#pragma unroll
    for (int c = 0; c < CPT; ++c) {
      if (rec[c] >> 16) {
        const int j = rec[c] & 0xFFFFu;
        const float2 a = S[j];
        S[j] = make_float2(a.x + acc[c].x, a.y + acc[c].y);
      }
    }
  }
}

}  // namespace blink
