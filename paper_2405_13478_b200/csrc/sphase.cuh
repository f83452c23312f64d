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
                                          const uint16_t *__restrict__ scat, int b0, int cnt, int tid,
                                          const float2 *__restrict__ corr = nullptr) {
#pragma unroll
  for (int q = 0; q < PF; ++q) {
    const int i = q * THREADS + tid;
    r.sc[q] = kScatDropped;
    if (i < cnt) {
      r.sc[q] = scat[b0 + i];
      r.v[q] = __ldcs(vis + b0 + i);               // streamed once: evict-first
    }
  }
  if (corr != nullptr) {   // pre-gridding corrections fused at load: V * F[ch][bl] (blink_correct.cu), F from L2
#pragma unroll
    for (int q = 0; q < PF; ++q) {
      const int i = q * THREADS + tid;
      if (i < cnt) {
        const float2 f = __ldg(corr + b0 + i), v = r.v[q];
        r.v[q] = make_float2(v.x * f.x - v.y * f.y, v.x * f.y + v.y * f.x);
      }
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

// Per-cell sums of one pass.  Cells are ordered by descending length, so the lanes of a warp own
// cells of (nearly) equal length: each thread walks its own cell, rank by rank, reading
// stage[roff[r] + k] -- consecutive threads read consecutive slots (no bank conflicts, no atomics)
// -- and adds in ascending baseline order.  roff is read four ranks at a time.  The cell records
// of a pass are fetched into registers BEFORE the scatter and its barrier (sums_prefetch), so no
// table latency is exposed between the barrier and the first shared-memory read; the tables are
// zero-padded to n_can_max, so the prefetch needs no bound from memory.
template <int THREADS> struct SumsRegs { uint32_t rec[kGridCellsPerThread]; };

template <int THREADS>
__device__ __forceinline__ void sums_prefetch(SumsRegs<THREADS> &sr, const uint32_t *__restrict__ cellrec,
                                              int n_can_max, int tid) {
#pragma unroll
  for (int c = 0; c < kGridCellsPerThread; ++c) {
    const int k = tid + c * THREADS;
    sr.rec[c] = k < n_can_max ? __ldg(cellrec + k) : 0u;
  }
}

__device__ __forceinline__ void sum_cell(uint32_t rec, int k, const uint16_t *__restrict__ roff,
                                         const float2 *stage, float2 *S) {
  const int j = rec & 0xFFFFu, len = rec >> 16;
  const float2 *__restrict__ col = stage + k;
  float ax = 0.f, ay = 0.f;
  int r = 0;
  for (; r + 4 <= len; r += 4) {
    const ushort4 o = *reinterpret_cast<const ushort4 *>(roff + r);     // roff stride is 4-aligned
    const float2 v0 = col[o.x], v1 = col[o.y], v2 = col[o.z], v3 = col[o.w];
    ax += v0.x; ay += v0.y;
    ax += v1.x; ay += v1.y;
    ax += v2.x; ay += v2.y;
    ax += v3.x; ay += v3.y;
  }
  for (; r < len; ++r) {
    const float2 v = col[roff[r]];
    ax += v.x; ay += v.y;
  }
  const float2 a = S[j];
  S[j] = make_float2(a.x + ax, a.y + ay);
}

template <int THREADS>
__device__ __forceinline__ void sums_run(const SumsRegs<THREADS> &sr, const uint32_t *__restrict__ cellrec,
                                         const uint16_t *__restrict__ roff, int n_can_max,
                                         const float2 *stage, float2 *S, int tid) {
#pragma unroll
  for (int c = 0; c < kGridCellsPerThread; ++c)
    if (sr.rec[c] >> 16) sum_cell(sr.rec[c], tid + c * THREADS, roff, stage, S);
  for (int k = tid + kGridCellsPerThread * THREADS; k < n_can_max; k += THREADS) {
    const uint32_t rec = cellrec[k];
    if (rec >> 16) sum_cell(rec, k, roff, stage, S);
  }
}

}  // namespace blink
