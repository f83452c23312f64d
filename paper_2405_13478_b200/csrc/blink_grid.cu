// blink_grid.cu -- steps a1/a2: gridding (listing :462-489).
//
// The paper's kernel is one thread per visibility with atomicAdd on the global grid and a separate
// zero-initialisation; it names the atomics as a cost and plans a deterministic
// parallel reduction.  Because the array geometry is fixed across snapshots,
// the plan has already sorted every channel's baselines by destination cell, so here gridding is an
// ATOMIC-FREE sort-by-table + segmented sum:
//
//   phase S  the snapshot's visibilities are read ONCE, coalesced, in input order, and each is
//            dropped (as V or conj(V)) into its precomputed slot of a cell-sorted stage in shared
//            memory; then one thread per canonical (half-plane) cell adds up its contiguous
//            segment in ascending baseline order -> S[j].  Baselines are taken in passes of
//            `stage_cap` so the stage fits next to everything else.
//   phase P  the dense N x N grid is written exactly: first the whole snapshot (or part) is
//            zero-filled by bulk asynchronous copies from a constant zero buffer in shared memory
//            (cp.async.bulk shared -> global, TMA engine; issued by one thread BEFORE phase S so the
//            fill drains while the sums are formed), then, once the fill has completed, the occupied
//            cells are stored on top: S[j] at canonical cells, conj(S[j]) at the mirrored cells.
//            No memset is needed and the grid is never read.
//
// One CTA works on one (snapshot, part) item at a time and strides over items (persistent grid),
// "part" splitting a snapshot's bands when there are few snapshots.
#include <algorithm>

#include "blink_internal.h"
#include "sphase.cuh"

namespace blink {

struct GridParams {
  const float2 *vis;
  float2 *uv;
  const ChannelInfo *chinfo;
  const uint16_t *scat, *roff;
  const uint32_t *cellrec;
  const int32_t *nact;
  const int32_t *pcell, *pcode, *pband;
  int n_bl, n_ch, n_snap, n_bands, band_cells, parts, n_can_max, n_pass, roff_stride, dbg, ch0;
  long long grid_cells;  // N*N
};

template <int THREADS, int PF, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) k_grid(const GridParams p) {
  constexpr int CAP = THREADS * PF;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float2 *zero = reinterpret_cast<float2 *>(smem_raw);           // [band_cells]
  float2 *S = zero + p.band_cells;                               // [n_can_max]
  float2 *stage = S + p.n_can_max;                               // [CAP]
  const int tid = threadIdx.x;

  {
    float4 *z4 = reinterpret_cast<float4 *>(smem_raw);
    for (int i = tid; i < p.band_cells / 2; i += THREADS) z4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  fence_async_smem();
  __syncthreads();

  const int bands_per_part = (p.n_bands + p.parts - 1) / p.parts;
  const long long n_items = (long long)p.n_snap * p.parts;
  const uint32_t band_bytes = (uint32_t)p.band_cells * sizeof(float2);
  PassRegs<PF> regs;
  if (blockIdx.x < n_items) {   // prefetch pass 0 of the first item
    const int s = (int)(blockIdx.x / p.parts);
    pass_load<THREADS, PF>(regs, p.vis + (size_t)s * p.n_bl, p.scat + (size_t)((s + p.ch0) % p.n_ch) * p.n_bl, 0,
                           min(CAP, p.n_bl), tid);
  }
  for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int s = (int)(item / p.parts), part = (int)(item % p.parts);
    const int ch = (s + p.ch0) % p.n_ch;
    const ChannelInfo ci = p.chinfo[ch];
    const float2 *__restrict__ vis = p.vis + (size_t)s * p.n_bl;
    const uint16_t *__restrict__ scat = p.scat + (size_t)ch * p.n_bl;
    const int b_lo = part * bands_per_part;
    const int b_hi = min(p.n_bands, b_lo + bands_per_part);
    float2 *__restrict__ grid = p.uv + (size_t)s * p.grid_cells;

    // ---- phase P, first half: zero-fill this part; drains while phase S runs -----------------
    if (tid == 0 && !(p.dbg & 1)) {
      for (int b = b_lo; b < b_hi; ++b) bulk_store(grid + (size_t)b * p.band_cells, zero, band_bytes);
      bulk_commit();
    }

    // ---- phase S: table-driven sort into the rank-major stage, then per-cell sums -----------
    for (int j = tid; j < p.n_can_max; j += THREADS) S[j] = make_float2(0.f, 0.f);
    for (int pass = 0; pass < p.n_pass; ++pass) {
      const size_t cp = (size_t)ch * p.n_pass + pass;
      const uint32_t *__restrict__ cellrec = p.cellrec + cp * max(p.n_can_max, 1);
      SumsRegs<THREADS> sr;
      sums_prefetch<THREADS>(sr, cellrec, p.n_can_max, tid);
      if (!(p.dbg & 4)) pass_scatter<PF>(regs, stage);
      __syncthreads();
      // loads of the next pass (or of the next item's first pass) fly during the sums and phase P
      if (pass + 1 < p.n_pass) {
        const int b0 = (pass + 1) * CAP;
        pass_load<THREADS, PF>(regs, vis, scat, b0, min(CAP, p.n_bl - b0), tid);
      } else if (item + gridDim.x < n_items) {
        const int s2 = (int)((item + gridDim.x) / p.parts);
        pass_load<THREADS, PF>(regs, p.vis + (size_t)s2 * p.n_bl, p.scat + (size_t)((s2 + p.ch0) % p.n_ch) * p.n_bl,
                               0, min(CAP, p.n_bl), tid);
      }
      if (!(p.dbg & 2)) sums_run<THREADS>(sr, cellrec, p.roff + cp * p.roff_stride, p.n_can_max, stage, S, tid);
      if (pass + 1 == p.n_pass && tid == 0) bulk_wait_all();   // the zero fill has landed
      __syncthreads();
    }

    // ---- phase P, second half: occupied cells on top of the zeros -----------------------------
    const int32_t *__restrict__ pband = p.pband + (size_t)ch * (p.n_bands + 1);
    const int32_t *__restrict__ pcell = p.pcell + (size_t)ch * 2 * p.n_bl;
    const int32_t *__restrict__ pcode = p.pcode + (size_t)ch * 2 * p.n_bl;
    const int e0 = pband[b_lo], e1 = pband[b_hi];
    for (int e = e0 + tid; e < e1 && !(p.dbg & 8); e += THREADS) {
      const int code = pcode[e];
      const float2 v = S[code & kPlaceMask];
      const int flag = code >> kPlaceShift;
      float2 o;
      if (flag == kPlaceDirect) o = v;
      else if (flag == kPlaceConj) o = make_float2(v.x, -v.y);
      else o = make_float2(v.x + v.x, 0.f);
      grid[pcell[e]] = o;
    }
    __syncthreads();  // S is rewritten by the next item
  }
}

template <int THREADS, int PF, int MINB>
static int launch_grid_v(const blink_plan *p, const GridParams &g0, cudaStream_t st) {
  GridParams g = g0;
  const size_t smem = p->grid_smem;
  if (smem > (size_t)p->max_smem_optin) return BLINK_EUNSUPPORTED;
  static thread_local size_t smem_set = 0;
  if (smem > smem_set) {
    BLINK_CUDA_TRY(cudaFuncSetAttribute(k_grid<THREADS, PF, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                   "k_grid smem attribute");
    BLINK_CUDA_TRY(cudaFuncSetAttribute(k_grid<THREADS, PF, MINB>, cudaFuncAttributePreferredSharedMemoryCarveout, 100),
                   "k_grid carveout");
    smem_set = smem;
  }
  int occ = 1;
  BLINK_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_grid<THREADS, PF, MINB>, THREADS, smem),
                 "k_grid occupancy");
  const int resident = std::max(1, occ) * p->sm_count;
  // split snapshots into parts when there are too few of them to fill the machine evenly
  int parts = 1;
  while (parts < g.n_bands && (long long)g.n_snap * parts < 4LL * resident) parts *= 2;
  g.parts = parts;
  const long long n_items = (long long)g.n_snap * parts;
  const int blocks = (int)std::min<long long>(n_items, resident);
  if (blocks <= 0) return BLINK_OK;
  k_grid<THREADS, PF, MINB><<<blocks, THREADS, smem, st>>>(g);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_grid launch");
  return BLINK_OK;
}

int launch_grid(const blink_plan *p, const float2 *vis, int n_snap, int ch0, float2 *uv, cudaStream_t st) {
  GridParams g;
  g.vis = vis; g.uv = uv; g.chinfo = p->d_chinfo;
  g.scat = p->d_scat; g.roff = p->d_roff; g.cellrec = p->d_cellrec; g.nact = p->d_nact; g.pcell = p->d_pcell; g.pcode = p->d_pcode; g.pband = p->d_pband;
  g.n_bl = p->n_bl; g.n_ch = p->n_ch; g.n_snap = n_snap; g.ch0 = ch0;
  g.n_bands = p->n_bands; g.band_cells = p->band_cells; g.n_can_max = p->n_can_max;
  g.n_pass = p->n_pass; g.roff_stride = p->roff_stride; g.parts = 1;
  g.dbg = 0;
  if (const char *e = getenv("BLINK_GRID_DEBUG")) g.dbg = atoi(e);   // timing experiments only
  g.grid_cells = (long long)p->n_pix * p->n_pix;
  if (p->grid_threads == 512 && p->grid_prefetch == 16) return launch_grid_v<512, 16, 1>(p, g, st);
  if (p->grid_threads == 512 && p->grid_prefetch == 8) return launch_grid_v<512, 8, 2>(p, g, st);
  if (p->grid_threads == 256 && p->grid_prefetch == 8) return launch_grid_v<256, 8, 3>(p, g, st);
  return launch_grid_v<256, 16, 2>(p, g, st);
}

}  // namespace blink

extern "C" int blink_grid(const blink_plan *plan, const void *vis, int n_t, void *uv_grid, void *stream) {
  if (!plan || n_t < 0) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!vis || !uv_grid) return BLINK_EINVAL;
  if (((uintptr_t)vis & 7) || ((uintptr_t)uv_grid & 15)) return BLINK_EINVAL;
  return blink::launch_grid(plan, (const float2 *)vis, n_t * plan->n_ch, 0, (float2 *)uv_grid, (cudaStream_t)stream);
}
