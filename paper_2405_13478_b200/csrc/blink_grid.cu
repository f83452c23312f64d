// blink_grid.cu -- steps a1/a2: gridding (listing :462-489).
//
// The paper's kernel is one thread per visibility with atomicAdd on the global grid and a separate
// zero-initialisation; it names the atomics as a cost and plans a deterministic
// parallel reduction.  Because the array geometry is fixed across snapshots,
// the plan has already sorted every channel's baselines by destination cell, so here gridding is an
// ATOMIC-FREE segmented gather:
//
//   phase S  for each canonical (half-plane) cell j:  S[j] = sum over its baselines, in ascending
//            baseline order, of V or conj(V)                              -> shared memory
//   phase P  the dense N x N grid is composed band by band (32 KB) in shared memory -- zeros, S[j]
//            at canonical cells, conj(S[j]) at the mirrored cells -- and each band leaves the SM as
//            ONE bulk asynchronous copy (cp.async.bulk shared -> global, TMA engine); bands with no
//            occupied cell are bulk-copied from a constant zero band.  Every byte of uv_grid is
//            written exactly once, so no memset and no read-modify-write traffic exists.
//
// One CTA works on one (snapshot, part) item at a time and strides over items (persistent grid of
// a few CTAs per SM), "part" splitting a snapshot's bands when there are few snapshots.
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

struct GridParams {
  const float2 *vis;
  float2 *uv;
  const ChannelInfo *chinfo;
  const int32_t *src, *seg, *pcell, *pcode, *pband;
  int n_bl, n_ch, n_snap, n_bands, band_cells, parts, n_can_max;
  long long grid_cells;  // N*N
};

constexpr int kGridThreads = 512;

__global__ void __launch_bounds__(kGridThreads) k_grid(const GridParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float2 *zero = reinterpret_cast<float2 *>(smem_raw);           // [band_cells]
  float2 *band0 = zero + p.band_cells;                           // [2][band_cells]
  float2 *S = band0 + 2 * p.band_cells;                          // [n_can_max]
  const int tid = threadIdx.x;

  for (int i = tid; i < p.band_cells; i += kGridThreads) zero[i] = make_float2(0.f, 0.f);
  fence_async_smem();
  __syncthreads();

  const int bands_per_part = (p.n_bands + p.parts - 1) / p.parts;
  const long long n_items = (long long)p.n_snap * p.parts;
  int nbuf = 0;
  for (long long item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int s = (int)(item / p.parts), part = (int)(item % p.parts);
    const int ch = s % p.n_ch;
    const ChannelInfo ci = p.chinfo[ch];
    const float2 *__restrict__ vis = p.vis + (size_t)s * p.n_bl;
    const int32_t *__restrict__ seg = p.seg + (size_t)ch * (p.n_bl + 1);
    const int32_t *__restrict__ src = p.src + (size_t)ch * p.n_bl;

    // ---- phase S: segmented gather, fixed summation order --------------------------------
    for (int j = tid; j < ci.n_can; j += kGridThreads) {
      const int e0 = seg[j], e1 = seg[j + 1];
      float ar = 0.f, ai = 0.f;
      for (int e = e0; e < e1; ++e) {
        const int code = src[e];
        const float2 v = __ldg(vis + (code >> 1));
        ar += v.x;
        ai += (code & 1) ? -v.y : v.y;
      }
      S[j] = make_float2(ar, ai);
    }
    __syncthreads();

    // ---- phase P: compose and emit the bands of this part -----------------------------------
    const int32_t *__restrict__ pband = p.pband + (size_t)ch * (p.n_bands + 1);
    const int32_t *__restrict__ pcell = p.pcell + (size_t)ch * 2 * p.n_bl;
    const int32_t *__restrict__ pcode = p.pcode + (size_t)ch * 2 * p.n_bl;
    const int b_lo = part * bands_per_part;
    const int b_hi = min(p.n_bands, b_lo + bands_per_part);
    const uint32_t band_bytes = (uint32_t)p.band_cells * sizeof(float2);
    for (int b = b_lo; b < b_hi; ++b) {
      const int e0 = pband[b], e1 = pband[b + 1];
      float2 *dst = p.uv + (size_t)s * p.grid_cells + (size_t)b * p.band_cells;
      if (e0 == e1) {
        if (tid == 0) { bulk_store(dst, zero, band_bytes); bulk_commit(); }
        continue;
      }
      float2 *buf = band0 + (size_t)(nbuf & 1) * p.band_cells;
      ++nbuf;
      if (tid == 0) bulk_wait_read<1>();   // the copy that last read this buffer has drained
      __syncthreads();
      {
        float4 *b4 = reinterpret_cast<float4 *>(buf);
        for (int i = tid; i < p.band_cells / 2; i += kGridThreads) b4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
      __syncthreads();
      const int base = b * p.band_cells;
      for (int e = e0 + tid; e < e1; e += kGridThreads) {
        const int code = pcode[e];
        const float2 v = S[code & kPlaceMask];
        const int flag = code >> kPlaceShift;
        float2 o;
        if (flag == kPlaceDirect) o = v;
        else if (flag == kPlaceConj) o = make_float2(v.x, -v.y);
        else o = make_float2(v.x + v.x, 0.f);
        buf[pcell[e] - base] = o;
      }
      fence_async_smem();
      __syncthreads();
      if (tid == 0) { bulk_store(dst, buf, band_bytes); bulk_commit(); }
    }
    __syncthreads();  // S is rewritten by the next item
  }
  if (tid == 0) bulk_wait_all();
}

int launch_grid(const blink_plan *p, const float2 *vis, int n_t, float2 *uv, cudaStream_t st) {
  GridParams g;
  g.vis = vis; g.uv = uv; g.chinfo = p->d_chinfo;
  g.src = p->d_src; g.seg = p->d_seg; g.pcell = p->d_pcell; g.pcode = p->d_pcode; g.pband = p->d_pband;
  g.n_bl = p->n_bl; g.n_ch = p->n_ch; g.n_snap = n_t * p->n_ch;
  g.n_bands = p->n_bands; g.band_cells = p->band_cells; g.n_can_max = p->n_can_max;
  g.grid_cells = (long long)p->n_pix * p->n_pix;
  const size_t smem = sizeof(float2) * ((size_t)3 * p->band_cells + (size_t)p->n_can_max);
  if (smem > (size_t)p->max_smem_optin) return BLINK_EUNSUPPORTED;
  static thread_local size_t smem_set = 0;
  if (smem > smem_set) {
    BLINK_CUDA_TRY(cudaFuncSetAttribute(k_grid, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                   "k_grid smem attribute");
    smem_set = smem;
  }
  int occ = 1;
  BLINK_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_grid, kGridThreads, smem),
                 "k_grid occupancy");
  if (occ < 1) occ = 1;
  const int resident = occ * p->sm_count;
  // split snapshots into parts when there are too few of them to fill the machine evenly
  int parts = 1;
  while (parts < g.n_bands && (long long)g.n_snap * parts < 4LL * resident) parts *= 2;
  g.parts = parts;
  const long long n_items = (long long)g.n_snap * parts;
  const int blocks = (int)std::min<long long>(n_items, resident);
  if (blocks <= 0) return BLINK_OK;
  k_grid<<<blocks, kGridThreads, smem, st>>>(g);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_grid launch");
  return BLINK_OK;
}

}  // namespace blink

extern "C" int blink_grid(const blink_plan *plan, const void *vis, int n_t, void *uv_grid, void *stream) {
  if (!plan || n_t < 0) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!vis || !uv_grid) return BLINK_EINVAL;
  if (((uintptr_t)vis & 7) || ((uintptr_t)uv_grid & 15)) return BLINK_EINVAL;
  return blink::launch_grid(plan, (const float2 *)vis, n_t, (float2 *)uv_grid, (cudaStream_t)stream);
}
