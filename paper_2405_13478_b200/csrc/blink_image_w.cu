// blink_image_w.cu -- steps a3-a5 at N = 1024 as ONE persistent kernel with one WARP per 1024-point
// transform (wfft.cuh): weighting, batched 2-D inverse FFT, fftshift, normalisation, real part
// (PAPER.md:360, :372-376).  Same two passes and the same fusions as blink_image.cu (Hermitian
// half-plane columns, two real rows per complex row transform, shift as a sign on load), but:
//
//   * both passes run in the same cooperative launch by two groups of persistent CTAs: the first g_a
//     CTAs produce U[y][kx] (pass A: items of 8 columns), the others consume it (pass B: items of 8
//     row pairs); each group deals its snapshot-major item sequence round-robin.  The U of a snapshot
//     lives in a ring of R slots sized to stay in L2 (4 MB per slot at wu = 512, 32 MB in all): it is
//     written by pass A, read by pass B a few snapshots later, and never crosses HBM.  Per-snapshot
//     completion counters order the two passes and the reuse of a slot: pass B of snapshot s waits for
//     done_a[s], pass A of snapshot s for done_b[s - R]; every wait points at an earlier item of a
//     group that takes its items in order, so they cannot deadlock.
//   * pass A is SPARSE: a column of the uv plane holds a handful of occupied cells (MWA Phase I: 14
//     on average, 85 at most, of 1024), so the inner step of the 32 x 32 split is a sum over those
//     cells -- each adds val * w32^(a y1) to its residue class b = iy mod 32, lane = y1 -- and only
//     the outer step is a dense 32-point butterfly.  The cells of a column arrive sorted by (b, a)
//     from the plan as 16-byte records, copied into shared memory (cp.async) one item ahead; the
//     visibilities of a snapshot are prefetched into L2 two snapshots ahead.
//   * pass B: the two U rows of a warp's row pair arrive in its exchange tile by bulk copy (UBLKCP),
//     issued for the NEXT item as soon as the tile is free, so the loads overlap the outer butterfly
//     and the stores; a warp-wide store of one register is 128 contiguous bytes of an image row.
//
// Used by blink_grid_image and blink_image when warp_route_applies() (blink_image: the same kernel with
// the cell values read from the uv grid at the plan's occupied cells instead of summed from the
// visibilities); compact arrays keep the line kernels of blink_image.cu.
#include <algorithm>

#include "blink_internal.h"
#include "sgather.cuh"
#include "wfft.cuh"

namespace blink {
using namespace blinkfft;

constexpr int kWN = 1024;
constexpr int kWWarps = 8;                     // transforms per item
constexpr int kWThreads = 32 * kWWarps;
constexpr int kWTileStride = kWfTile + 2;      // complex slots between the warps' tiles (16-byte aligned)
constexpr int kWOStride = 9;                   // out-tile row stride (complex), pass A
constexpr int kWItemsB = kWN / 2 / kWWarps;    // pass-B items per snapshot
constexpr size_t kWXchBytes = sizeof(cf32) * kWWarps * kWTileStride;
constexpr size_t kWOutBytes = sizeof(cf32) * kWN * kWOStride;
constexpr size_t kWRegionBytes = kWXchBytes > kWOutBytes ? kWXchBytes : kWOutBytes;
constexpr size_t kWFixedBytes = kWRegionBytes + sizeof(cf32) * (1024 + 32) + 8 * kWWarps;

struct WParams {
  ImgParams ip;
  int n_snap, items_a, g_a, ring;   // items_a = wu / 8; CTAs 0 .. g_a - 1 run pass A; ring slots of U
  int *done_a, *done_b;             // per snapshot; zero at launch, zeroed again by the last CTA to finish
  int *finished;                    // CTAs that have finished (same protocol)
  const uint4 *vrec;                // pass-A cell records
  const float2 *uvsrc;              // blink_image: cell values come from this uv grid; NULL = from visibilities
};

__device__ __forceinline__ int ld_acquire(const int *p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ int ld_relaxed(const int *p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

struct WItem { int kind, snap, idx; };   // kind 0 = pass A, 1 = pass B, -1 = none

// pass B loads of one warp: rows y0 and y0 + N/2 of the snapshot's U into the warp's tile
__device__ __forceinline__ void issue_rows(const WParams &q, const WItem &it, int wv, cf32 *tile, uint64_t *bar) {
  const int wu = q.ip.wu, y0 = it.idx * kWWarps + wv;
  const float2 *U = q.ip.U + (size_t)(it.snap % q.ring) * kWN * wu;
  const uint32_t bytes = (uint32_t)wu * sizeof(cf32);
  fence_proxy_async_all();            // generic reads of the tile, and the acquired U, before the async copies
  mbar_expect_tx(bar, 2 * bytes);
  bulk_load(tile, U + (size_t)y0 * wu, bytes, bar);
  bulk_load(tile + wu, U + (size_t)(y0 + kWN / 2) * wu, bytes, bar);
}

__global__ void __launch_bounds__(kWThreads, 2) k_img1024(const WParams q) {
  constexpr int N = kWN;
  const ImgParams &p = q.ip;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cf32 *region = reinterpret_cast<cf32 *>(smem_raw);                 // exchange tiles / pass-A out tile
  cf32 *tws = reinterpret_cast<cf32 *>(smem_raw + kWRegionBytes);    // inner-step twiddles [n1][b]
  cf32 *w32 = tws + 1024;                                            // exp(2 pi i k / 32)
  uint64_t *bars = reinterpret_cast<uint64_t *>(w32 + 32);           // one mbarrier per warp
  cf32 *cv = reinterpret_cast<cf32 *>(smem_raw + kWFixedBytes);      // cell values of a pass-A item
  int32_t *ck = reinterpret_cast<int32_t *>(cv + p.cell_cap);        // their iy
  int32_t *s_off = ck + p.cell_cap;                                  // [3][12] column offsets of this / the next two items
  uint4 *recs = reinterpret_cast<uint4 *>(s_off + 48);               // cell records of the item, copied in one item ahead
  const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;
  cf32 *tile = region + wv * kWTileStride;
  uint64_t *bar = bars + wv;

  for (int i = tid; i < 1024; i += kWThreads) tws[i] = __ldg(p.tw32 + i);
  if (tid < 32) w32[tid] = __ldg(p.tw + tid * (N / 32));
  if (tid < kWWarps) mbar_init(bars + tid, 1);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();

  uint32_t parity = 0;
  bool pending = false;                  // this warp's tile holds (or is receiving) the rows of the next item
  // roles: the first g_a CTAs produce U (pass A), the others consume it (pass B); each group deals
  // its own item sequence (snapshot-major) round-robin
  const bool role_a = (int)blockIdx.x < q.g_a;
  const int G = role_a ? q.g_a : (int)gridDim.x - q.g_a;
  const int per = role_a ? q.items_a : kWItemsB;
  const int total = q.n_snap * per;
  const int j_first = role_a ? (int)blockIdx.x : (int)blockIdx.x - q.g_a;
  // column offsets (vcol) of item jj, one per thread 0..8
  auto load_off = [&](int jj) {
    const int sn = jj / per, ix = jj - sn * per;
    return __ldg(p.vcol + (size_t)((sn + p.ch0) % p.n_ch) * (p.wu + 1) + ix * kWWarps + tid);
  };
  // asynchronous copy of the cell records [e0, e1) of item jj into recs (16 bytes per thread and step)
  auto fetch_recs = [&](int jj, int e0, int e1) {
    const int sn = jj / per;
    const uint4 *g = q.vrec + (size_t)((sn + p.ch0) % p.n_ch) * 2 * p.n_bl + e0;
    for (int i = tid; i < e1 - e0; i += kWThreads)
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(recs + i)), "l"(g + i) : "memory");
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  if (role_a && j_first < total) {
    if (tid <= kWWarps) {
      s_off[tid] = load_off(j_first);
      if (j_first + G < total) s_off[12 + tid] = load_off(j_first + G);
    }
    __syncthreads();
    fetch_recs(j_first, s_off[0], s_off[kWWarps]);
  }
  bool dep_ok = false;                   // the item's ring slot is known to be free (checked at the previous item's end)
  int n_it = 0;
  for (int j = j_first; j < total; j += G, ++n_it) {
    WItem cur, nxt;
    cur.kind = role_a ? 0 : 1; cur.snap = j / per; cur.idx = j - cur.snap * per;
    nxt.kind = j + G < total ? cur.kind : -1; nxt.snap = (j + G) / per; nxt.idx = (j + G) - nxt.snap * per;
    const int s = cur.snap, ch = (s + p.ch0) % p.n_ch;
    cf32 t[32];
    if (cur.kind == 0) {
      // ------------------------------------------------------------------ pass A, 8 columns
      const int kx0 = cur.idx * kWWarps;
      bool nonzero = true;
      if (!dep_ok && tid == 0 && s >= q.ring) {   // the slot's previous snapshot must have been read completely
        const int *d = q.done_b + (s - q.ring);
        while (ld_acquire(d) < kWItemsB * kWWarps) __nanosleep(100);
      }
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      __syncthreads();                     // the item's records have landed
      {
        const int32_t *off = s_off + 12 * (n_it % 3);
        const int e0 = off[0], e1 = off[kWWarps];
        int voff = 0;                      // offsets of the item after next, in flight during this item
        if (tid <= kWWarps && j + 2 * G < total) voff = load_off(j + 2 * G);
        {   // cell values: sum of the cell's visibilities in ascending baseline order, weighted, placed.
            // One 16-byte record per cell: iy | flag << 16 | len << 18, weight, first source code,
            // second source code (len = 2) or the cell's segment in src (len > 2)
          const float2 *__restrict__ vis = p.vis + (size_t)(p.snap_base + s) * p.n_bl;
          if (q.uvsrc == nullptr && cur.idx == 0 && tid == 0 && s + 2 < q.n_snap && (p.n_bl & 1) == 0) {
            // the visibilities of a snapshot two rounds ahead: into L2 before their pass A needs them
            const float2 *nv = vis + (size_t)2 * p.n_bl;
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nv), "r"((uint32_t)(p.n_bl * sizeof(float2))) : "memory");
          }
          const int32_t *__restrict__ src = p.src + (size_t)ch * p.n_bl;
          const float2 *__restrict__ cf = p.corr ? p.corr + (size_t)ch * p.n_bl : nullptr;
          if (q.uvsrc != nullptr) {
            // blink_image: the occupied cells of the item's 8 columns straight from the uv grid (the
            // half-plane kx >= 0 only; empty cells are zero by contract and never read)
            const float2 *__restrict__ g = q.uvsrc + (size_t)(p.snap_base + s) * N * N + kx0;
            for (int e = e0 + tid; e < e1; e += kWThreads) {
              const uint4 r = recs[e - e0];
              const int iy = (int)(r.x & 0xffff), flag = (r.x >> 16) & 3;
              int c = 0;
              while (e >= off[c + 1]) ++c;
              const float w = __uint_as_float(r.y);
              const float2 v = __ldg(g + (size_t)iy * N + c);
              cv[e - e0] = mk(v.x * w, (flag == kPlaceDirect || flag == kPlaceConj) ? v.y * w : 0.f);
              ck[e - e0] = iy;
            }
          } else
          for (int e = e0 + tid; e < e1; e += kWThreads) {
            const uint4 r = recs[e - e0];
            const int flag = (r.x >> 16) & 3, len = (int)(r.x >> 18);
            const float w = __uint_as_float(r.y);
            const float2 v0 = ld_vis(vis, cf, r.z >> 1);
            float2 v1 = make_float2(0.f, 0.f);
            if (len == 2) v1 = ld_vis(vis, cf, r.w >> 1);
            float ar = v0.x, ai = (r.z & 1) ? -v0.y : v0.y;
            if (len == 2) {
              ar += v1.x;
              ai += (r.w & 1) ? -v1.y : v1.y;
            } else if (len > 2) {
              for (int qq = (int)r.w + 1; qq < (int)r.w + len; ++qq) {
                const int code = __ldg(src + qq);
                const float2 v = ld_vis(vis, cf, code >> 1);
                ar += v.x;
                ai += (code & 1) ? -v.y : v.y;
              }
            }
            cf32 o;
            if (flag == kPlaceDirect) o = mk(ar * w, ai * w);
            else if (flag == kPlaceConj) o = mk(ar * w, -ai * w);
            else o = mk((ar + ar) * w, 0.f);
            cv[e - e0] = o;
            ck[e - e0] = (int)(r.x & 0xffff);
          }
        }
        __syncthreads();
        if (nxt.kind == 0) {               // the record buffer is free: start the next item's copy
          const int32_t *noff = s_off + 12 * ((n_it + 1) % 3);
          fetch_recs(j + G, noff[0], noff[kWWarps]);
        }
        if (tid <= kWWarps) s_off[12 * ((n_it + 2) % 3) + tid] = voff;
        // sparse inner step, lane = y1
        const int c0 = off[wv] - e0, c1 = off[wv + 1] - e0;
        unsigned mask = 0;
        int bcur = -1;
        cf32 acc = mk(0.f, 0.f);
        for (int i = c0; i < c1; ++i) {
          const cf32 v = cv[i];
          const int iy = ck[i], b = iy & 31, a = iy >> 5;
          if (b != bcur) {
            if (bcur >= 0) {
              tile[bcur * kWfRow + lane] = cmul(acc, tws[bcur * 32 + lane]);
              mask |= 1u << bcur;
            }
            bcur = b;
            acc = mk(0.f, 0.f);
          }
          const cf32 w = w32[(a * lane) & 31];
          acc.x = fmaf(v.x, w.x, fmaf(-v.y, w.y, acc.x));
          acc.y = fmaf(v.x, w.y, fmaf(v.y, w.x, acc.y));
        }
        if (bcur >= 0) {
          tile[bcur * kWfRow + lane] = cmul(acc, tws[bcur * 32 + lane]);
          mask |= 1u << bcur;
        }
        __syncwarp();
        nonzero = mask != 0;
        if (nonzero) wf_get_masked(tile, lane, mask, t);
      }
      // outer step: t[b] -> U[lane + 32 y2] of this warp's column
      if (nonzero) {
        dft32(t);
      } else {
#pragma unroll
        for (int i = 0; i < 32; ++i) t[i] = mk(0.f, 0.f);
      }
      __syncthreads();                   // every warp has read its exchange tile: the region becomes the out tile
#pragma unroll
      for (int y2 = 0; y2 < 32; ++y2) region[(lane + 32 * y2) * kWOStride + wv] = t[y2];
      __syncthreads();
      float2 *__restrict__ U = p.U + (size_t)(s % q.ring) * N * p.wu + kx0;
      for (int idx = tid; idx < kWWarps * N; idx += kWThreads) {
        const int cc = idx & 7, y = idx >> 3;
        U[(size_t)y * p.wu + cc] = region[y * kWOStride + cc];
      }
      __syncthreads();
      if (tid == 0) {
        __threadfence();
        atomicAdd(q.done_a + s, 1);
        // the next item's slot.  Only AFTER this item has been signalled: with a short ring the
        // snapshot whose pass B frees that slot can be the very one this item belongs to.
        if (nxt.kind == 0 && nxt.snap >= q.ring) {
          const int *d = q.done_b + (nxt.snap - q.ring);
          while (ld_acquire(d) < kWItemsB * kWWarps) __nanosleep(100);
        }
      }
      dep_ok = true;                       // the other threads learn it at the next item's first barrier
      pending = false;
    } else {
      // ------------------------------------------------------------------ pass B, 8 row pairs
      const int wu = p.wu;
      if (!pending) {
        if (lane == 0) {
          const int *d = q.done_a + s;
          while (ld_acquire(d) < q.items_a) __nanosleep(100);
          issue_rows(q, cur, wv, tile, bar);
        }
      }
      mbar_wait(bar, parity);
      parity ^= 1u;
      // lane b holds Z[32 a + b]: a < 16 is the direct half (Z = A + i B), a >= 16 the mirrored half
      // (Z[k] = conj A[N-k] + i conj B[N-k]); columns at or beyond wu are zero
#pragma unroll
      for (int a = 0; a < 16; ++a) {
        const int kk = 32 * a + lane;
        const bool ok = kk < wu;
        const cf32 A = ok ? tile[kk] : mk(0.f, 0.f);
        const cf32 B = ok ? tile[wu + kk] : mk(0.f, 0.f);
        t[a] = mk(A.x - B.y, A.y + B.x);
      }
#pragma unroll
      for (int a = 16; a < 32; ++a) {
        const int m = N - 32 * a - lane;
        const bool ok = m < wu;
        const cf32 A = ok ? tile[m] : mk(0.f, 0.f);
        const cf32 B = ok ? tile[wu + m] : mk(0.f, 0.f);
        t[a] = mk(A.x + B.y, B.x - A.y);
      }
      __syncwarp();
      // this warp's share of the snapshot's U has been consumed: the bulk copies have completed (the
      // mbarrier said so) and the values are in registers, so a relaxed add is enough to let the slot go
      if (lane == 0) atomicAdd(q.done_b + s, 1);
      // the next item's pass-A counter: a relaxed load issued now, its round trip to L2 hidden behind the
      // inner butterflies; the acquire fence follows only if the count says the rows are there
      int cnt_next = 0;
      if (nxt.kind == 1 && lane == 0) cnt_next = ld_relaxed(q.done_a + nxt.snap);
      wf_inner(t, lane, [&](int i) { return tws[i]; });
      wf_put(tile, lane, t);
      __syncwarp();
      wf_get(tile, lane, t);
      __syncwarp();
      pending = false;
      if (nxt.kind == 1) {               // rows of the next item, if its pass A is already complete
        int ready = 0;
        if (lane == 0) {
          ready = cnt_next >= q.items_a;
          if (ready) {
            fence_acq_rel_gpu();
            issue_rows(q, nxt, wv, tile, bar);
          }
        }
        pending = __shfl_sync(0xffffffffu, ready, 0) != 0;
      }
      dft32(t);
      float *__restrict__ r0 = p.img + ((size_t)(p.snap_base + s) * N + cur.idx * kWWarps + wv) * N + lane;
      float *__restrict__ r1 = r0 + (size_t)(N / 2) * N;
#pragma unroll
      for (int n2 = 0; n2 < 32; ++n2) {
        __stcs(r0 + 32 * n2, t[n2].x);
        __stcs(r1 + 32 * n2, t[n2].y);
      }
    }
  }
  // The last CTA to get here clears the counters, so the next launch finds them zero without a memset:
  // a CTA takes its ticket after its last counter access, so once all tickets are out nobody reads or
  // bumps a counter any more.
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    s_off[47] = atomicAdd(q.finished, 1) == (int)gridDim.x - 1;     // s_off[36..47] are spare
  }
  __syncthreads();
  if (s_off[47]) {
    __threadfence();
    for (int i = tid; i < q.n_snap; i += kWThreads) {
      q.done_a[i] = 0;
      q.done_b[i] = 0;
    }
    if (tid == 0) *q.finished = 0;
  }
}

static int w_grid(const blink_plan *p) {
  int per_sm = 2;
  if (p->opt.tune[kTuneWarpCtasPerSm] > 0) per_sm = std::max(1, std::min(2, (int)p->opt.tune[kTuneWarpCtasPerSm]));
  return std::max(2, per_sm * p->sm_count);
}
static int w_ring(const blink_plan *p) {
  // slots of U between the two groups: enough that pass A rarely waits for pass B, small enough to
  // stay in L2 (default 32 MB at wu = 512)
  const size_t per_snap = sizeof(float2) * (size_t)p->n_pix * p->wu;
  int ring = (int)std::max<size_t>(4, std::min<size_t>(64, ((size_t)32 << 20) / per_snap));
  if (p->opt.warp_ring >= 2) ring = p->opt.warp_ring;
  return ring;
}

// scratch: ring of U slots, then the counters (finished + padding [64], done_a[n_snap], done_b[n_snap])
size_t warp_route_ring_bytes(const blink_plan *p) {
  return sizeof(float2) * (size_t)p->n_pix * p->wu * (size_t)w_ring(p);
}
size_t warp_route_scratch_bytes(const blink_plan *p, long long n_snap) {
  return warp_route_ring_bytes(p) + sizeof(int) * (size_t)(2 * n_snap + 64);
}

int launch_img1024(const blink_plan *p, ImgParams ip, int n_snap, cudaStream_t st) {
  if (n_snap <= 0) return BLINK_OK;
  const int grid = w_grid(p);
  WParams q;
  q.n_snap = n_snap;
  q.items_a = p->wu / kWWarps;
  q.ring = w_ring(p);
  {   // split of the grid between the passes (measured on MWA Phase I: pass A needs the larger share)
    double fa = 0.6;
    if (p->opt.tune[kTuneWarpFracA] > 0) fa = std::min(0.9, std::max(0.1, 0.01 * p->opt.tune[kTuneWarpFracA]));
    q.g_a = std::min(grid - 1, std::max(1, (int)(fa * grid + 0.5)));
  }
  const size_t ring_bytes = warp_route_ring_bytes(p);
  if (warp_route_scratch_bytes(p, n_snap) > p->scratch_bytes || n_snap > p->warp_snap_cap) return BLINK_ERESERVE;
  int *cnt = reinterpret_cast<int *>(reinterpret_cast<unsigned char *>(p->d_scratch) + ring_bytes);
  q.finished = cnt;
  q.done_a = cnt + 64;
  q.done_b = cnt + 64 + n_snap;
  q.vrec = p->d_vrec;
  q.uvsrc = ip.vis == nullptr ? ip.uv : nullptr;
  ip.snap_base = 0;
  ip.U = p->d_scratch;
  q.ip = ip;
  // on top of the fixed part: cell values + their iy, the record buffer, the offsets ring
  const size_t smem = kWFixedBytes + (size_t)ip.cell_cap * (sizeof(cf32) + sizeof(int32_t) + sizeof(uint4)) + 48 * sizeof(int32_t);
  if (p->max_smem_optin > 0 && smem > (size_t)p->max_smem_optin) return BLINK_EUNSUPPORTED;
  static std::atomic<uint64_t> attr{0};
  const int rc = ensure_max_smem(k_img1024, p, attr, "k_img1024 smem attribute");
  if (rc != BLINK_OK) return rc;
  void *args[] = {(void *)&q};
  // cooperative: the item sequences are dealt statically, so every CTA of the grid must be resident
  const cudaError_t le = cudaLaunchCooperativeKernel((const void *)k_img1024, dim3(grid), dim3(kWThreads), args, smem, st);
  if (le != cudaSuccess) {
    // the kernel is the only thing that returns its counters to zero; after a launch that did not go
    // through, put them back on this stream so the next call does not start from whatever they hold
    set_cuda_error(le, "k_img1024 launch");
    cudaMemsetAsync(cnt, 0, p->scratch_bytes - ring_bytes, st);
    cudaGetLastError();
    return BLINK_ECUDA;
  }
  return BLINK_OK;
}

// the route pays when the half-plane is wide and sparsely filled (MWA-like arrays); compact arrays
// (a station imaged at 1024^2: 48 columns holding 100 cells each) stay on the line kernels
bool warp_route_applies(const blink_plan *p) {
  if (p->n_pix != kWN || p->wu < 256 || p->wu % kWWarps) return false;
  if (p->seg_len_max > 0x3FFF) return false;          // the cell records carry the segment length in 14 bits
  const size_t smem = kWFixedBytes + (size_t)((p->vtile8_max + 3) / 4 * 4) * (sizeof(cf32) + sizeof(int32_t) + sizeof(uint4)) + 48 * sizeof(int32_t);
  return 2 * (smem + 1024) <= (size_t)228 * 1024 && (p->max_smem_optin <= 0 || smem <= (size_t)p->max_smem_optin);
}

}  // namespace blink
