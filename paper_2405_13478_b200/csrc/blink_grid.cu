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
#include <cstdio>

#include "blink_internal.h"
#include "sgather.cuh"
#include "sphase.cuh"

namespace blink {

struct GridParams {
  const float2 *vis;
  const float2 *corr;          // [n_ch][n_bl] correction factors applied as the visibilities are loaded, or NULL
  float2 *uv;
  const ChannelInfo *chinfo;
  const uint16_t *scat, *roff;
  const uint32_t *cellrec;
  const int32_t *nact;
  const int32_t *pcell, *pcode, *pband;
  int n_bl, n_ch, n_snap, n_bands, band_cells, parts, n_can_max, n_pass, roff_stride, ch0;
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
    const int ch = (s + p.ch0) % p.n_ch;
    pass_load<THREADS, PF>(regs, p.vis + (size_t)s * p.n_bl, p.scat + (size_t)ch * p.n_bl, 0, min(CAP, p.n_bl), tid,
                           p.corr ? p.corr + (size_t)ch * p.n_bl : nullptr);
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
    if (tid == 0) {
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
      pass_scatter<PF>(regs, stage);
      __syncthreads();
      // loads of the next pass (or of the next item's first pass) fly during the sums and phase P
      if (pass + 1 < p.n_pass) {
        const int b0 = (pass + 1) * CAP;
        pass_load<THREADS, PF>(regs, vis, scat, b0, min(CAP, p.n_bl - b0), tid, p.corr ? p.corr + (size_t)ch * p.n_bl : nullptr);
      } else if (item + gridDim.x < n_items) {
        const int s2 = (int)((item + gridDim.x) / p.parts);
        const int ch2 = (s2 + p.ch0) % p.n_ch;
        pass_load<THREADS, PF>(regs, p.vis + (size_t)s2 * p.n_bl, p.scat + (size_t)ch2 * p.n_bl, 0, min(CAP, p.n_bl), tid,
                               p.corr ? p.corr + (size_t)ch2 * p.n_bl : nullptr);
      }
      sums_run<THREADS>(sr, cellrec, p.roff + cp * p.roff_stride, p.n_can_max, stage, S, tid);
      if (pass + 1 == p.n_pass && tid == 0) bulk_wait_all();   // the zero fill has landed
      __syncthreads();
    }

    // ---- phase P, second half: occupied cells on top of the zeros -----------------------------
    const int32_t *__restrict__ pband = p.pband + (size_t)ch * (p.n_bands + 1);
    const int32_t *__restrict__ pcell = p.pcell + (size_t)ch * 2 * p.n_bl;
    const int32_t *__restrict__ pcode = p.pcode + (size_t)ch * 2 * p.n_bl;
    const int e0 = pband[b_lo], e1 = pband[b_hi];
    for (int e = e0 + tid; e < e1; e += THREADS) {
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


// ---------------------------------------------------------------------------------------------
// Ring route (small grids, many snapshots): phase S as in k_fused (blink_fused.cu, sgather.cuh) --
// the snapshot's visibilities stream through a ring of shared-memory buffers by bulk copies, each
// chunk with its gather table; cells are owned by warps, sums need no atomics and no barrier between
// chunks -- and because nothing else needs the shared memory here, the ring runs ahead across
// snapshots without ever draining.  Phase P as above: bulk zero fill, then the occupied cells.
static int ring_upload(void **dst, const void *src, size_t bytes, cudaStream_t st) {
  cudaError_t e = cudaMalloc(dst, std::max<size_t>(bytes, 16));
  if (e != cudaSuccess) {
    set_cuda_error(e, "ring table cudaMalloc");
    *dst = nullptr;
    return e == cudaErrorMemoryAllocation ? BLINK_ENOMEM : BLINK_ECUDA;
  }
  BLINK_CUDA_TRY(cudaMemcpyAsync(*dst, src, bytes, cudaMemcpyHostToDevice, st), "ring table upload");
  return BLINK_OK;
}

struct GridRingParams {
  const float2 *vis;
  const float2 *corr;          // CORR: [n_ch][n_bl] correction factors
  float2 *uv;
  const ChannelInfo *chinfo;
  const unsigned char *rtab;   // [n_ch][n_chunk][tab_stride]
  const uint32_t *rsize;       // [n_ch][n_chunk]
  const int2 *rplace;          // [n_ch][2 n_bl] {cell, slot | flag << 30}
  int n_bl, n_ch, n_snap, n_can_max, n_chunk, chunk_vis, nbuf, tab_stride, n_bands, band_cells, ch0;
  uint32_t buf_bytes, off_buf, off_S, off_bar, tab_off, f_off;
  long long grid_cells;
};

constexpr int kRingPlacePf = 10;   // placement records fetched per thread ahead of the barrier

template <bool CORR>
__global__ void __launch_bounds__(kFusedThreads, 1) k_grid_ring(const GridRingParams p) {
  constexpr int THREADS = kFusedThreads;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float2 *zero = reinterpret_cast<float2 *>(smem_raw);                        // [band_cells]
  float2 *S = reinterpret_cast<float2 *>(smem_raw + p.off_S);
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + p.off_bar);
  uint64_t *empty = full + p.nbuf;
  const uint32_t sm_base = smem_u32(smem_raw), S_base = sm_base + p.off_S;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t vis_bytes = p.tab_off;
  const uint32_t band_bytes = (uint32_t)p.band_cells * sizeof(float2);
  const int n_S = ((p.n_can_max + 15) & ~15) + 16;

  if constexpr (CORR) {
    // the 16 "zero visibility" slots behind chunk buffer 0's visibilities, and their factor partners
    float2 *z = reinterpret_cast<float2 *>(smem_raw + p.off_buf) + p.chunk_vis;
    if (tid < 16) z[tid] = make_float2(0.f, 0.f);
    else if (tid < 32) reinterpret_cast<float2 *>(reinterpret_cast<unsigned char *>(z) + p.f_off)[tid - 16] = make_float2(0.f, 0.f);
  }
  if (tid == 0) {
    for (int b = 0; b < p.nbuf; ++b) {
      mbar_init(full + b, 1);
      mbar_init(empty + b, kFusedWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  {
    float4 *z4 = reinterpret_cast<float4 *>(smem_raw);
    for (int i = tid; i < p.band_cells / 2; i += THREADS) z4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  for (int j = tid; j < n_S; j += THREADS) S[j] = make_float2(0.f, 0.f);
  fence_async_smem();
  __syncthreads();

  // this CTA's snapshots: s = blockIdx.x + k gridDim.x, k < K; their chunks form one sequence q
  const int K = (p.n_snap - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
  const int Q = K * p.n_chunk;
  uint32_t fphase = 0, ephase = 0;
  int pq = 0, pk = 0, pc = 0, pb = 0;        // producer (thread 0): next chunk to request
  auto produce = [&]() {
    mbar_wait(empty + pb, ((ephase >> pb) & 1u) ^ 1u);
    ephase ^= 1u << pb;
    const int s = (int)blockIdx.x + pk * (int)gridDim.x;
    const int cnt = min(p.chunk_vis, p.n_bl - pc * p.chunk_vis);
    const uint32_t vb = (uint32_t)cnt * sizeof(float2);
    const size_t cp = (size_t)((s + p.ch0) % p.n_ch) * p.n_chunk + pc;
    const uint32_t tb = __ldg(p.rsize + cp);
    unsigned char *dst = smem_raw + p.off_buf + (size_t)pb * p.buf_bytes;
    mbar_expect_tx(full + pb, (CORR ? 2 * vb : vb) + tb);
    bulk_load(dst, p.vis + (size_t)s * p.n_bl + (size_t)pc * p.chunk_vis, vb, full + pb);
    bulk_load(dst + vis_bytes, p.rtab + cp * p.tab_stride, tb, full + pb);
    if constexpr (CORR)
      bulk_load(dst + p.f_off, p.corr + (size_t)((s + p.ch0) % p.n_ch) * p.n_bl + (size_t)pc * p.chunk_vis, vb, full + pb);
    ++pq;
    if (++pc == p.n_chunk) { pc = 0; ++pk; }
    if (++pb == p.nbuf) pb = 0;
  };
  if (tid == 0)
    while (pq < min(p.nbuf, Q)) produce();

  int b = 0, q = 0;
  for (int k = 0; k < K; ++k) {
    const int s = (int)blockIdx.x + k * (int)gridDim.x;
    const int ch = (s + p.ch0) % p.n_ch;
    float2 *__restrict__ grid = p.uv + (size_t)s * p.grid_cells;
    // ---- phase P, first half: zero-fill the snapshot; drains while phase S runs ----------------
    if (tid == 0) {
      for (int bd = 0; bd < p.n_bands; ++bd) bulk_store(grid + (size_t)bd * p.band_cells, zero, band_bytes);
      bulk_commit();
    }
    const int n_place = p.chinfo[ch].n_place;
    const int2 *__restrict__ place = p.rplace + (size_t)ch * 2 * p.n_bl;
    int2 pr[kRingPlacePf];
#pragma unroll
    for (int i = 0; i < kRingPlacePf; ++i) {
      const int e = tid + i * THREADS;
      pr[i] = e < n_place ? __ldg(place + e) : make_int2(-1, 0);
    }
    // ---- phase S ----------------------------------------------------------------------------
    for (int c = 0; c < p.n_chunk; ++c, ++q) {
      mbar_wait(full + b, (fphase >> b) & 1u);
      fphase ^= 1u << b;
      consume_chunk<CORR>(sm_base + p.off_buf + (uint32_t)b * p.buf_bytes + vis_bytes, warp, lane, sm_base, S_base, p.f_off);
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + b);
      if (tid == 0 && pq < Q) produce();     // chunk q + nbuf into the buffer just released
      if (++b == p.nbuf) b = 0;
    }
    if (tid == 0) bulk_wait_all();            // the zero fill has landed
    __syncthreads();
    // ---- phase P, second half: occupied cells on top of the zeros -----------------------------
    auto put = [&](int2 r) {
      if (r.x < 0) return;
      const float2 v = S[r.y & 0x3FFFFFFF];
      const uint32_t flag = (uint32_t)r.y >> 30;
      float2 o;
      if (flag == kPlaceDirect) o = v;
      else if (flag == kPlaceConj) o = make_float2(v.x, -v.y);
      else o = make_float2(v.x + v.x, 0.f);
      grid[r.x] = o;
    };
#pragma unroll
    for (int i = 0; i < kRingPlacePf; ++i) put(pr[i]);
    for (int e = tid + kRingPlacePf * THREADS; e < n_place; e += THREADS) put(__ldg(place + e));
    __syncthreads();
    for (int j = tid; j < p.n_can_max; j += THREADS) S[j] = make_float2(0.f, 0.f);
    __syncthreads();
  }
}


// Shared-memory plan and tables of the ring route; corr = 1: every chunk carries its correction factors
// too (see fused_layout in blink_fused.cu for the buffer format).  Layout (bytes):
//   [0, band)               zero band (source of the bulk zero fill)
//   [off_first, +nbuf * B)  chunk buffers
//   [off_S, ...)            canonical cell sums + 16 zero slots
//   [off_bar, ...)          full[nbuf], empty[nbuf] mbarriers
// n_chunk is a multiple of nbuf, so chunk c of every snapshot lands in buffer c % nbuf and the ring
// never has to drain between snapshots.
int grid_ring_layout(blink_plan *p, int corr, cudaStream_t st) {
  GatherLayout &L = p->rl[corr];
  if (L.ok) return BLINK_OK;
  const int N = p->n_pix, n_bl = p->n_bl, n_ch = p->n_ch;
  if (p->opt.grid_ring == -1 || N > 512 || (n_bl & 1) || p->max_smem_optin <= 0 || p->n_can_max < 1 ||
      (int)p->gathers.size() != n_ch)
    return BLINK_OK;
  const int sink0 = (p->n_can_max + 15) & ~15, n_S = sink0 + 16;
  if (n_S > 0x7FFF) return BLINK_OK;
  const size_t band = (sizeof(float2) * (size_t)p->band_cells + 127) / 128 * 128;
  const size_t s_bytes = (sizeof(float2) * (size_t)n_S + 127) / 128 * 128;
  const size_t limit = (size_t)p->max_smem_optin;
  if (band + s_bytes + 1024 > limit) return BLINK_OK;
  const int zpad = corr ? 16 : 0;
  std::vector<std::vector<int>> owner(n_ch), slot(n_ch);
  for (int ch = 0; ch < n_ch; ++ch) assign_cells(p->gathers[ch], owner[ch], slot[ch]);

  std::vector<AbstractTable> tabs;
  int n_chunk = 0, C = 0, nbuf = 0;
  size_t tab_stride = 0, buf_bytes = 0;
  bool found = false;
  static const int kNbufOrder[3] = {3, 2, 4};
  for (int oi = 0; oi < 3 && !found; ++oi) {
    nbuf = kNbufOrder[oi];
    const size_t room = (limit - band - s_bytes - 16 * (size_t)nbuf - 64) / nbuf / 128 * 128;   // bytes per buffer
    for (n_chunk = nbuf; n_chunk <= 16 * nbuf && !found; n_chunk += nbuf) {
      C = (n_bl + n_chunk - 1) / n_chunk;
      C = (C + 1) & ~1;
      if (C > 0x7FFE || (n_bl + C - 1) / C != n_chunk) continue;
      const size_t data_bytes = sizeof(float2) * (size_t)(C + zpad) * (corr ? 2 : 1);
      if (data_bytes > room) continue;
      tabs.assign((size_t)n_ch * n_chunk, AbstractTable());
      std::atomic<bool> all_ok{true};
      parallel_for(n_ch * n_chunk, [&](int i) {
        if (!all_ok.load()) return;
        const int ch = i / n_chunk, c = i % n_chunk;
        bool ok = true;
        build_chunk_table(p->gathers[ch], owner[ch], slot[ch], c * C, std::min(n_bl, (c + 1) * C), sink0, tabs[i], ok);
        if (!ok) all_ok.store(false);
      });
      if (!all_ok.load()) continue;
      tab_stride = 0;
      for (const AbstractTable &t : tabs) tab_stride = std::max(tab_stride, t.bytes.size());
      buf_bytes = (data_bytes + tab_stride + 127) / 128 * 128;
      if (buf_bytes > room) continue;
      found = true;
      break;
    }
  }
  if (!found) return BLINK_OK;
  L.chunk_vis = C;
  L.n_chunk = n_chunk;
  L.nbuf = nbuf;
  L.tab_stride = (int)tab_stride;
  L.buf_bytes = (uint32_t)buf_bytes;
  L.off_first = (uint32_t)band;
  L.off_S = (uint32_t)(band + (size_t)nbuf * buf_bytes);
  L.off_bar = (uint32_t)(L.off_S + s_bytes);
  L.smem = L.off_bar + 16 * (size_t)nbuf + 16;
  L.tab_off = (uint32_t)(sizeof(float2) * (size_t)(C + zpad));
  L.f_off = corr ? (uint32_t)(L.tab_off + tab_stride) : 0u;
  if (L.smem > limit || L.smem > 0x7FFFu * 8u) return BLINK_OK;

  const uint32_t s_slot0 = L.off_S / 8;
  const uint32_t zslot0 = corr ? L.off_first / 8 + (uint32_t)C : s_slot0 + (uint32_t)sink0;
  std::vector<unsigned char> h_tab((size_t)n_ch * n_chunk * tab_stride, 0);
  std::vector<uint32_t> h_size((size_t)n_ch * n_chunk, 0);
  for (int ch = 0; ch < n_ch; ++ch)
    for (int c = 0; c < n_chunk; ++c) {
      const size_t cp = (size_t)ch * n_chunk + c;
      std::vector<unsigned char> &b = tabs[cp].bytes;
      finalize_chunk_table(b, (uint32_t)((L.off_first + (size_t)(c % nbuf) * buf_bytes) / 8), zslot0);
      std::memcpy(h_tab.data() + cp * tab_stride, b.data(), b.size());
      h_size[cp] = (uint32_t)b.size();
    }
  int rc;
  if ((rc = ring_upload((void **)&L.d_tab, h_tab.data(), h_tab.size(), st)) != BLINK_OK) return rc;
  if ((rc = ring_upload((void **)&L.d_size, h_size.data(), sizeof(uint32_t) * h_size.size(), st)) != BLINK_OK) return rc;
  BLINK_CUDA_TRY(cudaStreamSynchronize(st), "ring table upload sync");
  L.ok = true;
  return BLINK_OK;
}

int grid_ring_build(blink_plan *p, cudaStream_t st) {
  p->ring_path = 0;
  int rc = grid_ring_layout(p, 0, st);
  if (rc != BLINK_OK) return rc;
  if (!p->rl[0].ok) return BLINK_OK;
  const int N = p->n_pix, n_bl = p->n_bl, n_ch = p->n_ch;
  std::vector<std::vector<int>> owner(n_ch), slot(n_ch);
  for (int ch = 0; ch < n_ch; ++ch) assign_cells(p->gathers[ch], owner[ch], slot[ch]);
  // placement records: every canonical cell and its mirror, ascending cell index (coalesced-ish stores)
  std::vector<int2> h_place((size_t)n_ch * 2 * n_bl, make_int2(-1, 0));
  for (int ch = 0; ch < n_ch; ++ch) {
    const HostGather &g = p->gathers[ch];
    std::vector<std::pair<int32_t, int32_t>> pl;
    pl.reserve(2 * (size_t)g.n_can);
    for (int j = 0; j < g.n_can; ++j) {
      const int c = g.can_cell[j], ix = c % N, iy = c / N;
      const int cc = ((N - iy) % N) * N + ((N - ix) % N);
      if (cc == c) {
        pl.push_back({c, slot[ch][j] | (int32_t)((uint32_t)kPlaceBoth << 30)});
      } else {
        pl.push_back({c, slot[ch][j] | (int32_t)((uint32_t)kPlaceDirect << 30)});
        pl.push_back({cc, slot[ch][j] | (int32_t)((uint32_t)kPlaceConj << 30)});
      }
    }
    std::sort(pl.begin(), pl.end());
    for (size_t k = 0; k < pl.size(); ++k) h_place[(size_t)ch * 2 * n_bl + k] = make_int2(pl[k].first, pl[k].second);
  }
  if ((rc = ring_upload((void **)&p->d_rplace, h_place.data(), sizeof(int2) * h_place.size(), st)) != BLINK_OK) return rc;
  BLINK_CUDA_TRY(cudaStreamSynchronize(st), "ring table upload sync");
  p->ring_min_snap = p->opt.grid_ring_min_snap > 0 ? p->opt.grid_ring_min_snap : p->sm_count;
  p->ring_path = 1;
  return BLINK_OK;
}

template <bool CORR>
static int launch_grid_ring(const blink_plan *p, const float2 *vis, int n_snap, int ch0, float2 *uv, cudaStream_t st) {
  const GatherLayout &L = p->rl[CORR ? 1 : 0];
  GridRingParams g;
  g.vis = vis; g.corr = CORR ? p->d_corr : nullptr; g.uv = uv; g.chinfo = p->d_chinfo;
  g.rtab = L.d_tab; g.rsize = L.d_size; g.rplace = p->d_rplace;
  g.n_bl = p->n_bl; g.n_ch = p->n_ch; g.n_snap = n_snap; g.n_can_max = p->n_can_max; g.n_chunk = L.n_chunk;
  g.chunk_vis = L.chunk_vis; g.nbuf = L.nbuf; g.tab_stride = L.tab_stride; g.n_bands = p->n_bands;
  g.band_cells = p->band_cells; g.ch0 = ch0; g.buf_bytes = L.buf_bytes; g.off_buf = L.off_first;
  g.off_S = L.off_S; g.off_bar = L.off_bar; g.tab_off = L.tab_off; g.f_off = L.f_off;
  g.grid_cells = (long long)p->n_pix * p->n_pix;
  static std::atomic<uint64_t> attr{0};
  const int rc = ensure_max_smem(k_grid_ring<CORR>, p, attr, "k_grid_ring smem attribute");
  if (rc != BLINK_OK) return rc;
  const int blocks = std::min(n_snap, p->sm_count);
  k_grid_ring<CORR><<<blocks, kFusedThreads, L.smem, st>>>(g);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_grid_ring launch");
  return BLINK_OK;
}

template <int THREADS, int PF, int MINB>
static int launch_grid_v(const blink_plan *p, const GridParams &g0, cudaStream_t st) {
  GridParams g = g0;
  const size_t smem = p->grid_smem;
  if (smem > (size_t)p->max_smem_optin) return BLINK_EUNSUPPORTED;
  static std::atomic<uint64_t> attr{0};
  const int rc = ensure_max_smem(k_grid<THREADS, PF, MINB>, p, attr, "k_grid smem attribute");
  if (rc != BLINK_OK) return rc;
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
  // many snapshots of a small grid: the ring route; few snapshots (or large grids): the band route,
  // which can split one snapshot over several CTAs
  // (the ring route reads the visibilities with bulk copies: 16-byte aligned base)
  if (p->ring_path == 1 && n_snap >= p->ring_min_snap && ((uintptr_t)vis & 15) == 0 && p->rl[p->corr_on ? 1 : 0].ok)
    return p->corr_on ? launch_grid_ring<true>(p, vis, n_snap, ch0, uv, st) : launch_grid_ring<false>(p, vis, n_snap, ch0, uv, st);
  GridParams g;
  g.vis = vis; g.corr = p->corr_on ? p->d_corr : nullptr; g.uv = uv; g.chinfo = p->d_chinfo;
  g.scat = p->d_scat; g.roff = p->d_roff; g.cellrec = p->d_cellrec; g.nact = p->d_nact; g.pcell = p->d_pcell; g.pcode = p->d_pcode; g.pband = p->d_pband;
  g.n_bl = p->n_bl; g.n_ch = p->n_ch; g.n_snap = n_snap; g.ch0 = ch0;
  g.n_bands = p->n_bands; g.band_cells = p->band_cells; g.n_can_max = p->n_can_max;
  g.n_pass = p->n_pass; g.roff_stride = p->roff_stride; g.parts = 1;
  g.grid_cells = (long long)p->n_pix * p->n_pix;
  return launch_grid_v<512, 16, 1>(p, g, st);
}

}  // namespace blink

extern "C" int blink_grid(const blink_plan *plan, const void *vis, int n_t, void *uv_grid, void *stream) {
  if (!plan || n_t < 0) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!vis || !uv_grid) return BLINK_EINVAL;
  if (((uintptr_t)vis & 7) || ((uintptr_t)uv_grid & 15)) return BLINK_EINVAL;
  int rc = check_device(plan);
  if (rc == BLINK_OK) rc = check_corrections_current(plan);
  if (rc != BLINK_OK) return rc;
  return blink::launch_grid(plan, (const float2 *)vis, n_t * plan->n_ch, 0, (float2 *)uv_grid, (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------------------
// blink_grid_validate: the input contract of blink_image checked cell by cell (see blink.h).
namespace blink {
__global__ void __launch_bounds__(256) k_grid_validate(const float2 *__restrict__ uv, const uint32_t *__restrict__ counts,
                                                       int N, int n_ch, long long n_cells_total,
                                                       unsigned long long *__restrict__ n_bad) {
  const long long NN = (long long)N * N;
  unsigned long long bad = 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_cells_total;
       i += (long long)gridDim.x * blockDim.x) {
    const long long s = i / NN;
    const int c = (int)(i - s * NN), iy = c / N, ix = c - iy * N;
    const int cm = ((N - iy) & (N - 1)) * N + ((N - ix) & (N - 1));
    const float2 g = uv[i], m = uv[s * NN + cm];
    const uint32_t cnt = counts[(size_t)(s % n_ch) * NN + c];
    const bool nonplan = cnt == 0 && !(g.x == 0.f && g.y == 0.f);
    const bool nonherm = !(g.x == m.x && g.y == -m.y);
    bad += (nonplan || nonherm) ? 1u : 0u;
  }
  for (int o = 16; o > 0; o >>= 1) bad += __shfl_down_sync(0xffffffffu, bad, o);
  if ((threadIdx.x & 31) == 0 && bad) atomicAdd(n_bad, bad);
}
}  // namespace blink

extern "C" int blink_grid_validate(const blink_plan *plan, const void *uv_grid, int n_t, int64_t *n_violations,
                                   void *stream) {
  if (!plan || n_t < 0 || !n_violations) return BLINK_EINVAL;
  *n_violations = 0;
  if (n_t == 0) return BLINK_OK;
  if (!uv_grid || ((uintptr_t)uv_grid & 7)) return BLINK_EINVAL;
  const int rc = check_device(plan);
  if (rc != BLINK_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  unsigned long long *d_bad = nullptr, h_bad = 0;
  BLINK_CUDA_TRY(cudaMalloc((void **)&d_bad, sizeof(*d_bad)), "blink_grid_validate cudaMalloc");
  const long long total = (long long)n_t * plan->n_ch * plan->n_pix * plan->n_pix;
  cudaError_t e = cudaMemsetAsync(d_bad, 0, sizeof(*d_bad), st);
  if (e == cudaSuccess) {
    blink::k_grid_validate<<<plan->sm_count * 8, 256, 0, st>>>((const float2 *)uv_grid, plan->d_counts, plan->n_pix, plan->n_ch,
                                                                total, d_bad);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h_bad, d_bad, sizeof(h_bad), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d_bad);
  if (e != cudaSuccess) {
    blink::set_cuda_error(e, "blink_grid_validate");
    return BLINK_ECUDA;
  }
  *n_violations = (int64_t)h_bad;
  return BLINK_OK;
}
