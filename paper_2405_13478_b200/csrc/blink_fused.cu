// blink_fused.cu -- blink_grid_image: steps a1-a5 in one call.
//
// Chunked route: the batch is cut into chunks of a few snapshots; each chunk is gridded into a
// small plan-owned uv scratch and imaged from it straight away, so the uv grids are written and
// read back while still resident in the 126 MB L2 and (ideally) never reach HBM: the DRAM traffic
// of a snapshot falls from 8 n_bl + 20 N^2 towards 8 n_bl + 4 N^2 bytes.
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdio>
#include <cstring>

// complex adds as packed fp32 pairs (fft_core.cuh, SASS FADD2) here too: pass B is issue-bound (42 % of
// the kernel's instructions, a warp ready and another one issuing a third of the time), and the packed
// form halves its adds -- station 0.403 -> 0.393 ms, sweep512 1.31 -> 1.25 ms.  (Round 1 measured the
// opposite, 0.419 -> 0.427 ms, when phase S still dominated the kernel.)  Phase S adds packed as well
// (sgather.cuh): 0.393 -> 0.392 ms.
#define BLINK_PHASE_S_PACKED
#include "blink_internal.h"
#include "fft_core.cuh"
#include "sgather.cuh"
#include "sphase.cuh"

#include "fused_kernel.cuh"

namespace blink {
using namespace blinkfft;

int fused_line_stride(int n_pix) { return ((n_pix + n_pix / 16 + 15) / 16) * 16 + 1; }

// the polyphase instances with D = 4 live in blink_fused_d4.cu (scalar complex adds)
int launch_fused_d4(const blink_plan *p, const FusedParams &fp, int nz, cudaStream_t st);

int fused_setup(blink_plan *p) {
  p->fused_path = 0;
  p->fused_chunk = p->chunk_snapshots;   // the two-kernel route chunks like blink_image
  return BLINK_OK;
}

int upload_table(void **dst, const void *src, size_t bytes, cudaStream_t st, const char *what) {
  cudaError_t e = cudaMalloc(dst, std::max<size_t>(bytes, 16));
  if (e != cudaSuccess) {
    set_cuda_error(e, what);
    *dst = nullptr;
    return e == cudaErrorMemoryAllocation ? BLINK_ENOMEM : BLINK_ECUDA;
  }
  BLINK_CUDA_TRY(cudaMemcpyAsync(*dst, src, bytes, cudaMemcpyHostToDevice, st), what);
  return BLINK_OK;
}

// Geometry of the shared-memory route, common to its table layouts.  The route applies to two-stage
// transforms (N <= 256 directly, 512 / 1024 as D x D sub-images of 256) whose bounding box fits, with
// 16-byte aligned snapshots (even n_bl) for the bulk copies.
struct FusedGeom {
  int Ns, D, sink0, n_S, LS, n_col;
  size_t region, region_al, s_bytes;
};

static bool fused_geom(const blink_plan *p, FusedGeom &g) {
  const int N = p->n_pix;
  if (p->opt.fused_route == -1 || N < 32 || (p->n_bl & 1) || p->max_smem_optin <= 0) return false;
  // polyphase route (see k_fused): a compact array on a large image is imaged as D x D interleaved
  // Ns x Ns sub-images, Ns = 256, when the bounding box fits the Ns transform
  g.Ns = N;
  g.D = 1;
  if (N > 256) {
    // (128-point sub-transforms were measured too: station 256^2 as 2 x 2 of 128^2 0.65 ms against
    // 0.42 ms direct, sweep512 as 4 x 4 1.92 ms against 1.36 ms as 2 x 2 of 256^2)
    g.Ns = 256;
    g.D = N / g.Ns;
    if (p->opt.polyphase == -1 || g.D > 4 || std::max(p->kx_max_all, p->ky_max_all) >= g.Ns / 2) return false;
  }
  g.sink0 = (p->n_can_max + 15) & ~15;                            // S[sink0 + b]: the always-zero slot of bank b
  g.n_S = g.sink0 + 16;
  if (g.n_S > 0x3FFF) return false;                               // 14-bit slot index in the phase-H records
  g.LS = fused_line_stride(g.Ns);
  g.n_col = p->kx_max_all + 1;
  if ((size_t)g.n_col * g.LS >= 0xFFFFu) return false;            // 16-bit line position
  const int T = g.Ns / 16, G = kFusedThreads / T;
  g.region = sizeof(float2) * ((size_t)g.n_col * g.LS + (size_t)G * (g.Ns + g.Ns / 16));
  g.region_al = (g.region + 127) / 128 * 128;
  g.s_bytes = sizeof(float2) * ((size_t)g.n_S + (g.D > 1 ? (size_t)g.D * (g.Ns / 2) : 0));   // sums (+ column phases)
  return true;
}

// One table layout of the route: corr = 0 plain, 1 = every chunk carries its correction factors too.
// Shared memory (bytes):
//   [0, region)             column lines + pass-B exchange lines; doubles as chunk buffers 1..nbuf-1
//   [off_first, +B)         chunk buffer 0 (dedicated)
//   [off_S, ...)            canonical cell sums, 16 zero slots (sinks), column phases
//   [off_bar, ...)          full[nbuf], empty[nbuf], region_free mbarriers
// A buffer holds V visibility slots, the chunk's gather table (tab_off = 8 V bytes in) and, with
// corr, V factor slots (f_off = 8 V + tab_stride bytes behind the visibilities); V = chunk_vis, or
// chunk_vis + 16 with corr: the 16 extra slots of buffer 0 and their factor partners are zeroed once
// by the kernel and never written again -- the "zero visibility" a padded table entry points at must
// have a finite factor behind it.
static int fused_layout_impl(blink_plan *p, GatherLayout &L, int corr, bool tc, cudaStream_t st) {
  if (L.ok) return BLINK_OK;
  FusedGeom g;
  if (!fused_geom(p, g) || (int)p->gathers.size() != p->n_ch) return BLINK_OK;
  if (tc) {
    // k_fused_tc: the aliased region is its 64 KB operand region, followed by the 64 KB constant matrix;
    // what is left holds up to two dedicated chunk buffers
    if (p->n_pix != 256 || g.D != 1 || std::max(p->kx_max_all, p->ky_max_all) > 63) return BLINK_OK;
    g.region = 65536;
    g.region_al = 131072;
  }
  const int n_bl = p->n_bl, n_ch = p->n_ch;
  const size_t limit = (size_t)p->max_smem_optin;
  const int zpad = corr ? 16 : 0;

  std::vector<std::vector<int>> owner(n_ch), slot(n_ch);
  for (int ch = 0; ch < n_ch; ++ch) assign_cells(p->gathers[ch], owner[ch], slot[ch]);

  const int force_chunks = std::abs(p->opt.tune[kTuneFusedChunks]);
  const bool two_buffers_ok = p->opt.tune[kTuneFusedChunks] < 0;   // (negative: also accept a ring of two buffers)
  std::vector<AbstractTable> tabs;
  int n_chunk = 0, C = 0, nbuf = 0, nded = 1;
  size_t tab_stride = 0, buf_bytes = 0;
  bool found = false;
  for (n_chunk = std::max(1, force_chunks); n_chunk <= 64 && !found; ++n_chunk) {
    C = (n_bl + n_chunk - 1) / n_chunk;
    C = (C + 1) & ~1;                                  // 16-byte multiples
    if (C > 0x7FFE) continue;                          // 15-bit slot index relative to the chunk
    if ((n_bl + C - 1) / C != n_chunk) continue;
    const size_t data_bytes = sizeof(float2) * (size_t)(C + zpad) * (corr ? 2 : 1);
    if (data_bytes + g.region_al + g.s_bytes > limit) continue;   // cannot fit whatever the tables
    tabs.assign((size_t)n_ch * n_chunk, AbstractTable());
    std::atomic<bool> all_ok{true};
    parallel_for(n_ch * n_chunk, [&](int i) {
      if (!all_ok.load()) return;
      const int ch = i / n_chunk, c = i % n_chunk;
      bool ok = true;
      build_chunk_table(p->gathers[ch], owner[ch], slot[ch], c * C, std::min(n_bl, (c + 1) * C), g.sink0, tabs[i], ok);
      if (!ok) all_ok.store(false);
    });
    if (!all_ok.load()) continue;
    tab_stride = 0;
    for (const AbstractTable &t : tabs) tab_stride = std::max(tab_stride, t.bytes.size());
    buf_bytes = (data_bytes + tab_stride + 127) / 128 * 128;
    const size_t tail = g.s_bytes + 16 * 8 + 128 + 64;  // sums, mbarriers (<= 8 buffers) and the kernel's own words
    if (g.region_al + buf_bytes + tail > limit) continue;
    nded = tc ? (int)std::min<size_t>(2, (limit - g.region_al - tail) / buf_bytes) : 1;
    nded = std::min(nded, n_chunk);
    nbuf = nded + (int)std::min<size_t>(8 - nded, g.region / buf_bytes);
    nbuf = std::min(nbuf, n_chunk);
    if (nbuf < 2 && n_chunk > 1) continue;             // the ring needs a second buffer
    // (measured on the station, k_fused_tc: 6 chunks in a ring of two 0.424 ms, 9 chunks in a ring of three 0.471 ms:
    // fewer, larger chunks mean fewer, fuller groups in phase S, which outweighs the deeper ring)
    (void)two_buffers_ok;   // (two dedicated + one aliased keep the copies ahead of the sums)
    const size_t total = g.region_al + (size_t)nded * buf_bytes + tail;
    if (total > limit || total > 0x7FFFu * 8u) continue;
    found = true;
    break;
  }
  if (!found) return BLINK_OK;

  L.chunk_vis = C;
  L.n_chunk = n_chunk;
  L.nbuf = nbuf;
  L.tab_stride = (int)tab_stride;
  L.buf_bytes = (uint32_t)buf_bytes;
  L.nded = nded;
  L.off_first = (uint32_t)g.region_al;
  L.off_S = (uint32_t)(g.region_al + (size_t)nded * buf_bytes);      // multiple of 128: slot s of S sits in bank s mod 16
  L.off_bar = (uint32_t)((L.off_S + g.s_bytes + 15) / 16 * 16);
  L.smem = L.off_bar + 16 * (size_t)nbuf + 128;
  L.tab_off = (uint32_t)(sizeof(float2) * (size_t)(C + zpad));
  L.f_off = corr ? (uint32_t)(L.tab_off + tab_stride) : 0u;

  const uint32_t s_slot0 = L.off_S / 8;
  const uint32_t zslot0 = corr ? L.off_first / 8 + (uint32_t)C : s_slot0 + (uint32_t)g.sink0;
  std::vector<unsigned char> h_tab((size_t)n_ch * n_chunk * tab_stride, 0);
  std::vector<uint32_t> h_size((size_t)n_ch * n_chunk, 0);
  for (int ch = 0; ch < n_ch; ++ch)
    for (int c = 0; c < n_chunk; ++c) {
      const size_t cp = (size_t)ch * n_chunk + c;
      std::vector<unsigned char> &b = tabs[cp].bytes;
      const int bi = c % nbuf;
      const uint32_t base_slot =
          (uint32_t)((bi < nded ? L.off_first + (uint32_t)bi * L.buf_bytes : (uint32_t)(bi - nded) * L.buf_bytes) / 8);
      finalize_chunk_table(b, base_slot, zslot0);
      std::memcpy(h_tab.data() + cp * tab_stride, b.data(), b.size());
      h_size[cp] = (uint32_t)b.size();
    }
  int rc;
  if ((rc = upload_table((void **)&L.d_tab, h_tab.data(), h_tab.size(), st, "fused table")) != BLINK_OK) return rc;
  if ((rc = upload_table((void **)&L.d_size, h_size.data(), sizeof(uint32_t) * h_size.size(), st, "fused table")) != BLINK_OK) return rc;
  BLINK_CUDA_TRY(cudaStreamSynchronize(st), "fused table upload sync");
  L.ok = true;
  return BLINK_OK;
}

int fused_layout(blink_plan *p, int corr, cudaStream_t st) { return fused_layout_impl(p, p->fl[corr], corr, false, st); }
int fused_layout_tc(blink_plan *p, int corr, cudaStream_t st) { return fused_layout_impl(p, p->tl[corr], corr, true, st); }

// Lay out shared memory, build and upload the tables of the route (plain layout; the layout with
// correction factors is built when blink_plan_apply_corrections first asks for it).
int fused_build(blink_plan *p, cudaStream_t st) {
  FusedGeom g;
  if (!fused_geom(p, g)) return BLINK_OK;
  const int N = p->n_pix, n_ch = p->n_ch, Ns = g.Ns, D = g.D, LS = g.LS, sink0 = g.sink0;
  int rc = fused_layout(p, 0, st);
  if (rc != BLINK_OK) return rc;
  if (!p->fl[0].ok) return BLINK_OK;
  p->fused_D = D;
  p->fused_threads = kFusedThreads;
  const std::vector<HostGather> &gathers = p->gathers;
  std::vector<std::vector<int>> owner(n_ch), slot(n_ch);
  for (int ch = 0; ch < n_ch; ++ch) assign_cells(gathers[ch], owner[ch], slot[ch]);

  // phase-H records: every bounding-box cell with kx >= 0, column by column; for D > 1 also the
  // complex weight of every record in every sub-image (a, b): w e^{2 pi i (kx a + ky b) / N}
  std::vector<std::vector<uint2>> hrecs(n_ch);
  std::vector<std::vector<float2>> hws(n_ch);       // [sub][record], records in hrecs order
  struct HCell { int kx, ky; double w; };
  std::vector<std::vector<HCell>> hcells(n_ch);
  p->h_max = 0;
  for (int ch = 0; ch < n_ch; ++ch) {
    const HostGather &g = gathers[ch];
    const ChannelInfo &ci = p->chinfo[ch];
    auto find_j = [&](int cell) -> int {
      auto it = std::lower_bound(g.can_cell.begin(), g.can_cell.end(), cell);
      return (it != g.can_cell.end() && *it == cell) ? (int)(it - g.can_cell.begin()) : -1;
    };
    auto pad16h = [](int i) { return i + (i >> 4); };
    if (g.n_can == 0) continue;
    for (int kx = 0; kx <= ci.kx_max; ++kx)
      for (int ky = -ci.ky_max; ky <= ci.ky_max; ++ky) {
        const int ix = kx, iy = (ky + N) % N;
        const bool canonical = (ky > 0) || (ky == 0 && kx >= 0);
        const int c = canonical ? iy * N + ix : ((N - iy) % N) * N + ((N - ix) % N);
        const int j = find_j(c);
        const uint32_t pos = (uint32_t)(kx * LS + pad16h((ky + Ns) % Ns));
        uint2 r;
        double wd = 0.0;
        if (j < 0) {
          r = make_uint2(pos | ((uint32_t)sink0 << 16), 0u);                    // a zero slot x 0
        } else {
          int cnt = g.seg_start[j + 1] - g.seg_start[j];
          if (c == 0) cnt *= 2;
          float w = ((kx + ky) & 1) ? -ci.inv_norm : ci.inv_norm;
          if (p->weighting == BLINK_UNIFORM) w /= (float)cnt;
          wd = (double)w;
          const uint32_t flag = c == 0 ? kPlaceBoth : (canonical ? kPlaceDirect : kPlaceConj);
          uint32_t wb;
          std::memcpy(&wb, &w, 4);
          r = make_uint2(pos | ((uint32_t)slot[ch][j] << 16) | (flag << 30), wb);
        }
        hrecs[ch].push_back(r);
        hcells[ch].push_back(HCell{kx, ky, wd});
      }
    p->h_max = std::max(p->h_max, (int)hrecs[ch].size());
  }
  std::vector<uint2> h_hrec((size_t)n_ch * std::max(p->h_max, 1), make_uint2(0xFFFFu, 0u));
  for (int ch = 0; ch < n_ch; ++ch)
    std::copy(hrecs[ch].begin(), hrecs[ch].end(), h_hrec.begin() + (size_t)ch * p->h_max);
  std::vector<float2> h_hw, h_pha;
  if (D > 1) {
    h_hw.assign((size_t)n_ch * D * std::max(p->h_max, 1), make_float2(0.f, 0.f));
    const double two_pi = 6.283185307179586476925286766559;
    for (int ch = 0; ch < n_ch; ++ch)
      for (int b = 0; b < D; ++b) {
        float2 *dst = h_hw.data() + ((size_t)ch * D + b) * p->h_max;
        for (size_t e = 0; e < hcells[ch].size(); ++e) {
          const HCell &hc = hcells[ch][e];
          const int m = ((hc.ky * b) % N + N) % N;               // phase index, exact in integers
          const double ang = two_pi * (double)m / (double)N;
          dst[e] = make_float2((float)(hc.w * std::cos(ang)), (float)(hc.w * std::sin(ang)));
        }
      }
    h_pha.resize((size_t)D * (Ns / 2));
    for (int a = 0; a < D; ++a)
      for (int k = 0; k < Ns / 2; ++k) {
        const double ang = two_pi * (double)((k * a) % N) / (double)N;
        h_pha[(size_t)a * (Ns / 2) + k] = make_float2((float)std::cos(ang), (float)std::sin(ang));
      }
  }

  if ((rc = upload_table((void **)&p->d_hrec, h_hrec.data(), sizeof(uint2) * h_hrec.size(), st, "fused table")) != BLINK_OK) return rc;
  if (D > 1) {
    if ((rc = upload_table((void **)&p->d_hw, h_hw.data(), sizeof(float2) * h_hw.size(), st, "fused table")) != BLINK_OK) return rc;
    if ((rc = upload_table((void **)&p->d_pha, h_pha.data(), sizeof(float2) * h_pha.size(), st, "fused table")) != BLINK_OK) return rc;
    std::vector<float2> h_tws(Ns);                  // exp(+2 pi i m / Ns), the sub-transforms' twiddles
    for (int m = 0; m < Ns; ++m) {
      const double ang = 6.283185307179586476925286766559 * (double)m / (double)Ns;
      h_tws[m] = make_float2((float)std::cos(ang), (float)std::sin(ang));
    }
    if ((rc = upload_table((void **)&p->d_tw_sub, h_tws.data(), sizeof(float2) * h_tws.size(), st, "fused table")) != BLINK_OK) return rc;
  }
  BLINK_CUDA_TRY(cudaStreamSynchronize(st), "fused table upload sync");
  p->fused_path = 1;
  return BLINK_OK;
}

// The NZ template argument of the k_fused instance the plan's current state selects (BLINK_Q_FUSED_NZ): the
// first transform stage reads only the NZ N/16-cell blocks next to DC on either side.  N <= 128: always 8
// (unpruned); sub-transforms of 256: 2, 3, 4 or 8 without corrections at D = 1, 3 or 8 otherwise.
int fused_nz_instance(const blink_plan *p) {
  const int n_sub = p->n_pix / p->fused_D;
  if (n_sub != 256) return 8;
  // band limit of the first transform stage, in units of N/16 cells
  const int reach = std::max(p->kx_max_all, p->ky_max_all) + 1, T = n_sub / 16;
  const int nz = (reach + T - 1) / T;
  if (p->fused_D == 1 && !p->corr_on) {   // (with corrections: the two instances that cover every band limit)
    if (nz <= 2) return 2;
    if (nz == 4) return 4;
  }
  return nz <= 3 ? 3 : 8;
}

template <bool CORR>
static int launch_fused_c(const blink_plan *p, const FusedParams &fp, cudaStream_t st) {
  const int nz = fused_nz_instance(p);
  if (p->fused_D == 2) return nz == 3 ? launch_fused_n<256, 3, 2, CORR>(p, fp, st) : launch_fused_n<256, 8, 2, CORR>(p, fp, st);
  if (p->fused_D == 4) return launch_fused_d4(p, fp, nz, st);
  switch (p->n_pix) {
    case 32: return launch_fused_n<32, 8, 1, CORR>(p, fp, st);
    case 64: return launch_fused_n<64, 8, 1, CORR>(p, fp, st);
    case 128: return launch_fused_n<128, 8, 1, CORR>(p, fp, st);
    case 256:
      if constexpr (!CORR) {
        if (nz == 2) return launch_fused_n<256, 2, 1, CORR>(p, fp, st);
        if (nz == 4) return launch_fused_n<256, 4, 1, CORR>(p, fp, st);
      }
      if (nz == 3) return launch_fused_n<256, 3, 1, CORR>(p, fp, st);
      return launch_fused_n<256, 8, 1, CORR>(p, fp, st);
    default: return BLINK_EUNSUPPORTED;
  }
}

static int launch_fused(const blink_plan *p, const float2 *vis, int n_t, float *img, cudaStream_t st) {
  if (p->tc_route && p->tl[p->corr_on ? 1 : 0].ok) return launch_fused_tc(p, vis, n_t, img, st);
  const GatherLayout &L = p->fl[p->corr_on ? 1 : 0];
  FusedParams fp;
  fp.vis = vis; fp.img = img; fp.chinfo = p->d_chinfo;
  fp.corr = p->corr_on ? p->d_corr : nullptr;
  fp.gtab = L.d_tab; fp.gsize = L.d_size; fp.hrec = p->d_hrec; fp.hw = p->d_hw; fp.pha = p->d_pha;
  fp.tw = p->fused_D > 1 ? p->d_tw_sub : p->d_tw;
  fp.n_bl = p->n_bl; fp.n_ch = p->n_ch; fp.n_snap = n_t * p->n_ch; fp.n_can_max = p->n_can_max;
  fp.n_chunk = L.n_chunk; fp.chunk_vis = L.chunk_vis; fp.nbuf = L.nbuf;
  fp.tab_stride = L.tab_stride; fp.n_col = p->kx_max_all + 1; fp.h_max = p->h_max;
  fp.buf_bytes = L.buf_bytes; fp.tab_off = L.tab_off; fp.f_off = L.f_off;
  fp.off_dedicated = L.off_first; fp.off_S = L.off_S; fp.off_bar = L.off_bar; fp.smem = (uint32_t)L.smem;
  return p->corr_on ? launch_fused_c<true>(p, fp, st) : launch_fused_c<false>(p, fp, st);
}

int launch_grid_image(const blink_plan *p, const float2 *vis, int n_t, float *img, cudaStream_t st) {
  if (fused_smem_route(p)) return launch_fused(p, vis, n_t, img, st);
  return launch_image_from_vis(p, vis, n_t * p->n_ch, img, st);
}

}  // namespace blink

extern "C" int blink_grid_image(const blink_plan *plan, const void *vis, int n_t, void *images, void *stream) {
  if (!plan || n_t < 0) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!vis || !images) return BLINK_EINVAL;
  if (((uintptr_t)vis & 15) || ((uintptr_t)images & 3)) return BLINK_EINVAL;
  int rc = check_device(plan);
  if (rc == BLINK_OK) rc = check_corrections_current(plan);
  if (rc != BLINK_OK) return rc;
  if (blink::scratch_need(plan, n_t, true) > plan->scratch_bytes) return BLINK_ERESERVE;
  return blink::launch_grid_image(plan, (const float2 *)vis, n_t, (float *)images, (cudaStream_t)stream);
}

#ifdef BLINK_TESTING_HOOKS   // libblink_testing.so only (build.py): libblink.so carries no host model and no probe
// Host emulation of phase S of k_fused for ONE channel (tests without a GPU): builds the gather
// tables exactly as fused_build does for chunks of chunk_vis baselines, then walks them the way a
// warp does over a byte-for-byte model of shared memory.
extern "C" int blink_host_fused_emulate(const int32_t *cell, int n_bl, int n_pix, int chunk_vis,
                                        const float *vis, float *sums, int32_t *stats) {
  using namespace blink;
  if (!cell || !vis || !sums || n_bl < 1 || chunk_vis < 2 || (chunk_vis & 1) || chunk_vis > 0x7FFE) return BLINK_EINVAL;
  HostGather g;
  int rc = build_gather_host(cell, n_bl, n_pix, g);
  if (rc != BLINK_OK) return rc;
  std::vector<int> owner, slot;
  assign_cells(g, owner, slot);
  const int sink0 = (g.n_can + 15) & ~15, n_S = sink0 + 16;
  const uint32_t s_slot0 = (uint32_t)((chunk_vis + 15) & ~15);        // S right after the chunk buffer
  if (s_slot0 + (uint32_t)n_S > 0x7FFFu) return BLINK_EUNSUPPORTED;
  std::vector<float> sm(2 * (size_t)(s_slot0 + n_S), 0.f);           // shared memory as float2 slots
  long groups = 0, rows = 0;
  for (int lo = 0; lo < n_bl; lo += chunk_vis) {
    const int hi = std::min(n_bl, lo + chunk_vis);
    AbstractTable t;
    bool ok = true;
    build_chunk_table(g, owner, slot, lo, hi, sink0, t, ok);
    if (!ok) return BLINK_EUNSUPPORTED;
    finalize_chunk_table(t.bytes, 0u, s_slot0 + (uint32_t)sink0);
    groups += t.groups;
    rows += t.rows;
    std::memcpy(sm.data(), vis + 2 * (size_t)lo, sizeof(float) * 2 * (size_t)(hi - lo));
    const unsigned char *tab = t.bytes.data();
    for (int w = 0; w < kFusedWarps; ++w) {
      uint32_t wx, lseq;
      std::memcpy(&wx, tab + 8 * w, 4);
      std::memcpy(&lseq, tab + 8 * w + 4, 4);
      size_t blk = wx & 0xFFFFFFu;
      for (int gi = 0; gi < (int)(wx >> 24); ++gi) {
        const int L = group_len(lseq, gi);
        const uint16_t *row = reinterpret_cast<const uint16_t *>(tab + blk);
        for (int lane = 0; lane < 32; ++lane) {
          float ax = 0.f, ay = 0.f;
          for (int r = 0; r < L; ++r) {
            const uint16_t e = row[(size_t)(r + 1) * 32 + lane];
            const float vx = sm[2 * (size_t)(e & 0x7FFF)], vy = sm[2 * (size_t)(e & 0x7FFF) + 1];
            if (r == 0) { ax = vx; ay = (e & 0x8000) ? -vy : vy; }
            else { ax += vx; ay += (e & 0x8000) ? -vy : vy; }
          }
          const size_t sj = 2 * ((size_t)s_slot0 + row[lane]);
          sm[sj] += ax;
          sm[sj + 1] += ay;
        }
        blk += (size_t)(L + 1) * 64;
      }
    }
  }
  for (int j = 0; j < g.n_can; ++j) {
    sums[2 * j] = sm[2 * ((size_t)s_slot0 + slot[j])];
    sums[2 * j + 1] = sm[2 * ((size_t)s_slot0 + slot[j]) + 1];
  }
  for (int b = 0; b < 16; ++b)                      // the zero slots must still be zero
    if (sm[2 * ((size_t)s_slot0 + sink0 + b)] != 0.f || sm[2 * ((size_t)s_slot0 + sink0 + b) + 1] != 0.f) return BLINK_EINVAL;
  if (stats) { stats[0] = g.n_can; stats[1] = (int32_t)groups; stats[2] = (int32_t)rows; }
  return BLINK_OK;
}
#endif  // BLINK_TESTING_HOOKS
