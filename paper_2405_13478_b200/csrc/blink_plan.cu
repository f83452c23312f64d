// blink_plan.cu -- plan creation: step a0, the uv-index precompute that exploits the fixed array
// geometry (the paper recomputes frequency, wavelength and the cell per thread
// per launch).  The fp64 index kernel and the integer count kernel run on the
// device; the cell-sorted gather / placement tables that make blink_grid atomic-free and
// deterministic (the paper's planned "parallel reduction") are sorted on the
// host once per plan.
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "blink_internal.h"

namespace blink {

static thread_local std::string g_cuda_err;
void set_cuda_error(cudaError_t e, const char *where) {
  g_cuda_err = std::string(where) + ": " + cudaGetErrorString(e);
  cudaGetLastError();  // clear sticky-free errors
}

void set_error_text(const char *text) { g_cuda_err = text; }

// ------------------------------------------------------------------------------------------
// K0: one thread per (channel, baseline).  Operation order is part of the contract (blink.h
// "Cell rule"): fp64, round-to-nearest intrinsics so that no FMA contraction can occur.
__global__ void k_uv_index(const double *__restrict__ ant, const int32_t *__restrict__ pi,
                           const int32_t *__restrict__ pj, const double *__restrict__ freq,
                           int n_bl, int n_ch, int N, double G, int32_t *__restrict__ cell,
                           uint32_t *__restrict__ counts) {
  const int bl = blockIdx.x * blockDim.x + threadIdx.x;
  const int ch = blockIdx.y;
  if (bl >= n_bl || ch >= n_ch) return;
  const double sc = __ddiv_rn(freq[ch], 299792458.0);
  const int i = pi[bl], j = pj[bl];
  const double de = __dsub_rn(ant[3 * j + 0], ant[3 * i + 0]);
  const double dn = __dsub_rn(ant[3 * j + 1], ant[3 * i + 1]);
  const double u = __dmul_rn(de, sc);
  const double v = __dmul_rn(dn, sc);
  const long long kx = llround(__dmul_rn(u, G));
  const long long ky = llround(__dmul_rn(v, G));
  const long long kmax = N / 2 - 1;
  int32_t c = -1;
  if (kx >= -kmax && kx <= kmax && ky >= -kmax && ky <= kmax) {
    const int ix = (int)((kx + N) % N), iy = (int)((ky + N) % N);
    const int cx = (N - ix) % N, cy = (N - iy) % N;
    c = iy * N + ix;
    uint32_t *cnt = counts + (size_t)ch * N * N;
    atomicAdd(cnt + c, 1u);                 // integer atomics: exact, order-independent
    atomicAdd(cnt + cy * N + cx, 1u);       // ("counter of the number of visibilities")
  }
  cell[(size_t)ch * n_bl + bl] = c;
}

int launch_index_kernel(blink_plan *p, const double *d_ant, const double *d_freq,
                        const int32_t *d_pi, const int32_t *d_pj, cudaStream_t st) {
  const int N = p->n_pix;
  const double G = (double)N * p->pixscale;
  BLINK_CUDA_TRY(cudaMemsetAsync(p->d_counts, 0, sizeof(uint32_t) * (size_t)p->n_ch * N * N, st),
                 "memset counts");
  dim3 grid((p->n_bl + 255) / 256, p->n_ch);
  k_uv_index<<<grid, 256, 0, st>>>(d_ant, d_pi, d_pj, d_freq, p->n_bl, p->n_ch, N, G, p->d_cell,
                                   p->d_counts);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_uv_index launch");
  return BLINK_OK;
}

// ------------------------------------------------------------------------------------------
// Host: canonical-cell gather table of one channel.  A kept baseline with cell c (centred
// coordinates kx, ky) contributes V to c and conj(V) to c*.  Exactly one of {c, c*} lies in the
// canonical half-plane (ky > 0, or ky == 0 and kx >= 0); the baseline is filed under that cell, as
// V (flag 0) or conj(V) (flag 1).  Sorting by (canonical cell, baseline) makes every cell's sum
// a contiguous segment in ascending-baseline order -- the oracle's summation order.
int build_gather_host(const int32_t *cell, int n_bl, int n_pix, HostGather &out) {
  const int N = n_pix;
  struct Ent { int32_t can; int32_t code; };
  std::vector<Ent> ents;
  ents.reserve(n_bl);
  for (int bl = 0; bl < n_bl; ++bl) {
    const int32_t c = cell[bl];
    if (c < 0) continue;
    if (c >= N * N) return BLINK_EINVAL;
    const int ix = c % N, iy = c / N;
    const int kx = ix < N / 2 ? ix : ix - N, ky = iy < N / 2 ? iy : iy - N;
    const bool canonical = (ky > 0) || (ky == 0 && kx >= 0);
    Ent e;
    if (canonical) {
      e.can = c;
      e.code = (bl << 1);
    } else {
      e.can = ((N - iy) % N) * N + ((N - ix) % N);
      e.code = (bl << 1) | 1;
    }
    ents.push_back(e);
  }
  std::stable_sort(ents.begin(), ents.end(), [](const Ent &a, const Ent &b) { return a.can < b.can; });
  out.n_kept = (int32_t)ents.size();
  out.src.resize(ents.size());
  out.can_cell.clear();
  out.seg_start.clear();
  for (size_t e = 0; e < ents.size(); ++e) {
    if (e == 0 || ents[e].can != ents[e - 1].can) {
      out.can_cell.push_back(ents[e].can);
      out.seg_start.push_back((int32_t)e);
    }
    out.src[e] = ents[e].code;
  }
  out.seg_start.push_back((int32_t)ents.size());
  out.n_can = (int32_t)out.can_cell.size();
  return BLINK_OK;
}

// Rank-major tables of the per-cell sums (blink_grid, blink_grid_image).  Pass q takes baselines
// [q cap, (q+1) cap).  Within a pass the cells that receive something are ordered by descending
// number of baselines (position k); the r-th baseline (ascending index) of the cell at position k
// has rank-major slot roff[r] + k.  Thread k then walks slots roff[r] + k, r = 0..len-1:
// consecutive threads touch consecutive slots, the lanes of a warp see near-equal trip counts,
// and the summation order is the oracle's (ascending baseline).
//   scat[bl]        slot | conj << 15 (0xFFFF = dropped)              -- scatter form (k_grid)
//   list[slot]      (bl - q cap) | conj << 15                          -- gather form (k_fused)
//   cellrec[k]      j | len << 16 (j = index of the canonical cell sum)
struct RankTables {
  int cap = 0, n_pass = 0, roff_stride = 0;
  std::vector<uint16_t> scat, list, roff;
  std::vector<uint32_t> cellrec;
  std::vector<int32_t> nact;
};

static void build_rank_tables(const std::vector<HostGather> &gathers, int n_ch, int n_bl, int ncm,
                              int cap, RankTables &t) {
  t.cap = cap;
  t.n_pass = std::max(1, (n_bl + cap - 1) / cap);
  const int n_pass = t.n_pass;
  t.scat.assign((size_t)n_ch * n_bl, kScatDropped);
  t.list.assign((size_t)n_ch * n_pass * cap, 0);
  t.cellrec.assign((size_t)n_ch * n_pass * ncm, 0);
  t.nact.assign((size_t)n_ch * n_pass, 0);
  std::vector<std::vector<uint16_t>> roffs((size_t)n_ch * n_pass);
  std::vector<int> maxlen_ch(n_ch, 0);
  parallel_for(n_ch, [&](int ch) {
    int maxlen = 0;
    const HostGather &g = gathers[ch];
    uint16_t *sc = t.scat.data() + (size_t)ch * n_bl;
    for (int q = 0; q < n_pass; ++q) {
      const int lo = q * cap, hi = std::min(n_bl, lo + cap);
      // per cell: entries of this pass are a contiguous sub-range of its (baseline-sorted) segment
      std::vector<std::array<int32_t, 3>> cells;   // {len, j, first entry}
      for (int j = 0; j < g.n_can; ++j) {
        int e0 = g.seg_start[j], e1 = g.seg_start[j + 1];
        while (e0 < e1 && (g.src[e0] >> 1) < lo) ++e0;
        int e2 = e0;
        while (e2 < e1 && (g.src[e2] >> 1) < hi) ++e2;
        if (e2 > e0) cells.push_back({e2 - e0, j, e0});
      }
      std::stable_sort(cells.begin(), cells.end(),
                       [](const std::array<int32_t, 3> &a, const std::array<int32_t, 3> &b) { return a[0] > b[0]; });
      const int n_act = (int)cells.size();
      t.nact[(size_t)ch * n_pass + q] = n_act;
      const int ml = n_act ? cells[0][0] : 0;
      maxlen = std::max(maxlen, ml);
      std::vector<uint16_t> &ro = roffs[(size_t)ch * n_pass + q];
      ro.assign(ml + 1, 0);
      int off = 0, nr = n_act;
      for (int r = 0; r < ml; ++r) {
        while (nr > 0 && cells[nr - 1][0] <= r) --nr;   // cells with len > r form a prefix
        ro[r] = (uint16_t)off;
        off += nr;
      }
      ro[ml] = (uint16_t)off;
      uint32_t *cr = t.cellrec.data() + ((size_t)ch * n_pass + q) * ncm;
      uint16_t *ls = t.list.data() + ((size_t)ch * n_pass + q) * cap;
      for (int k = 0; k < n_act; ++k) {
        cr[k] = (uint32_t)cells[k][1] | ((uint32_t)cells[k][0] << 16);
        for (int r = 0; r < cells[k][0]; ++r) {
          const int code = g.src[cells[k][2] + r];
          sc[code >> 1] = (uint16_t)((ro[r] + k) | ((code & 1) << 15));
          ls[ro[r] + k] = (uint16_t)(((code >> 1) - lo) | ((code & 1) << 15));
        }
      }
    }
    maxlen_ch[ch] = maxlen;
  });
  const int maxlen = *std::max_element(maxlen_ch.begin(), maxlen_ch.end());
  t.roff_stride = ((maxlen + 1 + 3) / 4) * 4;   // rows stay 8-byte aligned for ushort4 reads
  t.roff.assign((size_t)n_ch * n_pass * t.roff_stride, 0);
  for (size_t i = 0; i < roffs.size(); ++i)
    std::copy(roffs[i].begin(), roffs[i].end(), t.roff.begin() + i * t.roff_stride);
}

template <class T> static int dev_alloc(T **p, size_t n) {
  if (n == 0) n = 1;
  cudaError_t e = cudaMalloc((void **)p, n * sizeof(T));
  if (e != cudaSuccess) {
    set_cuda_error(e, "cudaMalloc");
    *p = nullptr;
    return e == cudaErrorMemoryAllocation ? BLINK_ENOMEM : BLINK_ECUDA;
  }
  return BLINK_OK;
}

static void plan_free(blink_plan *p) {
  if (!p) return;
  host_pipe_free(p);
  cudaFree(p->d_cell); cudaFree(p->d_counts); cudaFree(p->d_chinfo); cudaFree(p->d_src);
  cudaFree(p->d_seg); cudaFree(p->d_pcell); cudaFree(p->d_pcode); cudaFree(p->d_pband); cudaFree(p->d_scat); cudaFree(p->d_cellrec); cudaFree(p->d_roff); cudaFree(p->d_nact); cudaFree(p->d_wkey); cudaFree(p->d_wval); cudaFree(p->d_wcol);
  cudaFree(p->d_tw); cudaFree(p->d_scratch); cudaFree(p->d_vkey); cudaFree(p->d_vseg); cudaFree(p->d_vlen); cudaFree(p->d_vw); cudaFree(p->d_vcol); cudaFree(p->d_vrec); cudaFree(p->d_corr); cudaFree(p->d_tw32);
  cudaFree(p->d_tcref); cudaFree(p->d_cmat);
  res_route_free(p);
  cudaFree(p->d_hrec); cudaFree(p->d_hw); cudaFree(p->d_pha); cudaFree(p->d_tw_sub); cudaFree(p->d_rplace);
  for (int c = 0; c < 2; ++c) {
    cudaFree(p->fl[c].d_tab); cudaFree(p->fl[c].d_size); cudaFree(p->rl[c].d_tab); cudaFree(p->rl[c].d_size);
    cudaFree(p->tl[c].d_tab); cudaFree(p->tl[c].d_size);
  }
  delete p;
}

static bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

}  // namespace blink

using namespace blink;

extern "C" int blink_version(void) { return BLINK_VERSION; }

extern "C" const char *blink_strerror(int status) {
  switch (status) {
    case BLINK_OK: return "ok";
    case BLINK_EINVAL: return "invalid argument";
    case BLINK_ENOMEM: return "out of memory";
    case BLINK_ECUDA: return "CUDA error or no CUDA device";
    case BLINK_EUNSUPPORTED: return "not supported by this build";
    case BLINK_ERESERVE: return "plan scratch too small for this n_t: call blink_plan_reserve first";
    case BLINK_ECAPACITY: return "one snapshot's intermediate exceeds the built-in scratch of blink_image_static";
    default: return "unknown status";
  }
}

extern "C" const char *blink_last_cuda_error(void) { return g_cuda_err.c_str(); }

#ifdef BLINK_TESTING_HOOKS   // libblink_testing.so only (build.py): libblink.so carries no host model and no probe
extern "C" int blink_host_build_gather(const int32_t *cell, int n_bl, int n_pix, int32_t *n_can_out,
                                       int32_t *can_cell, int32_t *seg_start, int32_t *src) {
  if (!cell || n_bl < 0 || n_pix < 2 || (n_pix & 1) || !n_can_out || !can_cell || !seg_start || !src)
    return BLINK_EINVAL;
  HostGather g;
  int rc = build_gather_host(cell, n_bl, n_pix, g);
  if (rc != BLINK_OK) return rc;
  *n_can_out = g.n_can;
  std::copy(g.can_cell.begin(), g.can_cell.end(), can_cell);
  std::copy(g.seg_start.begin(), g.seg_start.end(), seg_start);
  std::copy(g.src.begin(), g.src.end(), src);
  return g.n_kept;
}
#endif  // BLINK_TESTING_HOOKS

extern "C" int blink_plan_create(blink_plan **out, const double *ant_enu_m, int n_ant,
                                 const double *freq_hz, int n_ch, int n_pix, double pixscale,
                                 int weighting, void *stream) {
  return blink_plan_create_opts(out, ant_enu_m, n_ant, freq_hz, n_ch, n_pix, pixscale, weighting, stream, nullptr);
}

extern "C" int blink_plan_create_opts(blink_plan **out, const double *ant_enu_m, int n_ant,
                                      const double *freq_hz, int n_ch, int n_pix, double pixscale,
                                      int weighting, void *stream, const blink_options *opts) try {
  blink_options opt = {};
  if (opts) {
    if (opts->struct_size != (int32_t)sizeof(blink_options)) return BLINK_EINVAL;
    opt = *opts;
    auto route_ok = [](int32_t v) { return v == 0 || v == -1; };
    if (!route_ok(opt.fused_route) || !route_ok(opt.polyphase) || !(route_ok(opt.warp_route) || opt.warp_route == 2) || !route_ok(opt.grid_ring) ||
        opt.warp_ring < 0 || opt.warp_ring == 1 || opt.grid_ring_min_snap < 0 || opt.image_chunk_mb < 0)
      return BLINK_EINVAL;
  }
  if (!out || !ant_enu_m || !freq_hz || n_ant < 2 || n_ant > 4096 || n_ch < 1 || n_ch > 65535 ||
      !(pixscale > 0.0) || (weighting != BLINK_NATURAL && weighting != BLINK_UNIFORM))
    return BLINK_EINVAL;
  if (n_pix < 2 || (n_pix & 1)) return BLINK_EINVAL;
  if (!is_pow2(n_pix) || n_pix < 32 || n_pix > 4096) return BLINK_EUNSUPPORTED;
  for (int c = 0; c < n_ch; ++c)
    if (!(freq_hz[c] > 0.0)) return BLINK_EINVAL;

  int dev = 0;
  BLINK_CUDA_TRY(cudaGetDevice(&dev), "cudaGetDevice");
  cudaStream_t st = (cudaStream_t)stream;
  blink_plan *p = new (std::nothrow) blink_plan();
  if (!p) return BLINK_ENOMEM;
  // the half-built plan goes away on every early return below AND when a host table runs out of memory
  // (std::bad_alloc unwinds through here to the handler at the end of this function)
  struct Guard {
    blink_plan *p;
    void drop() { plan_free(p); p = nullptr; }
    ~Guard() { if (p) plan_free(p); }
  } guard{p};
  p->device = dev;
  p->opt = opt;
  p->n_ant = n_ant;
  p->n_bl = n_ant * (n_ant - 1) / 2;
  p->n_ch = n_ch;
  p->n_pix = n_pix;
  p->pixscale = pixscale;
  p->weighting = weighting;
  cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&p->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  const int N = n_pix, n_bl = p->n_bl;
  const size_t NN = (size_t)N * N;

#define PLAN_TRY(expr)        \
  do {                        \
    int rc__ = (expr);        \
    if (rc__ != BLINK_OK) {   \
      guard.drop();           \
      return rc__;            \
    }                         \
  } while (0)
#define PLAN_CUDA(expr, where)              \
  do {                                      \
    cudaError_t e__ = (expr);               \
    if (e__ != cudaSuccess) {               \
      set_cuda_error(e__, where);           \
      guard.drop();                         \
      return BLINK_ECUDA;                   \
    }                                       \
  } while (0)

  p->h_ant.assign(ant_enu_m, ant_enu_m + (size_t)3 * n_ant);
  p->h_freq.assign(freq_hz, freq_hz + n_ch);
  // ---- inputs to the device, K0 --------------------------------------------------------
  std::vector<int32_t> pi(n_bl), pj(n_bl);
  {
    int bl = 0;
    for (int i = 0; i < n_ant; ++i)
      for (int j = i + 1; j < n_ant; ++j, ++bl) { pi[bl] = i; pj[bl] = j; }
  }
  double *d_ant = nullptr, *d_freq = nullptr;
  int32_t *d_pi = nullptr, *d_pj = nullptr;
  PLAN_TRY(dev_alloc(&p->d_cell, (size_t)n_ch * n_bl));
  PLAN_TRY(dev_alloc(&p->d_counts, (size_t)n_ch * NN));
  int rc = BLINK_OK;
  if ((rc = dev_alloc(&d_ant, (size_t)3 * n_ant)) || (rc = dev_alloc(&d_freq, (size_t)n_ch)) ||
      (rc = dev_alloc(&d_pi, (size_t)n_bl)) || (rc = dev_alloc(&d_pj, (size_t)n_bl))) {
    cudaFree(d_ant); cudaFree(d_freq); cudaFree(d_pi); cudaFree(d_pj);
    guard.drop();
    return rc;
  }
  std::vector<int32_t> h_cell((size_t)n_ch * n_bl);
  cudaError_t ce = cudaSuccess;
  auto step = [&](cudaError_t e) { if (ce == cudaSuccess) ce = e; };
  step(cudaMemcpyAsync(d_ant, ant_enu_m, sizeof(double) * 3 * n_ant, cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(d_freq, freq_hz, sizeof(double) * n_ch, cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(d_pi, pi.data(), sizeof(int32_t) * n_bl, cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(d_pj, pj.data(), sizeof(int32_t) * n_bl, cudaMemcpyHostToDevice, st));
  if (ce == cudaSuccess) rc = launch_index_kernel(p, d_ant, d_freq, d_pi, d_pj, st);
  step(cudaMemcpyAsync(h_cell.data(), p->d_cell, sizeof(int32_t) * h_cell.size(),
                       cudaMemcpyDeviceToHost, st));
  step(cudaStreamSynchronize(st));
  cudaFree(d_ant); cudaFree(d_freq); cudaFree(d_pi); cudaFree(d_pj);
  if (rc != BLINK_OK) { guard.drop(); return rc; }
  PLAN_CUDA(ce, "plan upload / index kernel");

  // ---- host: per-channel facts, gather and placement tables -------------------------------
  p->band_cells = (int)std::min<size_t>(NN, (size_t)kBandCellsDefault);
  p->n_bands = (int)(NN / p->band_cells);
  p->n_dropped.assign(n_ch, 0); p->wsum.assign(n_ch, 0); p->n_occ.assign(n_ch, 0);
  p->norm.assign(n_ch, 0.0); p->chinfo.assign(n_ch, ChannelInfo());
  std::vector<int32_t> h_src((size_t)n_ch * n_bl, 0), h_seg((size_t)n_ch * (n_bl + 1), 0);
  std::vector<int32_t> h_pcell((size_t)n_ch * 2 * n_bl, 0), h_pcode((size_t)n_ch * 2 * n_bl, 0);
  std::vector<int32_t> h_pband((size_t)n_ch * (p->n_bands + 1), 0);
  std::vector<HostGather> &gathers = p->gathers;
  gathers.assign(n_ch, HostGather());
  std::vector<int> ch_rc(n_ch, BLINK_OK);
  parallel_for(n_ch, [&](int ch) {
    HostGather &g = gathers[ch];
    if ((ch_rc[ch] = build_gather_host(h_cell.data() + (size_t)ch * n_bl, n_bl, N, g)) != BLINK_OK) return;
    ChannelInfo &ci = p->chinfo[ch];
    ci.n_kept = g.n_kept;
    ci.n_can = g.n_can;
    p->n_dropped[ch] = n_bl - g.n_kept;
    p->wsum[ch] = 2 * (int64_t)g.n_kept;
    std::copy(g.src.begin(), g.src.end(), h_src.begin() + (size_t)ch * n_bl);
    std::copy(g.seg_start.begin(), g.seg_start.end(), h_seg.begin() + (size_t)ch * (n_bl + 1));
    // placement: every canonical cell and its mirror, sorted by full-plane cell index
    std::vector<std::pair<int32_t, int32_t>> pl;
    pl.reserve(2 * (size_t)g.n_can);
    int kxm = 0, kym = 0;
    for (int j = 0; j < g.n_can; ++j) {
      const int c = g.can_cell[j], ix = c % N, iy = c / N;
      const int kx = ix < N / 2 ? ix : ix - N, ky = iy;  // canonical: ky >= 0
      kxm = std::max(kxm, std::abs(kx));
      kym = std::max(kym, ky);
      const int cc = ((N - iy) % N) * N + ((N - ix) % N);
      if (cc == c) {
        pl.push_back({c, j | (kPlaceBoth << kPlaceShift)});
      } else {
        pl.push_back({c, j | (kPlaceDirect << kPlaceShift)});
        pl.push_back({cc, j | (kPlaceConj << kPlaceShift)});
      }
    }
    std::sort(pl.begin(), pl.end());
    ci.n_place = (int32_t)pl.size();
    ci.kx_max = kxm;
    ci.ky_max = kym;
    p->n_occ[ch] = ci.n_place;
    p->norm[ch] = weighting == BLINK_NATURAL ? (double)p->wsum[ch] : (double)p->n_occ[ch];
    ci.inv_norm = p->norm[ch] > 0.0 ? (float)(1.0 / p->norm[ch]) : 0.0f;
    int32_t *pb = h_pband.data() + (size_t)ch * (p->n_bands + 1);
    size_t e = 0;
    for (int b = 0; b < p->n_bands; ++b) {
      pb[b] = (int32_t)e;
      const int64_t hi = (int64_t)(b + 1) * p->band_cells;
      while (e < pl.size() && pl[e].first < hi) ++e;
    }
    pb[p->n_bands] = (int32_t)pl.size();
    for (size_t k = 0; k < pl.size(); ++k) {
      h_pcell[(size_t)ch * 2 * n_bl + k] = pl[k].first;
      h_pcode[(size_t)ch * 2 * n_bl + k] = pl[k].second;
    }
  });
  for (int ch = 0; ch < n_ch; ++ch) {
    PLAN_TRY(ch_rc[ch]);
    const HostGather &g = gathers[ch];
    p->n_can_max = std::max(p->n_can_max, (int)g.n_can);
    for (int j = 0; j < g.n_can; ++j) p->seg_len_max = std::max(p->seg_len_max, g.seg_start[j + 1] - g.seg_start[j]);
    p->kx_max_all = std::max(p->kx_max_all, p->chinfo[ch].kx_max);
    p->ky_max_all = std::max(p->ky_max_all, p->chinfo[ch].ky_max);
  }
  if (p->n_can_max > kPlaceMask) { guard.drop(); return BLINK_EUNSUPPORTED; }

  // ---- gridder tables: rank-major stage slots, cells by descending per-pass length ------------
  {
    // CTA shape: 512 threads x 16 visibilities in registers, one CTA per SM (256 x 16 x 2, 512 x 8 x 2 and
    // 256 x 8 x 3 measured slower in round 1)
    p->grid_nbuf = 3;
    p->grid_threads = 512;
    p->grid_prefetch = 16;
    p->grid_ctas_per_sm = 1;
    const int kStageCap = p->grid_threads * p->grid_prefetch;
    p->stage_cap = kStageCap;
    p->n_pass = (n_bl + kStageCap - 1) / kStageCap;
    if (p->n_pass < 1) p->n_pass = 1;
    p->grid_smem = sizeof(float2) * ((size_t)p->band_cells + (size_t)p->n_can_max +
                                     (size_t)p->stage_cap) + 64;
    if (p->max_smem_optin > 0 && p->grid_smem > (size_t)p->max_smem_optin) { guard.drop(); return BLINK_EUNSUPPORTED; }
  }
  if (p->n_can_max > 0xFFFF || p->stage_cap > 0x7FFF) { guard.drop(); return BLINK_EUNSUPPORTED; }
  const int n_pass = p->n_pass, ncm = std::max(p->n_can_max, 1);
  RankTables rt;
  build_rank_tables(gathers, n_ch, n_bl, ncm, p->stage_cap, rt);
  p->roff_stride = rt.roff_stride;
  std::vector<uint16_t> &h_scat = rt.scat, &h_roff = rt.roff;
  std::vector<uint32_t> &h_cellrec = rt.cellrec;
  std::vector<int32_t> &h_nact = rt.nact;
  (void)n_pass;

  // twiddles exp(+2 pi i k / N), fp64 -> fp32
  std::vector<float2> h_tw(N);
  for (int k = 0; k < N; ++k) {
    const double a = 2.0 * 3.14159265358979323846264338327950288 * (double)k / (double)N;
    h_tw[k] = make_float2((float)cos(a), (float)sin(a));
  }

  PLAN_TRY(dev_alloc(&p->d_chinfo, (size_t)n_ch));
  PLAN_TRY(dev_alloc(&p->d_src, h_src.size()));
  PLAN_TRY(dev_alloc(&p->d_seg, h_seg.size()));
  PLAN_TRY(dev_alloc(&p->d_pcell, h_pcell.size()));
  PLAN_TRY(dev_alloc(&p->d_pcode, h_pcode.size()));
  PLAN_TRY(dev_alloc(&p->d_pband, h_pband.size()));
  PLAN_TRY(dev_alloc(&p->d_tw, (size_t)N));
  PLAN_TRY(dev_alloc(&p->d_scat, h_scat.size()));
  PLAN_TRY(dev_alloc(&p->d_cellrec, h_cellrec.size()));
  PLAN_TRY(dev_alloc(&p->d_roff, h_roff.size()));
  PLAN_TRY(dev_alloc(&p->d_nact, h_nact.size()));
  step(cudaMemcpyAsync(p->d_scat, h_scat.data(), sizeof(uint16_t) * h_scat.size(), cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_cellrec, h_cellrec.data(), sizeof(uint32_t) * h_cellrec.size(), cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_roff, h_roff.data(), sizeof(uint16_t) * h_roff.size(), cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_nact, h_nact.data(), sizeof(int32_t) * h_nact.size(), cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_chinfo, p->chinfo.data(), sizeof(ChannelInfo) * n_ch, cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_src, h_src.data(), sizeof(int32_t) * h_src.size(), cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_seg, h_seg.data(), sizeof(int32_t) * h_seg.size(), cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_pcell, h_pcell.data(), sizeof(int32_t) * h_pcell.size(), cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_pcode, h_pcode.data(), sizeof(int32_t) * h_pcode.size(), cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_pband, h_pband.data(), sizeof(int32_t) * h_pband.size(), cudaMemcpyHostToDevice, st));
  step(cudaMemcpyAsync(p->d_tw, h_tw.data(), sizeof(float2) * N, cudaMemcpyHostToDevice, st));
  std::vector<float2> h_tw32(32 * 32);
  if (N == 1024) {   // inner-step twiddles of the warp-per-transform kernels, [n1][b]
    for (int n1 = 0; n1 < 32; ++n1)
      for (int b = 0; b < 32; ++b) {
        const double a = 2.0 * 3.14159265358979323846264338327950288 * (double)(b * n1) / 1024.0;
        h_tw32[n1 * 32 + b] = make_float2((float)cos(a), (float)sin(a));
      }
    PLAN_TRY(dev_alloc(&p->d_tw32, h_tw32.size()));
    step(cudaMemcpyAsync(p->d_tw32, h_tw32.data(), sizeof(float2) * h_tw32.size(), cudaMemcpyHostToDevice, st));
  }
  step(cudaStreamSynchronize(st));
  PLAN_CUDA(ce, "plan table upload");
  PLAN_TRY(image_setup(p));
  PLAN_TRY(fused_setup(p));
  {
    // pass-A-from-visibilities tables (any N): every occupied cell with kx >= 0, by column
    std::vector<int32_t> h_vkey((size_t)n_ch * 2 * n_bl, 0), h_vseg((size_t)n_ch * 2 * n_bl, 0),
        h_vlen((size_t)n_ch * 2 * n_bl, 0), h_vcol((size_t)n_ch * (p->wu + 1), 0);
    std::vector<float> h_vw((size_t)n_ch * 2 * n_bl, 0.f);
    std::vector<uint4> h_vrec((size_t)n_ch * 2 * n_bl, make_uint4(0, 0, 0, 0));
    struct VEnt { int32_t key, seg, len; float w; };
    for (int ch = 0; ch < n_ch; ++ch) {
      const HostGather &g = gathers[ch];
      const float inv_norm = p->chinfo[ch].inv_norm;
      std::vector<VEnt> ent;
      for (int j = 0; j < g.n_can; ++j) {
        const int c = g.can_cell[j], ix = c % N, iy = c / N;
        const int kx = ix < N / 2 ? ix : ix - N, ky = iy;
        const int len = g.seg_start[j + 1] - g.seg_start[j];
        const int cnt = c == 0 ? 2 * len : len;
        float w = ((kx + ky) & 1) ? -inv_norm : inv_norm;
        if (weighting == BLINK_UNIFORM) w /= (float)cnt;
        if (kx >= 0)
          ent.push_back({(kx << 16) | iy, g.seg_start[j], len | ((c == 0 ? kPlaceBoth : kPlaceDirect) << 24), w});
        if (kx <= 0 && c != 0)
          ent.push_back({((-kx) << 16) | ((N - iy) % N), g.seg_start[j], len | (kPlaceConj << 24), w});
      }
      // within a column: by iy mod 32, then iy / 32 -- the order the warp-per-column pass A
      // (blink_image_w.cu) consumes; the line-scatter kernels do not care
      auto vorder = [](int32_t key) { return ((key >> 16) << 16) | ((key & 31) << 11) | ((key & 0xffff) >> 5); };
      std::sort(ent.begin(), ent.end(), [&](const VEnt &a, const VEnt &b) { return vorder(a.key) < vorder(b.key); });
      int32_t *vc = h_vcol.data() + (size_t)ch * (p->wu + 1);
      size_t e = 0;
      for (int kx = 0; kx < p->wu; ++kx) {
        vc[kx] = (int32_t)e;
        while (e < ent.size() && (ent[e].key >> 16) == kx) ++e;
      }
      vc[p->wu] = (int32_t)ent.size();
      const size_t base = (size_t)ch * 2 * n_bl;
      for (size_t k = 0; k < ent.size(); ++k) {
        h_vkey[base + k] = ent[k].key; h_vseg[base + k] = ent[k].seg;
        h_vlen[base + k] = ent[k].len; h_vw[base + k] = ent[k].w;
        {   // one 16-byte record per cell for the warp-per-column pass A (blink_image_w.cu)
          const int len = ent[k].len & 0xFFFFFF, flag = ent[k].len >> 24;
          uint32_t wbits;
          memcpy(&wbits, &ent[k].w, 4);
          h_vrec[base + k] = make_uint4((uint32_t)(ent[k].key & 0xffff) | ((uint32_t)flag << 16) | ((uint32_t)len << 18), wbits,
                                        (uint32_t)g.src[ent[k].seg],
                                        len == 2 ? (uint32_t)g.src[ent[k].seg + 1] : (uint32_t)ent[k].seg);
        }
      }
      for (int kx = 0; kx < p->wu; kx += 8) p->vtile8_max = std::max(p->vtile8_max, vc[std::min(kx + 8, p->wu)] - vc[kx]);
    }
    PLAN_TRY(dev_alloc(&p->d_vkey, h_vkey.size()));
    PLAN_TRY(dev_alloc(&p->d_vseg, h_vseg.size()));
    PLAN_TRY(dev_alloc(&p->d_vlen, h_vlen.size()));
    PLAN_TRY(dev_alloc(&p->d_vw, h_vw.size()));
    PLAN_TRY(dev_alloc(&p->d_vcol, h_vcol.size()));
    PLAN_TRY(dev_alloc(&p->d_vrec, h_vrec.size()));
    step(cudaMemcpyAsync(p->d_vrec, h_vrec.data(), sizeof(uint4) * h_vrec.size(), cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(p->d_vkey, h_vkey.data(), sizeof(int32_t) * h_vkey.size(), cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(p->d_vseg, h_vseg.data(), sizeof(int32_t) * h_vseg.size(), cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(p->d_vlen, h_vlen.data(), sizeof(int32_t) * h_vlen.size(), cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(p->d_vw, h_vw.data(), sizeof(float) * h_vw.size(), cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(p->d_vcol, h_vcol.data(), sizeof(int32_t) * h_vcol.size(), cudaMemcpyHostToDevice, st));
    step(cudaStreamSynchronize(st));
    PLAN_CUDA(ce, "vis-route table upload");
    PLAN_TRY(res_route_build(p, st));
    p->warp_route = (p->res_route != 1 && p->opt.warp_route != -1 && warp_route_applies(p)) ? 1 : 0;
  }
  PLAN_TRY(fused_build(p, st));
  PLAN_TRY(fused_tc_build(p, st));
  PLAN_TRY(grid_ring_build(p, st));
  if (weighting == BLINK_UNIFORM) {
    // canonical cells are exactly the occupied half-plane cells with ky > 0 or (ky == 0, kx >= 0);
    // pass A of blink_image works on columns kx >= 0 and all ky, so list every occupied cell with
    // kx >= 0 (canonical cells with kx >= 0, and mirrors of canonical cells with kx < 0 -- and of
    // kx == 0, ky > 0).  count = segment length (+ mirror symmetry: count[c] == count[c*]).
    std::vector<int32_t> h_wkey((size_t)n_ch * 2 * n_bl, 0), h_wcol((size_t)n_ch * (p->wu + 1), 0);
    std::vector<float> h_wval((size_t)n_ch * 2 * n_bl, 0.f);
    for (int ch = 0; ch < n_ch; ++ch) {
      const HostGather &g = gathers[ch];
      std::vector<std::pair<int32_t, float>> ent;
      for (int j = 0; j < g.n_can; ++j) {
        const int c = g.can_cell[j], ix = c % N, iy = c / N;
        const int kx = ix < N / 2 ? ix : ix - N;
        int cnt = g.seg_start[j + 1] - g.seg_start[j];
        if (c == 0) cnt *= 2;                       // DC holds V and conj(V) of each baseline
        const float w = 1.0f / (float)cnt;
        if (kx >= 0) ent.push_back({(kx << 16) | iy, w});
        if (kx <= 0 && c != 0) ent.push_back({((-kx) << 16) | ((N - iy) % N), w});
      }
      std::sort(ent.begin(), ent.end());
      int32_t *wc = h_wcol.data() + (size_t)ch * (p->wu + 1);
      size_t e = 0;
      for (int kx = 0; kx < p->wu; ++kx) {
        wc[kx] = (int32_t)e;
        while (e < ent.size() && (ent[e].first >> 16) == kx) ++e;
      }
      wc[p->wu] = (int32_t)ent.size();
      for (size_t k = 0; k < ent.size(); ++k) {
        h_wkey[(size_t)ch * 2 * n_bl + k] = ent[k].first;
        h_wval[(size_t)ch * 2 * n_bl + k] = ent[k].second;
      }
    }
    PLAN_TRY(dev_alloc(&p->d_wkey, h_wkey.size()));
    PLAN_TRY(dev_alloc(&p->d_wval, h_wval.size()));
    PLAN_TRY(dev_alloc(&p->d_wcol, h_wcol.size()));
    step(cudaMemcpyAsync(p->d_wkey, h_wkey.data(), sizeof(int32_t) * h_wkey.size(), cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(p->d_wval, h_wval.data(), sizeof(float) * h_wval.size(), cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(p->d_wcol, h_wcol.data(), sizeof(int32_t) * h_wcol.size(), cudaMemcpyHostToDevice, st));
    step(cudaStreamSynchronize(st));
    PLAN_CUDA(ce, "weight table upload");
  }
#undef PLAN_TRY
#undef PLAN_CUDA
  guard.p = nullptr;
  *out = p;
  return BLINK_OK;
} catch (const std::bad_alloc &) {
  return BLINK_ENOMEM;                      // host memory for the plan tables; the guard has freed the plan
} catch (...) {
  blink::set_error_text("blink_plan_create: unexpected C++ exception");
  return BLINK_ECUDA;
}

extern "C" int blink_plan_destroy(blink_plan *plan) {
  plan_free(plan);
  return BLINK_OK;
}

// blink_plan_refresh: step a0 again for new antenna coordinates (a tracking array's projected baselines
// move with hour angle), everything else as at creation.  The index kernel runs on the
// device, the table packing on the host cores (one channel per thread); the new tables replace the old
// ones once they are complete (its scratch included, sized as the old plan's was); the host staging is kept.
extern "C" int blink_plan_refresh(blink_plan *p, const double *ant_enu_m, void *stream) {
  if (!p || !ant_enu_m) return BLINK_EINVAL;
  int rc = check_device(p);
  if (rc != BLINK_OK) return rc;
  blink_plan *q = nullptr;
  blink_options opt = p->opt;
  rc = blink_plan_create_opts(&q, ant_enu_m, p->n_ant, p->h_freq.data(), p->n_ch, p->n_pix, p->pixscale, p->weighting,
                              stream, opt.struct_size ? &opt : nullptr);
  if (rc != BLINK_OK) return rc;
  // scratch for the new bounding box, while the old plan is still whole: a failure here (BLINK_ENOMEM for a
  // wider half-plane) must leave the caller with the plan it had.  Both scratches exist until the swap.
  if (p->reserved_n_t > 0 && (rc = image_reserve(q, p->reserved_n_t)) != BLINK_OK) {
    plan_free(q);
    return rc;
  }
  // kernels already queued still read the old tables
  cudaError_t e = cudaDeviceSynchronize();
  if (e != cudaSuccess) {
    set_cuda_error(e, "blink_plan_refresh sync");
    plan_free(q);
    return BLINK_ECUDA;
  }
  std::swap(*p, *q);                       // p: the new tables; q: the old ones, about to be freed
  std::swap(p->hp, q->hp);                 // the host staging depends on n_ch, n_bl, N only
  p->corr_stale = (q->corr_on || q->corr_stale) ? 1 : 0;   // the factors went with the old geometry
  plan_free(q);
  return BLINK_OK;
}

extern "C" int blink_plan_reserve(blink_plan *plan, int n_t) {
  if (!plan || n_t < 0) return BLINK_EINVAL;
  int rc = check_device(plan);
  if (rc != BLINK_OK) return rc;
  return image_reserve(plan, n_t);
}

extern "C" int blink_plan_read(const blink_plan *p, int what, int ch, void *dst, size_t bytes) {
  if (!p || !dst || ch < 0 || ch >= p->n_ch) return BLINK_EINVAL;
  const void *src = nullptr;
  size_t need = 0;
  if (what == BLINK_Q_CELL_IDX) {
    need = sizeof(int32_t) * (size_t)p->n_bl;
    src = p->d_cell + (size_t)ch * p->n_bl;
  } else if (what == BLINK_Q_COUNTS) {
    need = sizeof(uint32_t) * (size_t)p->n_pix * p->n_pix;
    src = p->d_counts + (size_t)ch * p->n_pix * p->n_pix;
  } else if (what == BLINK_Q_CORR && p->d_corr) {
    need = sizeof(float2) * (size_t)p->n_bl;
    src = p->d_corr + (size_t)ch * p->n_bl;
  } else {
    return BLINK_EINVAL;
  }
  if (bytes != need) return BLINK_EINVAL;
  BLINK_CUDA_TRY(cudaMemcpy(dst, src, need, cudaMemcpyDeviceToHost), "blink_plan_read");
  return BLINK_OK;
}

extern "C" int blink_plan_query(const blink_plan *p, int what, int index, void *out) {
  if (!p || !out) return BLINK_EINVAL;
  const int ch = index & 0xffff;
  const bool per_ch = what == BLINK_Q_N_DROPPED || what == BLINK_Q_WSUM || what == BLINK_Q_N_OCC ||
                      what == BLINK_Q_BBOX || what == BLINK_Q_NORM;
  if (per_ch && ch >= p->n_ch) return BLINK_EINVAL;
  switch (what) {
    case BLINK_Q_N_ANT: *(int32_t *)out = p->n_ant; break;
    case BLINK_Q_N_BL: *(int32_t *)out = p->n_bl; break;
    case BLINK_Q_N_CH: *(int32_t *)out = p->n_ch; break;
    case BLINK_Q_N_PIX: *(int32_t *)out = p->n_pix; break;
    case BLINK_Q_N_DROPPED: *(int64_t *)out = p->n_dropped[ch]; break;
    case BLINK_Q_WSUM: *(int64_t *)out = p->wsum[ch]; break;
    case BLINK_Q_N_OCC: *(int64_t *)out = p->n_occ[ch]; break;
    case BLINK_Q_BBOX:
      ((int32_t *)out)[0] = p->chinfo[ch].kx_max;
      ((int32_t *)out)[1] = p->chinfo[ch].ky_max;
      break;
    case BLINK_Q_NORM: *(double *)out = p->norm[ch]; break;
    case BLINK_Q_CELL_IDX: *(const int32_t **)out = p->d_cell; break;
    case BLINK_Q_COUNTS: *(const uint32_t **)out = p->d_counts; break;
    case BLINK_Q_IMAGE_PATH: *(int32_t *)out = p->image_path; break;
    case BLINK_Q_SCRATCH_BYTES: *(int64_t *)out = (int64_t)p->scratch_bytes; break;
    case BLINK_Q_IMAGE_CHUNK: *(int32_t *)out = p->chunk_snapshots; break;
    case BLINK_Q_FUSED_PATH: *(int32_t *)out = fused_smem_route(p) ? 1 : ((p->warp_route || p->res_route == 1) ? 2 : 0); break;
    case BLINK_Q_WARP_KERNEL: *(int32_t *)out = p->res_route == 1 ? 2 : (p->warp_route ? 1 : (p->res_route == 2 ? 3 : 0)); break;
    case BLINK_Q_FUSED_CHUNK: *(int32_t *)out = p->fused_chunk; break;
    case BLINK_Q_CORR: *(const void **)out = p->d_corr; break;
    case BLINK_Q_CORR_FUSED: *(int32_t *)out = p->corr_on; break;
    case BLINK_Q_TENSOR_ROUTE: *(int32_t *)out = (fused_smem_route(p) && p->tc_route && p->tl[p->corr_on ? 1 : 0].ok) ? 1 : 0; break;
    case BLINK_Q_FUSED_NZ: {
      const bool tc = p->tc_route && p->tl[p->corr_on ? 1 : 0].ok;
      *(int32_t *)out = (fused_smem_route(p) && !tc) ? fused_nz_instance(p) : 0;
      break;
    }
    case BLINK_Q_FUSED_D: *(int32_t *)out = fused_smem_route(p) ? p->fused_D : 0; break;
    default: return BLINK_EINVAL;
  }
  return BLINK_OK;
}
