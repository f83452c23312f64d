// blink_image_r.cu -- steps a1-a5 at N = 1024 for wide, sparsely filled uv planes (MWA-like arrays) as
// ONE kernel in which a snapshot's intermediate never leaves the SM: gridding (cell sums), weighting,
// 2-D inverse DFT, fftshift, normalisation, real part.
//
// The image rows are dealt by residue class: y = 32 y' + r.  For one class r (a "unit" of work: 32 image
// rows = 16 row pairs) the column pass needs, per column kx >= 0 of the half-plane,
//
//   U[32 y' + r][kx] = sum_c w32^(c y') * B_r[c][kx],   B_r[c][kx] = sum_{cells (iy, kx), iy mod 32 = c} G[iy][kx] w1024^(iy r)
//
// i.e. the plan's occupied cells (7e3 of 5e5 for MWA Phase I) each times one unit-modulus factor, summed into
// 32 bins per column, then ONE dense 32-point butterfly per column: a 32 x 512 complex tile = 128 KB of
// shared memory, where the row pass (two real image rows per 1024-point complex transform, one warp per
// transform, wfft.cuh's 32 x 32 split) picks it up.  So per unit a CTA of 16 warps runs
//
//   S  bins:    warp w owns the 32 columns {32 ((w + b) mod 16) + b}.  The columns' non-empty bins
//               ("entries") are dealt to its lanes by the plan so that every lane has the same number of
//               cells (longest entry first to the least loaded lane); a lane walks its own list, cell q of
//               lane l at position 32 q + l (consecutive lanes read consecutive slots), adds
//               G_j w32^(a_j r) and, at the last cell of an entry, stores the sum times w1024^(c r) into the
//               tile.  Empty bins are never written: the plan's per-column bin mask says which to read.
//               The image stores of the PREVIOUS unit (64 per lane, still in registers) are issued four
//               per step inside this loop, so they do not arrive at the memory pipe as one burst.
//   A  columns: lane = column; masked loads of its bins, dft32 in registers, and in place of the bins the
//               row-pass operands Z = U[y] + i U[y + 512] (rows p) and conj U[y] + i conj U[y + 512]
//               (rows 16 + p, the mirrored half kx < 0).  A column's 32 slots are private to its lane, so
//               S and A of a warp are ordered by __syncwarp alone.
//   B  rows:    after ALL columns (one mbarrier, 16 arrivals), warp p transforms row pair p: 32 loads per
//               lane, dft32, twiddles, exchange through the warp's own two tile rows (XOR swizzle, conflict
//               free), dft32, 64 coalesced streaming stores of 128 bytes.
//
// The tile of the next unit may be written once every warp has finished with its exchange (second mbarrier,
// arrived on half-way through B), so the outer butterflies and the stores of one unit overlap the bins and
// columns of the next.  The cell values G (sum of the cell's visibilities in ascending baseline order x
// weight x fftshift sign / norm, exactly as in blink_image_w.cu) are formed once per snapshot and kept in
// shared memory.  Units are dealt in contiguous runs, T = 32 n_snap units over the CTAs, so the CTAs finish
// together; no scratch in HBM, no inter-CTA traffic, no cooperative launch.
//
// Algorithmic HBM bytes per snapshot: 8 n_bl (visibilities, read once per CTA that touches the snapshot)
// + 4 N^2 (the image, written once) = SURVEY 8(d)'s B_fused.
#include <algorithm>
#include <cstring>
#include <map>

#include "blink_internal.h"
#include "sgather.cuh"
#include "fft_core.cuh"

namespace blink {
using namespace blinkfft;

constexpr int kRN = 1024;
constexpr int kRW = 512;                        // columns of the tile (kx = 0 .. 511)
constexpr int kRWarps = 16;
constexpr int kRThreads = 32 * kRWarps;
constexpr int kRHdr = 4;                        // ints per (channel, warp) header: first position, first entry slot, steps, -
constexpr int kRHdrRows = kRWarps + 1;          // + one row {positions, entry slots}
constexpr size_t kROffTw = sizeof(cf32) * 32 * kRW;                 // tile first
constexpr size_t kROffW32 = kROffTw + sizeof(cf32) * 1024;
constexpr size_t kROffHdr = kROffW32 + sizeof(cf32) * 32;
constexpr size_t kROffBar = kROffHdr + sizeof(int32_t) * kRHdrRows * kRHdr;
constexpr size_t kROffCv = (kROffBar + 16 + 15) / 16 * 16;
constexpr size_t kRBytesPerPos = sizeof(cf32) + sizeof(uint8_t);     // + 2 bytes per entry slot

struct RParams {
  ImgParams ip;
  int n_snap, cap, ecap;
  const uint4 *rrec;        // [n_ch][cap] iy | flag << 10 | kx << 12 | len << 21, weight, source 0, source 1 / segment (len 0 = padding)
  const uint8_t *rca;       // [n_ch][cap] iy >> 5 of the cell at this position | 32 if it is the last of its entry
  const uint16_t *res;      // [n_ch][ecap] tile slot c * 512 + kx of a lane's n-th entry at [32 n + lane] behind the warp's base
  const int32_t *rhdr;      // [n_ch][17][kRHdr]
  const uint32_t *rmask;    // [n_ch][512] non-empty bins of the column
  const float2 *uvsrc;      // blink_image: cell values from this uv grid; NULL = from the visibilities
};

// value of one cell: weighted sum of its visibilities in ascending baseline order (or the uv grid's cell)
__device__ __forceinline__ cf32 cell_from_vis(const uint4 r, const float2 v0, const float2 v1, const float2 *__restrict__ vis,
                                              const float2 *__restrict__ cf, const int32_t *__restrict__ src) {
  const int flag = (r.x >> 10) & 3, len = (int)(r.x >> 21);
  const float w = __uint_as_float(r.y);
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
  if (flag == kPlaceDirect) return mk(ar * w, ai * w);
  if (flag == kPlaceConj) return mk(ar * w, -ai * w);
  return mk((ar + ar) * w, 0.f);
}

// the image stores of one unit: t[n2] of lane n1 is pixel x = n1 + 32 n2 of rows y (real part) and y + 512 (imaginary part)
struct ROut { float *r0, *r1; };
template <int I> __device__ __forceinline__ void store4(const ROut &o, const cf32 *t) {      // stores 4 I .. 4 I + 3 of 64
  __stcs(o.r0 + 32 * (2 * I), t[2 * I].x);
  __stcs(o.r1 + 32 * (2 * I), t[2 * I].y);
  __stcs(o.r0 + 32 * (2 * I + 1), t[2 * I + 1].x);
  __stcs(o.r1 + 32 * (2 * I + 1), t[2 * I + 1].y);
}

template <bool DEFER> __global__ void __launch_bounds__(kRThreads, 1) k_img1024r(const RParams q) {
  constexpr int N = kRN;
  const ImgParams &p = q.ip;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cf32 *Z = reinterpret_cast<cf32 *>(smem_raw);                       // [32][512] bins -> row-pass operands -> exchange tiles
  cf32 *twB = reinterpret_cast<cf32 *>(smem_raw + kROffTw);           // [n1][b] exp(2 pi i b n1 / 1024)
  cf32 *w32 = reinterpret_cast<cf32 *>(smem_raw + kROffW32);          // exp(2 pi i k / 32)
  int32_t *hdr = reinterpret_cast<int32_t *>(smem_raw + kROffHdr);
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + kROffBar); // [0] columns done, [1] exchange tiles free
  cf32 *cv = reinterpret_cast<cf32 *>(smem_raw + kROffCv);            // cell values of the snapshot, by position
  uint16_t *es = reinterpret_cast<uint16_t *>(cv + q.cap);            // entry slots -> tile slot
  uint8_t *ca = reinterpret_cast<uint8_t *>(es + q.ecap);             // position -> iy >> 5 | last << 5
  const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;

  for (int i = tid; i < 1024; i += kRThreads) twB[i] = __ldg(p.tw32 + i);
  if (tid < 32) w32[tid] = __ldg(p.tw + tid * (N / 32));
  if (tid < 2) mbar_init(bars + tid, kRWarps);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();

  const long long T = (long long)q.n_snap * 32;
  const long long u0 = T * blockIdx.x / gridDim.x, u1 = T * (blockIdx.x + 1) / gridDim.x;
  const int kcol = 32 * ((wv + lane) & 15) + lane;       // this lane's column in phases S / A
  uint32_t ph_a = 0, ph_b = 0, cmask = 0;
  int s_cur = -1;
  cf32 t[32];
  ROut out = {nullptr, nullptr};           // rows of the unit whose pixels are still in t[] (NULL: none)
  for (long long u = u0; u < u1; ++u) {
    const int s = (int)(u >> 5), r = (int)(u & 31);
    if (s != s_cur) {
      // ---------------------------------------------------------------- G: the snapshot's cell values
      // (every warp is past the columns barrier of the previous unit, so nobody reads the old ones)
      if (out.r0 != nullptr) {
#pragma unroll
        for (int n2 = 0; n2 < 32; ++n2) {
          __stcs(out.r0 + 32 * n2, t[n2].x);
          __stcs(out.r1 + 32 * n2, t[n2].y);
        }
        out.r0 = nullptr;
      }
      s_cur = s;
      const int ch = (s + p.ch0) % p.n_ch;
      const int32_t *gh = q.rhdr + (size_t)ch * kRHdrRows * kRHdr;
      for (int i = tid; i < kRHdrRows * kRHdr; i += kRThreads) hdr[i] = __ldg(gh + i);
      cmask = __ldg(q.rmask + (size_t)ch * kRW + kcol);
      const int npos = __ldg(gh + kRWarps * kRHdr), nes = __ldg(gh + kRWarps * kRHdr + 1);
      {
        const uint4 *ge = reinterpret_cast<const uint4 *>(q.res + (size_t)ch * q.ecap);
        for (int i = tid; i < (nes + 7) / 8; i += kRThreads) reinterpret_cast<uint4 *>(es)[i] = __ldg(ge + i);
        const uint4 *ga = reinterpret_cast<const uint4 *>(q.rca + (size_t)ch * q.cap);
        for (int i = tid; i < (npos + 15) / 16; i += kRThreads) reinterpret_cast<uint4 *>(ca)[i] = __ldg(ga + i);
      }
      const uint4 *__restrict__ rec = q.rrec + (size_t)ch * q.cap;
      if (q.uvsrc != nullptr) {
        // blink_image: the plan's occupied cells with kx >= 0 straight from the uv grid (empty cells are
        // zero by contract and never read)
        const float2 *__restrict__ g = q.uvsrc + (size_t)(p.snap_base + s) * N * N;
        for (int i = tid; i < npos; i += kRThreads) {
          const uint4 rr = __ldg(rec + i);
          const int iy = (int)(rr.x & 1023), flag = (rr.x >> 10) & 3, kx = (rr.x >> 12) & 511;
          const float w = __uint_as_float(rr.y);
          float2 v = make_float2(0.f, 0.f);
          if (rr.x >> 21) v = __ldg(g + (size_t)iy * N + kx);
          cv[i] = mk(v.x * w, (flag == kPlaceDirect || flag == kPlaceConj) ? v.y * w : 0.f);
        }
      } else {
        const float2 *__restrict__ vis = p.vis + (size_t)(p.snap_base + s) * p.n_bl;
        const int32_t *__restrict__ src = p.src + (size_t)ch * p.n_bl;
        const float2 *__restrict__ cf = p.corr ? p.corr + (size_t)ch * p.n_bl : nullptr;
        for (int i0 = tid; i0 < npos; i0 += 8 * kRThreads) {       // eight cells per thread in flight
          uint4 rr[8];
          float2 v0[8], v1[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int i = i0 + j * kRThreads;
            rr[j] = i < npos ? __ldg(rec + i) : make_uint4(0, 0, 0, 0);
          }
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int len = (int)(rr[j].x >> 21);
            v0[j] = v1[j] = make_float2(0.f, 0.f);
            if (len >= 1) v0[j] = ld_vis(vis, cf, rr[j].z >> 1);
            if (len == 2) v1[j] = ld_vis(vis, cf, rr[j].w >> 1);
          }
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int i = i0 + j * kRThreads;
            if (i < npos) cv[i] = (rr[j].x >> 21) ? cell_from_vis(rr[j], v0[j], v1[j], vis, cf, src) : mk(0.f, 0.f);
          }
        }
      }
      __syncthreads();
    }
    if (u > u0) {                          // every warp has left its exchange tile of the previous unit
      mbar_wait(bars + 1, ph_b);
      ph_b ^= 1u;
    }
    {
      // -------------------------------------------------------------- S: the bins of this warp's columns
      const int32_t *h = hdr + wv * kRHdr;
      const int L = h[2];
      const cf32 *cvp = cv + h[0] + lane;
      const uint8_t *cap_ = ca + h[0] + lane;
      const uint16_t *esp = es + h[1] + lane;
      const cf32 *twr = twB + r * 32;                                 // w1024^(c r), c = 0 .. 31
      cf32 acc = mk(0.f, 0.f);
      auto step = [&](int qq) {
        const cf32 v = cvp[32 * qq];
        const int m = cap_[32 * qq];
        const cf32 w = w32[((m & 31) * r) & 31];
        acc.x = fmaf(v.x, w.x, fmaf(-v.y, w.y, acc.x));
        acc.y = fmaf(v.x, w.y, fmaf(v.y, w.x, acc.y));
        if (m & 32) {                                                  // last cell of an entry
          const int slot = *esp;
          esp += 32;
          Z[slot] = cmul(acc, twr[slot >> 9]);
          acc = mk(0.f, 0.f);
        }
      };
      const bool have = DEFER && out.r0 != nullptr;
      // sixteen steps with the 64 stores of the previous unit spread among them, then the rest
#define BLINK_R_STEP(I)             \
  if (I < L) step(I);               \
  if (have) store4<I>(out, t);
      BLINK_R_STEP(0) BLINK_R_STEP(1) BLINK_R_STEP(2) BLINK_R_STEP(3) BLINK_R_STEP(4) BLINK_R_STEP(5) BLINK_R_STEP(6) BLINK_R_STEP(7)
      BLINK_R_STEP(8) BLINK_R_STEP(9) BLINK_R_STEP(10) BLINK_R_STEP(11) BLINK_R_STEP(12) BLINK_R_STEP(13) BLINK_R_STEP(14) BLINK_R_STEP(15)
#undef BLINK_R_STEP
      for (int qq = 16; qq < L; ++qq) step(qq);
      __syncwarp();
      // -------------------------------------------------------------- A: this lane's column, in place
      cf32 *zc = Z + kcol;
      if (__any_sync(0xffffffffu, cmask != 0)) {
#pragma unroll
        for (int c = 0; c < 32; ++c) t[c] = ((cmask >> c) & 1u) ? zc[c * kRW] : mk(0.f, 0.f);
        dft32(t);                                                     // t[y'] = U[32 y' + r][kcol]
#pragma unroll
        for (int pp = 0; pp < 16; ++pp) {
          const cf32 A = t[pp], B = t[pp + 16];
          zc[pp * kRW] = mk(A.x - B.y, A.y + B.x);                    // U[y] + i U[y + 512]
          zc[(16 + pp) * kRW] = mk(A.x + B.y, B.x - A.y);             // conj U[y] + i conj U[y + 512]
        }
      } else {
#pragma unroll
        for (int c = 0; c < 32; ++c) zc[c * kRW] = mk(0.f, 0.f);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bars + 0);
    }
    mbar_wait(bars + 0, ph_a);
    ph_a ^= 1u;
    {
      // -------------------------------------------------------------- B: row pair p = wv
      // lane b holds Z[32 a + b]: a < 16 from row p (kx = 32 a + b), a >= 16 the mirrored half from row
      // 16 + p at kx = 1024 - 32 a - b (kx = 512 does not exist: zero)
      const cf32 *za = Z + wv * kRW + lane;
      const cf32 *zm = Z + (16 + wv) * kRW - lane;
#pragma unroll
      for (int a = 0; a < 16; ++a) t[a] = za[32 * a];
      t[16] = lane == 0 ? mk(0.f, 0.f) : zm[512];
#pragma unroll
      for (int a = 17; a < 32; ++a) t[a] = zm[32 * (32 - a)];
      __syncwarp();
      dft32(t);
#pragma unroll
      for (int n1 = 1; n1 < 32; ++n1) t[n1] = cmul(t[n1], twB[n1 * 32 + lane]);
      // exchange through the warp's own two rows: element (b, n1) at row (b < 16 ? p : 16 + p), slot
      // (b mod 16) * 32 + (n1 xor b): 8-byte stores by b and loads by n1 are both conflict-free
      cf32 *th = Z + ((lane & 16) ? (16 + wv) * kRW : wv * kRW) + (lane & 15) * 32;
#pragma unroll
      for (int n1 = 0; n1 < 32; ++n1) th[n1 ^ lane] = t[n1];
      __syncwarp();
#pragma unroll
      for (int b = 0; b < 32; ++b) t[b] = Z[(b < 16 ? wv * kRW : (16 + wv) * kRW) + (b & 15) * 32 + (lane ^ b)];
      __syncwarp();
      if (lane == 0) mbar_arrive(bars + 1);
      dft32(t);
      // the pixels stay in t[]: they are stored during phase S of the next unit (or below, after the last)
      out.r0 = p.img + ((size_t)(p.snap_base + s) * N + 32 * wv + r) * N + lane;
      out.r1 = out.r0 + (size_t)(N / 2) * N;
      if constexpr (!DEFER) {
#pragma unroll
        for (int n2 = 0; n2 < 32; ++n2) {
          __stcs(out.r0 + 32 * n2, t[n2].x);
          __stcs(out.r1 + 32 * n2, t[n2].y);
        }
        out.r0 = nullptr;
      }
    }
  }
  if (out.r0 != nullptr) {
#pragma unroll
    for (int n2 = 0; n2 < 32; ++n2) {
      __stcs(out.r0 + 32 * n2, t[n2].x);
      __stcs(out.r1 + 32 * n2, t[n2].y);
    }
  }
}

// ---- plan side ----------------------------------------------------------------------------------------
struct RCell { int k, iy, seg, len, flag; float w; };
struct RTables {
  std::vector<uint4> rec;
  std::vector<uint8_t> ca;
  std::vector<uint16_t> es;
  std::vector<int32_t> hdr;
  std::vector<uint32_t> mask;
};

// the tables of one channel
static void res_tables(const HostGather &g, int N, int weighting, float inv_norm, RTables &o) {
  std::vector<RCell> cells;
  for (int j = 0; j < g.n_can; ++j) {
    const int c = g.can_cell[j], ix = c % N, iy = c / N;
    const int kx = ix < N / 2 ? ix : ix - N, ky = iy;
    const int len = g.seg_start[j + 1] - g.seg_start[j];
    const int cnt = c == 0 ? 2 * len : len;
    float w = ((kx + ky) & 1) ? -inv_norm : inv_norm;
    if (weighting == BLINK_UNIFORM) w /= (float)cnt;
    if (kx >= 0) cells.push_back({kx, iy, g.seg_start[j], len, c == 0 ? kPlaceBoth : kPlaceDirect, w});
    if (kx <= 0 && c != 0) cells.push_back({-kx, (N - iy) % N, g.seg_start[j], len, kPlaceConj, w});
  }
  // entries (column, bin) per owning warp; the cells of an entry in ascending iy
  std::vector<std::map<int, std::vector<int>>> ent(kRWarps);
  std::sort(cells.begin(), cells.end(), [](const RCell &a, const RCell &b) { return a.k != b.k ? a.k < b.k : a.iy < b.iy; });
  o.mask.assign(kRW, 0u);
  for (int i = 0; i < (int)cells.size(); ++i) {
    const int k = cells[i].k, c = cells[i].iy & 31;
    ent[((k >> 5) - (k & 31)) & 15][c * kRW + k].push_back(i);
    o.mask[k] |= 1u << c;
  }
  o.hdr.assign((size_t)kRHdrRows * kRHdr, 0);
  o.rec.clear(); o.ca.clear(); o.es.clear();
  for (int w = 0; w < kRWarps; ++w) {
    // longest entry first to the lane with the fewest cells so far (ties: fewest entries, lowest lane)
    std::vector<std::pair<int, int>> order;      // (-len, slot)
    for (auto &kv : ent[w]) order.push_back({-(int)kv.second.size(), kv.first});
    std::sort(order.begin(), order.end());
    std::vector<std::vector<int>> mine(32);      // slots of each lane's entries, in the order it walks them
    int load[32] = {0};
    for (auto &od : order) {
      int best = 0;
      for (int l = 1; l < 32; ++l)
        if (load[l] < load[best] || (load[l] == load[best] && mine[l].size() < mine[best].size())) best = l;
      mine[best].push_back(od.second);
      load[best] += -od.first;
    }
    int L = 0, EL = 0;
    for (int l = 0; l < 32; ++l) { L = std::max(L, load[l]); EL = std::max(EL, (int)mine[l].size()); }
    int32_t *h = o.hdr.data() + (size_t)w * kRHdr;
    h[0] = (int32_t)o.rec.size(); h[1] = (int32_t)o.es.size(); h[2] = L; h[3] = EL;
    const size_t r0 = o.rec.size(), e0 = o.es.size();
    o.rec.resize(r0 + (size_t)32 * L, make_uint4(0, 0, 0, 0));
    o.ca.resize(r0 + (size_t)32 * L, 0);
    o.es.resize(e0 + (size_t)32 * EL, 0);
    for (int l = 0; l < 32; ++l) {
      int qpos = 0;
      for (size_t n = 0; n < mine[l].size(); ++n) {
        const std::vector<int> &cl = ent[w][mine[l][n]];
        o.es[e0 + 32 * n + l] = (uint16_t)mine[l][n];
        for (size_t i = 0; i < cl.size(); ++i, ++qpos) {
          const RCell &c = cells[cl[i]];
          uint32_t wbits;
          memcpy(&wbits, &c.w, 4);
          o.rec[r0 + 32 * (size_t)qpos + l] =
              make_uint4((uint32_t)c.iy | ((uint32_t)c.flag << 10) | ((uint32_t)c.k << 12) | ((uint32_t)c.len << 21), wbits,
                         (uint32_t)g.src[c.seg], c.len == 2 ? (uint32_t)g.src[c.seg + 1] : (uint32_t)c.seg);
          o.ca[r0 + 32 * (size_t)qpos + l] = (uint8_t)((c.iy >> 5) | (i + 1 == cl.size() ? 32 : 0));
        }
      }
    }
  }
  o.hdr[(size_t)kRWarps * kRHdr] = (int32_t)o.rec.size();
  o.hdr[(size_t)kRWarps * kRHdr + 1] = (int32_t)o.es.size();
}

static size_t res_smem(int cap, int ecap) { return kROffCv + (size_t)cap * kRBytesPerPos + (size_t)ecap * sizeof(uint16_t); }

void res_route_free(blink_plan *p) {
  cudaFree(p->d_rrec); cudaFree(p->d_rca); cudaFree(p->d_res); cudaFree(p->d_rhdr); cudaFree(p->d_rmask);
  p->d_rrec = nullptr; p->d_rca = nullptr; p->d_res = nullptr; p->d_rhdr = nullptr; p->d_rmask = nullptr;
  p->res_route = 0;
}

// Residue-class route of blink_grid_image / blink_image at N = 1024: applies when every channel's occupied
// half-plane cells (9 bytes per position, 2 per entry slot) fit in shared memory beside the 128 KB tile.
int res_route_build(blink_plan *p, cudaStream_t st) {
  p->res_route = 0;
  if (p->n_pix != kRN || p->opt.warp_route == -1 || p->opt.warp_route == 2) return BLINK_OK;
  if (p->wu > kRW || p->seg_len_max > 2047 || p->max_smem_optin <= 0) return BLINK_OK;
  const int n_ch = p->n_ch;
  std::vector<RTables> tb(n_ch);
  parallel_for(n_ch, [&](int ch) { res_tables(p->gathers[ch], p->n_pix, p->weighting, p->chinfo[ch].inv_norm, tb[ch]); });
  int cap = 16, ecap = 16;
  for (int ch = 0; ch < n_ch; ++ch) {
    cap = std::max(cap, ((int)tb[ch].rec.size() + 15) / 16 * 16);
    ecap = std::max(ecap, ((int)tb[ch].es.size() + 15) / 16 * 16);
  }
  if (ecap > 0xFFFF || res_smem(cap, ecap) > (size_t)p->max_smem_optin) return BLINK_OK;
  std::vector<uint4> h_rec((size_t)n_ch * cap, make_uint4(0, 0, 0, 0));
  std::vector<uint8_t> h_ca((size_t)n_ch * cap, 0);
  std::vector<uint16_t> h_es((size_t)n_ch * ecap, 0);
  std::vector<int32_t> h_hdr((size_t)n_ch * kRHdrRows * kRHdr, 0);
  std::vector<uint32_t> h_mask((size_t)n_ch * kRW, 0u);
  for (int ch = 0; ch < n_ch; ++ch) {
    std::copy(tb[ch].rec.begin(), tb[ch].rec.end(), h_rec.begin() + (size_t)ch * cap);
    std::copy(tb[ch].ca.begin(), tb[ch].ca.end(), h_ca.begin() + (size_t)ch * cap);
    std::copy(tb[ch].es.begin(), tb[ch].es.end(), h_es.begin() + (size_t)ch * ecap);
    std::copy(tb[ch].hdr.begin(), tb[ch].hdr.end(), h_hdr.begin() + (size_t)ch * kRHdrRows * kRHdr);
    std::copy(tb[ch].mask.begin(), tb[ch].mask.end(), h_mask.begin() + (size_t)ch * kRW);
  }
  int rc;
  if ((rc = upload_table((void **)&p->d_rrec, h_rec.data(), sizeof(uint4) * h_rec.size(), st, "residue route records")) != BLINK_OK) return rc;
  if ((rc = upload_table((void **)&p->d_rca, h_ca.data(), h_ca.size(), st, "residue route cells")) != BLINK_OK) return rc;
  if ((rc = upload_table((void **)&p->d_res, h_es.data(), sizeof(uint16_t) * h_es.size(), st, "residue route entries")) != BLINK_OK) return rc;
  if ((rc = upload_table((void **)&p->d_rhdr, h_hdr.data(), sizeof(int32_t) * h_hdr.size(), st, "residue route headers")) != BLINK_OK) return rc;
  if ((rc = upload_table((void **)&p->d_rmask, h_mask.data(), sizeof(uint32_t) * h_mask.size(), st, "residue route masks")) != BLINK_OK) return rc;
  BLINK_CUDA_TRY(cudaStreamSynchronize(st), "residue route upload");
  p->res_cap = cap;
  p->res_ecap = ecap;
  p->res_route = 1;
  return BLINK_OK;
}

int launch_img1024r(const blink_plan *p, ImgParams ip, int n_snap, cudaStream_t st) {
  if (n_snap <= 0) return BLINK_OK;
  RParams q;
  q.n_snap = n_snap;
  q.cap = p->res_cap;
  q.ecap = p->res_ecap;
  q.rrec = p->d_rrec; q.rca = p->d_rca; q.res = p->d_res; q.rhdr = p->d_rhdr; q.rmask = p->d_rmask;
  q.uvsrc = ip.vis == nullptr ? ip.uv : nullptr;
  ip.snap_base = 0;
  q.ip = ip;
  const size_t smem = res_smem(p->res_cap, p->res_ecap);
  static std::atomic<uint64_t> attr{0};
  static std::atomic<uint64_t> attr1{0};
  const bool defer = p->opt.tune[kTuneWarpCtasPerSm] == 2;
  const int rc = defer ? ensure_max_smem(k_img1024r<true>, p, attr, "k_img1024r smem attribute")
                       : ensure_max_smem(k_img1024r<false>, p, attr1, "k_img1024r smem attribute");
  if (rc != BLINK_OK) return rc;
  // one CTA per SM; fewer when there are fewer units than that
  const long long units = (long long)n_snap * 32;
  const int grid = (int)std::min<long long>(p->sm_count, units);
  if (defer) k_img1024r<true><<<grid, kRThreads, smem, st>>>(q);
  else k_img1024r<false><<<grid, kRThreads, smem, st>>>(q);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_img1024r launch");
  return BLINK_OK;
}

}  // namespace blink
