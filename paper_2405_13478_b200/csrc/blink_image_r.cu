// blink_image_r.cu -- steps a1-a5 at N = 1024 for wide, sparsely filled uv planes (MWA-like arrays) as
// ONE kernel in which a snapshot's intermediate never leaves the SM: gridding (cell sums), weighting,
// 2-D inverse DFT, fftshift, normalisation, real part.
//
// The image rows are dealt by residue class: y = 64 y' + r.  For one class r (a "unit" of work: 16 image
// rows = 8 row pairs y, y + 512) the column pass needs, per column kx >= 0 of the half-plane,
//
//   U[64 y' + r][kx] = sum_c w16^(c y') * B_r[c][kx],   B_r[c][kx] = sum_{cells (iy, kx), iy mod 16 = c} G[iy][kx] w1024^(iy r)
//
// i.e. the plan's occupied cells (7e3 of 5e5 for MWA Phase I) each times one unit-modulus factor, summed into
// 16 bins per column, then ONE dense 16-point butterfly per column: a 16 x 512 complex tile = 64 KB of
// shared memory, where the row pass (two real image rows per 1024-point complex transform, one warp per
// transform, wfft.cuh's 32 x 32 split) picks it up.  A CTA of 24 warps is split by role over a ring of
// two such tiles (full / empty mbarriers), so that the table walk of one unit overlaps the butterflies of
// another on every scheduler; after the split the producers give registers to the consumers
// (setmaxnreg: 16 x 32 x 64 + 8 x 32 x 112 = the 768 x 80 the CTA was launched with):
//
//   producers (warps 0-15), per unit:
//   S  bins:    warp w owns the 32 columns {32 ((w + b) mod 16) + b}.  The columns' non-empty bins
//               ("entries") are dealt to its lanes by the plan so that every lane has the same number of
//               cells (longest entry first to the least loaded lane, preferring a lane whose store lands in
//               a free bank); a lane walks its own list -- cell q of lane l at position 32 q + l: value and
//               32-bit descriptor (iy, last-of-entry flag, tile slot) in shared memory -- adds
//               G_j w1024^(iy_j r) and, at the last cell of an entry, stores the sum into the tile.  The
//               factor comes from the special-function unit, not from a table (see bins4).  Empty bins are
//               never written: the plan's per-column bin mask says which to read.
//   A  columns: lane = column; masked loads of its bins, dft16 in registers, and in place of the bins the
//               row-pass operands Z = U[y] + i U[y + 512] (rows p) and conj U[y] + i conj U[y + 512]
//               (rows 8 + p, the mirrored half kx < 0).  A column's 16 slots are private to its lane, so
//               S and A of a warp are ordered by __syncwarp alone.
//   G  (once per snapshot) every producer lane forms the values of ITS cells: the sum of the cell's
//               visibilities in ascending baseline order x weight x fftshift sign / norm, exactly as in
//               blink_image_w.cu.  Values and descriptors are lane-private and a warp's positions are the
//               same for every channel, so a snapshot change needs no barrier.
//   consumers (warps 16-23), per unit:
//   B  rows:    warp p transforms row pair p: 32 loads per lane, dft32, twiddles, exchange through the warp's
//               own two tile rows (16-byte stores, 8-byte loads, XOR swizzle: conflict free), tile released,
//               dft32, 64 coalesced streaming stores of 128 bytes.
//
// Units are dealt in contiguous runs, T = 64 n_snap units over the CTAs, so the CTAs finish together; no
// scratch in HBM, no inter-CTA traffic, no cooperative launch.
//
// Algorithmic HBM bytes per snapshot: 8 n_bl (visibilities, read once per CTA that touches the snapshot)
// + 4 N^2 (the image, written once) = SURVEY 8(d)'s B_fused.
#include <algorithm>
#include <array>
#include <cmath>
#include <complex>
#include <cstring>
#include <map>

#include "blink_internal.h"
#include "sgather.cuh"
#include "fft_core.cuh"

namespace blink {
using namespace blinkfft;

constexpr int kRN = 1024;
constexpr int kRW = 512;                        // columns of a tile (kx = 0 .. 511)
constexpr int kRRows = 16;                      // rows of a tile = image rows per unit
constexpr int kRUnits = kRN / kRRows;           // units (residue classes) per snapshot
constexpr int kRProd = 16, kRCons = 8;          // producer / consumer warps
constexpr int kRThreads = 32 * (kRProd + kRCons);
constexpr int kRLmax = 16;                      // most cells in a lane's list
constexpr int kRHdr = 2;                        // ints per (channel, producer warp) header: first position, steps
constexpr int kRRegsProd = 64, kRRegsCons = 112;// registers per thread after the role split: 16 x 32 x 64 + 8 x 32 x 112 = 768 x 80, the launch allocation
constexpr size_t kRTile = sizeof(cf32) * kRRows * kRW;
constexpr size_t kROffTw = 2 * kRTile;                              // the two tiles first
constexpr size_t kROffBar = kROffTw + sizeof(cf32) * 1024;
constexpr size_t kROffCv = kROffBar + 64;
// k_cols_res (N = 2048 / 4096, column pass only): two tiles of 8 rows x 1024 columns
constexpr int kCW = 1024, kCRows = 8, kCLmax = 32, kCThreads = 32 * kRProd;
constexpr size_t kCTile = sizeof(cf32) * kCRows * kCW;
constexpr size_t kCOffCv = 2 * kCTile + 64;

struct RParams {
  ImgParams ip;
  int n_snap, cap;
  const uint4 *rrec;        // [n_ch][cap] iy | flag << 10 | kx << 12 | len << 21, weight, source 0, source 1 / segment (len 0 = padding)
  const uint32_t *rmeta;    // [n_ch][cap] last-of-entry | 8 (tile slot c * 512 + kx) | iy << 22 (0 = padding)
  const int32_t *rhdr;      // [n_ch][kRProd][kRHdr]
  const uint32_t *rmask;    // [n_ch][tile columns] non-empty bins of the column
  const int16_t *rcols;     // k_cols_res: [16][32][2] the two columns of every lane (the same for all channels)
  const float2 *uvsrc;      // blink_image: cell values from this uv grid; NULL = from the visibilities
};

// Packing of a cell record's first word for an N = 2^LOGN grid with 2^LOGW tile columns:
// iy | flag << LOGN | kx << (LOGN + 2) | len << (LOGN + 2 + LOGW); the descriptor carries iy in its top LOGN bits
template <int LOGN, int LOGW> struct RPack {
  static constexpr int kFlagSh = LOGN, kKxSh = LOGN + 2, kLenSh = LOGN + 2 + LOGW;
  static constexpr uint32_t kIyMask = (1u << LOGN) - 1u, kKxMask = (1u << LOGW) - 1u, kLenMax = (1u << (32 - kLenSh)) - 1u;
  static constexpr uint32_t kAngleMask = ~0u << (32 - LOGN);
};

// value of one cell: weighted sum of its visibilities in ascending baseline order
template <class PK>
__device__ __forceinline__ cf32 cell_from_vis(const uint4 r, const float2 v0, const float2 v1, const float2 *__restrict__ vis,
                                              const float2 *__restrict__ cf, const int32_t *__restrict__ src) {
  const int flag = (r.x >> PK::kFlagSh) & 3, len = (int)(r.x >> PK::kLenSh);
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

// Phase G of a lane: descriptors and values of ITS L cells (positions base + 32 i) of snapshot s, channel ch
template <class PK>
__device__ __forceinline__ void cells_of_snapshot(const ImgParams &p, const float2 *__restrict__ uvsrc, const uint4 *__restrict__ rec,
                                                  const uint32_t *__restrict__ gm, cf32 *__restrict__ cvw, uint32_t *__restrict__ mp,
                                                  int L, int s, int ch, int n_pix) {
  for (int i = 0; i < L; ++i) mp[32 * i] = __ldg(gm + 32 * i);
  if (uvsrc != nullptr) {
    // blink_image: the plan's occupied cells with kx >= 0 straight from the uv grid (empty cells are
    // zero by contract and never read)
    const float2 *__restrict__ g = uvsrc + (size_t)s * n_pix * n_pix;
    for (int i = 0; i < L; ++i) {
      const uint4 rr = __ldg(rec + 32 * i);
      const int iy = (int)(rr.x & PK::kIyMask), flag = (rr.x >> PK::kFlagSh) & 3, kx = (rr.x >> PK::kKxSh) & PK::kKxMask;
      const float w = __uint_as_float(rr.y);
      float2 v = make_float2(0.f, 0.f);
      if (rr.x >> PK::kLenSh) v = __ldg(g + (size_t)iy * n_pix + kx);
      cvw[32 * i] = mk(v.x * w, (flag == kPlaceDirect || flag == kPlaceConj) ? v.y * w : 0.f);
    }
  } else {
    const float2 *__restrict__ vis = p.vis + (size_t)s * p.n_bl;
    const int32_t *__restrict__ src = p.src + (size_t)ch * p.n_bl;
    const float2 *__restrict__ cf = p.corr ? p.corr + (size_t)ch * p.n_bl : nullptr;
    for (int i0 = 0; i0 < L; i0 += 4) {            // four cells in flight
      uint4 rr[4];
      float2 v0[4], v1[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) rr[j] = i0 + j < L ? __ldg(rec + 32 * (i0 + j)) : make_uint4(0, 0, 0, 0);
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int len = (int)(rr[j].x >> PK::kLenSh);
        v0[j] = v1[j] = make_float2(0.f, 0.f);
        if (len >= 1) v0[j] = ld_vis(vis, cf, rr[j].z >> 1);
        if (len == 2) v1[j] = ld_vis(vis, cf, rr[j].w >> 1);
      }
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (i0 + j < L) cvw[32 * (i0 + j)] = (rr[j].x >> PK::kLenSh) ? cell_from_vis<PK>(rr[j], v0[j], v1[j], vis, cf, src) : mk(0.f, 0.f);
    }
  }
}

// wait of a warp that is ahead of the others: sleep between polls, so that the polling takes neither issue
// slots nor the shared-memory pipe from the warps it is waiting for
__device__ __forceinline__ void mbar_wait_idle(uint64_t *bar, uint32_t parity) {
  for (;;) {
    uint32_t done;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    if (done) break;
    __nanosleep(100);
  }
}

// steps Q0 .. Q0 + 3 of a lane's list: acc += G w1024^(iy r); an entry's last cell stores the sum.
// The factor comes from the special-function unit, not from a table: shared-memory bandwidth is what
// binds this kernel, and a 1024-entry table walked at stride iy r costs 5 wavefronts per step.  The
// descriptor carries iy in its top 10 bits, so the 32-bit product with r IS the angle as a signed
// binary fraction of a turn (mod 1 by overflow, in [-1/2, 1/2) where sin.approx / cos.approx are at
// their best: absolute error 2^-21.4, against 2^-24 for the table -- the image is a sum of ~7e3 such
// terms with unrelated errors, so this stays 1e2 below the 1e-4-of-peak bar; measured in DESIGN.md).
template <class PK>
__device__ __forceinline__ void bins4(const int Q0, const uint32_t *__restrict__ mp, const cf32 *__restrict__ cvp,
                                      unsigned char *__restrict__ zb, int r, int L, cf32 &acc) {
  cf32 v[4], w[4];
  uint32_t m[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const bool on = Q0 + j < L;                      // warp-uniform
    m[j] = on ? mp[32 * (Q0 + j)] : 0u;
    v[j] = on ? cvp[32 * (Q0 + j)] : mk(0.f, 0.f);
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int32_t P = (int32_t)((m[j] & PK::kAngleMask) * (uint32_t)r);           // turns * 2^32
    const float ang = (float)P * 1.4629180792671596e-9f;                          // 2 pi / 2^32
    w[j] = mk(__cosf(ang), __sinf(ang));
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    acc.x = fmaf(v[j].x, w[j].x, fmaf(-v[j].y, w[j].y, acc.x));
    acc.y = fmaf(v[j].x, w[j].y, fmaf(v[j].y, w[j].x, acc.y));
    if (m[j] & 1u) {
      *reinterpret_cast<cf32 *>(zb + (m[j] & 0xFFF8u)) = acc;
      acc = mk(0.f, 0.f);
    }
  }
}

__global__ void __launch_bounds__(kRThreads, 1) k_img1024r(const RParams q) {
  constexpr int N = kRN;
  using PK = RPack<10, 9>;
  const ImgParams &p = q.ip;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cf32 *twB = reinterpret_cast<cf32 *>(smem_raw + kROffTw);           // [n1][b] exp(2 pi i b n1 / 1024)
  uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + kROffBar); // full[2], empty[2]
  cf32 *cv = reinterpret_cast<cf32 *>(smem_raw + kROffCv);            // cell values of the snapshot, by position
  uint32_t *cmeta = reinterpret_cast<uint32_t *>(cv + q.cap);         // their descriptors (fixed per channel)
  const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;

  for (int i = tid; i < 1024; i += kRThreads) {
    twB[i] = __ldg(p.tw32 + i);
  }
  if (tid < 2) mbar_init(bars + tid, kRProd);
  else if (tid < 4) mbar_init(bars + tid, kRCons);
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();

  const long long T = (long long)q.n_snap * kRUnits;
  const long long u0 = T * blockIdx.x / gridDim.x, u1 = T * (blockIdx.x + 1) / gridDim.x;
  if (wv < kRProd) {
    // =================================================================== producers
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRRegsProd));
    const int k0 = 32 * ((wv + lane) & 15) + lane;          // this lane's column
    uint32_t cmask = 0;
    const cf32 *cvp = cv;
    uint32_t *mp = cmeta;
    int L = 0, s_cur = -1;
    long long n = 0;
    for (long long u = u0; u < u1; ++u, ++n) {
      const int s = (int)(u / kRUnits), r = (int)(u % kRUnits);
      if (s != s_cur) {
        // -------------------------------------------------------------- G: this lane's cells of the snapshot
        s_cur = s;
        const int ch = (s + p.ch0) % p.n_ch;
        const int32_t *gh = q.rhdr + ((size_t)ch * kRProd + wv) * kRHdr;
        const int base = __ldg(gh) + lane;
        L = __ldg(gh + 1);
        cmask = __ldg(q.rmask + (size_t)ch * kRW + k0);
        cvp = cv + base;
        mp = cmeta + base;
        cells_of_snapshot<PK>(p, q.uvsrc, q.rrec + (size_t)ch * q.cap + base, q.rmeta + (size_t)ch * q.cap + base, cv + base, mp, L,
                              p.snap_base + s, ch, N);
      }
      const int buf = (int)(n & 1);
      unsigned char *zbytes = smem_raw + buf * kRTile;
      if (n >= 2) mbar_wait_idle(bars + 2 + buf, (uint32_t)((n >> 1) - 1) & 1u);     // the consumers have left this tile
      // ---------------------------------------------------------------- S: the bins of this warp's columns
      {
        cf32 acc = mk(0.f, 0.f);
        if (L > 0) bins4<PK>(0, mp, cvp, zbytes, r, L, acc);
        if (L > 4) bins4<PK>(4, mp, cvp, zbytes, r, L, acc);
        if (L > 8) bins4<PK>(8, mp, cvp, zbytes, r, L, acc);
        if (L > 12) bins4<PK>(12, mp, cvp, zbytes, r, L, acc);
      }
      __syncwarp();
      // ---------------------------------------------------------------- A: this lane's column, in place
      {
        cf32 *zc = reinterpret_cast<cf32 *>(zbytes) + k0;
        cf32 t[16];
        if (__any_sync(0xffffffffu, cmask != 0)) {
#pragma unroll
          for (int c = 0; c < 16; ++c) t[c] = ((cmask >> c) & 1u) ? zc[c * kRW] : mk(0.f, 0.f);
          dft16(t);                                                   // t[y'] = U[64 y' + r][k]
#pragma unroll
          for (int pp = 0; pp < 8; ++pp) {
            const cf32 A = t[pp], B = t[pp + 8];
            zc[pp * kRW] = mk(A.x - B.y, A.y + B.x);                  // U[y] + i U[y + 512]
            zc[(8 + pp) * kRW] = mk(A.x + B.y, B.x - A.y);            // conj U[y] + i conj U[y + 512]
          }
        } else {
#pragma unroll
          for (int c = 0; c < 16; ++c) zc[c * kRW] = mk(0.f, 0.f);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bars + buf);
    }
  } else {
    // =================================================================== consumers: row pair p
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRRegsCons));
    const int pr = wv - kRProd;
    long long n = 0;
    for (long long u = u0; u < u1; ++u, ++n) {
      const int s = (int)(u / kRUnits), r = (int)(u % kRUnits);
      const int buf = (int)(n & 1);
      cf32 *zb = reinterpret_cast<cf32 *>(smem_raw + buf * kRTile);
      mbar_wait(bars + buf, (uint32_t)(n >> 1) & 1u);
      // lane b holds Z[32 a + b]: a < 16 from row p (kx = 32 a + b), a >= 16 the mirrored half from row
      // 8 + p at kx = 1024 - 32 a - b (kx = 512 does not exist: zero)
      cf32 t[32];
      const cf32 *za = zb + pr * kRW + lane;
      const cf32 *zm = zb + (8 + pr) * kRW - lane;
#pragma unroll
      for (int a = 0; a < 16; ++a) t[a] = za[32 * a];
      t[16] = lane == 0 ? mk(0.f, 0.f) : zm[512];
#pragma unroll
      for (int a = 17; a < 32; ++a) t[a] = zm[32 * (32 - a)];
      __syncwarp();
      dft32(t);
#pragma unroll
      for (int n1 = 1; n1 < 32; ++n1) t[n1] = cmul(t[n1], twB[n1 * 32 + lane]);
      // exchange through the warp's own two rows (1024 slots, no room for padding): lane b writes its
      // pairs (n1 = 2 j, 2 j + 1) as 16 bytes at pair slot j xor (b mod 16) of row segment b, lane n1
      // reads element (b, n1) from pair slot (n1 / 2) xor (b mod 16): 16-byte stores (per quarter warp) and
      // 8-byte loads (per half warp) are both conflict-free, and every address is one XOR from a lane constant
      {
        unsigned char *seg = reinterpret_cast<unsigned char *>(zb + ((lane & 16) ? (8 + pr) * kRW : pr * kRW)) + (lane & 15) * 256;
        const uint32_t wx = (uint32_t)(lane & 15) << 4;
#pragma unroll
        for (int j = 0; j < 16; ++j)
          *reinterpret_cast<float4 *>(seg + (wx ^ (uint32_t)(j << 4))) = make_float4(t[2 * j].x, t[2 * j].y, t[2 * j + 1].x, t[2 * j + 1].y);
      }
      __syncwarp();
      {
        const unsigned char *row0 = reinterpret_cast<const unsigned char *>(zb + pr * kRW);
        const unsigned char *row1 = reinterpret_cast<const unsigned char *>(zb + (8 + pr) * kRW);
        const uint32_t rx = ((uint32_t)(lane >> 1) << 4) | ((uint32_t)(lane & 1) << 3);
#pragma unroll
        for (int b = 0; b < 16; ++b) {
          const uint32_t o = (rx ^ (uint32_t)(b << 4)) + (uint32_t)(b * 256);
          t[b] = *reinterpret_cast<const cf32 *>(row0 + o);
          t[b + 16] = *reinterpret_cast<const cf32 *>(row1 + o);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bars + 2 + buf);
      dft32(t);
      float *__restrict__ r0 = p.img + ((size_t)(p.snap_base + s) * N + kRUnits * pr + r) * N + lane;
      float *__restrict__ r1 = r0 + (size_t)(N / 2) * N;
#pragma unroll
      for (int n2 = 0; n2 < 32; ++n2) {
        __stcs(r0 + 32 * n2, t[n2].x);
        __stcs(r1 + 32 * n2, t[n2].y);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------
// k_cols_res: the column pass (steps a1-a3 and the first half of a4) of the two-kernel routes at N = 2048 /
// 4096 for sparse half-planes at most 1024 columns wide (MWA Phase II: 7.5e3 occupied cells of 3.5e6), by
// the same residue classes: y = (N / 8) y' + r, eight bins per column (iy mod 8), dft8, and the eight rows
// U[(N / 8) y' + r][0 .. wu) of a unit leave the 8 x 1024 tile as bulk copies into the plan's U scratch,
// where k_image_rows picks them up.  The direct sums of k_cols_from_vis cost N complex multiply-adds per
// cell and column; here a cell costs N / 8 (one per unit) plus its column's butterflies.  One persistent CTA
// of 16 warps per SM, every warp in phases S and A (two columns per lane, dealt by the plan so that the
// warps carry the same number of cells), two tiles so that a unit's copies drain during the next unit.
template <int LOGN>
__global__ void __launch_bounds__(kCThreads, 1) k_cols_res(const RParams q) {
  constexpr int N = 1 << LOGN, R = N / kCRows;
  using PK = RPack<LOGN, 10>;
  const ImgParams &p = q.ip;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cf32 *cv = reinterpret_cast<cf32 *>(smem_raw + kCOffCv);            // cell values of the snapshot, by position
  uint32_t *cmeta = reinterpret_cast<uint32_t *>(cv + q.cap);         // their descriptors (fixed per channel)
  const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;
  const int k0 = __ldg(q.rcols + (wv * 32 + lane) * 2), k1 = __ldg(q.rcols + (wv * 32 + lane) * 2 + 1);
  const long long T = (long long)q.n_snap * R;
  const long long u0 = T * blockIdx.x / gridDim.x, u1 = T * (blockIdx.x + 1) / gridDim.x;
  uint32_t cmask0 = 0, cmask1 = 0;
  const cf32 *cvp = cv;
  uint32_t *mp = cmeta;
  int L = 0, s_cur = -1;
  long long n = 0;
  for (long long u = u0; u < u1; ++u, ++n) {
    const int sl = (int)(u / R), r = (int)(u % R);
    if (sl != s_cur) {
      // ---------------------------------------------------------------- G: this lane's cells of the snapshot
      s_cur = sl;
      const int s = p.snap_base + sl, ch = (s + p.ch0) % p.n_ch;
      const int32_t *gh = q.rhdr + ((size_t)ch * kRProd + wv) * kRHdr;
      const int base = __ldg(gh) + lane;
      L = __ldg(gh + 1);
      cmask0 = __ldg(q.rmask + (size_t)ch * kCW + k0);
      cmask1 = __ldg(q.rmask + (size_t)ch * kCW + k1);
      cvp = cv + base;
      mp = cmeta + base;
      cells_of_snapshot<PK>(p, q.uvsrc, q.rrec + (size_t)ch * q.cap + base, q.rmeta + (size_t)ch * q.cap + base, cv + base, mp, L, s,
                            ch, N);
    }
    const int buf = (int)(n & 1);
    unsigned char *zb = smem_raw + buf * kCTile;
    // (this tile was last read by the copies of unit n - 2: complete before the barrier of unit n - 1)
    // ------------------------------------------------------------------ S: the bins of this warp's columns
    {
      cf32 acc = mk(0.f, 0.f);
      for (int q0 = 0; q0 < L; q0 += 4) bins4<PK>(q0, mp, cvp, zb, r, L, acc);
    }
    __syncwarp();
    // ------------------------------------------------------------------ A: this lane's two columns, in place
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      cf32 *zc = reinterpret_cast<cf32 *>(zb) + (j ? k1 : k0);
      const uint32_t cm = j ? cmask1 : cmask0;
      cf32 t[kCRows];
#pragma unroll
      for (int c = 0; c < kCRows; ++c) t[c] = ((cm >> c) & 1u) ? zc[c * kCW] : mk(0.f, 0.f);
      if (cm != 0) dft8(t);                                           // t[y'] = U[(N / 8) y' + r][k]
#pragma unroll
      for (int c = 0; c < kCRows; ++c) zc[c * kCW] = t[c];
    }
    fence_async_smem();                                // the tile's generic writes before the copy engine reads it
    if (tid == 0 && n >= 1) bulk_wait_read<0>();       // the previous unit's copies have read the other tile: free for the next unit
    __syncthreads();                                   // the one barrier of a unit
    if (tid == 0) {
      float2 *__restrict__ U = p.U + ((size_t)sl * N + r) * p.wu;
#pragma unroll
      for (int y1 = 0; y1 < kCRows; ++y1)
        bulk_store(U + (size_t)y1 * R * p.wu, reinterpret_cast<cf32 *>(zb) + y1 * kCW, (uint32_t)(p.wu * sizeof(cf32)));
      bulk_commit();
    }
  }
  if (tid == 0) bulk_wait_all();
}

// ---- plan side ----------------------------------------------------------------------------------------
struct RCell { int k, iy, seg, len, flag; float w; };
struct RTables {                       // per producer warp: L steps, 32 L records / descriptors (lane-interleaved)
  std::vector<uint4> rec[kRProd];
  std::vector<uint32_t> meta[kRProd];
  int L[kRProd] = {0};
  std::vector<uint32_t> mask;
  bool ok = true;
};

// geometry of a residue-class kernel's tables: N = 2^logn grid, 2^logw tile columns, `rows` bins per column
// (= tile rows = rows of the column butterfly), longest lane list, and the producer warp that owns each column
// (the lane is always kx mod 32, so that a warp's column accesses hit 32 different banks)
struct RGeom {
  int logn, logw, rows, lmax;
  std::vector<int> owner;          // [2^logw] warp of column kx
};

static void half_plane_cells(const HostGather &g, int N, int weighting, float inv_norm, std::vector<RCell> &cells) {
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
  std::sort(cells.begin(), cells.end(), [](const RCell &a, const RCell &b) { return a.k != b.k ? a.k < b.k : a.iy < b.iy; });
}

// the tables of one channel
static void res_tables(const HostGather &g, const RGeom &gm, int weighting, float inv_norm, RTables &o) {
  const int N = 1 << gm.logn, W = 1 << gm.logw;
  std::vector<RCell> cells;
  half_plane_cells(g, N, weighting, inv_norm, cells);
  // entries (column, bin) per owning warp; the cells of an entry in ascending iy
  std::vector<std::map<int, std::vector<int>>> ent(kRProd);
  o.mask.assign(W, 0u);
  for (int i = 0; i < (int)cells.size(); ++i) {
    const int k = cells[i].k, c = cells[i].iy & (gm.rows - 1);
    ent[gm.owner[k]][c * W + k].push_back(i);
    o.mask[k] |= 1u << c;
  }
  for (int w = 0; w < kRProd; ++w) {
    // longest entry first to the lane with the fewest cells so far (ties: lowest lane)
    std::vector<std::pair<int, int>> order;      // (-len, slot)
    for (auto &kv : ent[w]) order.push_back({-(int)kv.second.size(), kv.first});
    std::sort(order.begin(), order.end());
    // Among the lanes within one cell of the lightest, one whose half-warp has no other entry ending at
    // the same step in the same bank pair (the tile store of that step is then conflict-free).
    std::vector<std::vector<int>> mine(32);      // slots of each lane's entries, in the order it walks them
    int load[32] = {0};
    std::vector<std::array<unsigned char, 32>> used;    // [end step][half-warp * 16 + bank pair]
    for (auto &od : order) {
      const int len = -od.first, bank = od.second & 15;
      int lo = load[0];
      for (int l = 1; l < 32; ++l) lo = std::min(lo, load[l]);
      int best = -1, best_cost = 1 << 30;
      for (int l = 0; l < 32; ++l) {
        if (load[l] > lo + 1) continue;
        const size_t end = (size_t)load[l] + len - 1;
        const int clash = end < used.size() ? used[end][(l >> 4) * 16 + bank] : 0;
        const int cost = clash * 4 + (load[l] - lo);
        if (cost < best_cost) { best_cost = cost; best = l; }
      }
      const size_t end = (size_t)load[best] + len - 1;
      if (used.size() <= end) used.resize(end + 1, std::array<unsigned char, 32>{});
      ++used[end][(best >> 4) * 16 + bank];
      mine[best].push_back(od.second);
      load[best] += len;
    }
    int L = 0;
    for (int l = 0; l < 32; ++l) L = std::max(L, load[l]);
    if (L > gm.lmax) { o.ok = false; return; }
    o.L[w] = L;
    const size_t r0 = 0;
    o.rec[w].assign((size_t)32 * L, make_uint4(0, 0, 0, 0));
    o.meta[w].assign((size_t)32 * L, 0u);
    for (int l = 0; l < 32; ++l) {
      int qpos = 0;
      for (size_t n = 0; n < mine[l].size(); ++n) {
        const std::vector<int> &cl = ent[w][mine[l][n]];
        for (size_t i = 0; i < cl.size(); ++i, ++qpos) {
          const RCell &c = cells[cl[i]];
          uint32_t wbits;
          memcpy(&wbits, &c.w, 4);
          o.rec[w][r0 + 32 * (size_t)qpos + l] =
              make_uint4((uint32_t)c.iy | ((uint32_t)c.flag << gm.logn) | ((uint32_t)c.k << (gm.logn + 2)) |
                             ((uint32_t)c.len << (gm.logn + 2 + gm.logw)), wbits,
                         (uint32_t)g.src[c.seg], c.len == 2 ? (uint32_t)g.src[c.seg + 1] : (uint32_t)c.seg);
          o.meta[w][r0 + 32 * (size_t)qpos + l] = ((uint32_t)c.iy << (32 - gm.logn)) | (i + 1 == cl.size() ? 1u : 0u) | (uint32_t)(8 * mine[l][n]);
        }
      }
    }
  }
}

static size_t res_smem(int cap) { return kROffCv + (size_t)cap * (sizeof(cf32) + sizeof(uint32_t)); }

void res_route_free(blink_plan *p) {
  cudaFree(p->d_rrec); cudaFree(p->d_rmeta); cudaFree(p->d_rhdr); cudaFree(p->d_rmask); cudaFree(p->d_rcols);
  p->d_rrec = nullptr; p->d_rmeta = nullptr; p->d_rhdr = nullptr; p->d_rmask = nullptr; p->d_rcols = nullptr;
  p->res_route = 0;
}

static size_t cols_smem(int cap) { return kCOffCv + (size_t)cap * (sizeof(cf32) + sizeof(uint32_t)); }

// k_img1024r: column 32 a + b belongs to warp (a - b) mod 16
static RGeom geom_1024() {
  RGeom gm{10, 9, kRRows, kRLmax, std::vector<int>(kRW)};
  for (int k = 0; k < kRW; ++k) gm.owner[k] = ((k >> 5) - (k & 31)) & 15;
  return gm;
}

// k_cols_res: 1024 tile columns, two per lane.  For every b = kx mod 32 the 32 columns 32 a + b go, heaviest
// first (occupied cells over all channels), to the warp with the fewest cells so far that still has a free
// slot for this b -- the column density of a centrally condensed array falls by 10x from kx = 0 outwards.
static RGeom geom_cols(const std::vector<HostGather> &gathers, int N, std::vector<int16_t> &cols) {
  const int logn = N == 2048 ? 11 : 12;
  RGeom gm{logn, 10, kCRows, kCLmax, std::vector<int>(kCW, 0)};
  std::vector<long long> wcol(kCW, 0);
  for (const HostGather &g : gathers)
    for (int j = 0; j < g.n_can; ++j) {
      const int ix = g.can_cell[j] % N, kx = ix < N / 2 ? ix : ix - N;
      if (std::abs(kx) < kCW) ++wcol[std::abs(kx)];
    }
  long long load[kRProd] = {0};
  cols.assign((size_t)kRProd * 32 * 2, 0);
  for (int b = 0; b < 32; ++b) {
    int order[32], used[kRProd] = {0};
    for (int a = 0; a < 32; ++a) order[a] = 32 * a + b;
    std::sort(order, order + 32, [&](int x, int y) { return wcol[x] != wcol[y] ? wcol[x] > wcol[y] : x < y; });
    for (int i = 0; i < 32; ++i) {
      int best = -1;
      for (int w = 0; w < kRProd; ++w)
        if (used[w] < 2 && (best < 0 || load[w] < load[best])) best = w;
      gm.owner[order[i]] = best;
      cols[((size_t)best * 32 + b) * 2 + used[best]] = (int16_t)order[i];
      ++used[best];
      load[best] += wcol[order[i]];
    }
  }
  return gm;
}

// Residue-class routes.  N = 1024 (res_route 1, k_img1024r: the whole of blink_grid_image / blink_image)
// applies when every lane's list of cells is at most kRLmax long (8192 occupied half-plane cells in all,
// dealt evenly) and the cell values fit in shared memory beside the tiles; N = 2048 / 4096 (res_route 2,
// k_cols_res: the column pass of the two-kernel routes) when the half-plane is at most 1024 columns wide
// and its cells fit beside the two 8 x 1024 tiles.
int res_route_build(blink_plan *p, cudaStream_t st) {
  p->res_route = 0;
  if (p->opt.warp_route == -1 || p->opt.warp_route == 2 || p->max_smem_optin <= 0) return BLINK_OK;
  const int N = p->n_pix, route = N == kRN ? 1 : ((N == 2048 || N == 4096) ? 2 : 0);
  if (route == 0) return BLINK_OK;
  std::vector<int16_t> h_cols;
  const RGeom gm = route == 1 ? geom_1024() : geom_cols(p->gathers, N, h_cols);
  const int W = 1 << gm.logw;
  // wide, sparsely filled half-planes only: a compact array (a station imaged at 1024^2: 40 columns, 14 baselines
  // per cell) is faster on the line kernels (measured 6.8 ms against 8.3 ms per 4000 snapshots)
  if (p->wu < 256 || p->wu > W || p->seg_len_max > (int)((1u << (32 - (gm.logn + 2 + gm.logw))) - 1u)) return BLINK_OK;
  const int n_ch = p->n_ch;
  std::vector<RTables> tb(n_ch);
  parallel_for(n_ch, [&](int ch) { res_tables(p->gathers[ch], gm, p->weighting, p->chinfo[ch].inv_norm, tb[ch]); });
  // A warp's positions start at the same place for every channel (its longest list over the channels
  // decides): its lanes rewrite their own values at a snapshot change while other warps still walk theirs.
  int base[kRProd + 1] = {0};
  for (int ch = 0; ch < n_ch; ++ch)
    if (!tb[ch].ok) return BLINK_OK;
  for (int w = 0; w < kRProd; ++w) {
    int lmax = 0;
    for (int ch = 0; ch < n_ch; ++ch) lmax = std::max(lmax, tb[ch].L[w]);
    base[w + 1] = base[w] + 32 * lmax;
  }
  const int cap = std::max(16, base[kRProd]);
  if ((route == 1 ? res_smem(cap) : cols_smem(cap)) > (size_t)p->max_smem_optin) return BLINK_OK;
  std::vector<uint4> h_rec((size_t)n_ch * cap, make_uint4(0, 0, 0, 0));
  std::vector<uint32_t> h_meta((size_t)n_ch * cap, 0u);
  std::vector<int32_t> h_hdr((size_t)n_ch * kRProd * kRHdr, 0);
  std::vector<uint32_t> h_mask((size_t)n_ch * W, 0u);
  for (int ch = 0; ch < n_ch; ++ch) {
    for (int w = 0; w < kRProd; ++w) {
      std::copy(tb[ch].rec[w].begin(), tb[ch].rec[w].end(), h_rec.begin() + (size_t)ch * cap + base[w]);
      std::copy(tb[ch].meta[w].begin(), tb[ch].meta[w].end(), h_meta.begin() + (size_t)ch * cap + base[w]);
      h_hdr[((size_t)ch * kRProd + w) * kRHdr] = base[w];
      h_hdr[((size_t)ch * kRProd + w) * kRHdr + 1] = tb[ch].L[w];
    }
    std::copy(tb[ch].mask.begin(), tb[ch].mask.end(), h_mask.begin() + (size_t)ch * W);
  }
  int rc;
  if ((rc = upload_table((void **)&p->d_rrec, h_rec.data(), sizeof(uint4) * h_rec.size(), st, "residue route records")) != BLINK_OK) return rc;
  if ((rc = upload_table((void **)&p->d_rmeta, h_meta.data(), sizeof(uint32_t) * h_meta.size(), st, "residue route descriptors")) != BLINK_OK) return rc;
  if ((rc = upload_table((void **)&p->d_rhdr, h_hdr.data(), sizeof(int32_t) * h_hdr.size(), st, "residue route headers")) != BLINK_OK) return rc;
  if ((rc = upload_table((void **)&p->d_rmask, h_mask.data(), sizeof(uint32_t) * h_mask.size(), st, "residue route masks")) != BLINK_OK) return rc;
  if (route == 2 &&
      (rc = upload_table((void **)&p->d_rcols, h_cols.data(), sizeof(int16_t) * h_cols.size(), st, "residue route columns")) != BLINK_OK)
    return rc;
  BLINK_CUDA_TRY(cudaStreamSynchronize(st), "residue route upload");
  p->res_cap = cap;
  p->res_route = route;
  return BLINK_OK;
}

int launch_img1024r(const blink_plan *p, ImgParams ip, int n_snap, cudaStream_t st) {
  if (n_snap <= 0) return BLINK_OK;
  RParams q;
  q.n_snap = n_snap;
  q.cap = p->res_cap;
  q.rrec = p->d_rrec; q.rmeta = p->d_rmeta; q.rhdr = p->d_rhdr; q.rmask = p->d_rmask; q.rcols = nullptr;
  q.uvsrc = ip.vis == nullptr ? ip.uv : nullptr;
  ip.snap_base = 0;
  q.ip = ip;
  const size_t smem = res_smem(p->res_cap);
  static std::atomic<uint64_t> attr{0};
  const int rc = ensure_max_smem(k_img1024r, p, attr, "k_img1024r smem attribute");
  if (rc != BLINK_OK) return rc;
  // one CTA per SM; fewer when there are fewer units than that
  const long long units = (long long)n_snap * kRUnits;
  const int grid = (int)std::min<long long>(p->sm_count, units);
  k_img1024r<<<grid, kRThreads, smem, st>>>(q);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_img1024r launch");
  return BLINK_OK;
}

template <int LOGN> static int launch_cols_res_n(const blink_plan *p, const RParams &q, cudaStream_t st) {
  static std::atomic<uint64_t> attr{0};
  const int rc = ensure_max_smem(k_cols_res<LOGN>, p, attr, "k_cols_res smem attribute");
  if (rc != BLINK_OK) return rc;
  const long long units = (long long)q.n_snap * ((1 << LOGN) / kCRows);
  const int grid = (int)std::min<long long>(p->sm_count, units);
  k_cols_res<LOGN><<<grid, kCThreads, cols_smem(p->res_cap), st>>>(q);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_cols_res launch");
  return BLINK_OK;
}

// pass A of a chunk of n_snap snapshots (ip.snap_base = the chunk's first) into the plan's U scratch
int launch_cols_res(const blink_plan *p, const ImgParams &ip, int n_snap, cudaStream_t st) {
  if (n_snap <= 0) return BLINK_OK;
  RParams q;
  q.n_snap = n_snap;
  q.cap = p->res_cap;
  q.rrec = p->d_rrec; q.rmeta = p->d_rmeta; q.rhdr = p->d_rhdr; q.rmask = p->d_rmask; q.rcols = p->d_rcols;
  q.uvsrc = ip.vis == nullptr ? ip.uv : nullptr;
  q.ip = ip;
  return p->n_pix == 2048 ? launch_cols_res_n<11>(p, q, st) : launch_cols_res_n<12>(p, q, st);
}

}  // namespace blink

#ifdef BLINK_TESTING_HOOKS   // libblink_testing.so only (build.py): libblink.so carries no host model and no probe
// Host model of the residue-class kernels for ONE channel and ONE snapshot (tests without a GPU): builds the
// tables exactly as res_route_build does and walks them the way the kernels do -- phase G (cell values from
// the records), phase S (lane lists -> bins; the tile starts as NaN, so a bin read that was never written
// shows), phase A (masked bins -> column DFT; at N = 1024 also the row-pass operands in place) and the row
// pass -- in fp64 with direct DFT sums instead of the butterflies, for the listed units.  N = 1024:
// k_img1024r (16 rows per unit); N = 2048 / 4096: k_cols_res (8 rows per unit, columns dealt to warps by
// cell count), followed by a plain Hermitian row sum in place of k_image_rows.
extern "C" int blink_host_residue_emulate(const int32_t *cell, int n_bl, int n_pix, int weighting, const float *vis, int n_units,
                                          const int32_t *units, float *rows, int32_t *stats) {
  using namespace blink;
  if (!cell || !vis || !rows || !units || n_bl < 1 || n_units < 0 || (weighting != BLINK_NATURAL && weighting != BLINK_UNIFORM))
    return BLINK_EINVAL;
  if (n_pix != 1024 && n_pix != 2048 && n_pix != 4096) return BLINK_EUNSUPPORTED;
  const int N = n_pix;
  HostGather g;
  int rc = build_gather_host(cell, n_bl, N, g);
  if (rc != BLINK_OK) return rc;
  long long wsum = 0, n_occ = 0;
  for (int j = 0; j < g.n_can; ++j) {
    wsum += 2LL * (g.seg_start[j + 1] - g.seg_start[j]);
    n_occ += g.can_cell[j] == 0 ? 1 : 2;
  }
  const double norm = weighting == BLINK_NATURAL ? (double)wsum : (double)n_occ;
  const float inv_norm = norm > 0.0 ? (float)(1.0 / norm) : 0.f;
  std::vector<int16_t> cols;
  const RGeom gm = N == kRN ? geom_1024() : geom_cols(std::vector<HostGather>{g}, N, cols);
  const int W = 1 << gm.logw, ROWS = gm.rows, n_classes = N / ROWS, len_sh = gm.logn + 2 + gm.logw;
  RTables tb;
  res_tables(g, gm, weighting, inv_norm, tb);
  if (!tb.ok) return BLINK_EUNSUPPORTED;
  typedef std::complex<double> cd;
  const double tau = 6.283185307179586476925286766559;
  // phase G
  std::vector<cd> cv[kRProd];
  int lmax = 0, npos = 0;
  for (int w = 0; w < kRProd; ++w) {
    lmax = std::max(lmax, tb.L[w]);
    npos += 32 * tb.L[w];
    cv[w].assign((size_t)32 * tb.L[w], cd(0.0, 0.0));
    for (size_t i = 0; i < cv[w].size(); ++i) {
      const uint4 r = tb.rec[w][i];
      const int flag = (r.x >> gm.logn) & 3, len = (int)(r.x >> len_sh);
      if (len == 0) continue;
      float wt;
      memcpy(&wt, &r.y, 4);
      double ar = 0.0, ai = 0.0;
      for (int q = 0; q < len; ++q) {
        const int code = q == 0 ? (int)r.z : (len == 2 ? (int)r.w : g.src[(int)r.w + q]);
        const int bl = code >> 1;
        ar += vis[2 * bl];
        ai += (code & 1) ? -(double)vis[2 * bl + 1] : (double)vis[2 * bl + 1];
      }
      if (flag == kPlaceDirect) cv[w][i] = cd(ar * wt, ai * wt);
      else if (flag == kPlaceConj) cv[w][i] = cd(ar * wt, -ai * wt);
      else cv[w][i] = cd(2.0 * ar * wt, 0.0);
    }
  }
  if (stats) { stats[0] = npos; stats[1] = lmax; stats[2] = g.n_can; }
  const double nan = std::nan("");
  const uint32_t angle_mask = ~0u << (32 - gm.logn);
  std::vector<cd> tile((size_t)ROWS * W), Z(N);
  // the kernels' column ownership: k_img1024r warp w, lane b: column 32 ((w + b) mod 16) + b; k_cols_res: the dealt table
  auto column_of = [&](int w, int b, int j) { return N == kRN ? 32 * ((w + b) & 15) + b : (int)cols[((size_t)w * 32 + b) * 2 + j]; };
  const int cpl = N == kRN ? 1 : 2;
  for (int iu = 0; iu < n_units; ++iu) {
    const int r = units[iu];
    if (r < 0 || r >= n_classes) return BLINK_EINVAL;
    std::fill(tile.begin(), tile.end(), cd(nan, nan));
    // phase S
    for (int w = 0; w < kRProd; ++w)
      for (int l = 0; l < 32; ++l) {
        cd acc(0.0, 0.0);
        for (int q = 0; q < tb.L[w]; ++q) {
          const uint32_t m = tb.meta[w][(size_t)32 * q + l];
          const int32_t P = (int32_t)((m & angle_mask) * (uint32_t)r);
          const double ang = (double)P * (tau / 4294967296.0);
          acc += cv[w][(size_t)32 * q + l] * cd(cos(ang), sin(ang));
          if (m & 1u) {
            tile[(m & 0xFFF8u) >> 3] = acc;
            acc = cd(0.0, 0.0);
          }
        }
      }
    // phase A
    for (int w = 0; w < kRProd; ++w)
      for (int b = 0; b < 32; ++b)
        for (int j = 0; j < cpl; ++j) {
          const int k = column_of(w, b, j);
          if ((k & 31) != b || gm.owner[k] != w) return BLINK_EINVAL;      // a lane's columns sit in its own bank
          std::vector<cd> t(ROWS), U(ROWS);
          for (int c = 0; c < ROWS; ++c) t[c] = ((tb.mask[k] >> c) & 1u) ? tile[(size_t)c * W + k] : cd(0.0, 0.0);
          for (int y1 = 0; y1 < ROWS; ++y1) {
            cd a(0.0, 0.0);
            for (int c = 0; c < ROWS; ++c) a += t[c] * std::polar(1.0, tau * (double)((c * y1) % ROWS) / ROWS);
            U[y1] = a;
          }
          if (N == kRN) {
            for (int pp = 0; pp < ROWS / 2; ++pp) {
              const cd A = U[pp], B = U[pp + ROWS / 2];
              tile[(size_t)pp * W + k] = A + cd(0.0, 1.0) * B;
              tile[(size_t)(ROWS / 2 + pp) * W + k] = std::conj(A) + cd(0.0, 1.0) * std::conj(B);
            }
          } else {
            for (int y1 = 0; y1 < ROWS; ++y1) tile[(size_t)y1 * W + k] = U[y1];
          }
        }
    if (N == kRN) {
      // phase B of k_img1024r
      for (int pr = 0; pr < ROWS / 2; ++pr) {
        for (int kk = 0; kk < N; ++kk) {
          if (kk < W) Z[kk] = tile[(size_t)pr * W + kk];
          else if (kk == W) Z[kk] = cd(0.0, 0.0);
          else Z[kk] = tile[(size_t)(ROWS / 2 + pr) * W + (N - kk)];
        }
        float *r0 = rows + ((size_t)iu * ROWS + pr) * N, *r1 = rows + ((size_t)iu * ROWS + ROWS / 2 + pr) * N;
        for (int x = 0; x < N; ++x) {
          cd a(0.0, 0.0);
          for (int kk = 0; kk < N; ++kk) a += Z[kk] * std::polar(1.0, tau * (double)((kk * x) % N) / N);
          r0[x] = (float)a.real();      // image row 64 pr + r
          r1[x] = (float)a.imag();      // image row 64 pr + r + 512
        }
      }
    } else {
      // in place of k_image_rows: I[y][x] = Re U[y][0] + 2 Re sum_{kx > 0} U[y][kx] e^{2 pi i kx x / N}
      std::vector<cd> ph(N);
      for (int m = 0; m < N; ++m) ph[m] = std::polar(1.0, tau * (double)m / N);
      for (int y1 = 0; y1 < ROWS; ++y1) {
        float *ro = rows + ((size_t)iu * ROWS + y1) * N;       // image row (N / 8) y1 + r
        for (int x = 0; x < N; ++x) {
          double a = tile[(size_t)y1 * W].real();
          for (int kk = 1; kk < W; ++kk) a += 2.0 * (tile[(size_t)y1 * W + kk] * ph[(int)(((long long)kk * x) % N)]).real();
          ro[x] = (float)a;
        }
      }
    }
  }
  return BLINK_OK;
}
#endif  // BLINK_TESTING_HOOKS
