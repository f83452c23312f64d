// blink_fused.cu -- blink_grid_image: steps a1-a5 in one call.
//
// Chunked route: the batch is cut into chunks of a few snapshots; each chunk is gridded into a
// small plan-owned uv scratch and imaged from it straight away, so the uv grids are written and
// read back while still resident in the 126 MB L2 and (ideally) never reach HBM: the DRAM traffic
// of a snapshot falls from 8 n_bl + 20 N^2 towards 8 n_bl + 4 N^2 bytes.
#include <algorithm>

#include "blink_internal.h"
#include "fft_core.cuh"
#include "sphase.cuh"

namespace blink {
using namespace blinkfft;

// ---------------------------------------------------------------------------------------------
// Shared-memory route.  One persistent CTA per SM images one snapshot at a time without the uv
// grid ever leaving the SM:
//   phase S   the snapshot's visibilities arrive in shared memory in INPUT order, in chunks of
//             `chunk_vis` baselines, by bulk asynchronous copies (cp.async.bulk global -> shared,
//             completion on an mbarrier; no thread instructions, no registers).  For every chunk
//             one thread per canonical (half-plane) cell walks the plan's rank-major gather list
//             -- (local baseline | conj << 15), two ranks per 32-bit word -- and adds its
//             visibilities in ascending baseline order into S[j].  No atomics, no scatter.
//             Chunk buffers: one dedicated (so the first chunk of the NEXT snapshot streams in
//             during passes A and B) plus as many as fit in the space of the column lines and the
//             pass-B exchange lines, which are idle during phase S.
//   phase H   the occupied cells with kx >= 0 are written, already weighted, normalised and
//             sign-flipped for the fftshift, into per-column lines in shared memory (the grid is
//             exactly Hermitian by construction, so the half-plane is all that is needed);
//   pass A    column transforms along ky, in place in the lines, loads pruned to the bounding box;
//   pass B    row transforms, two real image rows per complex transform, read from the lines across
//             columns and stored to global memory straight from the last butterfly stage.
// A transform is owned by T = N/16 <= 16 lanes of one warp, so the exchanges inside it need only
// __syncwarp.  The last-stage twiddles depend only on the lane, so they live in registers for the
// whole kernel.
struct FusedParams {
  const float2 *vis;
  float *img;
  const ChannelInfo *chinfo;
  const uint2 *frec;        // [n_ch][n_chunk][n_can_max]  {j | len << 16, ranks 0,1 of the gather list}
  const uint32_t *fpair;    // [n_ch][n_chunk][chunk_vis]  rows q >= 1: ranks 2q, 2q+1
  const int2 *frow;         // [n_ch][n_chunk][frow_stride] row q: {offset into fpair, cells with len > 2q}
  const int32_t *hpos, *hcode;
  const float *hw;
  const float2 *tw;
  int n_bl, n_ch, n_snap, n_can_max, n_chunk, chunk_vis, nbuf, frow_stride, n_col, h_max;
  uint32_t off_dedicated, off_S, off_bar;   // byte offsets into dynamic shared memory
};

constexpr int kHPer = 5;       // phase-H table entries fetched per thread at a time
constexpr int kCellsPf = 5;    // cells per thread whose records are prefetched ahead of the data

int fused_line_stride(int n_pix) { return ((n_pix + n_pix / 16 + 15) / 16) * 16 + 1; }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!done);
}
// bulk copy global -> shared of `bytes` (multiple of 16, both addresses 16-byte aligned); SASS UBLKCP
__device__ __forceinline__ void bulk_load(void *sdst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(sdst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// one gather-list entry: add (conj-flagged) visibility e of the chunk to the accumulator
__device__ __forceinline__ void add_entry(const float2 *__restrict__ buf, uint32_t e, float &ax, float &ay) {
  const float2 v = buf[e & 0x7FFFu];
  ax += v.x;
  ay += __uint_as_float(__float_as_uint(v.y) ^ ((e & 0x8000u) << 16));
}

template <int N, int THREADS>
__global__ void __launch_bounds__(THREADS, 1) k_fused(const FusedParams p) {
  constexpr int T = N / 16;             // lanes per transform
  constexpr int G = THREADS / T;        // transforms in flight per CTA
  constexpr int LS = ((LineSize<N>::value + 15) / 16) * 16 + 1;
  constexpr int LSB = LineSize<N>::value;
  using F = Fft<N>;
  static_assert(F::NSTAGE == 2 && T <= 32, "shared-memory route needs a two-stage warp-local transform");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float2 *lines = reinterpret_cast<float2 *>(smem_raw);                       // [n_col][LS]
  float2 *X = lines + (size_t)p.n_col * LS;                                   // exchange lines [G][LSB]
  float2 *S = reinterpret_cast<float2 *>(smem_raw + p.off_S);                 // [n_can_max]
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + p.off_bar);         // [nbuf]
  const int tid = threadIdx.x;
  const int grp = tid / T, t = tid % T;
  const uint32_t chunk_bytes = (uint32_t)p.chunk_vis * sizeof(float2);
  // chunk c of every snapshot lives in buffer c % nbuf; buffer 0 is the dedicated one, the others
  // alias the lines / exchange area
  auto buf_of = [&](int b) -> float2 * {
    return reinterpret_cast<float2 *>(b == 0 ? smem_raw + p.off_dedicated : smem_raw + (size_t)(b - 1) * chunk_bytes);
  };
  auto issue = [&](int s, int c) {      // one thread
    const int b = c % p.nbuf;
    const int cnt = min(p.chunk_vis, p.n_bl - c * p.chunk_vis);
    const uint32_t bytes = (uint32_t)cnt * sizeof(float2);
    mbar_expect_tx(bar + b, bytes);
    bulk_load(buf_of(b), p.vis + (size_t)s * p.n_bl + (size_t)c * p.chunk_vis, bytes, bar + b);
  };

  if (tid == 0) {
    for (int b = 0; b < p.nbuf; ++b) mbar_init(bar + b, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // last-stage twiddles w^(r k), k fixed per lane: registers for the whole kernel
  constexpr int R1 = F::template radix<1>();
  constexpr int NB1 = 16 / R1;
  cf32 tw1[NB1][R1 > 1 ? R1 : 2];
#pragma unroll
  for (int b = 0; b < NB1; ++b) F::template twiddles<1>(tw1[b], t + b * T, p.tw);
  __syncthreads();
  if (tid == 0 && blockIdx.x < p.n_snap) issue(blockIdx.x, 0);
  const int c_last0 = ((p.n_chunk - 1) / p.nbuf) * p.nbuf;   // last chunk of a snapshot in buffer 0
  uint32_t phase = 0;                                        // bit b: parity of the next wait on buffer b

  for (int s = blockIdx.x; s < p.n_snap; s += gridDim.x) {
    const int ch = s % p.n_ch;
    const ChannelInfo ci = p.chinfo[ch];
    // the lines / exchange area is idle until phase H: fill it with this snapshot's next chunks
    if (tid == 0)
      for (int c = 1; c < min(p.n_chunk, p.nbuf); ++c) issue(s, c);

    // ---- phase S ----------------------------------------------------------------------------
    for (int j = tid; j < p.n_can_max; j += THREADS) S[j] = make_float2(0.f, 0.f);
    __syncthreads();
    for (int c = 0; c < p.n_chunk; ++c) {
      const int b = c % p.nbuf;
      const size_t cp = (size_t)ch * p.n_chunk + c;
      const uint2 *__restrict__ frec = p.frec + cp * max(p.n_can_max, 1);
      const uint32_t *__restrict__ fpair = p.fpair + cp * p.chunk_vis;
      const int2 *__restrict__ frow = p.frow + cp * p.frow_stride;
      // table records first: they do not depend on the data, so their latency hides behind the wait
      uint2 rec[kCellsPf];
      uint32_t pr1[kCellsPf];
      const int2 row1 = __ldg(frow + 1);
#pragma unroll
      for (int q = 0; q < kCellsPf; ++q) {
        const int k = tid + q * THREADS;
        rec[q] = k < p.n_can_max ? __ldg(frec + k) : make_uint2(0u, 0u);
        pr1[q] = k < row1.y ? __ldg(fpair + row1.x + k) : 0u;
      }
      mbar_wait(bar + b, (phase >> b) & 1u);
      phase ^= 1u << b;
      const float2 *__restrict__ buf = buf_of(b);
      auto sum_cell = [&](uint2 rc, uint32_t p1, int k) {
        const int len = rc.x >> 16;
        if (len == 0) return;
        float ax = 0.f, ay = 0.f;
        add_entry(buf, rc.y & 0xFFFFu, ax, ay);
        if (len > 1) add_entry(buf, rc.y >> 16, ax, ay);
        if (len > 2) add_entry(buf, p1 & 0xFFFFu, ax, ay);
        if (len > 3) add_entry(buf, p1 >> 16, ax, ay);
        for (int q = 2; 2 * q < len; ++q) {
          const uint32_t pq = __ldg(fpair + __ldg(frow + q).x + k);
          add_entry(buf, pq & 0xFFFFu, ax, ay);
          if (2 * q + 1 < len) add_entry(buf, pq >> 16, ax, ay);
        }
        const int j = rc.x & 0xFFFFu;
        const float2 a = S[j];
        S[j] = make_float2(a.x + ax, a.y + ay);
      };
#pragma unroll
      for (int q = 0; q < kCellsPf; ++q) sum_cell(rec[q], pr1[q], tid + q * THREADS);
      for (int k = tid + kCellsPf * THREADS; k < p.n_can_max; k += THREADS)
        sum_cell(__ldg(frec + k), k < row1.y ? __ldg(fpair + row1.x + k) : 0u, k);
      __syncthreads();                  // buffer b is free, S is consistent
      if (tid == 0) {
        if (c + p.nbuf < p.n_chunk) issue(s, c + p.nbuf);
        else if (c == c_last0 && s + (int)gridDim.x < p.n_snap) issue(s + gridDim.x, 0);
      }
    }

    // ---- phase H: zero the bounding-box rows of the lines, then drop in the occupied cells ------
    const int kym = ci.ky_max, nrow = 2 * kym + 1;
    for (int e = tid; e < nrow * p.n_col; e += THREADS) {
      const int c = e / nrow, iy = (e % nrow - kym + N) & (N - 1);
      lines[c * LS + pad16(iy)] = make_float2(0.f, 0.f);
    }
    {
      const size_t hb = (size_t)ch * 2 * p.n_bl;
      for (int e0 = 0; e0 < p.h_max; e0 += kHPer * THREADS) {
        int code[kHPer], pos[kHPer];
        float w[kHPer];
#pragma unroll
        for (int c = 0; c < kHPer; ++c) {          // independent table loads, issued together
          const int e = e0 + c * THREADS + tid;
          pos[c] = e < p.h_max ? __ldg(p.hpos + hb + e) : -1;
          code[c] = e < p.h_max ? __ldg(p.hcode + hb + e) : 0;
          w[c] = e < p.h_max ? __ldg(p.hw + hb + e) : 0.f;
        }
        if (e0 == 0) __syncthreads();               // the zero fill above is complete
#pragma unroll
        for (int c = 0; c < kHPer; ++c) {
          if (pos[c] < 0) continue;                  // tables are padded with pos = -1
          const float2 v = S[code[c] & kPlaceMask];
          const int flag = code[c] >> kPlaceShift;
          float2 o;
          if (flag == kPlaceDirect) o = make_float2(v.x * w[c], v.y * w[c]);
          else if (flag == kPlaceConj) o = make_float2(v.x * w[c], -v.y * w[c]);
          else o = make_float2((v.x + v.x) * w[c], 0.f);
          lines[pos[c]] = o;
        }
      }
      if (p.h_max == 0) __syncthreads();
    }
    __syncthreads();

    // ---- pass A: columns kx = 0..kx_max, in place ----------------------------------------------
    for (int c0 = 0; c0 <= ci.kx_max; c0 += G) {
      const int c = c0 + grp;
      const bool act = c <= ci.kx_max;            // uniform per transform group (T lanes)
      float2 *line = lines + (size_t)(act ? c : 0) * LS;
      cf32 v[16];
      if (act)
        F::template load<0>(v, t, [&](int idx) {
          return (idx <= kym || idx >= N - kym) ? line[pad16(idx)] : mk(0.f, 0.f);
        });
      __syncwarp();
      if (act) {
        F::template compute<0>(v, t, p.tw);
        F::template store<0>(v, t, [&](int idx, cf32 x) { line[pad16(idx)] = x; });
      }
      __syncwarp();
      if (act) {
        F::template load<1>(v, t, [&](int idx) { return line[pad16(idx)]; });
        F::template compute_tw<1>(v, tw1);
      }
      __syncwarp();
      if (act) F::template store<1>(v, t, [&](int idx, cf32 x) { line[pad16(idx)] = x; });
    }
    __syncthreads();

    // ---- pass B: row pairs (y, y + N/2) --------------------------------------------------------
    const int kxm = ci.kx_max;
    float2 *xl = X + (size_t)grp * LSB;
    float *__restrict__ img = p.img + (size_t)s * N * N;
    for (int q0 = 0; q0 < N / 2; q0 += G) {
      const bool act = q0 + grp < N / 2;
      const int y0 = act ? q0 + grp : 0, y1 = y0 + N / 2;
      const int o0 = pad16(y0), o1 = pad16(y1);
      cf32 v[16];
      if (act) {
        // stage-0 inputs Z[idx], idx = t + r*T: r < 8 direct half (a + i b), r >= 8 mirrored half
        // (conj a + i conj b at k = N - idx) -- static per r, branch-free, all loads in flight
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          float2 a[8], b[8];
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const int idx = t + (8 * h + q) * T;
            const int k = h == 0 ? idx : N - idx;
            const bool ok = k <= kxm;
            a[q] = ok ? lines[k * LS + o0] : make_float2(0.f, 0.f);
            b[q] = ok ? lines[k * LS + o1] : make_float2(0.f, 0.f);
          }
#pragma unroll
          for (int q = 0; q < 8; ++q)
            v[8 * h + q] = h == 0 ? mk(a[q].x - b[q].y, a[q].y + b[q].x) : mk(a[q].x + b[q].y, b[q].x - a[q].y);
        }
        F::template compute<0>(v, t, p.tw);
      }
      __syncwarp();                                   // previous round's reads of xl are done
      if (act) F::template store<0>(v, t, [&](int idx, cf32 x) { xl[pad16(idx)] = x; });
      __syncwarp();
      if (act) {
        F::template load<1>(v, t, [&](int idx) { return xl[pad16(idx)]; });
        F::template compute_tw<1>(v, tw1);
        float *__restrict__ r0 = img + (size_t)y0 * N, *__restrict__ r1 = img + (size_t)y1 * N;
        F::template store<1>(v, t, [&](int x, cf32 z) { __stcs(r0 + x, z.x); __stcs(r1 + x, z.y); });
      }
    }
    // generic-proxy writes to the lines / exchange area are ordered before the next snapshot's
    // bulk copies into the same bytes
    fence_async_smem();
    __syncthreads();
  }
}

// shared-memory plan of the route; returns false if it does not fit.  Layout (bytes):
//   [0, region)            column lines + pass-B exchange lines; doubles as chunk buffers 1..nbuf-1
//   [off_dedicated, +C*8)  chunk buffer 0
//   [off_S, +n_can_max*8)  canonical cell sums
//   [off_bar, +nbuf*8)     mbarriers
static bool fused_layout(blink_plan *p, int threads) {
  const int N = p->n_pix, T = N / 16, G = threads / std::max(T, 1);
  const size_t region = sizeof(float2) * ((size_t)(p->kx_max_all + 1) * fused_line_stride(N) + (size_t)G * (N + N / 16));
  const size_t region_al = (region + 127) / 128 * 128;
  const size_t s_bytes = (sizeof(float2) * (size_t)std::max(p->n_can_max, 1) + 15) / 16 * 16;
  const size_t limit = (size_t)p->max_smem_optin;
  for (int n_chunk = 1; n_chunk <= 64; ++n_chunk) {
    int C = (p->n_bl + n_chunk - 1) / n_chunk;
    C = (C + 1) & ~1;                              // 16-byte multiples
    if (C > 0x8000) continue;                      // 15-bit local baseline index
    const size_t cb = sizeof(float2) * (size_t)C;
    const int nbuf = 1 + (int)std::min<size_t>(7, region / cb);
    if (nbuf < 2 && n_chunk > 1) continue;         // the ring needs a second buffer
    const size_t total = region_al + cb + s_bytes + 8 * (size_t)nbuf + 64;
    if (total > limit) continue;
    p->fused_chunk_vis = C;
    p->fused_n_chunk = (p->n_bl + C - 1) / C;
    p->fused_nbuf = std::min(nbuf, std::max(p->fused_n_chunk, 1));
    p->fused_off_dedicated = (uint32_t)region_al;
    p->fused_off_S = (uint32_t)(region_al + cb);
    p->fused_off_bar = (uint32_t)(region_al + cb + s_bytes);
    p->fused_smem = region_al + cb + s_bytes + 8 * (size_t)p->fused_nbuf + 16;
    return true;
  }
  return false;
}

int fused_setup(blink_plan *p) {
  p->fused_path = 0;
  p->fused_chunk = p->chunk_snapshots;   // the two-kernel route chunks like blink_image
  // shared-memory route: two-stage transforms (N <= 256), everything resident in one SM, and
  // 16-byte aligned snapshots (even n_bl) for the bulk copies
  int want = 1;
  if (const char *e = getenv("BLINK_FUSED_SMEM")) want = atoi(e);
  if (want && p->n_pix <= 256 && p->n_pix >= 32 && (p->n_bl & 1) == 0 && p->max_smem_optin > 0) {
    p->fused_threads = 512;
    if (fused_layout(p, p->fused_threads)) p->fused_path = 1;
  }
  return BLINK_OK;
}

template <int N>
static int launch_fused_n(const blink_plan *p, const FusedParams &fp, cudaStream_t st) {
  constexpr int THREADS = 512;
  static thread_local size_t smem_set = 0;
  if (p->fused_smem > smem_set) {
    BLINK_CUDA_TRY(cudaFuncSetAttribute(k_fused<N, THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)p->fused_smem), "k_fused smem attribute");
    BLINK_CUDA_TRY(cudaFuncSetAttribute(k_fused<N, THREADS>, cudaFuncAttributePreferredSharedMemoryCarveout, 100),
                   "k_fused carveout");
    smem_set = p->fused_smem;
  }
  const int blocks = std::min(fp.n_snap, p->sm_count);
  if (blocks <= 0) return BLINK_OK;
  k_fused<N, THREADS><<<blocks, THREADS, p->fused_smem, st>>>(fp);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_fused launch");
  return BLINK_OK;
}

static int launch_fused(const blink_plan *p, const float2 *vis, int n_t, float *img, cudaStream_t st) {
  FusedParams fp;
  fp.vis = vis; fp.img = img; fp.chinfo = p->d_chinfo;
  fp.frec = p->d_frec; fp.fpair = p->d_fpair; fp.frow = p->d_frow;
  fp.hpos = p->d_hpos; fp.hcode = p->d_hcode; fp.hw = p->d_hw; fp.tw = p->d_tw;
  fp.n_bl = p->n_bl; fp.n_ch = p->n_ch; fp.n_snap = n_t * p->n_ch; fp.n_can_max = p->n_can_max;
  fp.n_chunk = p->fused_n_chunk; fp.chunk_vis = p->fused_chunk_vis; fp.nbuf = p->fused_nbuf;
  fp.frow_stride = p->frow_stride; fp.n_col = p->kx_max_all + 1; fp.h_max = p->h_max;
  fp.off_dedicated = p->fused_off_dedicated; fp.off_S = p->fused_off_S; fp.off_bar = p->fused_off_bar;
  switch (p->n_pix) {
    case 32: return launch_fused_n<32>(p, fp, st);
    case 64: return launch_fused_n<64>(p, fp, st);
    case 128: return launch_fused_n<128>(p, fp, st);
    case 256: return launch_fused_n<256>(p, fp, st);
    default: return BLINK_EUNSUPPORTED;
  }
}

int fused_reserve(blink_plan *p, int n_t) { return image_reserve(p, n_t); }

int launch_grid_image(const blink_plan *p, const float2 *vis, int n_t, float *img, cudaStream_t st) {
  if (p->fused_path == 1) return launch_fused(p, vis, n_t, img, st);
  return launch_image_from_vis(p, vis, n_t * p->n_ch, img, st);
}

}  // namespace blink

extern "C" int blink_grid_image(const blink_plan *plan, const void *vis, int n_t, void *images, void *stream) {
  if (!plan || n_t < 0) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!vis || !images) return BLINK_EINVAL;
  if (((uintptr_t)vis & 7) || ((uintptr_t)images & 3)) return BLINK_EINVAL;
  blink_plan *mp = const_cast<blink_plan *>(plan);
  int rc = blink::image_reserve(mp, n_t);
  if (rc != BLINK_OK) return rc;
  return blink::launch_grid_image(plan, (const float2 *)vis, n_t, (float *)images, (cudaStream_t)stream);
}
