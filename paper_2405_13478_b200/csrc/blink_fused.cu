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
//   phase S   as in k_grid: visibilities -> rank-major stage -> S[j] (canonical half-plane sums);
//   phase H   the occupied cells with kx >= 0 are written, already weighted, normalised and
//             sign-flipped for the fftshift, into per-column lines in shared memory (the grid is
//             exactly Hermitian by construction, so the half-plane is all that is needed);
//   pass A    column transforms along ky, in place in the lines, loads pruned to the bounding box;
//   pass B    row transforms, two real image rows per complex transform, read from the lines across
//             columns and stored to global memory straight from the last butterfly stage.
// A transform is owned by T = N/16 <= 16 lanes of one warp, so the exchanges inside it need only
// __syncwarp.  The next snapshot's visibilities are prefetched into registers during phase S and
// stay in flight through passes A and B.
struct FusedParams {
  const float2 *vis;
  float *img;
  const ChannelInfo *chinfo;
  const uint16_t *scat, *roff;
  const uint32_t *cellrec;
  const int32_t *nact, *hpos, *hcode, *hcount;
  const float *hw;
  const float2 *tw;
  int n_bl, n_ch, n_snap, n_can_max, n_pass, roff_stride, n_col, ky_max_all, h_max;
};

constexpr int kHPer = 5;   // phase-H table entries fetched per thread at a time

int fused_line_stride(int n_pix) { return ((n_pix + n_pix / 16 + 15) / 16) * 16 + 1; }

template <int N, int THREADS, int PF>
__global__ void __launch_bounds__(THREADS, 1) k_fused(const FusedParams p) {
  constexpr int CAP = THREADS * PF;
  constexpr int T = N / 16;             // lanes per transform
  constexpr int G = THREADS / T;        // transforms in flight per CTA
  constexpr int LS = ((LineSize<N>::value + 15) / 16) * 16 + 1;
  constexpr int LSB = LineSize<N>::value;
  using F = Fft<N>;
  static_assert(F::NSTAGE == 2 && T <= 32, "shared-memory route needs a two-stage warp-local transform");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2 *S = reinterpret_cast<float2 *>(smem_raw);              // [n_can_max]
  float2 *lines = S + p.n_can_max;                               // [n_col][LS]
  float2 *X = lines + (size_t)p.n_col * LS;                      // stage [CAP] / exchange lines [G][LSB]
  const int tid = threadIdx.x;
  const int grp = tid / T, t = tid % T;

  PassRegs<PF> regs;
  if (blockIdx.x < p.n_snap)
    pass_load<THREADS, PF>(regs, p.vis + (size_t)blockIdx.x * p.n_bl,
                           p.scat + (size_t)(blockIdx.x % p.n_ch) * p.n_bl, 0, min(CAP, p.n_bl), tid);
  for (int s = blockIdx.x; s < p.n_snap; s += gridDim.x) {
    const int ch = s % p.n_ch;
    const ChannelInfo ci = p.chinfo[ch];
    const float2 *__restrict__ vis = p.vis + (size_t)s * p.n_bl;
    const uint16_t *__restrict__ scat = p.scat + (size_t)ch * p.n_bl;

    // ---- phase S ----------------------------------------------------------------------------
    for (int j = tid; j < p.n_can_max; j += THREADS) S[j] = make_float2(0.f, 0.f);
    for (int pass = 0; pass < p.n_pass; ++pass) {
      const size_t cp = (size_t)ch * p.n_pass + pass;
      const uint32_t *__restrict__ cellrec = p.cellrec + cp * max(p.n_can_max, 1);
      SumsRegs<THREADS> sr;
      sums_prefetch<THREADS>(sr, cellrec, p.n_can_max, tid);
      pass_scatter<PF>(regs, X);
      __syncthreads();
      if (pass + 1 < p.n_pass) {
        const int b0 = (pass + 1) * CAP;
        pass_load<THREADS, PF>(regs, vis, scat, b0, min(CAP, p.n_bl - b0), tid);
      } else if (s + (int)gridDim.x < p.n_snap) {
        const int s2 = s + gridDim.x;
        pass_load<THREADS, PF>(regs, p.vis + (size_t)s2 * p.n_bl, p.scat + (size_t)(s2 % p.n_ch) * p.n_bl,
                               0, min(CAP, p.n_bl), tid);
      }
      sums_run<THREADS>(sr, cellrec, p.roff + cp * p.roff_stride, p.n_can_max, X, S, tid);
      __syncthreads();
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
        F::template compute<1>(v, t, p.tw);
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
        F::template compute<1>(v, t, p.tw);
        float *__restrict__ r0 = img + (size_t)y0 * N, *__restrict__ r1 = img + (size_t)y1 * N;
        F::template store<1>(v, t, [&](int x, cf32 z) { __stcs(r0 + x, z.x); __stcs(r1 + x, z.y); });
      }
    }
    __syncthreads();   // X becomes the stage of the next snapshot
  }
}

size_t fused_smem_bytes(const blink_plan *p, int threads, int prefetch) {
  const int N = p->n_pix, T = N / 16, G = threads / std::max(T, 1);
  const size_t x = std::max((size_t)threads * prefetch, (size_t)G * (N + N / 16));
  return sizeof(float2) * ((size_t)p->n_can_max + (size_t)(p->kx_max_all + 1) * fused_line_stride(N) + x) + 16;
}

int fused_setup(blink_plan *p) {
  p->fused_path = 0;
  p->fused_chunk = p->chunk_snapshots;   // the two-kernel route chunks like blink_image
  // shared-memory route: two-stage transforms (N <= 256) and everything resident in one SM.
  // Its stage capacity must equal the gridder's (the scatter tables are built for one capacity).
  int want = 1;
  if (const char *e = getenv("BLINK_FUSED_SMEM")) want = atoi(e);
  if (want && p->n_pix <= 256 && p->n_pix >= 32) {
    const int threads = 512, prefetch = p->stage_cap / 512;
    if (prefetch * 512 == p->stage_cap && (prefetch == 8 || prefetch == 16)) {
      const size_t smem = fused_smem_bytes(p, threads, prefetch);
      if (p->max_smem_optin > 0 && smem <= (size_t)p->max_smem_optin) {
        p->fused_path = 1;
        p->fused_threads = threads;
        p->fused_prefetch = prefetch;
        p->fused_smem = smem;
      }
    }
  }
  return BLINK_OK;
}

template <int N, int PF>
static int launch_fused_n(const blink_plan *p, const FusedParams &fp, cudaStream_t st) {
  constexpr int THREADS = 512;
  static thread_local size_t smem_set = 0;
  if (p->fused_smem > smem_set) {
    BLINK_CUDA_TRY(cudaFuncSetAttribute(k_fused<N, THREADS, PF>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)p->fused_smem), "k_fused smem attribute");
    BLINK_CUDA_TRY(cudaFuncSetAttribute(k_fused<N, THREADS, PF>, cudaFuncAttributePreferredSharedMemoryCarveout, 100),
                   "k_fused carveout");
    smem_set = p->fused_smem;
  }
  const int blocks = std::min(fp.n_snap, p->sm_count);
  if (blocks <= 0) return BLINK_OK;
  k_fused<N, THREADS, PF><<<blocks, THREADS, p->fused_smem, st>>>(fp);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_fused launch");
  return BLINK_OK;
}

static int launch_fused(const blink_plan *p, const float2 *vis, int n_t, float *img, cudaStream_t st) {
  FusedParams fp;
  fp.vis = vis; fp.img = img; fp.chinfo = p->d_chinfo; fp.scat = p->d_scat; fp.roff = p->d_roff;
  fp.cellrec = p->d_cellrec; fp.nact = p->d_nact; fp.hpos = p->d_hpos; fp.hcode = p->d_hcode;
  fp.hcount = p->d_hcount; fp.hw = p->d_hw; fp.tw = p->d_tw;
  fp.n_bl = p->n_bl; fp.n_ch = p->n_ch; fp.n_snap = n_t * p->n_ch; fp.n_can_max = p->n_can_max;
  fp.n_pass = p->n_pass; fp.roff_stride = p->roff_stride; fp.n_col = p->kx_max_all + 1;
  fp.ky_max_all = p->ky_max_all; fp.h_max = p->h_max;
  const bool pf16 = p->fused_prefetch == 16;
  switch (p->n_pix) {
    case 32: return pf16 ? launch_fused_n<32, 16>(p, fp, st) : launch_fused_n<32, 8>(p, fp, st);
    case 64: return pf16 ? launch_fused_n<64, 16>(p, fp, st) : launch_fused_n<64, 8>(p, fp, st);
    case 128: return pf16 ? launch_fused_n<128, 16>(p, fp, st) : launch_fused_n<128, 8>(p, fp, st);
    case 256: return pf16 ? launch_fused_n<256, 16>(p, fp, st) : launch_fused_n<256, 8>(p, fp, st);
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
