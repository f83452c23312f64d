// blink_dynspec.cu -- the stage right after imaging: subtraction of a
// running reference image and transposition of the image cube into per-pixel dynamic spectra.
//
//   "imaging artefacts like side-lobes can be removed by subtracting a reference image of the same
//    field (formed as a combination of previous images or prepared prior to the processing)"
//    (PAPER.md:76); the reference "can be the preceding dirty image, some form of an average of the
//    sequence of previous images ... or a model image"; "once the data cube of images
//    ... are created, dynamic spectra from all pixels (i.e time series in different directions in
//    the sky) will be formed".
//
// The paper prints no formula; readings DESIGN.md c21-c23.  Per channel and pixel, R_0 handed in:
//     D_t = I_t - R_t,   R_{t+1} = (1 - alpha) R_t + alpha I_t,   dyn[y][x][ch][t] = D_t
// alpha = 1: preceding image; alpha = 0: fixed model image; in between: exponential running average.
//
// Pure streaming work, 8 bytes per voxel (read the image once, write the spectrum once).  A thread
// owns one pixel of a 256-pixel tile: it loads 32 time steps of its pixel (each load instruction of a
// warp is 128 contiguous bytes of an image row, 32 loads in flight per thread, issued one tile ahead
// so that they overlap the previous tile's barrier and stores), runs the recurrence
// in registers and drops the differences into a [32 t][256 pixel] shared tile (row stride 257, so both
// the pixel-major writes and the time-major reads are bank-conflict free); then each warp writes, for
// 32 pixels in turn, the 32 time steps of one pixel: 128 contiguous bytes of that pixel's spectrum.
// A CTA walks all channels of its group, so the (channel, time) plane of a pixel is written by one
// CTA in address order and partially covered 32-byte sectors at channel boundaries merge in L2.
#include <cmath>
#include <cstdlib>

#include "blink_internal.h"
#include "sgather.cuh"

namespace blink {

constexpr int kDsPix = 256;          // pixels per CTA = threads per CTA
constexpr int kDsT = 32;             // time steps per tile
constexpr int kDsStride = kDsPix + 1;

template <int MINB>
__global__ void __launch_bounds__(kDsPix, MINB) k_dynspec(const float *__restrict__ img, float *__restrict__ ref,
                                                    float *__restrict__ dyn, int n_t, int n_ch, long long nn,
                                                    int ch_per, float alpha) {
  __shared__ float tile[kDsT * kDsStride];
  const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;
  const long long pix0 = (long long)blockIdx.x * kDsPix, pix = pix0 + tid;
  const int ch_begin = blockIdx.y * ch_per, ch_end = min(n_ch, ch_begin + ch_per);
  const float beta = 1.0f - alpha;
  const long long t_stride = (long long)n_ch * nn;
  const int total = (ch_end - ch_begin) * ((n_t + kDsT - 1) / kDsT);
  // tiles q = 0 .. total-1 run channel-major; the loads of tile q + 1 (and the reference of a channel
  // about to start) are issued as soon as tile q's differences sit in shared memory -- v is dead by
  // then -- so they are in flight during the barrier and the store phase of tile q
  float v[kDsT];
  float r_next = 0.0f;
  auto issue = [&](int ch, int t0) {
    const float *__restrict__ src = img + (long long)ch * nn + pix + (long long)t0 * t_stride;
#pragma unroll
    for (int k = 0; k < kDsT; ++k) v[k] = (t0 + k < n_t) ? __ldcs(src + (long long)k * t_stride) : 0.0f;
    if (t0 == 0 && ref) r_next = ref[(long long)ch * nn + pix];
  };
  if (total > 0) issue(ch_begin, 0);
  float R = 0.0f;
  int ch = ch_begin, t0 = 0;
  for (int q = 0; q < total; ++q) {
    if (t0 == 0) R = r_next;
#pragma unroll
    for (int k = 0; k < kDsT; ++k) {
      tile[k * kDsStride + tid] = v[k] - R;
      if (t0 + k < n_t) R = fmaf(alpha, v[k], beta * R);
    }
    if (t0 + kDsT >= n_t && ref) ref[(long long)ch * nn + pix] = R;
    const bool last_tile = t0 + kDsT >= n_t;
    const int ch_n = last_tile ? ch + 1 : ch, t0_n = last_tile ? 0 : t0 + kDsT;
    if (q + 1 < total) issue(ch_n, t0_n);
    __syncthreads();
    if (t0 + lane < n_t) {
      float *__restrict__ dst = dyn + ((pix0 + wv * 32) * n_ch + ch) * (long long)n_t + t0 + lane;
      const long long p_stride = (long long)n_ch * n_t;
#pragma unroll 8
      for (int pp = 0; pp < 32; ++pp) __stcs(dst + pp * p_stride, tile[lane * kDsStride + wv * 32 + pp]);
    }
    __syncthreads();
    ch = ch_n;
    t0 = t0_n;
  }
}

// Same work with the loads done by the copy engine and no CTA-wide barrier.  A ninth warp is the
// producer: per tile it posts one bulk copy (cp.async.bulk, SASS UBLKCP) of P pixels per time step into
// a ring of [T t][P pixel] stages, completion counted by a `full` mbarrier per stage; it re-arms a
// stage once the consumer warps have arrived on its `empty` mbarrier.  A consumer warp owns 32
// pixels for the whole kernel and works IN PLACE on its T x 32 corner of the stage: recurrence with
// lane = pixel, the difference of (time k, pixel p) written back to column p ^ (k mod 32) of row k (a
// permutation of the 32 banks, and the row's inputs have all been read by then), __syncwarp, then
// stores with lane = time step reading column pp ^ lane of rows lane + 32 m (again a permutation):
// 128 contiguous bytes of one pixel's spectrum per instruction, T / 32 instructions back to back per
// pixel, no bank conflict in either direction and no second buffer.  The other stage(s) are in flight
// while a warp works on one; warps drift apart, so loads, arithmetic and stores of different warps
// overlap.  Needs 16-byte aligned image rows (any torch allocation).
// Template parameters: P pixels per CTA (P / 32 consumer warps), T time steps per tile (a multiple of
// 32; a pixel's run of T * 4 bytes is written by T / 32 back-to-back store instructions), STAGES.
template <int P, int T, int STAGES>
struct DsCfg {
  static constexpr int kWarps = P / 32;
  static constexpr size_t kSmem = sizeof(float) * STAGES * T * P + 16 * STAGES;
};

template <int P, int T, int STAGES, int MINB>
__global__ void __launch_bounds__(P + 32, MINB) k_dynspec_tma(const float *__restrict__ img, float *__restrict__ ref,
                                                              float *__restrict__ dyn, int n_t, int n_ch, long long nn,
                                                              int ch_per, float alpha) {
  constexpr int CW = P / 32;
  extern __shared__ __align__(128) unsigned char ds_smem[];
  float *in = reinterpret_cast<float *>(ds_smem);                    // [stage][T t][P pixels]
  uint64_t *full = reinterpret_cast<uint64_t *>(in + STAGES * T * P);
  uint64_t *empty = full + STAGES;
  const int tid = threadIdx.x, lane = tid & 31, wv = tid >> 5;
  const long long pix0 = (long long)blockIdx.x * P;
  const int ch_begin = blockIdx.y * ch_per, ch_end = min(n_ch, ch_begin + ch_per);
  const int n_tt = (n_t + T - 1) / T, total = (ch_end - ch_begin) * n_tt;
  if (tid < STAGES) {
    mbar_init(full + tid, 1);
    mbar_init(empty + tid, CW);
  }
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  __syncthreads();
  if (wv == CW) {
    // ---------------------------------------------------------------- producer warp (lane k = time steps t0 + k + 32 m)
    int ch = ch_begin, t0 = 0;
    for (int q = 0; q < total; ++q) {
      const int st = q % STAGES;
      if (q >= STAGES) {
        mbar_wait(empty + st, (uint32_t)(q / STAGES - 1) & 1u);
        fence_async_smem();                // the consumers' generic reads before the copy engine overwrites the stage
      }
      const int rows = min(T, n_t - t0);
      if (lane == 0) mbar_expect_tx(full + st, (uint32_t)rows * P * sizeof(float));
      __syncwarp();
#pragma unroll
      for (int m = 0; m < T / 32; ++m) {
        const int k = lane + 32 * m;
        if (k < rows)
          bulk_load(in + (st * T + k) * P, img + ((long long)(t0 + k) * n_ch + ch) * nn + pix0, P * sizeof(float), full + st);
      }
      if (t0 + T >= n_t) { ++ch; t0 = 0; } else { t0 += T; }
    }
    return;
  }
  // ------------------------------------------------------------------ consumer warps
  const float beta = 1.0f - alpha;
  const long long pix = pix0 + tid;
  const long long p_stride = (long long)n_ch * n_t;
  float R = 0.0f, r_next = (ref && total > 0) ? ref[(long long)ch_begin * nn + pix] : 0.0f;
  int ch = ch_begin, t0 = 0;
  for (int q = 0; q < total; ++q) {
    const int st = q % STAGES;
    mbar_wait(full + st, (uint32_t)(q / STAGES) & 1u);
    if (t0 == 0) R = r_next;
    float *__restrict__ x = in + st * T * P + wv * 32;   // this warp's corner: x[k * P + column]
    if (t0 + T <= n_t) {
#pragma unroll
      for (int k = 0; k < T; ++k) {
        const float v = x[k * P + lane];
        x[k * P + (lane ^ (k & 31))] = v - R;
        R = fmaf(alpha, v, beta * R);
      }
    } else {
#pragma unroll
      for (int k = 0; k < T; ++k) {
        if (t0 + k < n_t) {
          const float v = x[k * P + lane];
          x[k * P + (lane ^ (k & 31))] = v - R;
          R = fmaf(alpha, v, beta * R);
        }
      }
    }
    __syncwarp();
    const bool last_tile = t0 + T >= n_t;
    if (last_tile && ref) {
      ref[(long long)ch * nn + pix] = R;
      if (ch + 1 < ch_end) r_next = ref[(long long)(ch + 1) * nn + pix];
    }
    {
      float *__restrict__ dst = dyn + ((pix0 + wv * 32) * n_ch + ch) * (long long)n_t + t0 + lane;
      const float *__restrict__ row = x + lane * P;
#pragma unroll 4
      for (int pp = 0; pp < 32; ++pp, dst += p_stride) {
#pragma unroll
        for (int m = 0; m < T / 32; ++m)
          if (t0 + lane + 32 * m < n_t) __stcs(dst + 32 * m, row[32 * m * P + (pp ^ lane)]);
      }
    }
    __syncwarp();                          // the warp is done with its corner of the stage
    if (lane == 0) mbar_arrive(empty + st);
    if (last_tile) { ++ch; t0 = 0; } else { t0 += T; }
  }
}

template <int P, int T, int STAGES, int MINB>
static int launch_dynspec_tma(const blink_plan *p, const float *images, float *ref_state, float *dynspec, int n_t, double alpha,
                              cudaStream_t st) {
  const long long nn = (long long)p->n_pix * p->n_pix;
  const int tiles = (int)(nn / P);
  // enough CTAs for a few rounds per SM; a CTA keeps whole channels.  When a pixel's time row is not a
  // whole number of 32-byte sectors, an even channel count per CTA keeps the group boundaries on
  // sector boundaries for even n_t.
  const int target = p->sm_count * 24;      // measured 6 / 12 / 24 / 48 / 96 per SM: 0.358 / 0.331 / 0.325 / 0.328 / 0.325 ms (station cube)
  int groups = std::min(p->n_ch, (target + tiles - 1) / tiles);
  int ch_per = (p->n_ch + groups - 1) / groups;
  if ((n_t & 7) && (ch_per & 1) && ch_per < p->n_ch) ++ch_per;
  groups = (p->n_ch + ch_per - 1) / ch_per;
  constexpr size_t smem = DsCfg<P, T, STAGES>::kSmem;
  static std::atomic<uint64_t> attr{0};
  const int rc = ensure_max_smem(k_dynspec_tma<P, T, STAGES, MINB>, p, attr, "k_dynspec_tma smem attribute", false);
  if (rc != BLINK_OK) return rc;
  k_dynspec_tma<P, T, STAGES, MINB><<<dim3(tiles, groups), P + 32, smem, st>>>(images, ref_state, dynspec, n_t, p->n_ch, nn, ch_per,
                                                                               (float)alpha);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_dynspec_tma launch");
  return BLINK_OK;
}

}  // namespace blink

extern "C" int blink_dynspec(const blink_plan *p, const void *images, int n_t, double alpha, void *ref_state,
                             void *dynspec, void *stream) {
  using namespace blink;
  if (!p || n_t < 0 || !(alpha >= 0.0 && alpha <= 1.0)) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!images || !dynspec || images == dynspec) return BLINK_EINVAL;
  if (((uintptr_t)images & 3) || ((uintptr_t)dynspec & 3) || ((uintptr_t)ref_state & 3)) return BLINK_EINVAL;
  const long long nn = (long long)p->n_pix * p->n_pix;     // a multiple of 256 for every supported N (>= 32)
  if (nn % kDsPix) return BLINK_EUNSUPPORTED;
  const int route = p->opt.tune[kTuneDynspecRoute];   // 1 = register loads even for aligned cubes
  { const int rc = check_device(p); if (rc != BLINK_OK) return rc; }
  cudaStream_t st = (cudaStream_t)stream;
  if (route != 1 && ((uintptr_t)images & 15) == 0) {
    const float *im = (const float *)images;
    float *rs = (float *)ref_state, *ds = (float *)dynspec;
    // tile shape: 128 pixels x 64 time steps, two stages, three CTAs per SM.  Measured on the station
    // cube (n_t = 100), ms per call: <256,32,3> 0.368, <128,32,3> 0.378, <128,64,3> 0.335, <128,64,2> 0.331,
    // <64,64,3> 0.338, <256,64,2> 0.376, <64,128,2> 0.393, <128,128,3> 0.492, <64,128,3> 0.505: longer runs
    // per pixel on the write side pay until too few consumer warps are left per SM.
    return launch_dynspec_tma<128, 64, 2, 3>(p, im, rs, ds, n_t, alpha, st);
  }
  const int tiles = (int)(nn / kDsPix);
  const int target = p->sm_count * 12;
  int groups = std::min(p->n_ch, (target + tiles - 1) / tiles);
  int ch_per = (p->n_ch + groups - 1) / groups;
  if ((n_t & 7) && (ch_per & 1) && ch_per < p->n_ch) ++ch_per;
  groups = (p->n_ch + ch_per - 1) / ch_per;
  k_dynspec<3><<<dim3(tiles, groups), kDsPix, 0, st>>>((const float *)images, (float *)ref_state, (float *)dynspec, n_t, p->n_ch, nn,
                                                       ch_per, (float)alpha);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_dynspec launch");
  return BLINK_OK;
}
