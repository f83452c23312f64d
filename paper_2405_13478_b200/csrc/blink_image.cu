// blink_image.cu -- steps a3-a5: weighting, batched 2-D inverse FFT, fftshift, normalisation, real
// part (the paper calls cufftPlanMany / ExecC2C, then takes the real part
// and shifts in separate steps).  Hand-written Stockham transforms (fft_core.cuh), fused with
// everything around them:
//
//   pass A (columns, along ky): reads only the half-plane kx = 0..kx_max of the plan's bounding box
//     and its mirror, forms H = (G[k] + conj(G[-k])) / 2 -- so the REAL PART of the transform is
//     produced by a Hermitian (half-size) transform --, applies the uniform weight 1/count, the
//     normalisation 1/norm and the fftshift as the sign (-1)^(kx+ky) ON LOAD, then U[y][kx] =
//     sum_ky H[ky][kx] w^(ky y).
//   pass B (rows, along kx): two real rows per complex transform: Z = U[y] + i U[y'] extended by
//     Hermitian symmetry, z = IFFT(Z), image[y] = Re z, image[y'] = Im z, stored coalesced straight
//     from the last butterfly stage.
//
// U lives in a small plan-owned scratch (two-pass path) sized to stay L2-resident between the two
// launches of a chunk of snapshots.
#include <algorithm>
#include <cstdio>

#include "blink_internal.h"
#include "fft_core.cuh"

namespace blink {
using namespace blinkfft;

template <int N> struct ImgCfg {
  static constexpr int T = N / 16;                                   // threads per transform
  static constexpr int LS = ((LineSize<N>::value + 15) / 16) * 16 + 1;  // line stride, = 1 mod 16
  static constexpr int CT_MAX = (1024 / T) < 16 ? (1024 / T) : 16;   // columns per CTA, pass A
  static constexpr int RP_MAX = (N / 2) < (512 / T) ? (N / 2) : (512 / T > 0 ? 512 / T : 1);
};

// run stages 1.. of the transform; stage 0's load is done by the caller
// BM: inputs r of the first-stage butterflies outside this mask are known to be zero (never read)
template <int N, unsigned BM = 0xFFFFu, class Store>
__device__ __forceinline__ void fft_tail(cf32 *v, int t, cf32 *line, const cf32 *__restrict__ tw, Store st) {
  using F = Fft<N>;
  // N >= 512: every stride is 1 or a multiple of 16, so the padded-line accesses take immediate offsets
  constexpr bool kLine = N >= 512;
  if constexpr (BM == 0xFFFFu) F::template compute<0>(v, t, tw);
  else F::template compute0_pruned<BM>(v);
  if constexpr (kLine) F::template store_line<0>(v, t, line);
  else F::template store<0>(v, t, [&](int idx, cf32 x) { line[pad16(idx)] = x; });
  __syncthreads();
  if constexpr (kLine) F::template load_line<1>(v, t, line);
  else F::template load<1>(v, t, [&](int idx) { return line[pad16(idx)]; });
  F::template compute<1>(v, t, tw);
  if constexpr (F::NSTAGE == 2) {
    F::template store<1>(v, t, st);
  } else {
    __syncthreads();
    if constexpr (kLine) F::template store_line<1>(v, t, line);
    else F::template store<1>(v, t, [&](int idx, cf32 x) { line[pad16(idx)] = x; });
    __syncthreads();
    if constexpr (kLine) F::template load_line<2>(v, t, line);
    else F::template load<2>(v, t, [&](int idx) { return line[pad16(idx)]; });
    F::template compute<2>(v, t, tw);
    F::template store<2>(v, t, st);
  }
}

template <int N, int CT>
__global__ void __launch_bounds__(CT * (N / 16)) k_image_cols(const ImgParams p) {
  using C = ImgCfg<N>;
  constexpr int THREADS = CT * C::T;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cf32 *lines = reinterpret_cast<cf32 *>(smem_raw);
  const int tid = threadIdx.x;
  const int sl = blockIdx.y, s = p.snap_base + sl, ch = (s + p.ch0) % p.n_ch;
  const ChannelInfo ci = p.chinfo[ch];
  const int kx0 = blockIdx.x * CT;
  const float2 *__restrict__ G = p.uv + (size_t)s * N * N;

  // thread -> fixed column c, rows ky = -ky_max + r0 + i*RS: no div/mod or 64-bit index math in the
  // loop, 4 rows (8 independent 8-byte loads) in flight per thread.  Rows of the bounding box are
  // always written (zeros included), so only the rows outside it need an explicit zero fill.
  constexpr int RS = THREADS / CT;
  const int c = tid % CT, r0 = tid / CT, kx = kx0 + c, kym = ci.ky_max;
  cf32 *myline = lines + c * C::LS;
  if (kx > ci.kx_max) {
    for (int i = r0; i < N; i += RS) myline[pad16(i)] = mk(0.f, 0.f);
  } else {
    for (int i = kym + 1 + r0; i < N - kym; i += RS) myline[pad16(i)] = mk(0.f, 0.f);
    const float2 *__restrict__ Ga = G + kx;
    const float2 *__restrict__ Gb = G + ((N - kx) & (N - 1));
    const float w0 = 0.5f * ci.inv_norm;
    for (int ky = -kym + r0; ky <= kym; ky += 4 * RS) {
      float2 a[4], b[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int kyu = ky + u * RS;
        if (kyu <= kym) {
          const int iy = kyu & (N - 1);
          a[u] = __ldcs(Ga + iy * N);
          b[u] = __ldcs(Gb + ((N - iy) & (N - 1)) * N);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int kyu = ky + u * RS;
        if (kyu <= kym) {
          const float w = ((kx + kyu) & 1) ? -w0 : w0;
          myline[pad16(kyu & (N - 1))] = mk((a[u].x + b[u].x) * w, (a[u].y - b[u].y) * w);
        }
      }
    }
  }
  __syncthreads();
  if (p.uniform) {   // sparse 1/count on the occupied cells of these columns
    const int32_t *__restrict__ wcol = p.wcol + (size_t)ch * (p.wu + 1);
    const int e0 = wcol[kx0], e1 = wcol[min(kx0 + CT, p.wu)];
    const int32_t *__restrict__ wkey = p.wkey + (size_t)ch * 2 * p.n_bl;
    const float *__restrict__ wval = p.wval + (size_t)ch * 2 * p.n_bl;
    for (int e = e0 + tid; e < e1; e += THREADS) {
      const int key = wkey[e];
      const float w = wval[e];
      cf32 *q = lines + ((key >> 16) - kx0) * C::LS + pad16(key & 0xffff);
      *q = mk(q->x * w, q->y * w);
    }
    __syncthreads();
  }

  const int t = tid / CT;
  cf32 *line = myline;
  cf32 v[16];
  Fft<N>::template load<0>(v, t, [&](int idx) { return line[pad16(idx)]; });
  __syncthreads();
  float2 *__restrict__ U = p.U + (size_t)sl * N * p.wu + kx0 + c;
  fft_tail<N>(v, t, line, p.tw, [&](int y, cf32 x) { U[(size_t)y * p.wu] = x; });
}

// Pass A of blink_grid_image (two-kernel route): the column lines are filled straight from the
// visibilities -- every occupied cell of these columns sums its own (short) segment of the
// cell-sorted baseline list, in ascending baseline order, and is stored weighted, normalised and
// sign-flipped -- so the dense uv grid is never written or read.
template <int N, int CT>
__global__ void __launch_bounds__(CT * (N / 16)) k_cols_from_vis(const ImgParams p) {
  using C = ImgCfg<N>;
  constexpr int THREADS = CT * C::T;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cf32 *lines = reinterpret_cast<cf32 *>(smem_raw);
  const int tid = threadIdx.x;
  const int sl = blockIdx.y, s = p.snap_base + sl, ch = (s + p.ch0) % p.n_ch;
  const int kx0 = blockIdx.x * CT;
  const int32_t *__restrict__ vcol = p.vcol + (size_t)ch * (p.wu + 1);
  const int e0 = vcol[kx0], e1 = vcol[min(kx0 + CT, p.wu)];
  // Sparse tiles: when none of the CT columns holds more than direct_max occupied cells, the
  // column transforms are cheaper as direct sums U[y] = sum_cells H exp(+2 pi i ky y / N).  One
  // column per W warps; a lane owns 16 outputs y = y0 + 32 i and steps its twiddle by w^(32 ky).
  constexpr int W = THREADS / 32 / CT;            // warps per column (N / 512)
  if constexpr (W >= 1) {
    int nmax = 0;
#pragma unroll
    for (int c = 0; c < CT; ++c) nmax = max(nmax, __ldg(vcol + kx0 + c + 1) - __ldg(vcol + kx0 + c));
    if (nmax <= p.direct_max) {
      const int wv = tid >> 5, lane = tid & 31, c = wv % CT, part = wv / CT;
      const int c0 = __ldg(vcol + kx0 + c), n_c = __ldg(vcol + kx0 + c + 1) - c0;
      const size_t tb = (size_t)ch * 2 * p.n_bl;
      cf32 val = mk(0.f, 0.f);
      int iy = 0;
      if (lane < n_c) {                            // lane l forms the l-th cell of the column
        const int e = c0 + lane;
        const float2 *__restrict__ vis = p.vis + (size_t)s * p.n_bl;
        const float2 *__restrict__ cf = p.corr ? p.corr + (size_t)ch * p.n_bl : nullptr;
        const int32_t *__restrict__ src = p.src + (size_t)ch * p.n_bl;
        const int st = __ldg(p.vseg + tb + e), lf = __ldg(p.vlen + tb + e);
        const float w = __ldg(p.vw + tb + e);
        iy = __ldg(p.vkey + tb + e) & 0xffff;
        const int len = lf & 0xFFFFFF, flag = lf >> 24;
        float ar = 0.f, ai = 0.f;
        for (int q = st; q < st + len; ++q) {
          const int code = __ldg(src + q);
          const float2 v = ld_vis(vis, cf, code >> 1);
          ar += v.x;
          ai += (code & 1) ? -v.y : v.y;
        }
        if (flag == kPlaceDirect) val = mk(ar * w, ai * w);
        else if (flag == kPlaceConj) val = mk(ar * w, -ai * w);
        else val = mk((ar + ar) * w, 0.f);
      }
      const int y0 = part * (N / W) + lane;
      cf32 acc[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) acc[i] = mk(0.f, 0.f);
      for (int k = 0; k < n_c; ++k) {
        const cf32 vk = mk(__shfl_sync(0xffffffffu, val.x, k), __shfl_sync(0xffffffffu, val.y, k));
        const int ik = __shfl_sync(0xffffffffu, iy, k);
        const cf32 step = __ldg(p.tw + ((ik * 32) & (N - 1)));
        cf32 t = cmul(vk, __ldg(p.tw + ((ik * y0) & (N - 1))));
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          acc[i] = cadd(acc[i], t);
          t = cmul(t, step);
        }
      }
      cf32 *line = lines + c * C::LS;
#pragma unroll
      for (int i = 0; i < 16; ++i) line[pad16(y0 + 32 * i)] = acc[i];
      __syncthreads();
      float2 *__restrict__ U = p.U + (size_t)sl * N * p.wu + kx0;
      for (int idx = tid; idx < CT * N; idx += THREADS) {
        const int cc = idx % CT, y = idx / CT;
        U[(size_t)y * p.wu + cc] = lines[cc * C::LS + pad16(y)];
      }
      return;
    }
  }
  for (int i = tid; i < CT * C::LS; i += THREADS) lines[i] = mk(0.f, 0.f);
  __syncthreads();
  {
    const size_t tb = (size_t)ch * 2 * p.n_bl;
    const float2 *__restrict__ vis = p.vis + (size_t)s * p.n_bl;
    const float2 *__restrict__ cf = p.corr ? p.corr + (size_t)ch * p.n_bl : nullptr;
    const int32_t *__restrict__ src = p.src + (size_t)ch * p.n_bl;
    for (int e = e0 + tid; e < e1; e += THREADS) {
      const int key = __ldg(p.vkey + tb + e), st = __ldg(p.vseg + tb + e), lf = __ldg(p.vlen + tb + e);
      const float w = __ldg(p.vw + tb + e);
      const int len = lf & 0xFFFFFF, flag = lf >> 24;
      float ar = 0.f, ai = 0.f;
      for (int q = st; q < st + len; ++q) {
        const int code = __ldg(src + q);
        const float2 v = ld_vis(vis, cf, code >> 1);
        ar += v.x;
        ai += (code & 1) ? -v.y : v.y;
      }
      cf32 o;
      if (flag == kPlaceDirect) o = mk(ar * w, ai * w);
      else if (flag == kPlaceConj) o = mk(ar * w, -ai * w);
      else o = mk((ar + ar) * w, 0.f);
      lines[((key >> 16) - kx0) * C::LS + pad16(key & 0xffff)] = o;
    }
  }
  __syncthreads();
  const int c = tid % CT, t = tid / CT;
  cf32 *line = lines + c * C::LS;
  cf32 v[16];
  Fft<N>::template load<0>(v, t, [&](int idx) { return line[pad16(idx)]; });
  __syncthreads();
  float2 *__restrict__ U = p.U + (size_t)sl * N * p.wu + kx0 + c;
  fft_tail<N>(v, t, line, p.tw, [&](int y, cf32 x) { U[(size_t)y * p.wu] = x; });
}

// NZ < 8: the half-plane is narrower than NZ N / 16 columns, so of the 16 inputs of a first-stage butterfly
// only r < NZ (direct half) and r >= 16 - NZ (mirrored half) can be non-zero: the others are neither loaded
// nor added
template <int N, int RP, int NZ = 8>
__global__ void __launch_bounds__(RP * (N / 16)) k_image_rows(const ImgParams p) {
  using C = ImgCfg<N>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cf32 *lines = reinterpret_cast<cf32 *>(smem_raw);
  const int tid = threadIdx.x;
  const int sl = blockIdx.y, s = p.snap_base + sl, ch = (s + p.ch0) % p.n_ch;
  const int kxm = p.chinfo[ch].kx_max;
  const int pr = tid / C::T, t = tid % C::T;
  const int y0 = blockIdx.x * RP + pr, y1 = y0 + N / 2;
  const float2 *__restrict__ U0 = p.U + ((size_t)sl * N + y0) * p.wu;
  const float2 *__restrict__ U1 = p.U + ((size_t)sl * N + y1) * p.wu;
  cf32 *line = lines + pr * C::LS;
  cf32 v[16];
  // stage-0 inputs Z[idx], idx = t + r*T: r < 8 is the direct half (Z = a + i b), r >= 8 the mirrored
  // half (Z = conj a + i conj b at k = N - idx) -- static per r, so the 32 loads are branch-free and
  // all in flight together
  {
    float2 a[16], b[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      if (r >= NZ && r < 16 - NZ) continue;
      const int idx = t + r * C::T;
      const int k = r < 8 ? idx : N - idx;
      const bool ok = k <= kxm;
      a[r] = ok ? __ldg(U0 + k) : make_float2(0.f, 0.f);
      b[r] = ok ? __ldg(U1 + k) : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      if (r >= NZ && r < 16 - NZ) continue;
      v[r] = r < 8 ? mk(a[r].x - b[r].y, a[r].y + b[r].x) : mk(a[r].x + b[r].y, b[r].x - a[r].y);
    }
  }
  float *__restrict__ r0 = p.img + ((size_t)s * N + y0) * N;
  float *__restrict__ r1 = p.img + ((size_t)s * N + y1) * N;
  fft_tail<N, BandMask<NZ>::value>(v, t, line, p.tw, [&](int x, cf32 z) { __stcs(r0 + x, z.x); __stcs(r1 + x, z.y); });
}

template <int N, int CT, int RP>
static int run_image_cfg(const blink_plan *p, ImgParams ip, int n_snap, cudaStream_t st) {
  using C = ImgCfg<N>;
  const bool from_vis = ip.vis != nullptr;
  const size_t smem_a = sizeof(cf32) * CT * C::LS, smem_b = sizeof(cf32) * RP * C::LS;
  if (std::max(smem_a, smem_b) > (size_t)p->max_smem_optin) return BLINK_EUNSUPPORTED;
  static std::atomic<uint64_t> attr_a{0}, attr_v{0}, attr_b{0};
  int rc = ensure_max_smem(k_image_cols<N, CT>, p, attr_a, "k_image_cols smem attribute");
  if (rc == BLINK_OK) rc = ensure_max_smem(k_cols_from_vis<N, CT>, p, attr_v, "k_cols_from_vis smem attribute");
  if (rc == BLINK_OK) rc = ensure_max_smem(k_image_rows<N, RP>, p, attr_b, "k_image_rows smem attribute");
  // a half-plane at most N / 4 columns wide: the row transforms' first stage pruned to 4 + 4 of 16 inputs
  constexpr bool kNarrow = N >= 2048;
  static std::atomic<uint64_t> attr_b4{0};
  const bool narrow = kNarrow && p->kx_max_all < N / 4;
  if constexpr (kNarrow)
    if (rc == BLINK_OK && narrow) rc = ensure_max_smem(k_image_rows<N, RP, 4>, p, attr_b4, "k_image_rows smem attribute");
  if (rc != BLINK_OK) return rc;
  const size_t per_snap = sizeof(float2) * (size_t)N * p->wu;
  const int chunk = (int)std::min<size_t>((size_t)std::max(1, p->chunk_snapshots), p->scratch_bytes / per_snap);
  if (chunk < 1) return BLINK_ENOMEM;
  for (int base = 0; base < n_snap; base += chunk) {
    const int cs = std::min(chunk, n_snap - base);
    ip.snap_base = base;
    if (p->res_route == 2) {                // sparse half-plane at N = 2048 / 4096: column pass by residue class
      rc = launch_cols_res(p, ip, cs, st);
      if (rc != BLINK_OK) return rc;
    } else if (from_vis) k_cols_from_vis<N, CT><<<dim3(p->wu / CT, cs), CT * C::T, smem_a, st>>>(ip);
    else k_image_cols<N, CT><<<dim3(p->wu / CT, cs), CT * C::T, smem_a, st>>>(ip);
    if constexpr (kNarrow) {
      if (narrow) k_image_rows<N, RP, 4><<<dim3(N / 2 / RP, cs), RP * C::T, smem_b, st>>>(ip);
      else k_image_rows<N, RP><<<dim3(N / 2 / RP, cs), RP * C::T, smem_b, st>>>(ip);
    } else {
      k_image_rows<N, RP><<<dim3(N / 2 / RP, cs), RP * C::T, smem_b, st>>>(ip);
    }
  }
  BLINK_CUDA_TRY(cudaGetLastError(), "k_image launch");
  return BLINK_OK;
}

// default tile shapes per N; N = 512 / 1024 also carry alternatives selectable through the plan
template <int N> static int run_image_n(const blink_plan *p, const ImgParams &ip, int n_snap, cudaStream_t st) {
  using C = ImgCfg<N>;
  if constexpr (N == 1024) {
    const int ct = p->img_ct ? p->img_ct : 8, rp = p->img_rp ? p->img_rp : 2;
    if (ct == 16) return run_image_cfg<N, 16, 2>(p, ip, n_snap, st);
    if (ct == 4) return rp == 1 ? run_image_cfg<N, 4, 1>(p, ip, n_snap, st) : run_image_cfg<N, 4, 2>(p, ip, n_snap, st);
    if (ct == 2) return run_image_cfg<N, 2, 2>(p, ip, n_snap, st);
    if (rp == 8) return run_image_cfg<N, 8, 8>(p, ip, n_snap, st);
    if (rp == 4) return run_image_cfg<N, 8, 4>(p, ip, n_snap, st);
    if (rp == 1) return run_image_cfg<N, 8, 1>(p, ip, n_snap, st);
    return run_image_cfg<N, 8, 2>(p, ip, n_snap, st);
  } else if constexpr (N == 512) {
    if (p->img_ct == 16) return run_image_cfg<N, 16, 8>(p, ip, n_snap, st);
    return run_image_cfg<N, 8, 8>(p, ip, n_snap, st);
  } else if constexpr (N <= 256) {
    constexpr int RP = (N / 2) < (256 / C::T) ? (N / 2) : (256 / C::T);
    return run_image_cfg<N, 16, RP>(p, ip, n_snap, st);
  } else {
    return run_image_cfg<N, C::CT_MAX, (256 / C::T > 0 ? 256 / C::T : 1)>(p, ip, n_snap, st);
  }
}


int image_setup(blink_plan *p) {
  p->wu = ((p->kx_max_all + 1 + 15) / 16) * 16;   // multiple of every column-tile width
  p->img_ct = p->opt.tune[kTuneImageCt];
  p->img_rp = p->opt.tune[kTuneImageRp];
  p->image_path = 1;
  // snapshots per launch pair.  Fewer and larger launches win over keeping U L2-resident: every launch pair
  // costs ~40 us of start-up and tail (measured per 480 MWA-II snapshots at 4096^2: 60 MB -> 19.2 ms,
  // 512 MB -> 14.2 ms, 2 GB -> 12.3 ms, 8 GB -> 12.2 ms)
  size_t budget = (size_t)2048 << 20;
  if (p->opt.image_chunk_mb > 0) budget = (size_t)p->opt.image_chunk_mb << 20;
  const size_t per_snap = sizeof(float2) * (size_t)p->n_pix * p->wu;
  // a chunk's snapshots are the launch's gridDim.y: at most 65535
  p->chunk_snapshots = (int)std::min<size_t>(65535, std::max<size_t>(1, budget / per_snap));
  return BLINK_OK;
}

// Device scratch of a call of n_t time steps.  The shared-memory route of blink_grid_image needs none;
// the two-kernel routes hold U of one chunk of snapshots; the warp route a ring of U slots plus two
// completion counters per snapshot.
size_t scratch_need(const blink_plan *p, long long n_t, bool fused) {
  if (fused && fused_smem_route(p)) return 0;
  if (p->res_route == 1) return 0;
  const long long n_snap = std::max<long long>(n_t * p->n_ch, 1);
  if (p->warp_route) return warp_route_scratch_bytes(p, n_snap);
  const size_t per_snap = sizeof(float2) * (size_t)p->n_pix * p->wu;
  return per_snap * (size_t)std::min<long long>(n_snap, p->chunk_snapshots);
}

int image_reserve(blink_plan *p, int n_t) {
  p->reserved_n_t = std::max(p->reserved_n_t, n_t);
  const long long n_snap = std::max<long long>((long long)n_t * p->n_ch, 1);
  const size_t need = std::max(scratch_need(p, n_t, false), scratch_need(p, n_t, true));
  if (need <= p->scratch_bytes && (!p->warp_route || n_snap <= p->warp_snap_cap)) return BLINK_OK;
  if (p->d_scratch) {
    BLINK_CUDA_TRY(cudaDeviceSynchronize(), "scratch regrow sync");
    cudaFree(p->d_scratch);
    p->d_scratch = nullptr;
    p->scratch_bytes = 0;
  }
  cudaError_t e = cudaMalloc((void **)&p->d_scratch, need);
  if (e != cudaSuccess) {
    set_cuda_error(e, "scratch cudaMalloc");
    return e == cudaErrorMemoryAllocation ? BLINK_ENOMEM : BLINK_ECUDA;
  }
  p->scratch_bytes = need;
  if (p->warp_route) {
    // the route's completion counters follow the ring; the kernel leaves them zero behind itself
    const size_t ring = warp_route_ring_bytes(p);
    BLINK_CUDA_TRY(cudaMemset(reinterpret_cast<unsigned char *>(p->d_scratch) + ring, 0, need - ring), "scratch counters");
    // cudaMemset on device memory may return before the fill has run, and it runs on the legacy default
    // stream: a k_img1024 launch on a non-blocking stream (the host pipe's, a torch side stream) is not
    // ordered after it.  Reserve is allowed to synchronise; the hot call is not.
    BLINK_CUDA_TRY(cudaDeviceSynchronize(), "scratch counters sync");
    p->warp_snap_cap = n_snap;
  }
  return BLINK_OK;
}

static int launch_image_impl(const blink_plan *p, const float2 *uv, const float2 *vis, int n_snap, int ch0, float *img, cudaStream_t st) {
  ImgParams ip;
  ip.vis = vis; ip.corr = (vis != nullptr && p->corr_on) ? p->d_corr : nullptr; ip.src = p->d_src; ip.vkey = p->d_vkey; ip.vseg = p->d_vseg; ip.vlen = p->d_vlen;
  ip.vcol = p->d_vcol; ip.vw = p->d_vw; ip.tw32 = p->d_tw32;
  ip.cell_cap = (std::max(p->vtile8_max, 1) + 3) / 4 * 4;
  ip.uv = uv; ip.img = img; ip.U = p->d_scratch; ip.chinfo = p->d_chinfo;
  ip.wkey = p->d_wkey; ip.wval = p->d_wval; ip.wcol = p->d_wcol; ip.n_bl = p->n_bl;
  ip.tw = p->d_tw; ip.n_ch = p->n_ch; ip.wu = p->wu; ip.uniform = p->weighting == BLINK_UNIFORM;
  ip.snap_base = 0;
  ip.ch0 = ch0;
  ip.direct_max = p->opt.tune[kTuneDirectMax] > 0 ? std::min(32, p->opt.tune[kTuneDirectMax] - 1) : 12;
  if (p->res_route == 1)                    // residue-class kernel, intermediate in shared memory (blink_image_r.cu)
    return launch_img1024r(p, ip, n_snap, st);
  if (p->warp_route)                        // persistent warp-per-transform kernel (blink_image_w.cu)
    return launch_img1024(p, ip, n_snap, st);
  switch (p->n_pix) {
    case 32: return run_image_n<32>(p, ip, n_snap, st);
    case 64: return run_image_n<64>(p, ip, n_snap, st);
    case 128: return run_image_n<128>(p, ip, n_snap, st);
    case 256: return run_image_n<256>(p, ip, n_snap, st);
    case 512: return run_image_n<512>(p, ip, n_snap, st);
    case 1024: return run_image_n<1024>(p, ip, n_snap, st);
    case 2048: return run_image_n<2048>(p, ip, n_snap, st);
    case 4096: return run_image_n<4096>(p, ip, n_snap, st);
    default: return BLINK_EUNSUPPORTED;
  }
}

int launch_image(const blink_plan *p, const float2 *uv, int n_snap, int ch0, float *img, cudaStream_t st) {
  return launch_image_impl(p, uv, nullptr, n_snap, ch0, img, st);
}

int launch_image_from_vis(const blink_plan *p, const float2 *vis, int n_snap, float *img, cudaStream_t st) {
  return launch_image_impl(p, nullptr, vis, n_snap, 0, img, st);
}

// ------------------------------------------------------------------------------------------
// blink_image_static (blink.h): the line kernels above with their intermediate U in memory that nobody
// allocates at run time.  For callers who may not enter the CUDA allocator when they need images (a
// real-time loop that cannot afford cudaMalloc's device-wide stall, a GPU whose memory another component
// already owns, a "no allocation after start-up" rule): the scratch is part of the library image.
//
// The array is a device object; in HOST code its name is only a handle the runtime maps to an address.
// Passing `g_static_U` itself to a kernel would hand it a host-side pointer (a fault, or -- where the GPU
// can reach host memory -- silent use of the wrong bytes), so the launcher asks the runtime for the real
// device address once per device and passes that.
static __device__ __align__(256) unsigned char g_static_U[BLINK_STATIC_SCRATCH_BYTES];

constexpr int kStaticMaxDevices = 64;
static std::atomic<float2 *> g_static_U_addr[kStaticMaxDevices];   // device address of g_static_U, per device ordinal

// set-up, once per device, with that device current: cudaGetSymbolAddress resolves the symbol in the
// CURRENT device's copy of the module.  Two threads racing here both get the same answer.
static int static_scratch_addr(int device, float2 **out) {
  if (device < 0 || device >= kStaticMaxDevices) return BLINK_EUNSUPPORTED;
  float2 *a = g_static_U_addr[device].load(std::memory_order_acquire);
  if (a == nullptr) {
    void *ptr = nullptr;
    BLINK_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_static_U), "blink_image_static: cudaGetSymbolAddress(g_static_U)");
    if (ptr == nullptr) return BLINK_ECUDA;
    a = static_cast<float2 *>(ptr);
    g_static_U_addr[device].store(a, std::memory_order_release);
  }
  *out = a;
  return BLINK_OK;
}

template <int N, int CT, int RP>
static int run_image_static_cfg(const blink_plan *p, ImgParams ip, int n_snap, int chunk, cudaStream_t st) {
  using C = ImgCfg<N>;
  const size_t smem_a = sizeof(cf32) * CT * C::LS, smem_b = sizeof(cf32) * RP * C::LS;
  if (std::max(smem_a, smem_b) > (size_t)p->max_smem_optin) return BLINK_EUNSUPPORTED;
  // per-device kernel attributes: part of the first call's set-up, like the address above
  static std::atomic<uint64_t> attr_a{0}, attr_b{0}, attr_b4{0};
  int rc = ensure_max_smem(k_image_cols<N, CT>, p, attr_a, "k_image_cols smem attribute");
  if (rc == BLINK_OK) rc = ensure_max_smem(k_image_rows<N, RP>, p, attr_b, "k_image_rows smem attribute");
  constexpr bool kNarrow = N >= 2048;
  const bool narrow = kNarrow && p->kx_max_all < N / 4;
  if constexpr (kNarrow)
    if (rc == BLINK_OK && narrow) rc = ensure_max_smem(k_image_rows<N, RP, 4>, p, attr_b4, "k_image_rows smem attribute");
  if (rc != BLINK_OK) return rc;
  for (int base = 0; base < n_snap; base += chunk) {   // stream order keeps a pair's row pass ahead of the next column pass
    const int cs = std::min(chunk, n_snap - base);
    ip.snap_base = base;
    k_image_cols<N, CT><<<dim3(p->wu / CT, cs), CT * C::T, smem_a, st>>>(ip);
    if constexpr (kNarrow) {
      if (narrow) k_image_rows<N, RP, 4><<<dim3(N / 2 / RP, cs), RP * C::T, smem_b, st>>>(ip);
      else k_image_rows<N, RP><<<dim3(N / 2 / RP, cs), RP * C::T, smem_b, st>>>(ip);
    } else {
      k_image_rows<N, RP><<<dim3(N / 2 / RP, cs), RP * C::T, smem_b, st>>>(ip);
    }
  }
  BLINK_CUDA_TRY(cudaGetLastError(), "blink_image_static launch");
  return BLINK_OK;
}

// the default tile shapes of run_image_n (no tuning slots: this entry point has one configuration per N)
template <int N> static int run_image_static_n(const blink_plan *p, const ImgParams &ip, int n_snap, int chunk, cudaStream_t st) {
  using C = ImgCfg<N>;
  if constexpr (N == 1024) return run_image_static_cfg<N, 8, 2>(p, ip, n_snap, chunk, st);
  else if constexpr (N == 512) return run_image_static_cfg<N, 8, 8>(p, ip, n_snap, chunk, st);
  else if constexpr (N <= 256) return run_image_static_cfg<N, 16, ((N / 2) < (256 / C::T) ? (N / 2) : (256 / C::T))>(p, ip, n_snap, chunk, st);
  else return run_image_static_cfg<N, C::CT_MAX, (256 / C::T > 0 ? 256 / C::T : 1)>(p, ip, n_snap, chunk, st);
}

static int launch_image_static(const blink_plan *p, const float2 *uv, int n_snap, float *img, cudaStream_t st) {
  const size_t per_snap = sizeof(float2) * (size_t)p->n_pix * p->wu;
  if (per_snap > (size_t)BLINK_STATIC_SCRATCH_BYTES) {
    char msg[200];
    snprintf(msg, sizeof msg, "blink_image_static: one snapshot's intermediate is %zu bytes (8 x N = %d x wu = %d), "
             "the built-in scratch holds %u", per_snap, p->n_pix, p->wu, (unsigned)BLINK_STATIC_SCRATCH_BYTES);
    set_error_text(msg);
    return BLINK_ECAPACITY;
  }
  float2 *U = nullptr;
  int rc = static_scratch_addr(p->device, &U);
  if (rc != BLINK_OK) return rc;
  // a chunk's snapshots are the launch's gridDim.y: at most 65535
  const int chunk = (int)std::min<size_t>(65535, (size_t)BLINK_STATIC_SCRATCH_BYTES / per_snap);
  ImgParams ip = {};
  ip.uv = uv; ip.img = img; ip.U = U; ip.chinfo = p->d_chinfo;
  ip.wkey = p->d_wkey; ip.wval = p->d_wval; ip.wcol = p->d_wcol; ip.n_bl = p->n_bl;
  ip.tw = p->d_tw; ip.n_ch = p->n_ch; ip.wu = p->wu; ip.uniform = p->weighting == BLINK_UNIFORM;
  ip.snap_base = 0; ip.ch0 = 0;
  switch (p->n_pix) {
    case 32: return run_image_static_n<32>(p, ip, n_snap, chunk, st);
    case 64: return run_image_static_n<64>(p, ip, n_snap, chunk, st);
    case 128: return run_image_static_n<128>(p, ip, n_snap, chunk, st);
    case 256: return run_image_static_n<256>(p, ip, n_snap, chunk, st);
    case 512: return run_image_static_n<512>(p, ip, n_snap, chunk, st);
    case 1024: return run_image_static_n<1024>(p, ip, n_snap, chunk, st);
    case 2048: return run_image_static_n<2048>(p, ip, n_snap, chunk, st);
    case 4096: return run_image_static_n<4096>(p, ip, n_snap, chunk, st);
    default: return BLINK_EUNSUPPORTED;
  }
}

}  // namespace blink

extern "C" int blink_image_static(const blink_plan *plan, const void *uv_grid, int n_t, void *images, void *stream) {
  if (!plan || n_t < 0) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!uv_grid || !images) return BLINK_EINVAL;
  if (((uintptr_t)uv_grid & 7) || ((uintptr_t)images & 3)) return BLINK_EINVAL;
  int rc = check_device(plan);
  if (rc != BLINK_OK) return rc;
  return blink::launch_image_static(plan, (const float2 *)uv_grid, n_t * plan->n_ch, (float *)images, (cudaStream_t)stream);
}

extern "C" int blink_image(const blink_plan *plan, const void *uv_grid, int n_t, void *images, void *stream) {
  if (!plan || n_t < 0) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!uv_grid || !images) return BLINK_EINVAL;
  if (((uintptr_t)uv_grid & 7) || ((uintptr_t)images & 3)) return BLINK_EINVAL;
  int rc = check_device(plan);
  if (rc != BLINK_OK) return rc;
  if (blink::scratch_need(plan, n_t, false) > plan->scratch_bytes) return BLINK_ERESERVE;
  return blink::launch_image(plan, (const float2 *)uv_grid, n_t * plan->n_ch, 0, (float *)images, (cudaStream_t)stream);
}
