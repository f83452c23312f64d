// blink_correct.cu -- pre-gridding corrections of PAPER.md section 4.2 (:142-156): (i) cable-length
// phase, (ii) calibration in phase and amplitude, (iii) geometric phase rotation of the phase centre
// (SURVEY.md section 8(f) item f2).  The paper names the three steps and says they are GPU kernels
// run post-correlation (:156) but prints no formula; the readings are DESIGN.md c18-c20:
//
//   measured V_ij = a_i conj(a_j) V_ij(true),   a_i(nu) = g_i(nu) exp(-2 pi i nu L_i / c)
//   F[ch][bl(i,j)] = exp(+2 pi i (u l0 + v m0 + w (n0 - 1))) / (a_i conj(a_j))
//
// with (u, v, w) = (r_j - r_i) nu / c, un-snapped.  Gains, cable lengths, geometry and pointing are
// fixed across the snapshots of a plan, so -- like the uv indices -- everything that depends on them
// is folded into ONE table at plan time (k_corr_table, fp64) and the per-snapshot work is a single
// complex multiply per visibility (k_correct), a pure streaming kernel: 16 bytes per visibility
// against HBM, the 8-byte factors stay in L2 (8.4 MB for the 256-antenna station, 32 channels).
#include <cmath>
#include <vector>

#include "blink_internal.h"

namespace blink {

constexpr double kSpeedOfLight = 299792458.0;

// one thread per (channel, baseline); all arithmetic fp64, result rounded once to complex64
__global__ void k_corr_table(const double *__restrict__ ant, const int32_t *__restrict__ pi,
                             const int32_t *__restrict__ pj, const double *__restrict__ freq,
                             const double2 *__restrict__ gains, const double *__restrict__ cable,
                             double l0, double m0, double n0m1, int n_ant, int n_bl, int n_ch,
                             float2 *__restrict__ F) {
  const int bl = blockIdx.x * blockDim.x + threadIdx.x, ch = blockIdx.y;
  if (bl >= n_bl) return;
  const int i = pi[bl], j = pj[bl];
  const double sc = freq[ch] / kSpeedOfLight;
  const double u = (ant[3 * j] - ant[3 * i]) * sc, v = (ant[3 * j + 1] - ant[3 * i + 1]) * sc,
               w = (ant[3 * j + 2] - ant[3 * i + 2]) * sc;
  // phase in cycles: + geometric rotation, + (L_i - L_j) nu / c from 1 / (a_i conj a_j)
  double cyc = u * l0 + v * m0 + w * n0m1 + (cable[i] - cable[j]) * sc;
  cyc -= rint(cyc);
  double sn, cs;
  sincospi(2.0 * cyc, &sn, &cs);
  const double2 gi = gains[(size_t)ch * n_ant + i], gj = gains[(size_t)ch * n_ant + j];
  // d = g_i conj(g_j);  F = (cs + i sn) / d = (cs + i sn) conj(d) / |d|^2
  const double dr = gi.x * gj.x + gi.y * gj.y, di = gi.y * gj.x - gi.x * gj.y;
  const double inv = 1.0 / (dr * dr + di * di);
  const double fr = (cs * dr + sn * di) * inv, fi = (sn * dr - cs * di) * inv;
  F[(size_t)ch * n_bl + bl] = make_float2((float)fr, (float)fi);
}

// out = in * F.  A thread owns table entries (two visibilities = 16 bytes each), keeps the factor in
// registers and walks the time steps, four loads in flight: every access is a coalesced 16-byte
// streaming load or store and the table is read once per launch.
__global__ void __launch_bounds__(256) k_correct(const float4 *__restrict__ in, const float4 *__restrict__ F,
                                                 float4 *__restrict__ out, int n_t, long long tab_pair) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < tab_pair; k += stride) {
    const float4 f = __ldg(F + k);
    const float4 *__restrict__ src = in + k;
    float4 *__restrict__ dst = out + k;
    int t = 0;
    for (; t + 4 <= n_t; t += 4) {
      float4 a[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) a[r] = __ldcs(src + (long long)(t + r) * tab_pair);
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        float4 o;
        o.x = a[r].x * f.x - a[r].y * f.y;
        o.y = a[r].x * f.y + a[r].y * f.x;
        o.z = a[r].z * f.z - a[r].w * f.w;
        o.w = a[r].z * f.w + a[r].w * f.z;
        __stcs(dst + (long long)(t + r) * tab_pair, o);
      }
    }
    for (; t < n_t; ++t) {
      const float4 a = __ldcs(src + (long long)t * tab_pair);
      float4 o;
      o.x = a.x * f.x - a.y * f.y;
      o.y = a.x * f.y + a.y * f.x;
      o.z = a.z * f.z - a.w * f.w;
      o.w = a.z * f.w + a.w * f.z;
      __stcs(dst + (long long)t * tab_pair, o);
    }
  }
}

// same, one visibility per thread and step (odd n_ch * n_bl or buffers not 16-byte aligned)
__global__ void __launch_bounds__(256) k_correct1(const float2 *__restrict__ in, const float2 *__restrict__ F,
                                                  float2 *__restrict__ out, int n_t, long long tab) {
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < tab; k += stride) {
    const float2 f = __ldg(F + k);
    for (int t = 0; t < n_t; ++t) {
      const float2 a = __ldcs(in + (long long)t * tab + k);
      __stcs(out + (long long)t * tab + k, make_float2(a.x * f.x - a.y * f.y, a.x * f.y + a.y * f.x));
    }
  }
}

}  // namespace blink

extern "C" int blink_plan_set_corrections(blink_plan *p, const double *gains, const double *cable_len_m,
                                          double l0, double m0, void *stream) try {
  using namespace blink;
  if (!p) return BLINK_EINVAL;
  const double r2 = l0 * l0 + m0 * m0;
  if (!(r2 < 1.0)) return BLINK_EINVAL;
  const int n_ant = p->n_ant, n_ch = p->n_ch, n_bl = p->n_bl;
  std::vector<double> h_g((size_t)n_ch * n_ant * 2), h_c(n_ant, 0.0);
  for (size_t k = 0; k < (size_t)n_ch * n_ant; ++k) {
    const double re = gains ? gains[2 * k] : 1.0, im = gains ? gains[2 * k + 1] : 0.0;
    const double a2 = re * re + im * im;
    if (!std::isfinite(a2) || !(a2 > 0.0)) return BLINK_EINVAL;
    h_g[2 * k] = re; h_g[2 * k + 1] = im;
  }
  if (cable_len_m)
    for (int a = 0; a < n_ant; ++a) {
      if (!std::isfinite(cable_len_m[a])) return BLINK_EINVAL;
      h_c[a] = cable_len_m[a];
    }
  std::vector<int32_t> pi(n_bl), pj(n_bl);
  {
    int bl = 0;
    for (int i = 0; i < n_ant; ++i)
      for (int j = i + 1; j < n_ant; ++j, ++bl) { pi[bl] = i; pj[bl] = j; }
  }
  cudaStream_t st = (cudaStream_t)stream;
  BLINK_CUDA_TRY(cudaSetDevice(p->device), "cudaSetDevice");
  double *d_ant = nullptr, *d_freq = nullptr, *d_g = nullptr, *d_c = nullptr;
  int32_t *d_pi = nullptr, *d_pj = nullptr;
  float2 *d_F = nullptr;
  cudaError_t ce = cudaSuccess;
  auto step = [&](cudaError_t e) { if (ce == cudaSuccess) ce = e; };
  step(cudaMalloc((void **)&d_ant, sizeof(double) * 3 * n_ant));
  step(cudaMalloc((void **)&d_freq, sizeof(double) * n_ch));
  step(cudaMalloc((void **)&d_g, sizeof(double) * h_g.size()));
  step(cudaMalloc((void **)&d_c, sizeof(double) * n_ant));
  step(cudaMalloc((void **)&d_pi, sizeof(int32_t) * n_bl));
  step(cudaMalloc((void **)&d_pj, sizeof(int32_t) * n_bl));
  step(cudaMalloc((void **)&d_F, sizeof(float2) * (size_t)n_ch * n_bl));
  if (ce == cudaSuccess) {
    step(cudaMemcpyAsync(d_ant, p->h_ant.data(), sizeof(double) * 3 * n_ant, cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(d_freq, p->h_freq.data(), sizeof(double) * n_ch, cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(d_g, h_g.data(), sizeof(double) * h_g.size(), cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(d_c, h_c.data(), sizeof(double) * n_ant, cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(d_pi, pi.data(), sizeof(int32_t) * n_bl, cudaMemcpyHostToDevice, st));
    step(cudaMemcpyAsync(d_pj, pj.data(), sizeof(int32_t) * n_bl, cudaMemcpyHostToDevice, st));
  }
  if (ce == cudaSuccess) {
    const double n0m1 = std::sqrt(1.0 - r2) - 1.0;
    k_corr_table<<<dim3((n_bl + 255) / 256, n_ch), 256, 0, st>>>(d_ant, d_pi, d_pj, d_freq, (const double2 *)d_g, d_c, l0, m0,
                                                                n0m1, n_ant, n_bl, n_ch, d_F);
    step(cudaGetLastError());
    step(cudaStreamSynchronize(st));
  }
  cudaFree(d_ant); cudaFree(d_freq); cudaFree(d_g); cudaFree(d_c); cudaFree(d_pi); cudaFree(d_pj);
  if (ce != cudaSuccess) {
    cudaFree(d_F);
    set_cuda_error(ce, "blink_plan_set_corrections");
    return ce == cudaErrorMemoryAllocation ? BLINK_ENOMEM : BLINK_ECUDA;
  }
  if (p->d_corr) {
    cudaDeviceSynchronize();          // an earlier table may still be in use by queued blink_correct calls
    cudaFree(p->d_corr);
  }
  p->d_corr = d_F;
  return BLINK_OK;
} catch (const std::bad_alloc &) {
  return BLINK_ENOMEM;                      // host tables; the plan keeps the state it had
} catch (...) {
  blink::set_error_text("blink_plan_set_corrections: unexpected C++ exception");
  return BLINK_ECUDA;
}

extern "C" int blink_correct(const blink_plan *p, const void *vis_in, int n_t, void *vis_out, void *stream) {
  using namespace blink;
  if (!p || n_t < 0) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!vis_in || !vis_out || !p->d_corr) return BLINK_EINVAL;
  if (((uintptr_t)vis_in & 7) || ((uintptr_t)vis_out & 7)) return BLINK_EINVAL;
  { const int rc = check_device(p); if (rc != BLINK_OK) return rc; }
  cudaStream_t st = (cudaStream_t)stream;
  const long long tab = (long long)p->n_ch * p->n_bl;
  const int blocks = p->sm_count * 8;
  if ((tab & 1) == 0 && (((uintptr_t)vis_in | (uintptr_t)vis_out) & 15) == 0)
    k_correct<<<blocks, 256, 0, st>>>((const float4 *)vis_in, (const float4 *)p->d_corr, (float4 *)vis_out, n_t, tab / 2);
  else
    k_correct1<<<blocks, 256, 0, st>>>((const float2 *)vis_in, p->d_corr, (float2 *)vis_out, n_t, tab);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_correct launch");
  return BLINK_OK;
}

// f2 as SURVEY.md section 8(f) words it: the corrections FUSED AT LOAD.  on = 1: blink_grid and
// blink_grid_image multiply every visibility by its factor as they read it -- in shared memory on the
// bulk-copy routes (the factors of a chunk ride in the same buffer as its visibilities and gather
// table; their table layouts are built here, on first use), in registers on the others -- so no
// separate 16-byte-per-visibility pass exists and the visibilities cross HBM once.
extern "C" int blink_plan_apply_corrections(blink_plan *p, int on, void *stream) try {
  using namespace blink;
  if (!p || (on != 0 && on != 1)) return BLINK_EINVAL;
  int rc = check_device(p);
  if (rc != BLINK_OK) return rc;
  if (on && !p->d_corr) return BLINK_EINVAL;
  if (on) {
    cudaStream_t st = (cudaStream_t)stream;
    if (p->fused_path == 1 && (rc = fused_layout(p, 1, st)) != BLINK_OK) return rc;
    if (p->tc_route && (rc = fused_layout_tc(p, 1, st)) != BLINK_OK) return rc;
    if (p->ring_path == 1 && (rc = grid_ring_layout(p, 1, st)) != BLINK_OK) return rc;
  }
  p->corr_on = on;
  p->corr_stale = 0;                  // the caller has said what it wants after a refresh
  return BLINK_OK;
} catch (const std::bad_alloc &) {
  return BLINK_ENOMEM;                      // host tables; the plan keeps the state it had
} catch (...) {
  blink::set_error_text("blink_plan_apply_corrections: unexpected C++ exception");
  return BLINK_ECUDA;
}
