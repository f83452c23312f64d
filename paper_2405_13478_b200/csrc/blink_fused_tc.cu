// blink_fused_tc.cu -- host side of k_fused_tc (fused_tc_kernel.cuh): the tensor-core form of
// blink_grid_image's shared-memory route at N = 256 -- its plan tables and its launcher.
#include <algorithm>
#include <cmath>
#include <cstring>

#include "blink_internal.h"
#include "fft_core.cuh"
#include "sgather.cuh"
#include "sphase.cuh"

#include "fused_kernel.cuh"
#include "fused_tc_kernel.cuh"

namespace blink {

// fp32 -> bf16 bits, round to nearest even (the operands of the constant matrix are finite)
static uint16_t bf16_rn(float x) {
  uint32_t u;
  std::memcpy(&u, &x, 4);
  u += 0x7FFFu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}
static float bf16_to_float(uint16_t h) {
  const uint32_t u = (uint32_t)h << 16;
  float x;
  std::memcpy(&x, &u, 4);
  return x;
}

// Tables of the tensor-core route.
//   cmat   the constant matrix C[n][K], n = 0..127, K = 128: K-group kg = K / 8 in 0..15 holds, for parity
//          p = kg / 8 and trig = (kg / 4) % 2 (0 cos, 1 sin), the frequencies k = 2 (8 (kg % 4) + e) + p,
//          e = K % 8; value cos / sin (2 pi k n / 256), fp64 -> fp32 -> bf16 hi + bf16 lo.  Operand layout
//          [kg][n][e] (16-byte vectors), hi block then lo block.
//   refs   per channel, [16][512] cell references: thread tid of the kernel handles kx = tid % 64, parity
//          p = (tid / 64) % 2, block b = tid / 128; reference row 2 i + sg (i = 0..7, sg = 0: +ky, 1: -ky)
//          with ky = 2 (8 b + i) + p names the cell H[+-ky][kx] as {slot of its canonical sum in S | placement
//          flag << 14, weight}, weight = fftshift sign x 1/norm x (1/count if uniform) x (2 if kx > 0); an
//          empty cell points at a zero slot with weight 0; -ky for ky = 0 is empty.  Bit 16 of row 0 says that
//          the whole task is empty.
int fused_tc_build(blink_plan *p, cudaStream_t st) {
  p->tc_route = 0;
  if (p->fused_path != 1 || p->n_pix != 256 || p->fused_D != 1 || p->opt.tune[kTuneTensor] != 1) return BLINK_OK;
  if (std::max(p->kx_max_all, p->ky_max_all) > 63) return BLINK_OK;
  int rc = fused_layout_tc(p, 0, st);
  if (rc != BLINK_OK) return rc;
  if (!p->tl[0].ok) return BLINK_OK;
  const int N = 256, n_ch = p->n_ch;
  const double two_pi = 6.283185307179586476925286766559;

  std::vector<uint16_t> cm(2 * 16 * 128 * 8);
  for (int kg = 0; kg < 16; ++kg)
    for (int n = 0; n < 128; ++n)
      for (int e = 0; e < 8; ++e) {
        const int par = kg / 8, trig = (kg / 4) % 2, k = 2 * (8 * (kg % 4) + e) + par;
        const double ang = two_pi * (double)((k * n) % N) / (double)N;
        const float v = (float)(trig ? std::sin(ang) : std::cos(ang));
        const uint16_t hi = bf16_rn(v), lo = bf16_rn(v - bf16_to_float(hi));
        const size_t idx = ((size_t)kg * 128 + n) * 8 + e;
        cm[idx] = hi;
        cm[16 * 128 * 8 + idx] = lo;
      }

  const int sink0 = (p->n_can_max + 15) & ~15;
  std::vector<uint2> refs((size_t)n_ch * kTcRefRows * kFusedThreads);
  parallel_for(n_ch, [&](int ch) {
    const HostGather &g = p->gathers[ch];
    const ChannelInfo &ci = p->chinfo[ch];
    std::vector<int> owner, slot;
    assign_cells(g, owner, slot);
    auto find_j = [&](int cell) -> int {
      auto it = std::lower_bound(g.can_cell.begin(), g.can_cell.end(), cell);
      return (it != g.can_cell.end() && *it == cell) ? (int)(it - g.can_cell.begin()) : -1;
    };
    uint2 *out = refs.data() + (size_t)ch * kTcRefRows * kFusedThreads;
    for (int tid = 0; tid < kFusedThreads; ++tid) {
      const int kx = tid & 63, par = (tid >> 6) & 1, b = tid >> 7;
      bool any = false;
      for (int i = 0; i < 8; ++i)
        for (int sg = 0; sg < 2; ++sg) {
          const int ky = (2 * (8 * b + i) + par) * (sg ? -1 : 1);
          uint2 r = make_uint2((uint32_t)sink0, 0u);                 // a zero slot x 0
          if (kx <= ci.kx_max && std::abs(ky) <= ci.ky_max && !(sg == 1 && ky == 0) && g.n_can > 0) {
            const int ix = kx, iy = (ky + N) % N;
            const bool canonical = (ky > 0) || (ky == 0 && kx >= 0);
            const int c = canonical ? iy * N + ix : ((N - iy) % N) * N + ((N - ix) % N);
            const int j = find_j(c);
            if (j >= 0) {
              int cnt = g.seg_start[j + 1] - g.seg_start[j];
              if (c == 0) cnt *= 2;
              float w = ((kx + ky) & 1) ? -ci.inv_norm : ci.inv_norm;
              if (p->weighting == BLINK_UNIFORM) w /= (float)cnt;
              if (kx > 0) w *= 2.0f;                                 // c_kx: the mirrored half kx < 0
              const uint32_t flag = c == 0 ? kPlaceBoth : (canonical ? kPlaceDirect : kPlaceConj);
              uint32_t wb;
              std::memcpy(&wb, &w, 4);
              r = make_uint2((uint32_t)slot[j] | (flag << 14), wb);
              any = true;
            }
          }
          out[(size_t)(2 * i + sg) * kFusedThreads + tid] = r;
        }
      if (!any) out[tid].x |= 0x10000u;
    }
  });
  if ((rc = upload_table((void **)&p->d_cmat, cm.data(), cm.size() * sizeof(uint16_t), st, "tc table")) != BLINK_OK) return rc;
  if ((rc = upload_table((void **)&p->d_tcref, refs.data(), refs.size() * sizeof(uint2), st, "tc table")) != BLINK_OK) return rc;
  BLINK_CUDA_TRY(cudaStreamSynchronize(st), "tc table upload sync");
  p->tc_route = 1;
  return BLINK_OK;
}

int launch_fused_tc(const blink_plan *p, const float2 *vis, int n_t, float *img, cudaStream_t st) {
  const GatherLayout &L = p->tl[p->corr_on ? 1 : 0];
  FusedTcParams q;
  FusedParams &fp = q.f;
  fp.vis = vis; fp.img = img; fp.chinfo = p->d_chinfo;
  fp.corr = p->corr_on ? p->d_corr : nullptr;
  fp.gtab = L.d_tab; fp.gsize = L.d_size; fp.hrec = nullptr; fp.hw = nullptr; fp.pha = nullptr; fp.tw = nullptr;
  fp.n_bl = p->n_bl; fp.n_ch = p->n_ch; fp.n_snap = n_t * p->n_ch; fp.n_can_max = p->n_can_max;
  fp.n_chunk = L.n_chunk; fp.chunk_vis = L.chunk_vis; fp.nbuf = L.nbuf;
  fp.tab_stride = L.tab_stride; fp.n_col = 0; fp.h_max = 0;
  fp.buf_bytes = L.buf_bytes; fp.tab_off = L.tab_off; fp.f_off = L.f_off;
  fp.off_dedicated = L.off_first; fp.off_S = L.off_S; fp.off_bar = L.off_bar; fp.smem = (uint32_t)L.smem;
  fp.chunk_shift = (8 << 16) / std::max(fp.n_chunk, 1);
  q.refs = p->d_tcref;
  q.cmat = p->d_cmat;
  q.nded = L.nded;
  const int blocks = std::min(fp.n_snap, p->sm_count);
  if (blocks <= 0) return BLINK_OK;
  static std::atomic<uint64_t> attr0{0}, attr1{0};
  if (p->corr_on) {
    const int rc = ensure_max_smem(k_fused_tc<true>, p, attr1, "k_fused_tc smem attribute");
    if (rc != BLINK_OK) return rc;
    k_fused_tc<true><<<blocks, kFusedThreads, fp.smem, st>>>(q);
  } else {
    const int rc = ensure_max_smem(k_fused_tc<false>, p, attr0, "k_fused_tc smem attribute");
    if (rc != BLINK_OK) return rc;
    k_fused_tc<false><<<blocks, kFusedThreads, fp.smem, st>>>(q);
  }
  BLINK_CUDA_TRY(cudaGetLastError(), "k_fused_tc launch");
  return BLINK_OK;
}

}  // namespace blink
