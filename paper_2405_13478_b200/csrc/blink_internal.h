// blink_internal.h -- plan object shared by the libblink translation units (not part of the ABI).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <atomic>
#include <string>
#include <thread>
#include <vector>

#include "../../include/blink.h"
#include "../../include/blink_testing.h"

namespace blink {

// flags in the high bits of a placement code; low bits = index j of the canonical-cell sum S[j]
constexpr int kPlaceShift = 28;
constexpr int32_t kPlaceMask = (1 << kPlaceShift) - 1;
constexpr int32_t kPlaceDirect = 0;  // grid[cell] = S[j]
constexpr int32_t kPlaceConj = 1;    // grid[cell] = conj(S[j])
constexpr int32_t kPlaceBoth = 2;    // grid[cell] = S[j] + conj(S[j])   (self-conjugate cell: DC)

constexpr int kBandCellsDefault = 2048;  // cells (complex64) per output band of the gridder = 16 KB
constexpr uint16_t kScatDropped = 0xFFFFu;  // scatter code of a baseline outside the grid
constexpr int kGridCellsPerThread = 5;      // register accumulators per thread in the per-cell sums

struct ChannelInfo {   // mirrored on the device, one per channel
  int32_t n_kept;      // baselines inside the grid
  int32_t n_can;       // distinct canonical (half-plane) cells
  int32_t n_place;     // occupied cells in the full plane
  int32_t kx_max, ky_max;
  float inv_norm;      // 1 / image normalisation
};

// blink_options::tune[] slots (0 = default), private to this version
enum TuneSlot {
  kTuneWarpFracA = 0,     // warp route: percent of the grid's CTAs that run pass A (default 60)
  kTuneWarpCtasPerSm = 1, // warp route: resident CTAs per SM
  kTuneFusedChunks = 2,   // shared-memory route: smallest number of chunks per snapshot tried
  kTuneImageCt = 3,       // two-pass imaging: columns per CTA (pass A)
  kTuneImageRp = 4,       // two-pass imaging: row pairs per CTA (pass B)
  kTuneDirectMax = 5,     // two-kernel route: most cells per column for the direct-sum column transform, +1 (default 13)
  kTuneDynspecRoute = 6,  // blink_dynspec: 1 = register-load kernel even for aligned cubes
  kTuneTensor = 7         // 1 = the shared-memory route at N = 256 runs its transforms on the tensor cores (k_fused_tc);
                          // default off: measured 0.422 ms against 0.403 ms for k_fused on the station
};

struct HostGather {    // cell-sorted tables of one channel (see blink_host_build_gather)
  int32_t n_kept = 0, n_can = 0;
  std::vector<int32_t> can_cell, seg_start, src;
};

// Shared-memory plan and device tables of one set of phase-S gather tables (sgather.cuh): chunks of
// chunk_vis baselines stream through a ring of nbuf buffers, each chunk with its gather table
// (tab_off bytes behind the visibilities) and -- when the pre-gridding corrections are fused in --
// its correction factors (f_off bytes behind the visibilities; 0 = none).
struct GatherLayout {
  int chunk_vis = 0, n_chunk = 0, nbuf = 0, tab_stride = 0, nded = 1;   // nded: dedicated (un-aliased) buffers
  uint32_t buf_bytes = 0, off_first = 0, off_S = 0, off_bar = 0, tab_off = 0, f_off = 0;
  size_t smem = 0;
  unsigned char *d_tab = nullptr;   // [n_ch][n_chunk][tab_stride]
  uint32_t *d_size = nullptr;       // [n_ch][n_chunk] bytes of each table (multiple of 16)
  bool ok = false;
};

// blink_grid_image_host (blink_host.cu): three streams over a ring of device staging buffers
struct HostPipe {
  static constexpr int kDepth = 3;
  int chunk_t = 0;                                  // time steps per chunk the buffers are sized for (0 = not reserved)
  float2 *d_vis[kDepth] = {};
  float *d_img[kDepth] = {};
  cudaStream_t st[3] = {};                          // in, compute, out
  cudaEvent_t in_done[kDepth] = {}, cmp_done[kDepth] = {}, out_done[kDepth] = {}, start = nullptr, done[3] = {};
};

}  // namespace blink

struct blink_plan {
  int n_ant = 0, n_bl = 0, n_ch = 0, n_pix = 0, weighting = 0;
  double pixscale = 0.0;
  int device = 0;
  int sm_count = 148;
  int max_smem_optin = 0;
  blink_options opt = {};           // as given to blink_plan_create_opts (zeros = defaults)
  blink::HostPipe hp;               // staging of blink_grid_image_host

  // inputs kept for blink_plan_set_corrections
  std::vector<double> h_ant, h_freq;
  float2 *d_corr = nullptr;         // [n_ch][n_bl] correction factors F (blink_correct.cu), NULL until set
  int corr_on = 0;                  // 1 = blink_grid / blink_grid_image multiply by F as they load (blink_plan_apply_corrections)
  int corr_stale = 0;               // 1 = the fused corrections were on when blink_plan_refresh dropped the table: the gridding
                                    // calls refuse (BLINK_EINVAL) until blink_plan_apply_corrections is called again
  std::vector<blink::HostGather> gathers;   // per-channel cell-sorted tables, kept for lazily built layouts

  // per-channel facts (host)
  std::vector<int64_t> n_dropped, wsum, n_occ;
  std::vector<double> norm;
  std::vector<blink::ChannelInfo> chinfo;

  // device tables
  int32_t *d_cell = nullptr;        // [n_ch][n_bl]
  uint32_t *d_counts = nullptr;     // [n_ch][N][N]
  blink::ChannelInfo *d_chinfo = nullptr;  // [n_ch]
  int32_t *d_src = nullptr;         // [n_ch][n_bl]      (bl << 1) | conj, sorted by (can cell, bl)
  int32_t *d_seg = nullptr;         // [n_ch][n_bl + 1]  CSR offsets of canonical cells into d_src
  int32_t *d_pcell = nullptr;       // [n_ch][2 n_bl]    occupied full-plane cells, ascending
  int32_t *d_pcode = nullptr;       // [n_ch][2 n_bl]    j | flag << kPlaceShift
  int32_t *d_pband = nullptr;       // [n_ch][n_bands+1] CSR of d_pcell by output band
  uint16_t *d_scat = nullptr;       // [n_ch][n_bl]      slot in its pass's rank-major stage | conj << 15
  uint32_t *d_cellrec = nullptr;    // [n_ch][n_pass][n_can_max] j | len << 16, by descending len
  uint16_t *d_roff = nullptr;       // [n_ch][n_pass][roff_stride] stage offset of rank r
  int32_t *d_nact = nullptr;        // [n_ch][n_pass]    cells with >= 1 baseline in the pass
  int roff_stride = 0;
  int stage_cap = 0;                // baselines staged in shared memory per pass
  int n_pass = 0;                   // ceil(n_bl / stage_cap)
  int grid_nbuf = 3;                // band buffers in flight per CTA
  int grid_ctas_per_sm = 1;
  int grid_threads = 512, grid_prefetch = 16;  // CTA shape: stage_cap = threads * prefetch
  size_t grid_smem = 0;
  float2 *d_tw = nullptr;           // [N] exp(+2 pi i k / N)
  // uniform weighting: sparse per-column list of the occupied half-plane cells and 1/count
  int32_t *d_wkey = nullptr;        // [n_ch][2 n_bl] (kx << 16) | iy, sorted by kx then iy
  float *d_wval = nullptr;          // [n_ch][2 n_bl] 1 / count
  int32_t *d_wcol = nullptr;        // [n_ch][wu + 1] CSR by column kx
  int img_ct = 0, img_rp = 0;       // tuning: columns per CTA (pass A), row pairs per CTA (pass B)
  int n_bands = 0;                  // bands per snapshot = N*N / band_cells
  int band_cells = 0;
  int n_can_max = 0;
  int kx_max_all = 0, ky_max_all = 0;

  // blink_image scratch (two-pass path): U[chunk][N][wu] complex64
  int wu = 0;                       // padded half-plane width
  float2 *d_scratch = nullptr;
  size_t scratch_bytes = 0;
  int reserved_n_t = 0;             // largest n_t blink_plan_reserve has been asked for
  int image_path = 1;
  int chunk_snapshots = 0;

  // blink_grid_image
  int fused_path = 0;               // 1 = shared-memory single kernel, 0 = chunked grid + image
  int fused_chunk = 0;              // snapshots per chunk of the chunked route
  // two-kernel route of blink_grid_image: pass A straight from the visibilities.  Occupied cells
  // with kx >= 0, sorted by column: where they go, which segment of d_src feeds them, weight
  int32_t *d_vkey = nullptr;        // [n_ch][2 n_bl] (kx << 16) | iy
  int32_t *d_vseg = nullptr;        // [n_ch][2 n_bl] first entry in d_src (channel-relative)
  int32_t *d_vlen = nullptr;        // [n_ch][2 n_bl] entries | flag << 24
  float *d_vw = nullptr;            // [n_ch][2 n_bl] sign * (1/norm) * (1/count if uniform)
  int32_t *d_vcol = nullptr;        // [n_ch][wu + 1] CSR by column
  uint4 *d_vrec = nullptr;          // [n_ch][2 n_bl] packed cell records: iy | flag << 16 | len << 18, weight, source 0, source 1 / segment
  int vtile8_max = 0;               // most cells in any 8-column tile of any channel
  float2 *d_tw32 = nullptr;         // [32][32] exp(+2 pi i b n1 / 1024) (wfft.cuh), N = 1024 only
  int warp_route = 0;               // 1 = blink_grid_image takes the warp-per-transform kernel (blink_image_w.cu)
  int seg_len_max = 0;              // most baselines in any canonical cell of any channel
  int warp_ring = 0;                // slots of U in the warp route's ring
  long long warp_snap_cap = 0;      // snapshots per call the warp route's counters in scratch are sized for
  // residue-class route at N = 1024 (blink_image_r.cu): the intermediate stays in shared memory, no scratch
  int res_route = 0;                // 1 = blink_grid_image / blink_image take k_img1024r (N = 1024); 2 = the column pass of the
                                    // two-kernel routes is k_cols_res (N = 2048 / 4096)
  int16_t *d_rcols = nullptr;       // [16][32][2] columns of every lane of k_cols_res
  int res_cap = 0;                  // positions per channel of its tables
  uint4 *d_rrec = nullptr;          // [n_ch][res_cap] cell records, lane-interleaved lists per producer warp
  uint32_t *d_rmeta = nullptr;      // [n_ch][res_cap] cell descriptors (iy, last-of-entry, tile slot)
  int32_t *d_rhdr = nullptr;        // [n_ch][8][2] per-warp headers
  uint32_t *d_rmask = nullptr;      // [n_ch][512] non-empty bins per column
  // blink_grid, ring route (see grid_ring_build in blink_grid.cu): phase S as in k_fused
  int ring_path = 0;                // 1 = k_grid_ring available
  int ring_min_snap = 0;            // fewer snapshots per call take the band route
  blink::GatherLayout rl[2];        // [0] plain, [1] with correction factors (built by blink_plan_apply_corrections)
  int2 *d_rplace = nullptr;         // [n_ch][2 n_bl] {cell, slot of S | flag << 30}, ascending cell

  // shared-memory route (see fused_build in blink_fused.cu)
  int h_max = 0;                    // phase-H records per channel (padded with pos = 0xFFFF)
  int fused_threads = 512;
  blink::GatherLayout fl[2];        // [0] plain, [1] with correction factors; off_first = the dedicated buffer 0
  // tensor-core form of the route (k_fused_tc, fused_tc_kernel.cuh): N = 256, bounding box inside |k| < 64
  int tc_route = 0;                 // 1 = blink_grid_image takes k_fused_tc
  blink::GatherLayout tl[2];        // its phase-S layouts ([0] plain, [1] with correction factors)
  uint2 *d_tcref = nullptr;         // [n_ch][16][512] phase-H cell references
  uint4 *d_cmat = nullptr;          // [4096] the constant cosine / sine matrix, bf16 hi | lo, operand layout
  uint2 *d_hrec = nullptr;          // [n_ch][h_max] {line position | j << 16 | flag << 30, weight}
  int fused_D = 1;                  // polyphase route: the image is fused_D x fused_D interleaved sub-images of n_pix / fused_D
  float2 *d_hw = nullptr;           // [n_ch][fused_D][h_max] complex phase-H weights of the sub-image rows
  float2 *d_pha = nullptr;          // [fused_D][n_pix / fused_D / 2] column phases of the sub-image columns
  float2 *d_tw_sub = nullptr;       // [n_pix / fused_D] twiddles of the sub-transforms

};

namespace blink {

// arguments of the imaging kernels (blink_image.cu, blink_image_w.cu)
struct ImgParams {
  const float2 *uv;
  float *img;
  float2 *U;
  const ChannelInfo *chinfo;
  const int32_t *wkey, *wcol;
  const float *wval;
  // pass A straight from visibilities (blink_grid_image, two-kernel route)
  const float2 *vis;
  const int32_t *src, *vkey, *vseg, *vlen, *vcol;
  const float *vw;
  const float2 *tw, *tw32;
  int n_ch, n_bl, wu, uniform, snap_base, ch0, direct_max, cell_cap;
  const float2 *corr;   // [n_ch][n_bl] correction factors applied to the visibilities as they are loaded, or NULL
};

#if defined(__CUDACC__)
// one visibility, corrected at load when a factor table is given (f2 fused: V * F, blink_correct.cu)
__device__ __forceinline__ float2 ld_vis(const float2 *__restrict__ vis, const float2 *__restrict__ cf, int i) {
  float2 v = __ldg(vis + i);
  if (cf != nullptr) {
    const float2 f = __ldg(cf + i);
    v = make_float2(v.x * f.x - v.y * f.y, v.x * f.y + v.y * f.x);
  }
  return v;
}
#endif

// warp-per-transform persistent kernel at N = 1024 (blink_image_w.cu)
int launch_img1024(const blink_plan *p, ImgParams ip, int n_snap, cudaStream_t st);
bool warp_route_applies(const blink_plan *p);
size_t warp_route_scratch_bytes(const blink_plan *p, long long n_snap);
size_t warp_route_ring_bytes(const blink_plan *p);
// residue-class kernel at N = 1024 (blink_image_r.cu)
int res_route_build(blink_plan *p, cudaStream_t st);
void res_route_free(blink_plan *p);
int launch_img1024r(const blink_plan *p, ImgParams ip, int n_snap, cudaStream_t st);
int launch_cols_res(const blink_plan *p, const ImgParams &ip, int n_snap, cudaStream_t st);   // pass A of a chunk of n_snap snapshots

}  // namespace blink

namespace blink {

void set_cuda_error(cudaError_t e, const char *where);
void set_error_text(const char *text);   // a non-CUDA explanation, read back through blink_last_cuda_error
void host_pipe_free(blink_plan *p);
int build_gather_host(const int32_t *cell, int n_bl, int n_pix, HostGather &out);

// kernels' host launchers (each returns a blink_status)
int launch_index_kernel(blink_plan *p, const double *d_ant, const double *d_freq,
                        const int32_t *d_pi, const int32_t *d_pj, cudaStream_t st);
// n_snap consecutive snapshots whose first one is channel ch0 (channel of snapshot s = (ch0 + s) % n_ch)
int launch_grid(const blink_plan *p, const float2 *vis, int n_snap, int ch0, float2 *uv, cudaStream_t st);
int launch_image(const blink_plan *p, const float2 *uv, int n_snap, int ch0, float *img, cudaStream_t st);
int image_setup(blink_plan *p);
int image_reserve(blink_plan *p, int n_t);
// device scratch a call of n_t time steps needs: blink_image (fused = false) or blink_grid_image
size_t scratch_need(const blink_plan *p, long long n_t, bool fused);
int grid_ring_build(blink_plan *p, cudaStream_t st);
int grid_ring_layout(blink_plan *p, int corr, cudaStream_t st);
int fused_setup(blink_plan *p);
int fused_build(blink_plan *p, cudaStream_t st);
int fused_layout(blink_plan *p, int corr, cudaStream_t st);
int fused_layout_tc(blink_plan *p, int corr, cudaStream_t st);
int fused_tc_build(blink_plan *p, cudaStream_t st);
int launch_fused_tc(const blink_plan *p, const float2 *vis, int n_t, float *img, cudaStream_t st);
int upload_table(void **dst, const void *src, size_t bytes, cudaStream_t st, const char *what);
// true when blink_grid_image takes the shared-memory kernel in the plan's current state
inline bool fused_smem_route(const blink_plan *p) {
  return p->fused_path == 1 && (p->fl[p->corr_on ? 1 : 0].ok || (p->tc_route && p->tl[p->corr_on ? 1 : 0].ok));
}
int fused_line_stride(int n_pix);
int fused_nz_instance(const blink_plan *p);
int launch_grid_image(const blink_plan *p, const float2 *vis, int n_t, float *img, cudaStream_t st);
int launch_image_from_vis(const blink_plan *p, const float2 *vis, int n_snap, float *img, cudaStream_t st);

}  // namespace blink

// gridding calls after a refresh that dropped active corrections: refuse rather than grid uncorrected data
inline int check_corrections_current(const blink_plan *p) {
  if (!p->corr_stale) return BLINK_OK;
  blink::set_error_text("the plan applied corrections at load before blink_plan_refresh dropped their table: call "
                        "blink_plan_set_corrections and blink_plan_apply_corrections(plan, 1) again, or "
                        "blink_plan_apply_corrections(plan, 0) to grid uncorrected");
  return BLINK_EINVAL;
}

// hot calls: the plan's device must be current
inline int check_device(const blink_plan *p) {
  int d = -1;
  if (cudaGetDevice(&d) != cudaSuccess) return BLINK_ECUDA;
  return d == p->device ? BLINK_OK : BLINK_EINVAL;
}

#define BLINK_CUDA_TRY(expr, where)                 \
  do {                                              \
    cudaError_t e__ = (expr);                       \
    if (e__ != cudaSuccess) {                       \
      blink::set_cuda_error(e__, where);            \
      return BLINK_ECUDA;                           \
    }                                               \
  } while (0)

namespace blink {
// cudaFuncSetAttribute is per device: `done` holds one bit per device ordinal that has it.  The
// attribute is set to the device's opt-in maximum once, so no launch ever needs to raise it again.
template <class K> inline int ensure_max_smem(K kern, const blink_plan *p, std::atomic<uint64_t> &done, const char *what,
                                              bool carveout = true) {
  const uint64_t bit = 1ull << (p->device & 63);
  if (done.load(std::memory_order_acquire) & bit) return BLINK_OK;
  BLINK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, p->max_smem_optin), what);
  if (carveout) BLINK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100), what);
  done.fetch_or(bit, std::memory_order_release);
  return BLINK_OK;
}
}  // namespace blink

#include "parallel_for.h"
