// fused_kernel.cuh -- k_fused, the shared-memory route of blink_grid_image (see blink_fused.cu for the
// whole picture), as a header so that its instantiations can live in translation units that choose
// different forms of the complex arithmetic (fft_core.cuh: BLINK_SCALAR_COMPLEX; sgather.cuh:
// BLINK_PHASE_S_PACKED).  Include after blink_internal.h, fft_core.cuh, sgather.cuh, sphase.cuh.
#pragma once

#include <algorithm>

namespace blink {
using namespace blinkfft;

// ---------------------------------------------------------------------------------------------
// Shared-memory route.  One persistent CTA per SM images one snapshot at a time without the uv
// grid ever leaving the SM:
//   phase S   the snapshot's visibilities arrive in shared memory in INPUT order, in chunks of
//             `chunk_vis` baselines, by bulk asynchronous copies (cp.async.bulk global -> shared,
//             completion on an mbarrier; no thread instructions, no registers), each chunk together
//             with the plan's gather table for that (channel, chunk), so every table access in the
//             inner loop is a shared-memory read.  Every canonical (half-plane) cell is OWNED by one
//             warp for the whole kernel, so the sums need no atomics and no barriers between warps:
//             per chunk a warp walks its cells in groups of 32 (one cell per lane, grouped by
//             descending number of baselines in the chunk, rows padded with a pointer to a zero slot)
//             and adds each group's sums into S[j].  Chunk buffers form a ring with full/empty
//             mbarriers: buffer 0 is dedicated (so the first chunk of the NEXT snapshot streams in
//             during phase H and passes A and B), the others alias the column lines and the pass-B
//             exchange lines, which are idle during phase S.  Thread 0 is the producer.
//   phase H   every cell of the bounding box with kx >= 0 is written -- weighted, normalised and
//             sign-flipped for the fftshift, zero where no baseline lands -- into per-column lines in
//             shared memory (the grid is exactly Hermitian by construction, so the half-plane is all
//             that is needed);
//   pass A    column transforms along ky, in place in the lines, loads pruned to the bounding box;
//   pass B    row transforms, two real image rows per complex transform, read from the lines across
//             columns and stored to global memory straight from the last butterfly stage.
// A transform is owned by T = N/16 <= 16 lanes of one warp, so the exchanges inside it need only
// __syncwarp.  The last-stage twiddles depend only on the lane, so they live in registers for the
// whole kernel.
constexpr int kHPer = 7;              // phase-H records fetched per thread ahead of the barrier

struct FusedParams {
  const float2 *vis;
  const float2 *corr;         // CORR: [n_ch][n_bl] correction factors, copied chunk by chunk beside the visibilities
  float *img;
  const ChannelInfo *chinfo;
  const unsigned char *gtab;  // [n_ch][n_chunk][tab_stride] phase-S gather tables (see fused_build)
  const uint32_t *gsize;      // [n_ch][n_chunk] bytes of each table (multiple of 16)
  const uint2 *hrec;          // [n_ch][h_max] {pos | j << 16 | flag << 30, weight}; pos 0xFFFF = padding
  const float2 *hw;           // D > 1: [n_ch][D][h_max] complex phase-H weights of the sub-image rows b (see k_fused)
  const float2 *pha;          // D > 1: [D][N/2] column phases e^{2 pi i kx a / (D N)} of the sub-image columns a
  const float2 *tw;
  int n_bl, n_ch, n_snap, n_can_max, n_chunk, chunk_vis, nbuf, tab_stride, n_col, h_max;
  uint32_t buf_bytes, off_dedicated, off_S, off_bar;   // byte offsets into dynamic shared memory
  uint32_t tab_off, f_off, smem;                       // table / factors behind a buffer's visibilities; launch smem bytes
  int chunk_shift;                                     // k_fused_tc: floor(8 * 65536 / n_chunk): (c * this) >> 16 = 8 c / n_chunk
};



// NZ: the first radix-16 stage of both passes reads inputs r = 0..NZ-1 and 16-NZ..15 only (the
// bounding box reaches at most NZ * N/16 - 1 cells from the origin); NZ = 8 reads everything.
//
// D > 1 (polyphase route for compact arrays on large images): the image has D N x D N pixels but the
// bounding box still fits an N x N transform (|k| < N/2).  Writing X = D x' + a, Y = D y' + b,
//   I[Y][X] = sum_k (G[k] e^{2 pi i (kx a + ky b) / (D N)}) e^{2 pi i (kx (x' - N/2) + ky (y' - N/2)) / N},
// i.e. the image is D*D interleaved N x N images of the SAME cell sums, each with its own unit-modulus
// factor per cell (odd in k, so the modulated grid stays Hermitian and the two-rows-per-transform
// trick still holds).  The ky part of the factor is folded into the phase-H weight, the kx part is
// constant along a column, so it commutes with pass A and is applied when pass B loads the column
// values.  Phase S runs once per snapshot, phases H and A once per b, pass B once per (b, a) with the
// D transform groups of a row pair side by side in a warp; no transform longer than N is ever taken and no zero outside the bounding box is
// ever touched.
template <int N, int THREADS, int NZ, int D, bool CORR>
__global__ void __launch_bounds__(THREADS, 1) k_fused(const FusedParams p) {
  constexpr int T = N / 16;             // lanes per transform
  constexpr int G = THREADS / T;        // transforms in flight per CTA
  constexpr int LS = ((LineSize<N>::value + 15) / 16) * 16 + 1;
  constexpr int LSB = LineSize<N>::value;
  using F = Fft<N>;
  static_assert(F::NSTAGE == 2 && T <= 32, "shared-memory route needs a two-stage warp-local transform");
  static_assert(THREADS == kFusedThreads, "the gather tables are built for kFusedWarps warps");
  constexpr unsigned BM = BandMask<NZ>::value;
  constexpr int NZL = NZ >= 8 ? 8 : NZ;         // inputs read from each end of a first-stage butterfly
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float2 *lines = reinterpret_cast<float2 *>(smem_raw);                       // [n_col][LS]
  float2 *X = lines + (size_t)p.n_col * LS;                                   // exchange lines [G][LSB]
  float2 *S = reinterpret_cast<float2 *>(smem_raw + p.off_S);                 // [n_can_max up to 16 | 16 sinks]
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + p.off_bar);        // [nbuf]
  uint64_t *empty = full + p.nbuf;                                            // [nbuf]
  uint64_t *region_free = empty + p.nbuf;   // every warp has finished pass B: lines / exchange area reusable
  const uint32_t sm_base = smem_u32(smem_raw), S_base = sm_base + p.off_S;
  const int tid = threadIdx.x;
  const int warp = tid >> 5, lane = tid & 31;
  const int grp = tid / T, t = tid % T;
  const uint32_t vis_bytes = p.tab_off;
  // chunk c of every snapshot lives in buffer c % nbuf; buffer 0 is the dedicated one, the others
  // alias the lines / exchange area
  auto buf_of = [&](int b) -> unsigned char * {
    return b == 0 ? smem_raw + p.off_dedicated : smem_raw + (size_t)(b - 1) * p.buf_bytes;
  };
  uint32_t fphase = 0;                  // bit b: parity of the next wait on full[b]
  uint32_t ephase = 0;                  // producer only: bit b: parity of the last completed empty[b] phase
  uint32_t rphase = 0;                  // producer only: parity of the next wait on region_free
  auto produce = [&](int s, int c, int b) {    // thread 0 only; b = c % nbuf
    mbar_wait(empty + b, ((ephase >> b) & 1u) ^ 1u);   // every warp has let go of the buffer
    ephase ^= 1u << b;
    const int cnt = min(p.chunk_vis, p.n_bl - c * p.chunk_vis);
    const uint32_t vb = (uint32_t)cnt * sizeof(float2);
    const size_t cp = (size_t)(s % p.n_ch) * p.n_chunk + c;
    const uint32_t tb = __ldg(p.gsize + cp);
    unsigned char *dst = buf_of(b);
    mbar_expect_tx(full + b, (CORR ? 2 * vb : vb) + tb);
    bulk_load(dst, p.vis + (size_t)s * p.n_bl + (size_t)c * p.chunk_vis, vb, full + b);
    bulk_load(dst + vis_bytes, p.gtab + cp * p.tab_stride, tb, full + b);
    if constexpr (CORR)
      bulk_load(dst + p.f_off, p.corr + (size_t)(s % p.n_ch) * p.n_bl + (size_t)c * p.chunk_vis, vb, full + b);
  };

  if (tid == 0) {
    for (int b = 0; b < p.nbuf; ++b) {
      mbar_init(full + b, 1);
      mbar_init(empty + b, kFusedWarps);
    }
    mbar_init(region_free, kFusedWarps);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // S[0..n_can_max-1] cell sums; S[sink0 + b], b = 0..15: one always-zero slot per bank (sinks of
  // padded lanes and the "zero visibility" padded entries point at)
  const int n_S = ((p.n_can_max + 15) & ~15) + 16;
  for (int j = tid; j < n_S; j += THREADS) S[j] = make_float2(0.f, 0.f);
  if constexpr (CORR) {
    // the 16 "zero visibility" slots behind chunk buffer 0's visibilities, and their factor partners
    float2 *z = reinterpret_cast<float2 *>(smem_raw + p.off_dedicated) + p.chunk_vis;
    if (tid < 16) z[tid] = make_float2(0.f, 0.f);
    else if (tid < 32) reinterpret_cast<float2 *>(reinterpret_cast<unsigned char *>(z) + p.f_off)[tid - 16] = make_float2(0.f, 0.f);
  }
  const float2 *pha_s = S + n_S;        // D > 1: [D][N/2] column phases of the sub-images, right after the sums
  if constexpr (D > 1)
    for (int j = tid; j < D * (N / 2); j += THREADS) S[n_S + j] = __ldg(p.pha + j);
  // last-stage twiddles w^(r k), k fixed per lane: registers for the whole kernel
  constexpr int R1 = F::template radix<1>();
  constexpr int NB1 = 16 / R1;
  cf32 tw1[NB1][R1 > 1 ? R1 : 2];
#pragma unroll
  for (int b = 0; b < NB1; ++b) F::template twiddles<1>(tw1[b], t + b * T, p.tw);
  __syncthreads();
  if (tid == 0 && blockIdx.x < p.n_snap) produce(blockIdx.x, 0, 0);
  const int c_last0 = ((p.n_chunk - 1) / p.nbuf) * p.nbuf;   // last chunk of a snapshot in buffer 0

  for (int s = blockIdx.x; s < p.n_snap; s += gridDim.x) {
    const int ch = s % p.n_ch;
    const ChannelInfo ci = p.chinfo[ch];
    // the lines / exchange area is idle until phase H: fill it with this snapshot's next chunks, once
    // every warp has left pass B of the previous snapshot (the other warps start on chunk 0 meanwhile)
    if (tid == 0) {
      if (s != (int)blockIdx.x) {
        mbar_wait(region_free, rphase);
        rphase ^= 1u;
      }
      for (int c = 1; c < min(p.n_chunk, p.nbuf); ++c) produce(s, c, c);
    }

    // phase-H records do not depend on the sums: request them now, they arrive during phase S
    uint2 hr[kHPer];
    const uint2 *__restrict__ hrec = p.hrec + (size_t)ch * p.h_max;
#pragma unroll
    for (int q = 0; q < kHPer; ++q) {
      const int e = tid + q * THREADS;
      hr[q] = e < p.h_max ? __ldg(hrec + e) : make_uint2(0xFFFFu, 0u);
    }

    // ---- phase S ----------------------------------------------------------------------------
    for (int c = 0, b = 0; c < p.n_chunk; ++c) {
      mbar_wait(full + b, (fphase >> b) & 1u);
      fphase ^= 1u << b;
      consume_chunk<CORR>(smem_u32(buf_of(b)) + vis_bytes, warp, lane, sm_base, S_base, p.f_off);
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + b);    // this warp is done with the buffer
      if (tid == 0) {
        if (c + p.nbuf < p.n_chunk) produce(s, c + p.nbuf, b);
        else if (c == c_last0 && s + (int)gridDim.x < p.n_snap) produce(s + gridDim.x, 0, 0);
      }
      if (++b == p.nbuf) b = 0;
    }

    // ---- phase H: every bounding-box cell with kx >= 0, weighted, into the column lines --------
    const int kym = ci.ky_max;
    const int kxm = ci.kx_max;
    float2 *xl = X + (size_t)grp * LSB;
#pragma unroll 1
    for (int sub_b = 0; sub_b < D; ++sub_b) {
    {
      __syncthreads();                              // all sums done, all chunk buffers released (sub > 0: pass B done with the lines)
      auto place = [&](uint2 r, int e) {
        const uint32_t pos = r.x & 0xFFFFu;
        if (pos == 0xFFFFu) return;
        const float2 v = S[(r.x >> 16) & 0x3FFFu];
        const uint32_t flag = r.x >> 30;
        float2 o;
        if constexpr (D == 1) {
          const float w = __uint_as_float(r.y);
          if (flag == kPlaceDirect) o = make_float2(v.x * w, v.y * w);
          else if (flag == kPlaceConj) o = make_float2(v.x * w, -v.y * w);
          else o = make_float2((v.x + v.x) * w, 0.f);
        } else {
          const float2 w = __ldg(p.hw + ((size_t)ch * D + sub_b) * p.h_max + e);
          float2 z;
          if (flag == kPlaceDirect) z = v;
          else if (flag == kPlaceConj) z = make_float2(v.x, -v.y);
          else z = make_float2(v.x + v.x, 0.f);
          o = make_float2(z.x * w.x - z.y * w.y, z.x * w.y + z.y * w.x);
        }
        lines[pos] = o;
      };
#pragma unroll
      for (int q = 0; q < kHPer; ++q) place(hr[q], tid + q * THREADS);
      for (int e = tid + kHPer * THREADS; e < p.h_max; e += THREADS) place(__ldg(hrec + e), e);
    }
    __syncthreads();
    // the sums are consumed: clear them for the next snapshot (sink and zero slot stay zero)
    if (sub_b == D - 1)
      for (int j = tid; j < p.n_can_max; j += THREADS) S[j] = make_float2(0.f, 0.f);

    // ---- pass A: columns kx = 0..kx_max, in place ----------------------------------------------
    for (int c0 = 0; c0 <= ci.kx_max; c0 += G) {
      const int c = c0 + grp;
      const bool act = c <= ci.kx_max;            // uniform per transform group (T lanes)
      float2 *line = lines + (size_t)(act ? c : 0) * LS;
      cf32 v[16];
      if (act) {
        // stage-0 inputs idx = t + r*T: only r < NZL and r >= 16 - NZL can lie inside the bounding box
#pragma unroll
        for (int r = 0; r < 16; ++r) {
          if (r >= NZL && r < 16 - NZL) continue;
          const int idx = t + r * T;
          v[r] = (idx <= kym || idx >= N - kym) ? line[pad16(idx)] : mk(0.f, 0.f);
        }
      }
      __syncwarp();
      if (act) {
        F::template compute0_pruned<BM>(v);
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
    float *__restrict__ img = p.img + (size_t)s * (D * N) * (D * N) + (size_t)sub_b * (D * N);
    // items = (row pair, sub-image column a), a fastest: the D transform groups of one row pair are
    // neighbours in a warp (D = 2: its two half-warps), so a warp-wide store of one register covers
    // interleaved pixels D x' + a -- 128 contiguous bytes at D = 2.  a = grp % D is fixed per thread.
    const int my_a = D > 1 ? grp % D : 0;
    for (int q0 = 0; q0 < (N / 2) * D; q0 += G) {
      const bool act = q0 + grp < (N / 2) * D;
      const int y0 = act ? (q0 + grp) / D : 0, y1 = y0 + N / 2;
      const int o0 = pad16(y0), o1 = pad16(y1);
      cf32 v[16];
      if (act) {
        // stage-0 inputs Z[idx], idx = t + r*T: r < 8 direct half (a + i b), r >= 8 mirrored half
        // (conj a + i conj b at k = N - idx) -- static per r, branch-free, all loads in flight
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          float2 a[NZL], b[NZL];
#pragma unroll
          for (int q = 0; q < NZL; ++q) {
            const int r = h == 0 ? q : 16 - NZL + q;
            const int idx = t + r * T;
            const int k = h == 0 ? idx : N - idx;
            const bool ok = k <= kxm;
            a[q] = ok ? lines[k * LS + o0] : make_float2(0.f, 0.f);
            b[q] = ok ? lines[k * LS + o1] : make_float2(0.f, 0.f);
          }
#pragma unroll
          for (int q = 0; q < NZL; ++q) {
            const int r = h == 0 ? q : 16 - NZL + q;
            v[r] = h == 0 ? mk(a[q].x - b[q].y, a[q].y + b[q].x) : mk(a[q].x + b[q].y, b[q].x - a[q].y);
            if constexpr (D > 1) {
              // column phase e^{2 pi i kx a / (D N)} of sub-image a: kx = +k for the direct half, -k mirrored
              const int idx = t + r * T;
              const int k = h == 0 ? idx : N - idx;
              const float2 ph = pha_s[my_a * (N / 2) + (k & (N / 2 - 1))];
              v[r] = h == 0 ? cmul(v[r], mk(ph.x, ph.y)) : cmul(v[r], mk(ph.x, -ph.y));
            }
          }
        }
        F::template compute0_pruned<BM>(v);
      }
      __syncwarp();                                   // previous round's reads of xl are done
      if (act) F::template store<0>(v, t, [&](int idx, cf32 x) { xl[pad16(idx)] = x; });
      __syncwarp();
      if (act) {
        F::template load<1>(v, t, [&](int idx) { return xl[pad16(idx)]; });
        F::template compute_tw<1>(v, tw1);
        float *__restrict__ r0 = img + (size_t)y0 * (D * D * N) + my_a, *__restrict__ r1 = img + (size_t)y1 * (D * D * N) + my_a;
        F::template store<1>(v, t, [&](int x, cf32 z) { __stcs(r0 + D * x, z.x); __stcs(r1 + D * x, z.y); });
      }
    }
    }   // sub_b
    // generic-proxy writes to the lines / exchange area are ordered before the next snapshot's
    // bulk copies into the same bytes; no CTA-wide barrier: a warp that is done moves on to phase S
    // of the next snapshot (its own cell sums, the dedicated buffer) while others finish pass B
    fence_async_smem();
    __syncwarp();
    if (lane == 0) mbar_arrive(region_free);
  }
}

template <int N, int NZ, int D = 1, bool CORR = false>
static int launch_fused_n(const blink_plan *p, const FusedParams &fp, cudaStream_t st) {
  constexpr int THREADS = kFusedThreads;
  static std::atomic<uint64_t> attr{0};
  const int rc = ensure_max_smem(k_fused<N, THREADS, NZ, D, CORR>, p, attr, "k_fused smem attribute");
  if (rc != BLINK_OK) return rc;
  const int blocks = std::min(fp.n_snap, p->sm_count);
  if (blocks <= 0) return BLINK_OK;
  k_fused<N, THREADS, NZ, D, CORR><<<blocks, THREADS, fp.smem, st>>>(fp);
  BLINK_CUDA_TRY(cudaGetLastError(), "k_fused launch");
  return BLINK_OK;
}

}  // namespace blink
