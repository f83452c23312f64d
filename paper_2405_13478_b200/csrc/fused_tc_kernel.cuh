// fused_tc_kernel.cuh -- k_fused_tc: the shared-memory route of blink_grid_image at N = 256 with the
// two transform passes on the 5th-generation tensor cores (tcgen05.mma, accumulators in TMEM).
//
// The uv plane of a station snapshot is band-limited (|kx|, |ky| < 64 of 256; SKA-Low station: 41), so
// both passes of the inverse DFT (steps a4/a5; Eq. 4-5 :162-167) are dense
// contractions of the snapshot's cell sums against a CONSTANT cosine / sine matrix -- the one place on
// the path where a tensor-core contraction fits.  With H[ky][kx] the weighted,
// normalised, sign-flipped (fftshift) cell sums of the half-plane kx >= 0 (phase S as in k_fused),
//
//   pass A   U[y][kx]  = sum_ky H[ky][kx] e^{2 pi i ky y / N}
//   pass B   I[y][x]   = sum_kx c_kx Re(U[y][kx] e^{2 pi i kx x / N}),   c_0 = 1, c_kx = 2 (folded into H)
//
// Both use the parity of the frequency index as a radix-2 step, so every matrix has 128 rows:
//   U[y] = Ue[y] + Uo[y],  U[y + 128] = Ue[y] - Uo[y]      (Ue / Uo: even / odd ky, y < 128)
//   I[y][x] = Ie + Io,     I[y][x + 128] = Ie - Io          (Ie / Io: even / odd kx, x < 128)
// and the +-ky pairs are folded (Hs = H[ky] + H[-ky], Hd = H[ky] - H[-ky]) so that only k >= 0 appears:
//   Ue_r = sum_{ky even} Hs_r cos - Hd_i sin,   Ue_i = sum_{ky even} Hs_i cos + Hd_r sin     (same for Uo)
//   Ie   = sum_{kx even} U_r cos - U_i sin                                                    (same for Io)
// One constant matrix serves both passes: C[n][K], n = 0..127 (y in pass A, x in pass B), K = 128 columns
// (cos k even | sin k even | cos k odd | sin k odd), k = 0..63, angle 2 pi k n / 256.
//
// Precision.  The tensor cores take bf16 operands; every fp32 operand is split into bf16 hi + lo and a
// product is three MMAs, hi.hi + hi.lo + lo.hi, accumulated in fp32 in TMEM -- 2.7e-6 of the image
// peak on a station snapshot (numpy emulation and the GPU parity tests; bar 1e-4).
//
// Per snapshot, one persistent CTA of 512 threads per SM:
//   phase S    as k_fused: visibilities + gather tables stream through a ring of bulk-copied chunks, every
//              canonical cell is summed by the warp that owns it (optionally x correction factors)
//   phase H    thread (kx, parity, block of 8 ky) forms Hs / Hd of its 8 cells from the sums, splits them
//              and stores them as rows (kx, re) and (kx, im) of the pass-A operand B_H[128][128] (hi, lo)
//   MMA A      one thread: D_A[128 y][Ue_r | Ue_i | Uo_r | Uo_i] = C (cols of that parity) x B_H^T, 24 MMAs
//   per half t of the image rows (y = m + 128 t):
//     convert  warps read D_A from TMEM, form U = Ue +- Uo, split, store the pass-B operand (over B_H)
//     MMA B    TRANSPOSED: (Ie^T | Io^T) = C x (U-operand)^T, lanes = image column x, columns = the half's rows
//   store      (during the next phase S) warps read a unit and write I[y][x] = Ie + Io, I[y][x + 128] = Ie - Io:
//              a warp's store of one register is 128 contiguous bytes
// TMEM (512 columns): D_A 256 + half 0, then half 1 over D_A: the finished image (256 KB) sits in TMEM and
// is written out between the chunks of the NEXT snapshot's phase S, so image stores and visibility loads
// overlap.  Shared memory: operand region 64 KB (B_H, then the U-operand; idle during phase S, so chunk
// buffers alias it), C 64 KB, dedicated chunk buffers, cell sums.
#pragma once

#include <cuda_bf16.h>

namespace blink {

constexpr uint32_t kTcOper = 0;            // operand region: hi at +0, lo at +32768
constexpr uint32_t kTcOperBytes = 65536;
constexpr uint32_t kTcCmat = 65536;        // constant matrix: hi at +0, lo at +32768
constexpr uint32_t kTcFixedBytes = 131072; // operand region + constant matrix
constexpr int kTcRefRows = 16;             // cell references per phase-H task: 8 ky x (+ky, -ky)

struct FusedTcParams {
  FusedParams f;              // phase S and the common fields (hrec, hw, pha, tw unused)
  const uint2 *refs;          // [n_ch][16][512] {slot | flag << 14 | empty << 16, weight}
  const uint4 *cmat;          // [4096] the constant matrix in operand layout, hi then lo
  int nded;                   // dedicated chunk buffers (buffers 0 .. nded - 1)
};

__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {
  // K-major, no swizzle: core matrix = 8 rows x 16 bytes, contiguous; rows of a K-group 16 bytes apart
  // (stride-byte-offset between 8-row groups = 128), K-groups 128 rows x 16 bytes apart (leading-byte-
  // offset = 2048); descriptor version 1 (sm_100)
  return (uint64_t)((saddr >> 4) & 0x3FFFu) | ((uint64_t)(2048u >> 4) << 16) | ((uint64_t)(128u >> 4) << 32) | (1ull << 46);
}
// instruction descriptor: D fp32, A / B bf16, both K-major, M = 128
template <int NN> __device__ __forceinline__ uint32_t umma_idesc() {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(NN >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}"
               ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float *v) {
  uint32_t r[16];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                 "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, float *v) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr));
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// eight fp32 values -> eight bf16 (round to nearest even) and the eight bf16 of what the rounding lost
__device__ __forceinline__ void split8(const float *x, uint4 &hi, uint4 &lo) {
  uint32_t h[4], l[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const __nv_bfloat162 hb = __floats2bfloat162_rn(x[2 * i], x[2 * i + 1]);
    const float r0 = x[2 * i] - __low2float(hb), r1 = x[2 * i + 1] - __high2float(hb);
    const __nv_bfloat162 lb = __floats2bfloat162_rn(r0, r1);
    h[i] = reinterpret_cast<const uint32_t &>(hb);
    l[i] = reinterpret_cast<const uint32_t &>(lb);
  }
  hi = make_uint4(h[0], h[1], h[2], h[3]);
  lo = make_uint4(l[0], l[1], l[2], l[3]);
}
// operand element (row n, K-group kg) as a 16-byte vector: hi at base + (kg * 128 + n) * 16, lo 32 KB behind
__device__ __forceinline__ void store_split8(unsigned char *oper, int kg, int n, const float *x) {
  uint4 hi, lo;
  split8(x, hi, lo);
  uint4 *p = reinterpret_cast<uint4 *>(oper + ((size_t)kg * 128 + n) * 16);
  p[0] = hi;
  p[2048] = lo;                 // + 32768 bytes
}

// the three bf16 products of one K = 64 half (four K-steps of 16): A rows at a_base, B rows at b_base
// (byte addresses of the hi parts; lo parts 32 KB behind), into tmem_d; first = the accumulator starts here
template <int NN> __device__ __forceinline__ void umma_k64(uint32_t tmem_d, uint32_t a_base, uint32_t b_base) {
  const uint32_t idesc = umma_idesc<NN>();
#pragma unroll
  for (int prod = 0; prod < 3; ++prod) {
    const uint32_t a = a_base + (prod == 2 ? 32768u : 0u), b = b_base + (prod == 1 ? 32768u : 0u);
#pragma unroll
    for (int ks = 0; ks < 4; ++ks)
      umma_bf16(tmem_d, umma_desc(a + ks * 4096u), umma_desc(b + ks * 4096u), idesc, (prod | ks) != 0);
  }
}

template <bool CORR>
__global__ void __launch_bounds__(kFusedThreads, 1) k_fused_tc(const FusedTcParams q) {
  constexpr int THREADS = kFusedThreads, N = 256;
  const FusedParams &p = q.f;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char *oper = smem_raw + kTcOper;
  float2 *S = reinterpret_cast<float2 *>(smem_raw + p.off_S);
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + p.off_bar);        // [nbuf]
  uint64_t *empty = full + p.nbuf;                                            // [nbuf]
  uint64_t *bar_a = empty + p.nbuf;         // MMA A complete
  uint64_t *bar_b = bar_a + 1;              // [2] MMA B of half t (image rows 128 t .. 128 t + 127) complete
  uint32_t *tmem_ptr = reinterpret_cast<uint32_t *>(bar_b + 2);
  const uint32_t sm_base = smem_u32(smem_raw), S_base = sm_base + p.off_S;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t vis_bytes = p.tab_off;
  const int nded = q.nded;
  // chunk c of every snapshot lives in buffer c % nbuf; buffers 0 .. nded - 1 are dedicated, the others
  // alias the operand region
  auto buf_of = [&](int b) -> unsigned char * {
    return b < nded ? smem_raw + p.off_dedicated + (size_t)b * p.buf_bytes : smem_raw + (size_t)(b - nded) * p.buf_bytes;
  };
  uint32_t fphase = 0, ephase = 0, pa = 0, pb = 0;   // pb: parity of bar_b[] for the snapshot in flight
  auto produce = [&](int s, int c, int b) {    // thread 0 only; b = c % nbuf
    mbar_wait(empty + b, ((ephase >> b) & 1u) ^ 1u);
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
    // (an L2 prefetch of the chunk that follows this one into the same buffer: no gain, 0.426 against 0.422 ms;
    // of the whole next snapshot: 60 % of it read from DRAM twice)
  };

  if (tid == 0) {
    for (int b = 0; b < p.nbuf; ++b) {
      mbar_init(full + b, 1);
      mbar_init(empty + b, kFusedWarps);
    }
    mbar_init(bar_a, 1);
    mbar_init(bar_b, 1);
    mbar_init(bar_b + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {     // all of tensor memory: one CTA per SM
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_ptr)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  const int n_S = ((p.n_can_max + 15) & ~15) + 16;
  for (int j = tid; j < n_S; j += THREADS) S[j] = make_float2(0.f, 0.f);
  if constexpr (CORR) {
    float2 *z = reinterpret_cast<float2 *>(smem_raw + p.off_dedicated) + p.chunk_vis;
    if (tid < 16) z[tid] = make_float2(0.f, 0.f);
    else if (tid < 32) reinterpret_cast<float2 *>(reinterpret_cast<unsigned char *>(z) + p.f_off)[tid - 16] = make_float2(0.f, 0.f);
  }
  {   // the constant matrix, once
    uint4 *c = reinterpret_cast<uint4 *>(smem_raw + kTcCmat);
    for (int i = tid; i < 4096; i += THREADS) c[i] = __ldg(q.cmat + i);
  }
  fence_async_smem();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_ptr;
  const uint32_t oper_a = sm_base + kTcOper, cmat_a = sm_base + kTcCmat;
  if (tid == 0)
    for (int c = 0; c < min(nded, p.n_chunk); ++c)
      if ((int)blockIdx.x < p.n_snap) produce(blockIdx.x, c, c);

  // this thread's roles: phase H task (kx, parity, block) and TMEM quadrant / column part
  const int h_kx = tid & 63, h_p = (tid >> 6) & 1, h_b = tid >> 7;
  const int qd = warp & 3, part = warp >> 2, row = qd * 32 + lane;
  const uint32_t t_lane = tmem + ((uint32_t)(qd * 32) << 16);

  // The finished image of a snapshot stays in TMEM (all 512 columns: eight units of 32 rows, transposed) and is
  // written out unit by unit BETWEEN the chunks of the next snapshot's phase S, so that the image stores and
  // the visibility loads stream at the same time instead of taking turns at the HBM.
  float *img_prev = nullptr;               // image whose units are still in TMEM
  auto drain = [&](int u) {                // unit u -> image rows 32 u + 8 part + e, columns row and row + 128
    mbar_wait(bar_b + (u >> 2), pb ^ 1u);
    tc_fence_after();
    const uint32_t slot = t_lane + (u < 4 ? 256 : 0) + 32 * (u & 3);    // half 0 in columns 256.., half 1 over D_A
    float2 ie[4], io[4];
    tmem_ld8(slot + 8 * part, reinterpret_cast<float *>(ie));
    tmem_ld8(slot + 128 + 8 * part, reinterpret_cast<float *>(io));
    tmem_ld_wait();
    float *__restrict__ o = img_prev + (size_t)(32 * u + 8 * part) * N + row;
#pragma unroll
    for (int e = 0; e < 4; ++e) {          // packed fp32 pairs: one instruction per two pixels
      const float2 a = blinkfft::cadd(ie[e], io[e]), d = blinkfft::csub(ie[e], io[e]);
      o[(2 * e) * N] = a.x;
      o[(2 * e) * N + 128] = d.x;
      o[(2 * e + 1) * N] = a.y;
      o[(2 * e + 1) * N + 128] = d.y;
    }
  };
  // units to have drained after chunk c of the next phase S: spread evenly over the chunks
  auto drained_after = [&](int c) { return c + 1 >= p.n_chunk ? 8 : (int)(((uint32_t)(c + 1) * (uint32_t)p.chunk_shift) >> 16); };

  auto chunk_step = [&](int s, int c, int b) {   // chunk c of snapshot s (in buffer b): sums, release, refill
    mbar_wait(full + b, (fphase >> b) & 1u);
    fphase ^= 1u << b;
    consume_chunk<CORR>(smem_u32(buf_of(b)) + vis_bytes, warp, lane, sm_base, S_base, p.f_off);
    __syncwarp();
    if (lane == 0) mbar_arrive(empty + b);
    if (tid == 0) {
      if (c + p.nbuf < p.n_chunk) produce(s, c + p.nbuf, b);
      else if (b < nded && b < p.n_chunk && s + (int)gridDim.x < p.n_snap)
        produce(s + gridDim.x, b, b);        // the buffer's last chunk of this snapshot: next snapshot's chunk b
    }
  };

  for (int s = blockIdx.x; s < p.n_snap; s += gridDim.x) {
    const int ch = s % p.n_ch;
    // the operand region is idle until phase H: fill its chunk buffers once the previous snapshot's last
    // MMAs (which read it) are complete
    if (tid == 0) {
      if (img_prev != nullptr) mbar_wait(bar_b + 1, pb ^ 1u);
      for (int c = nded; c < min(p.n_chunk, p.nbuf); ++c) produce(s, c, c);
    }
    int next_u = 0;
    // the phase-H cell references do not depend on the sums: request them now, they arrive during phase S
    uint2 r[kTcRefRows];
    {
      const uint2 *__restrict__ refs = q.refs + (size_t)ch * (kTcRefRows * THREADS) + tid;
      r[0] = __ldg(refs);
      if (!(r[0].x & 0x10000u)) {
#pragma unroll
        for (int i = 1; i < kTcRefRows; ++i) r[i] = __ldg(refs + i * THREADS);
      }
    }
    // ---- phase S ----------------------------------------------------------------------------
    for (int c = 0, b = 0; c < p.n_chunk; ++c) {
      chunk_step(s, c, b);
      if (++b == p.nbuf) b = 0;
      if (img_prev != nullptr)               // the previous image leaves TMEM in step with the chunks
        for (const int want = drained_after(c); next_u < want; ++next_u) drain(next_u);
    }
    tc_fence_before();
    __syncthreads();                         // all sums done, every chunk buffer released, TMEM drained

    // ---- phase H: B_H rows (kx, re) = h_kx and (kx, im) = 64 + h_kx, K-groups of parity h_p, block h_b --
    {
      float hs_r[8], hs_i[8], nhd_i[8], hd_r[8];
      if (r[0].x & 0x10000u) {               // no occupied cell in this task
#pragma unroll
        for (int i = 0; i < 8; ++i) hs_r[i] = hs_i[i] = nhd_i[i] = hd_r[i] = 0.f;
      } else {
        auto cellv = [&](uint2 rr) -> float2 {
          const float2 v = S[rr.x & 0x3FFFu];
          const uint32_t flag = (rr.x >> 14) & 3u;
          const float w = __uint_as_float(rr.y);
          if (flag == kPlaceDirect) return make_float2(v.x * w, v.y * w);
          if (flag == kPlaceConj) return make_float2(v.x * w, -v.y * w);
          return make_float2((v.x + v.x) * w, 0.f);
        };
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float2 hp = cellv(r[2 * i]), hm = cellv(r[2 * i + 1]);
          hs_r[i] = hp.x + hm.x;
          hs_i[i] = hp.y + hm.y;
          nhd_i[i] = hm.y - hp.y;
          hd_r[i] = hp.x - hm.x;
        }
      }
      const int kg = h_p * 8 + h_b;          // K-group of the cosine columns; the sine columns are 4 groups on
      store_split8(oper, kg, h_kx, hs_r);
      store_split8(oper, kg + 4, h_kx, nhd_i);
      store_split8(oper, kg, 64 + h_kx, hs_i);
      store_split8(oper, kg + 4, 64 + h_kx, hd_r);
    }
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    // ---- MMA A: D_A cols [0,128) = Ue (re | im), [128,256) = Uo ----------------------------------
    if (tid == 32) {
      tc_fence_after();
      umma_k64<128>(tmem, cmat_a, oper_a);
      umma_k64<128>(tmem + 128, cmat_a + 4 * 4096u, oper_a + 4 * 4096u);
      umma_commit(bar_a);
    }
    // the sums are consumed: clear them for the next snapshot (the zero slots stay zero)
    for (int j = tid; j < p.n_can_max; j += THREADS) S[j] = make_float2(0.f, 0.f);
    // (taking the next snapshot's chunk 0 here, behind MMA A, was measured: 0.436 ms against 0.422 -- its copy
    // has not landed yet, the wait only moves)
    mbar_wait(bar_a, pa);
    pa ^= 1u;
    tc_fence_after();

    float *__restrict__ img = p.img + (size_t)s * N * N;
#pragma unroll 1
    for (int t = 0; t < 2; ++t) {
      // ---- convert: U = Ue +- Uo for kx in [16 part, 16 part + 16) of row `row`, into the operand region.  The
      // arithmetic of half 1 runs while the MMAs of half 0 are still reading the region; only its stores wait.
      {
        uint4 hi[4], lo[4];
        float ue[16], uo[16], x_e[8], x_o[8];
        tmem_ld16(t_lane + 16 * part, ue);
        tmem_ld16(t_lane + 128 + 16 * part, uo);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          x_e[e] = t ? ue[2 * e] - uo[2 * e] : ue[2 * e] + uo[2 * e];
          x_o[e] = t ? ue[2 * e + 1] - uo[2 * e + 1] : ue[2 * e + 1] + uo[2 * e + 1];
        }
        split8(x_e, hi[0], lo[0]);                    // cos, kx even
        split8(x_o, hi[2], lo[2]);                    // cos, kx odd
        tmem_ld16(t_lane + 64 + 16 * part, ue);
        tmem_ld16(t_lane + 192 + 16 * part, uo);
        tmem_ld_wait();
#pragma unroll
        for (int e = 0; e < 8; ++e) {      // the operand holds -U_i
          x_e[e] = t ? uo[2 * e] - ue[2 * e] : -(ue[2 * e] + uo[2 * e]);
          x_o[e] = t ? uo[2 * e + 1] - ue[2 * e + 1] : -(ue[2 * e + 1] + uo[2 * e + 1]);
        }
        split8(x_e, hi[1], lo[1]);                    // sin, kx even
        split8(x_o, hi[3], lo[3]);                    // sin, kx odd
        if (t == 1) {                      // half 0's MMAs must have finished reading the operand region
          mbar_wait(bar_b, pb);
          tc_fence_after();
        }
#pragma unroll
        for (int g = 0; g < 4; ++g) {
          uint4 *dst = reinterpret_cast<uint4 *>(oper + ((size_t)(4 * g + part) * 128 + row) * 16);
          dst[0] = hi[g];
          dst[2048] = lo[g];
        }
      }
      fence_async_smem();
      tc_fence_before();
      __syncthreads();
      // ---- MMA B, transposed: (Ie^T | Io^T) of image rows 128 t .. 128 t + 127: lanes = image column x (rows of
      // C), columns = image rows (rows of the U-operand).  Half 0 goes to TMEM columns 256.., half 1 over D_A,
      // which the second convert has just finished reading.
      if (tid == 32) {
        tc_fence_after();
        const uint32_t slot = tmem + (t ? 0 : 256);
        umma_k64<128>(slot, cmat_a, oper_a);
        umma_k64<128>(slot + 128, cmat_a + 4 * 4096u, oper_a + 4 * 4096u);
        umma_commit(bar_b + t);
      }
    }
    img_prev = img;
    pb ^= 1u;
  }
  if (img_prev != nullptr)
    for (int u = 0; u < 8; ++u) drain(u);
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
}

}  // namespace blink
