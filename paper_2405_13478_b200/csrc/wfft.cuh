// wfft.cuh -- warp-per-transform inverse FFT of 1024 points (step a4).
//
// One warp owns one transform, every lane 32 of its points in registers; the transform is the
// 32 x 32 Cooley-Tukey split of N = 1024 (sign e^{+...}, Eq. 4-5, unnormalised):
//
//   k = 32 a + b,  n = n1 + 32 n2   (a, b, n1, n2 = 0..31)
//   X[n1 + 32 n2] = sum_b w32^(b n2) * [ w1024^(b n1) * sum_a x[32 a + b] w32^(a n1) ]
//
//   inner  : lane b holds z[a] = x[32 a + b]; a 32-point butterfly in registers gives the bracket's
//            sum for n1 = 0..31, then the twiddle w1024^(b n1) from a table laid out [n1][b]
//   exchange: lane b writes row b of a 32 x 32 tile in shared memory (row stride 34 complex =
//            272 B: 16-byte stores of 8 lanes and 8-byte loads of 16 lanes are both conflict-free),
//            lane n1 reads column n1
//   outer  : lane n1 holds t[b]; a second 32-point butterfly gives X[n1 + 32 n2], n2 = 0..31, so a
//            warp-wide store of register n2 covers 32 consecutive outputs.
//
// Only __syncwarp() separates the phases.  The pieces are plain inline functions of (lane, data) so
// tests/host_fft_check.cpp runs the same index algebra lane by lane on the CPU.
#pragma once

#include "fft_core.cuh"

namespace blinkfft {

constexpr int kWfN = 1024;
constexpr int kWfRow = 34;                    // complex slots per exchange row
constexpr int kWfTile = 32 * kWfRow;          // complex slots per warp's exchange tile

struct alignas(16) cf32q { float x, y, z, w; };

// twiddle table for the inner step: tab[n1 * 32 + b] = exp(+2 pi i b n1 / 1024) (symmetric in b, n1)
// inner butterfly + twiddle for lane b.  `tw(i)` returns tab[i].
template <class TwLoad> BLINK_HD void wf_inner(cf32 *z, int b, TwLoad tw) {
  dft32(z);
#pragma unroll
  for (int n1 = 1; n1 < 32; ++n1) z[n1] = cmul(z[n1], tw(n1 * 32 + b));
}

// lane b writes its 32 values as row b (16-byte stores)
BLINK_HD void wf_put(cf32 *tile, int b, const cf32 *z) {
  cf32q *row = reinterpret_cast<cf32q *>(tile + b * kWfRow);
#pragma unroll
  for (int j = 0; j < 16; ++j) {
    cf32q q;
    q.x = z[2 * j].x; q.y = z[2 * j].y; q.z = z[2 * j + 1].x; q.w = z[2 * j + 1].y;
    row[j] = q;
  }
}

// lane n1 reads column n1
BLINK_HD void wf_get(const cf32 *tile, int n1, cf32 *t) {
#pragma unroll
  for (int b = 0; b < 32; ++b) t[b] = tile[b * kWfRow + n1];
}

// column n1 with rows outside `mask` known to be zero (never read)
BLINK_HD void wf_get_masked(const cf32 *tile, int n1, unsigned mask, cf32 *t) {
#pragma unroll
  for (int b = 0; b < 32; ++b) t[b] = ((mask >> b) & 1u) ? tile[b * kWfRow + n1] : mk(0.f, 0.f);
}

}  // namespace blinkfft
