// blink_fused_small.cu -- the k_fused instantiations for N <= 128 (blink_grid_image, shared-memory route).
// These sizes spend most of their time in phase S (the 32640 visibilities of a station snapshot against
// a 128^2 image), and both the gather sums and the butterflies measured faster with packed fp32 pairs
// (add.rn.f32x2, SASS FADD2: sweep128 0.382 -> 0.363 ms per 4000 snapshots), while k_fused<256> measured
// 2 % slower with either -- hence two translation units over one kernel header.
#define BLINK_PHASE_S_PACKED
#include "blink_internal.h"
#include "fft_core.cuh"
#include "sgather.cuh"
#include "sphase.cuh"
#include "fused_kernel.cuh"

namespace blink {

int launch_fused_small(const blink_plan *p, const FusedParams &fp, cudaStream_t st) {
  if (fp.corr) {
    switch (p->n_pix) {
      case 32: return launch_fused_n<32, 8, 1, true>(p, fp, st);
      case 64: return launch_fused_n<64, 8, 1, true>(p, fp, st);
      case 128: return launch_fused_n<128, 8, 1, true>(p, fp, st);
      default: return BLINK_EUNSUPPORTED;
    }
  }
  switch (p->n_pix) {
    case 32: return launch_fused_n<32, 8>(p, fp, st);
    case 64: return launch_fused_n<64, 8>(p, fp, st);
    case 128: return launch_fused_n<128, 8>(p, fp, st);
    default: return BLINK_EUNSUPPORTED;
  }
}

}  // namespace blink
