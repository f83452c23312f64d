// blink_fused_d4.cu -- the k_fused instantiations of the polyphase route with D = 4 (compact arrays imaged at
// 1024^2: sixteen interleaved 256^2 sub-images per snapshot).  Same kernel header as blink_fused.cu, but the
// complex adds as scalar FADDs: with packed fp32 pairs (FADD2) this instance measured 5.41 ms against
// 5.26 ms per 4000 sweep1024 snapshots, while D = 1 and D = 2 gain 2.5 % and 5 % from the packed form --
// hence two translation units over one kernel header.
#define BLINK_SCALAR_COMPLEX
#include "blink_internal.h"
#include "fft_core.cuh"
#include "sgather.cuh"
#include "sphase.cuh"
#include "fused_kernel.cuh"

namespace blink {

int launch_fused_d4(const blink_plan *p, const FusedParams &fp, int nz, cudaStream_t st) {
  if (fp.corr) return nz <= 3 ? launch_fused_n<256, 3, 4, true>(p, fp, st) : launch_fused_n<256, 8, 4, true>(p, fp, st);
  return nz <= 3 ? launch_fused_n<256, 3, 4, false>(p, fp, st) : launch_fused_n<256, 8, 4, false>(p, fp, st);
}

}  // namespace blink
