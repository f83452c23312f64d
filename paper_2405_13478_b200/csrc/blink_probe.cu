// blink_probe.cu -- in-run measurement of the fp32 ALU peak ("an fp32 FMA loop"),
// the denominator of bench.py's ALU side bound.  Not on the hot path: a register-only kernel whose
// threads run eight independent dependency chains of one instruction kind, so the fp32 pipe is the only
// limit.  bench.py times the launch with CUDA events and divides *flops by the time.
#ifdef BLINK_TESTING_HOOKS   // libblink_testing.so only (build.py): libblink.so carries no host model and no probe
#include "blink_internal.h"

namespace blink {

// OP 0: add.f32 (FADD, 1 flop)   1: fma.rn.f32 (FFMA, 2 flops)
//    2: add.rn.f32x2 (FADD2, 2 flops)   3: fma.rn.f32x2 (FFMA2, 4 flops)
template <int OP> __global__ void __launch_bounds__(256) k_probe_fp32(float *__restrict__ out, int iters, float a, float b) {
  constexpr int CH = 8;
  const int tid = blockIdx.x * blockDim.x + threadIdx.x;
  if constexpr (OP < 2) {
    float x[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) x[c] = (float)(tid + c) * 1e-9f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int u = 0; u < 8; ++u)
#pragma unroll
        for (int c = 0; c < CH; ++c) {
          if constexpr (OP == 0) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(x[c]) : "f"(b));
          else asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[c]) : "f"(a), "f"(b));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < CH; ++c) s += x[c];
    out[tid] = s;
  } else {
    unsigned long long x[CH];
    const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
    const unsigned long long ua = reinterpret_cast<const unsigned long long &>(a2), ub = reinterpret_cast<const unsigned long long &>(b2);
#pragma unroll
    for (int c = 0; c < CH; ++c) {
      const float2 v = make_float2((float)(tid + c) * 1e-9f, (float)(tid - c) * 1e-9f);
      x[c] = reinterpret_cast<const unsigned long long &>(v);
    }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int u = 0; u < 8; ++u)
#pragma unroll
        for (int c = 0; c < CH; ++c) {
          if constexpr (OP == 2) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(x[c]) : "l"(ub));
          else asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[c]) : "l"(ua), "l"(ub));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < CH; ++c) {
      const float2 v = reinterpret_cast<const float2 &>(x[c]);
      s += v.x + v.y;
    }
    out[tid] = s;
  }
}

}  // namespace blink

extern "C" int blink_probe_fp32(int op, int iters, void *out_dev, size_t out_floats, int64_t *flops, void *stream) {
  using namespace blink;
  if (op < 0 || op > 3 || iters < 1 || !out_dev || out_floats < 256 || !flops) return BLINK_EINVAL;
  const int blocks = (int)std::min<size_t>(out_floats / 256, 1u << 20);
  cudaStream_t st = (cudaStream_t)stream;
  float *out = (float *)out_dev;
  switch (op) {
    case 0: k_probe_fp32<0><<<blocks, 256, 0, st>>>(out, iters, 0.999f, 1e-7f); break;
    case 1: k_probe_fp32<1><<<blocks, 256, 0, st>>>(out, iters, 0.999f, 1e-7f); break;
    case 2: k_probe_fp32<2><<<blocks, 256, 0, st>>>(out, iters, 0.999f, 1e-7f); break;
    default: k_probe_fp32<3><<<blocks, 256, 0, st>>>(out, iters, 0.999f, 1e-7f); break;
  }
  BLINK_CUDA_TRY(cudaGetLastError(), "k_probe_fp32 launch");
  static const int kFlopsPerOp[4] = {1, 2, 2, 4};
  *flops = (int64_t)blocks * 256 * (int64_t)iters * 64 * kFlopsPerOp[op];
  return BLINK_OK;
}
#endif  // BLINK_TESTING_HOOKS
