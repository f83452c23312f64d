// fft_core.cuh -- register/shared-memory Stockham building blocks for the batched inverse FFT
// (step a4; the paper calls cuFFT/hipFFT PlanMany + ExecC2C, this is the
// hand-written replacement).  Inverse direction only: X[n] = sum_k x[k] exp(+2 pi i k n / N)
// (sign from Eq. 4-5), unnormalised.
//
// Every thread owns E = 16 complex points of one length-N transform (T = N/16 threads per
// transform).  A transform is 2 or 3 radix-{2,4,8,16} Stockham autosort stages; between stages the
// points are exchanged through a padded shared-memory line.  The per-thread phases (load / twiddle
// + butterfly / store) are plain inline functions usable from host code too, so the index algebra
// is unit-tested on the CPU (tests/host_fft_check.cpp) before it ever runs on a GPU.
#pragma once

#if defined(__CUDACC__)
#define BLINK_HD __host__ __device__ __forceinline__
#include <cuda_runtime.h>
typedef float2 cf32;
#else
#define BLINK_HD inline
struct cf32 { float x, y; };
#endif

namespace blinkfft {

BLINK_HD cf32 mk(float x, float y) { cf32 r; r.x = x; r.y = y; return r; }
#if defined(__CUDA_ARCH__) && !defined(BLINK_SCALAR_COMPLEX)
// sm_100a packed fp32 pairs (SASS FADD2): one issue slot per complex add; same rounding as two FADDs
__device__ __forceinline__ cf32 cadd(cf32 a, cf32 b) {
  unsigned long long r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(reinterpret_cast<const unsigned long long &>(a)), "l"(reinterpret_cast<const unsigned long long &>(b)));
  return reinterpret_cast<const cf32 &>(r);
}
__device__ __forceinline__ cf32 csub(cf32 a, cf32 b) {
  unsigned long long r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(reinterpret_cast<const unsigned long long &>(a)), "l"(reinterpret_cast<const unsigned long long &>(b)));
  return reinterpret_cast<const cf32 &>(r);
}
#else
BLINK_HD cf32 cadd(cf32 a, cf32 b) { return mk(a.x + b.x, a.y + b.y); }
BLINK_HD cf32 csub(cf32 a, cf32 b) { return mk(a.x - b.x, a.y - b.y); }
#endif
BLINK_HD cf32 cmul(cf32 a, cf32 b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
BLINK_HD cf32 cconj(cf32 a) { return mk(a.x, -a.y); }
BLINK_HD cf32 mul_i(cf32 a) { return mk(-a.y, a.x); }   // a * (+i)

#define BLINK_SQRT1_2 0.70710678118654752440f
#define BLINK_COS_PI_8 0.92387953251128675613f
#define BLINK_SIN_PI_8 0.38268343236508977173f

// ---- inverse DFT butterflies, natural-order in, natural-order out --------------------------
BLINK_HD void dft2(cf32 &a, cf32 &b) {
  cf32 t = a;
  a = cadd(t, b);
  b = csub(t, b);
}

BLINK_HD void dft4(cf32 &a, cf32 &b, cf32 &c, cf32 &d) {
  cf32 t0 = cadd(a, c), t1 = csub(a, c), t2 = cadd(b, d), t3 = mul_i(csub(b, d));
  a = cadd(t0, t2);
  c = csub(t0, t2);
  b = cadd(t1, t3);
  d = csub(t1, t3);
}

BLINK_HD void dft8(cf32 *v) {  // v[0..7]
  cf32 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
  cf32 o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
  dft4(e0, e1, e2, e3);
  dft4(o0, o1, o2, o3);
  // o[k] *= w8^k, w8 = exp(+i pi/4)
  o1 = mk(BLINK_SQRT1_2 * (o1.x - o1.y), BLINK_SQRT1_2 * (o1.x + o1.y));
  o2 = mul_i(o2);
  o3 = mk(-BLINK_SQRT1_2 * (o3.x + o3.y), BLINK_SQRT1_2 * (o3.x - o3.y));
  v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
  v[1] = cadd(e1, o1); v[5] = csub(e1, o1);
  v[2] = cadd(e2, o2); v[6] = csub(e2, o2);
  v[3] = cadd(e3, o3); v[7] = csub(e3, o3);
}

BLINK_HD void dft16(cf32 *v) {  // v[0..15]
  cf32 e[8], o[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
  dft8(e);
  dft8(o);
  // o[k] *= w16^k, w16 = exp(+i pi/8) = (C, S)
  const float C = BLINK_COS_PI_8, S = BLINK_SIN_PI_8, Q = BLINK_SQRT1_2;
  o[1] = cmul(o[1], mk(C, S));
  o[2] = mk(Q * (o[2].x - o[2].y), Q * (o[2].x + o[2].y));
  o[3] = cmul(o[3], mk(S, C));
  o[4] = mul_i(o[4]);
  o[5] = cmul(o[5], mk(-S, C));
  o[6] = mk(-Q * (o[6].x + o[6].y), Q * (o[6].x - o[6].y));
  o[7] = cmul(o[7], mk(-C, S));
#pragma unroll
  for (int k = 0; k < 8; ++k) { v[k] = cadd(e[k], o[k]); v[k + 8] = csub(e[k], o[k]); }
}

template <int R> BLINK_HD void dft(cf32 *v);
template <> BLINK_HD void dft<2>(cf32 *v) { dft2(v[0], v[1]); }
template <> BLINK_HD void dft<4>(cf32 *v) { dft4(v[0], v[1], v[2], v[3]); }
template <> BLINK_HD void dft<8>(cf32 *v) { dft8(v); }
template <> BLINK_HD void dft<16>(cf32 *v) { dft16(v); }
BLINK_HD void dft32(cf32 *v);
template <> BLINK_HD void dft<32>(cf32 *v) { dft32(v); }

// ---- pruned butterflies: inputs known to be zero at compile time --------------------------------
// dftp<R, M>(v) is dft<R>(v) for inputs whose bit in M is clear being zero (their v[] entries are
// never read).  Decimation in time: the even- and odd-indexed inputs are transformed separately
// with their own masks and combined; a half with no non-zero input costs nothing, and the other
// half's outputs are then copied (or negated) instead of added.  Used for the first stage of the
// image transforms, whose inputs vanish outside the plan's bounding box.
template <int A> BLINK_HD cf32 mul_w16(cf32 x) {   // x * exp(+i pi A / 8), A = 0..7
  if constexpr (A == 0) return x;
  else if constexpr (A == 4) return mul_i(x);
  else if constexpr (A == 2) return mk(BLINK_SQRT1_2 * (x.x - x.y), BLINK_SQRT1_2 * (x.x + x.y));
  else if constexpr (A == 6) return mk(-BLINK_SQRT1_2 * (x.x + x.y), BLINK_SQRT1_2 * (x.x - x.y));
  else if constexpr (A == 1) return cmul(x, mk(BLINK_COS_PI_8, BLINK_SIN_PI_8));
  else if constexpr (A == 3) return cmul(x, mk(BLINK_SIN_PI_8, BLINK_COS_PI_8));
  else if constexpr (A == 5) return cmul(x, mk(-BLINK_SIN_PI_8, BLINK_COS_PI_8));
  else return cmul(x, mk(-BLINK_COS_PI_8, BLINK_SIN_PI_8));
}

// 32-point butterfly: radix-2 decimation in time over two 16-point butterflies (used by the
// warp-per-transform kernels, wfft.cuh, where a lane owns 32 points of a 1024-point transform)
#define BLINK_COS_PI_16 0.98078528040323044913f
#define BLINK_SIN_PI_16 0.19509032201612826785f
#define BLINK_COS_3PI_16 0.83146961230254523708f
#define BLINK_SIN_3PI_16 0.55557023301960222474f

template <int A> BLINK_HD cf32 mul_w32(cf32 x) {   // x * exp(+i pi A / 16), A = 0..15
  if constexpr ((A & 1) == 0) return mul_w16<A / 2>(x);
  else if constexpr (A == 1) return cmul(x, mk(BLINK_COS_PI_16, BLINK_SIN_PI_16));
  else if constexpr (A == 3) return cmul(x, mk(BLINK_COS_3PI_16, BLINK_SIN_3PI_16));
  else if constexpr (A == 5) return cmul(x, mk(BLINK_SIN_3PI_16, BLINK_COS_3PI_16));
  else if constexpr (A == 7) return cmul(x, mk(BLINK_SIN_PI_16, BLINK_COS_PI_16));
  else if constexpr (A == 9) return cmul(x, mk(-BLINK_SIN_PI_16, BLINK_COS_PI_16));
  else if constexpr (A == 11) return cmul(x, mk(-BLINK_SIN_3PI_16, BLINK_COS_3PI_16));
  else if constexpr (A == 13) return cmul(x, mk(-BLINK_COS_3PI_16, BLINK_SIN_3PI_16));
  else return cmul(x, mk(-BLINK_COS_PI_16, BLINK_SIN_PI_16));
}

template <int K> struct Combine32 {
  BLINK_HD static void run(cf32 *v, const cf32 *e, const cf32 *o) {
    if constexpr (K < 16) {
      const cf32 t = mul_w32<K>(o[K]);
      v[K] = cadd(e[K], t);
      v[K + 16] = csub(e[K], t);
      Combine32<K + 1>::run(v, e, o);
    }
  }
};

BLINK_HD void dft32(cf32 *v) {  // v[0..31]
  cf32 e[16], o[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
  dft16(e);
  dft16(o);
  Combine32<0>::run(v, e, o);
}

constexpr unsigned prune_even(unsigned m, int r) {   // mask of the even-indexed inputs, compacted
  unsigned o = 0;
  for (int k = 0; k < r / 2; ++k) o |= ((m >> (2 * k)) & 1u) << k;
  return o;
}
constexpr unsigned prune_odd(unsigned m, int r) { return prune_even(m >> 1, r); }

template <int R, unsigned M> BLINK_HD void dftp(cf32 *v);

template <int R, int K, bool HAS_E, bool HAS_O> struct PruneCombine {
  BLINK_HD static void run(cf32 *v, const cf32 *e, const cf32 *o) {
    if constexpr (K < R / 2) {
      if constexpr (HAS_E && HAS_O) {
        const cf32 t = mul_w16<K * (16 / R)>(o[K]);
        v[K] = cadd(e[K], t);
        v[K + R / 2] = csub(e[K], t);
      } else if constexpr (HAS_E) {
        v[K] = e[K];
        v[K + R / 2] = e[K];
      } else {
        const cf32 t = mul_w16<K * (16 / R)>(o[K]);
        v[K] = t;
        v[K + R / 2] = mk(-t.x, -t.y);
      }
      PruneCombine<R, K + 1, HAS_E, HAS_O>::run(v, e, o);
    }
  }
};

template <int R, unsigned M> BLINK_HD void dftp(cf32 *v) {
  static_assert(R == 1 || R == 2 || R == 4 || R == 8 || R == 16, "radix");
  constexpr unsigned FULL = (1u << R) - 1u;
  if constexpr (R == 1 || (M & FULL) == 0) {
    return;
  } else if constexpr ((M & FULL) == FULL) {
    dft<R>(v);
  } else {
    constexpr unsigned EM = prune_even(M & FULL, R), OM = prune_odd(M & FULL, R);
    cf32 e[R / 2], o[R / 2];
#pragma unroll
    for (int k = 0; k < R / 2; ++k) {
      e[k] = ((EM >> k) & 1u) ? v[2 * k] : mk(0.f, 0.f);
      o[k] = ((OM >> k) & 1u) ? v[2 * k + 1] : mk(0.f, 0.f);
    }
    dftp<R / 2, EM>(e);
    dftp<R / 2, OM>(o);
    PruneCombine<R, 0, EM != 0, OM != 0>::run(v, e, o);
  }
}

// mask of a first-stage butterfly whose inputs r = NZ .. 15 - NZ are zero (band-limited line)
template <int NZ> struct BandMask {
  static constexpr unsigned value = NZ >= 8 ? 0xFFFFu : (((1u << NZ) - 1u) | (((1u << NZ) - 1u) << (16 - NZ)));
};

// ---- per-N stage plan ------------------------------------------------------------------------
template <int N> struct Radices;
template <> struct Radices<32>   { static constexpr int n = 2, r0 = 16, r1 = 2,  r2 = 1; };
template <> struct Radices<64>   { static constexpr int n = 2, r0 = 16, r1 = 4,  r2 = 1; };
template <> struct Radices<128>  { static constexpr int n = 2, r0 = 16, r1 = 8,  r2 = 1; };
template <> struct Radices<256>  { static constexpr int n = 2, r0 = 16, r1 = 16, r2 = 1; };
template <> struct Radices<512>  { static constexpr int n = 3, r0 = 16, r1 = 8,  r2 = 4; };
template <> struct Radices<1024> { static constexpr int n = 3, r0 = 16, r1 = 8,  r2 = 8; };
template <> struct Radices<2048> { static constexpr int n = 3, r0 = 16, r1 = 16, r2 = 8; };
template <> struct Radices<4096> { static constexpr int n = 3, r0 = 16, r1 = 16, r2 = 16; };

// shared-memory line padding: one extra complex slot per 16 keeps the stride-16 scatter of the
// first stage and the unit-stride gathers of later stages both conflict-free for 8-byte accesses
BLINK_HD int pad16(int i) { return i + (i >> 4); }
template <int N> struct LineSize { static constexpr int value = N + N / 16; };

template <int N> struct Fft {
  static constexpr int E = 16;
  static constexpr int T = N / E;  // threads per transform
  using RD = Radices<N>;
  static constexpr int NSTAGE = RD::n;

  template <int S> static constexpr int radix() { return S == 0 ? RD::r0 : (S == 1 ? RD::r1 : RD::r2); }
  template <int S> static constexpr int ns() { return S == 0 ? 1 : (S == 1 ? RD::r0 : RD::r0 * RD::r1); }

  // Phase 1 of stage S: v[b*R + r] = in[j + r * N/R], j = t + b*T.  `ld(idx)` returns the point
  // at natural index idx of this stage's input.
  template <int S, class Load> BLINK_HD static void load(cf32 *v, int t, Load ld) {
    constexpr int R = radix<S>();
#pragma unroll
    for (int b = 0; b < E / R; ++b) {
      const int j = t + b * T;
#pragma unroll
      for (int r = 0; r < R; ++r) v[b * R + r] = ld(j + r * (N / R));
    }
  }

  // Phase 2 of stage S: twiddle by w_{Ns R}^{r k}, k = j mod Ns, then the radix-R butterfly.
  // tw[m] = exp(+2 pi i m / N), m = 0..N-1.  Powers of the base twiddle are formed by a
  // depth <= 4 product tree from one table lookup.
  template <int S> BLINK_HD static void compute(cf32 *v, int t, const cf32 *tw) {
    constexpr int R = radix<S>();
    constexpr int Ns = ns<S>();
#pragma unroll
    for (int b = 0; b < E / R; ++b) {
      cf32 *x = v + b * R;
      if (Ns > 1) {
        const int j = t + b * T;
        const int k = j & (Ns - 1);
        cf32 w[R > 1 ? R : 2];
        w[1] = tw[k * (N / (Ns * R))];
        if (R > 2) { w[2] = cmul(w[1], w[1]); w[3] = cmul(w[2], w[1]); }
        if (R > 4) {
          w[4] = cmul(w[2], w[2]);
          w[5] = cmul(w[4], w[1]); w[6] = cmul(w[4], w[2]); w[7] = cmul(w[4], w[3]);
        }
        if (R > 8) {
          w[8] = cmul(w[4], w[4]);
#pragma unroll
          for (int r = 9; r < 16; ++r) w[r] = cmul(w[8], w[r - 8]);
        }
#pragma unroll
        for (int r = 1; r < R; ++r) x[r] = cmul(x[r], w[r]);
      }
      dft<R>(x);
    }
  }

  // Stage 0 (no twiddles) with inputs r outside the mask M known to be zero; radix 16 only.
  template <unsigned M> BLINK_HD static void compute0_pruned(cf32 *v) {
    static_assert(RD::r0 == 16, "first stage is radix 16");
    dftp<16, M>(v);
  }

  // The twiddles of butterfly j of stage S, w[r] = w_{Ns R}^{r k}, k = j mod Ns, each read straight
  // from the table (no product tree): for callers that keep them in registers across transforms.
  template <int S> BLINK_HD static void twiddles(cf32 *w, int j, const cf32 *tw) {
    constexpr int R = radix<S>();
    constexpr int Ns = ns<S>();
    const int k = j & (Ns - 1);
    w[0] = mk(1.f, 0.f);
#pragma unroll
    for (int r = 1; r < R; ++r) w[r] = tw[(r * k * (N / (Ns * R))) & (N - 1)];
  }

  // Phase 2 with caller-held twiddles: w[b][r] from twiddles<S>(w[b], t + b*T, tw).
  template <int S, int WR> BLINK_HD static void compute_tw(cf32 *v, const cf32 (*w)[WR]) {
    constexpr int R = radix<S>();
#pragma unroll
    for (int b = 0; b < E / R; ++b) {
      cf32 *x = v + b * R;
#pragma unroll
      for (int r = 1; r < R; ++r) x[r] = cmul(x[r], w[b][r]);
      dft<R>(x);
    }
  }

  // Phases 1 and 3 against a pad16 line in shared memory, with the padding strength-reduced: the R
  // accesses of a butterfly are a fixed stride apart in the PADDED line as well (strides that are
  // multiples of 16 gain stride/16 pad slots; the unit stride of stage 0's store stays inside one block
  // of 16), so a butterfly costs one address and R immediate offsets instead of R shift-add pairs.
  template <int S> BLINK_HD static void load_line(cf32 *v, int t, const cf32 *line) {
    constexpr int R = radix<S>();
    static_assert((N / R) % 16 == 0, "input stride must be a multiple of the padding period");
#pragma unroll
    for (int b = 0; b < E / R; ++b) {
      const cf32 *pb = line + pad16(t + b * T);
#pragma unroll
      for (int r = 0; r < R; ++r) v[b * R + r] = pb[r * (N / R + N / R / 16)];
    }
  }
  template <int S> BLINK_HD static void store_line(const cf32 *v, int t, cf32 *line) {
    constexpr int R = radix<S>();
    constexpr int Ns = ns<S>();
    static_assert(Ns == 1 || Ns % 16 == 0, "output stride must be 1 or a multiple of the padding period");
#pragma unroll
    for (int b = 0; b < E / R; ++b) {
      const int j = t + b * T;
      const int k = j & (Ns - 1);
      cf32 *pb = line + pad16((j - k) * R + k);
#pragma unroll
      for (int r = 0; r < R; ++r) pb[r * (Ns + Ns / 16)] = v[b * R + r];
    }
  }

  // Phase 3 of stage S: out[(j/Ns) Ns R + k + r Ns] = v[b*R + r].  `st(idx, val)`.
  template <int S, class Store> BLINK_HD static void store(const cf32 *v, int t, Store st) {
    constexpr int R = radix<S>();
    constexpr int Ns = ns<S>();
#pragma unroll
    for (int b = 0; b < E / R; ++b) {
      const int j = t + b * T;
      const int k = j & (Ns - 1);
      const int j0 = (j - k) * R + k;
#pragma unroll
      for (int r = 0; r < R; ++r) st(j0 + r * Ns, v[b * R + r]);
    }
  }
};

}  // namespace blinkfft
