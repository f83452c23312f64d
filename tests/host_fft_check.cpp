// Host-side check of the Stockham stage algebra in paper_2405_13478_b200/csrc/fft_core.cuh:
// emulates the T threads of one transform phase by phase (load all / compute / store all, with a
// padded line standing in for shared memory) and compares with a naive fp64 inverse DFT.
// Built and run by tests/test_host_logic.py (CPU only).  Prints "OK" or "FAIL ...".
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "../paper_2405_13478_b200/csrc/fft_core.cuh"
#include "../paper_2405_13478_b200/csrc/wfft.cuh"

using namespace blinkfft;

template <int N, int S> struct RunStages {
  static void run(std::vector<cf32> &line, const std::vector<cf32> &tw) {
    using F = Fft<N>;
    std::vector<cf32> regs(F::T * 16);
    for (int t = 0; t < F::T; ++t)
      F::template load<S>(&regs[t * 16], t, [&](int idx) { return line[pad16(idx)]; });
    for (int t = 0; t < F::T; ++t) F::template compute<S>(&regs[t * 16], t, tw.data());
    for (int t = 0; t < F::T; ++t)
      F::template store<S>(&regs[t * 16], t, [&](int idx, cf32 v) { line[pad16(idx)] = v; });
    if (S + 1 < F::NSTAGE) RunStages<N, (S + 1 < F::NSTAGE ? S + 1 : S)>::run_next(line, tw);
  }
  static void run_next(std::vector<cf32> &line, const std::vector<cf32> &tw) { run(line, tw); }
};

template <int N> int check() {
  std::vector<cf32> tw(N), line(LineSize<N>::value);
  for (int k = 0; k < N; ++k) {
    double a = 2.0 * M_PI * k / N;
    tw[k] = mk((float)cos(a), (float)sin(a));
  }
  std::vector<double> xr(N), xi(N);
  srand(1234 + N);
  for (int k = 0; k < N; ++k) {
    xr[k] = rand() / (double)RAND_MAX - 0.5;
    xi[k] = rand() / (double)RAND_MAX - 0.5;
    line[pad16(k)] = mk((float)xr[k], (float)xi[k]);
  }
  RunStages<N, 0>::run(line, tw);
  double maxerr = 0, maxref = 0;
  for (int n = 0; n < N; ++n) {
    double sr = 0, si = 0;
    for (int k = 0; k < N; ++k) {
      double a = 2.0 * M_PI * ((long long)k * n % N) / N;
      sr += (double)(float)xr[k] * cos(a) - (double)(float)xi[k] * sin(a);
      si += (double)(float)xr[k] * sin(a) + (double)(float)xi[k] * cos(a);
    }
    cf32 g = line[pad16(n)];
    maxerr = fmax(maxerr, fmax(fabs(g.x - sr), fabs(g.y - si)));
    maxref = fmax(maxref, fmax(fabs(sr), fabs(si)));
  }
  double rel = maxerr / maxref;
  printf("N=%d rel_err=%.3e\n", N, rel);
  return rel < 2e-6 ? 0 : 1;
}

// pruned butterfly against the full one on inputs that are zero outside the mask
template <unsigned M> int check_pruned() {
  cf32 a[16], b[16];
  for (int k = 0; k < 16; ++k) {
    const bool nz = (M >> k) & 1u;
    a[k] = nz ? mk(0.3f * k - 1.1f, 0.7f - 0.05f * k * k) : mk(0.f, 0.f);
    b[k] = nz ? a[k] : mk(1e30f, -1e30f);      // must never be read
  }
  dft<16>(a);
  dftp<16, M>(b);
  double err = 0;
  for (int k = 0; k < 16; ++k) err = fmax(err, fmax(fabs(a[k].x - b[k].x), fabs(a[k].y - b[k].y)));
  printf("pruned mask=%04x err=%.3e\n", M, err);
  return err < 1e-5 ? 0 : 1;
}

// warp-per-transform 1024-point split (wfft.cuh): 32 lanes emulated one after another, with the
// exchange tile standing in for shared memory; `nz_rows` < 32 also exercises wf_get_masked
static int check_warp1024(unsigned mask) {
  const int N = kWfN;
  std::vector<cf32> tab(32 * 32), tile(kWfTile, mk(1e30f, 1e30f));
  for (int n1 = 0; n1 < 32; ++n1)
    for (int b = 0; b < 32; ++b) {
      double a = 2.0 * M_PI * (b * n1) / N;
      tab[n1 * 32 + b] = mk((float)cos(a), (float)sin(a));
    }
  std::vector<double> xr(N, 0.0), xi(N, 0.0);
  srand(77);
  for (int k = 0; k < N; ++k)
    if ((mask >> (k & 31)) & 1u) { xr[k] = rand() / (double)RAND_MAX - 0.5; xi[k] = rand() / (double)RAND_MAX - 0.5; }
  for (int b = 0; b < 32; ++b) {
    if (!((mask >> b) & 1u)) continue;          // rows of absent residues are never written
    cf32 z[32];
    for (int a = 0; a < 32; ++a) z[a] = mk((float)xr[32 * a + b], (float)xi[32 * a + b]);
    wf_inner(z, b, [&](int i) { return tab[i]; });
    wf_put(tile.data(), b, z);
  }
  double maxerr = 0, maxref = 0;
  for (int n1 = 0; n1 < 32; ++n1) {
    cf32 t[32];
    if (mask == 0xFFFFFFFFu) wf_get(tile.data(), n1, t); else wf_get_masked(tile.data(), n1, mask, t);
    dft32(t);
    for (int n2 = 0; n2 < 32; ++n2) {
      const int n = n1 + 32 * n2;
      double sr = 0, si = 0;
      for (int k = 0; k < N; ++k) {
        double a = 2.0 * M_PI * ((long long)k * n % N) / N;
        sr += (double)(float)xr[k] * cos(a) - (double)(float)xi[k] * sin(a);
        si += (double)(float)xr[k] * sin(a) + (double)(float)xi[k] * cos(a);
      }
      maxerr = fmax(maxerr, fmax(fabs(t[n2].x - sr), fabs(t[n2].y - si)));
      maxref = fmax(maxref, fmax(fabs(sr), fabs(si)));
    }
  }
  printf("warp1024 mask=%08x rel_err=%.3e\n", mask, maxerr / maxref);
  return maxerr / maxref < 2e-6 ? 0 : 1;
}

int main() {
  int bad = 0;
  bad += check_warp1024(0xFFFFFFFFu);
  bad += check_warp1024(0x80010005u);
  bad += check_pruned<BandMask<1>::value>();
  bad += check_pruned<BandMask<2>::value>();
  bad += check_pruned<BandMask<3>::value>();
  bad += check_pruned<BandMask<4>::value>();
  bad += check_pruned<BandMask<5>::value>();
  bad += check_pruned<BandMask<7>::value>();
  bad += check_pruned<BandMask<8>::value>();
  bad += check_pruned<0x0001u>();
  bad += check_pruned<0x8421u>();
  bad += check<32>();
  bad += check<64>();
  bad += check<128>();
  bad += check<256>();
  bad += check<512>();
  bad += check<1024>();
  bad += check<2048>();
  bad += check<4096>();
  // small butterflies against the definition
  for (int R : {2, 4, 8, 16, 32}) {
    cf32 v[32];
    double xr[32], xi[32];
    for (int k = 0; k < R; ++k) { xr[k] = k * 0.37 - 1.0; xi[k] = 0.5 - k * k * 0.011; v[k] = mk((float)xr[k], (float)xi[k]); }
    if (R == 2) dft<2>(v); else if (R == 4) dft<4>(v); else if (R == 8) dft<8>(v); else if (R == 16) dft<16>(v); else dft<32>(v);
    for (int n = 0; n < R; ++n) {
      double sr = 0, si = 0;
      for (int k = 0; k < R; ++k) {
        double a = 2.0 * M_PI * k * n / R;
        sr += (float)xr[k] * cos(a) - (float)xi[k] * sin(a);
        si += (float)xr[k] * sin(a) + (float)xi[k] * cos(a);
      }
      if (fabs(v[n].x - sr) > 4e-5 || fabs(v[n].y - si) > 4e-5) { printf("FAIL dft%d n=%d\n", R, n); ++bad; }
    }
  }
  puts(bad ? "FAIL" : "OK");
  return bad;
}
