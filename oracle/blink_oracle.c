/*
 * blink_oracle.c -- CPU ORACLE for the BLINK imager hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain, slow, obviously-correct restatement of what the hot path computes,
 * written from /root/reference/PAPER.md (arxiv 2405.13478, Sokolowski et al., "High-Time Resolution
 * GPU Imager for FRB searches at low radio frequencies").  It shares NO code, header, table or
 * constant generator with the CUDA path under paper_2405_13478_b200/csrc/, and nothing in the
 * product may import, link or call it: only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may.
 *
 * Everything is fp64.  Visibilities arrive as the same complex64 arrays the GPU gets and are
 * promoted to double on load.  Steps follow SURVEY.md section 8(c) / DESIGN.md "Readings":
 *
 *   1. baseline -> cell        PAPER.md:350 (sec 5.2.1 "difference between the antenna positions
 *                              expressed in wavelengths"), Eq. 9 PAPER.md:202 (du = 1/(N_px dx)),
 *                              listing PAPER.md:477-478 (frequency / wavelength in double)
 *   2. in-grid test            reading c7 (paper silent)
 *   3. FFT-native cell index   PAPER.md:352 (indices chosen so no data move is needed before FFT)
 *   4. accumulate V and V*     PAPER.md:353-354, cell rule PAPER.md:211; Hermitian: reading c2
 *   5. weighting               PAPER.md:211-213, :360 (natural / uniform from the counter)
 *   6. inverse 2-D DFT, shift, normalise, real part
 *                              Eq. 4-5 PAPER.md:162-167 (sign), PAPER.md:374-376 (real part, shift)
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): lattice index map by brute force,
 * count invariants and the paper's baseline counts (Tables 1 and 3), exact Hermitian grid,
 * O(N^4) literal sum vs separable, numpy.fft.ifft2 special case, Parseval, unit source at phase
 * centre = 1, offset source at predicted pixel, direct Fourier sum on lattice arrays.
 * Parity vs the paper's own implementation: UNPINNED (its code and template images are absent).
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC blink_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C_M_PER_S 299792458.0 /* speed of light, exact SI value */
#define ORACLE_PI 3.14159265358979323846264338327950288

/* number of cross-correlation baselines, N_b = N_ant (N_ant - 1) / 2  (Table 3) */
int64_t oracle_n_baselines(int n_ant) { return (int64_t)n_ant * (n_ant - 1) / 2; }

/* baseline ordering of the boundary: bl(i,j) = i(2 n_ant - i - 1)/2 + (j - i - 1), 0 <= i < j */
int64_t oracle_baseline_index(int n_ant, int i, int j) {
  return (int64_t)i * (2 * (int64_t)n_ant - i - 1) / 2 + (j - i - 1);
}

/*
 * Steps 1-3 for one channel.  ant_enu_m: [n_ant][3] East, North, Up metres (Up ignored: coplanar /
 * zenith).  Outputs per baseline (length n_bl, any may be NULL):
 *   kx, ky      centred integer cell coordinates (always written, also for dropped baselines)
 *   cell        iy*N + ix of V, FFT-native order (DC at [0][0]); -1 if the baseline is dropped
 *   cell_conj   cell of V* at (-kx,-ky); -1 if dropped
 * Returns the number of dropped baselines, or -1 on bad arguments.
 */
int64_t oracle_uv_cells(const double *ant_enu_m, int n_ant, double freq_hz, int n_pix,
                        double pixscale, int64_t *kx_out, int64_t *ky_out, int32_t *cell,
                        int32_t *cell_conj) {
  if (!ant_enu_m || n_ant < 2 || n_pix < 2 || (n_pix & 1) || !(pixscale > 0.0) || !(freq_hz > 0.0))
    return -1;
  const int64_t N = n_pix;
  const double G = (double)n_pix * pixscale; /* 1/du, Eq. 9 */
  const double sc = freq_hz / ORACLE_C_M_PER_S; /* 1/lambda: one fp64 divide (reading c6) */
  const int64_t kmax = N / 2 - 1;
  int64_t n_dropped = 0, bl = 0;
  for (int i = 0; i < n_ant; ++i) {
    for (int j = i + 1; j < n_ant; ++j, ++bl) {
      /* b_ij = r_j - r_i (reading c10); subtract, then multiply; no FMA (-ffp-contract=off) */
      double de = ant_enu_m[3 * j + 0] - ant_enu_m[3 * i + 0];
      double dn = ant_enu_m[3 * j + 1] - ant_enu_m[3 * i + 1];
      double u = de * sc;
      double v = dn * sc;
      double ug = u * G;
      double vg = v * G;
      int64_t kx = llround(ug); /* nearest, ties away from zero (reading c5) */
      int64_t ky = llround(vg);
      if (kx_out) kx_out[bl] = kx;
      if (ky_out) ky_out[bl] = ky;
      int keep = (kx >= -kmax && kx <= kmax && ky >= -kmax && ky <= kmax);
      if (!keep) {
        ++n_dropped;
        if (cell) cell[bl] = -1;
        if (cell_conj) cell_conj[bl] = -1;
        continue;
      }
      int64_t ix = ((kx % N) + N) % N;
      int64_t iy = ((ky % N) + N) % N;
      int64_t cx = (N - ix) % N;
      int64_t cy = (N - iy) % N;
      if (cell) cell[bl] = (int32_t)(iy * N + ix);
      if (cell_conj) cell_conj[bl] = (int32_t)(cy * N + cx);
    }
  }
  return n_dropped;
}

/*
 * Step 4 for one snapshot.  vis: complex64 [n_bl] as interleaved float re,im.  grid: fp64
 * interleaved re,im [N*N] (zeroed here), count: uint32 [N*N] (zeroed here; may be NULL).
 * Baseline order bl = 0..n_bl-1; V into cell, then conj(V) into cell_conj.
 */
void oracle_grid(const int32_t *cell, const int32_t *cell_conj, int64_t n_bl, const float *vis,
                 int n_pix, double *grid, uint32_t *count) {
  const int64_t NN = (int64_t)n_pix * n_pix;
  memset(grid, 0, sizeof(double) * 2 * (size_t)NN);
  if (count) memset(count, 0, sizeof(uint32_t) * (size_t)NN);
  for (int64_t bl = 0; bl < n_bl; ++bl) {
    if (cell[bl] < 0) continue;
    double re = (double)vis[2 * bl], im = (double)vis[2 * bl + 1];
    int64_t c = cell[bl], cc = cell_conj[bl];
    grid[2 * c] += re;
    grid[2 * c + 1] += im;
    if (count) count[c] += 1u;
    grid[2 * cc] += re;
    grid[2 * cc + 1] += -im;
    if (count) count[cc] += 1u;
  }
}

/* Count grid only (step 4 without values); geometry is fixed so it holds for every t. */
void oracle_counts(const int32_t *cell, const int32_t *cell_conj, int64_t n_bl, int n_pix,
                   uint32_t *count) {
  const int64_t NN = (int64_t)n_pix * n_pix;
  memset(count, 0, sizeof(uint32_t) * (size_t)NN);
  for (int64_t bl = 0; bl < n_bl; ++bl) {
    if (cell[bl] < 0) continue;
    count[cell[bl]] += 1u;
    count[cell_conj[bl]] += 1u;
  }
}

/*
 * Step 5, in place.  weighting 0 = natural (grid unchanged, norm = sum of counts),
 * 1 = uniform (grid[c] /= count[c] where count>0, norm = number of occupied cells).
 * Returns norm (0 if the grid is empty).
 */
double oracle_weight(double *grid, const uint32_t *count, int n_pix, int weighting) {
  const int64_t NN = (int64_t)n_pix * n_pix;
  double norm = 0.0;
  if (weighting == 0) {
    for (int64_t c = 0; c < NN; ++c) norm += (double)count[c];
  } else {
    for (int64_t c = 0; c < NN; ++c) {
      if (count[c] > 0) {
        grid[2 * c] /= (double)count[c];
        grid[2 * c + 1] /= (double)count[c];
        norm += 1.0;
      }
    }
  }
  return norm;
}

/* exact-index twiddle table w[k] = exp(+2 pi i k / N), k = 0..N-1 (sign: reading c3) */
static double *make_twiddles(int n_pix) {
  double *w = (double *)malloc(sizeof(double) * 2 * (size_t)n_pix);
  if (!w) return NULL;
  for (int k = 0; k < n_pix; ++k) {
    double a = 2.0 * ORACLE_PI * (double)k / (double)n_pix;
    w[2 * k] = cos(a);
    w[2 * k + 1] = sin(a);
  }
  return w;
}

/*
 * Step 6, literal definition: for every pixel the full double sum over all N*N cells.  O(N^4);
 * used only for N <= 64 to pin the separable version.
 *   I[y][x] = (1/norm) Re sum_{iy,ix} G'[iy][ix] exp(+2 pi i (ix (x - N/2) + iy (y - N/2)) / N)
 * img: fp64 [N*N].  Returns max |Im| / norm over the image (Hermitian residual) via imag_max.
 */
int oracle_dft2_literal(const double *grid, int n_pix, double norm, double *img, double *imag_max) {
  const int64_t N = n_pix;
  double *w = make_twiddles(n_pix);
  if (!w) return -1;
  double imax = 0.0;
  for (int64_t y = 0; y < N; ++y) {
    int64_t ys = (y + N / 2) % N; /* (y - N/2) mod N */
    for (int64_t x = 0; x < N; ++x) {
      int64_t xs = (x + N / 2) % N;
      double sr = 0.0, si = 0.0;
      for (int64_t iy = 0; iy < N; ++iy) {
        for (int64_t ix = 0; ix < N; ++ix) {
          int64_t k = (ix * xs + iy * ys) % N;
          double gr = grid[2 * (iy * N + ix)], gi = grid[2 * (iy * N + ix) + 1];
          sr += gr * w[2 * k] - gi * w[2 * k + 1];
          si += gr * w[2 * k + 1] + gi * w[2 * k];
        }
      }
      img[y * N + x] = sr / norm;
      if (fabs(si / norm) > imax) imax = fabs(si / norm);
    }
  }
  if (imag_max) *imag_max = imax;
  free(w);
  return 0;
}

/*
 * Step 6, separable naive DFT: row pass (over ix) then column pass (over iy).  Rows of the grid
 * that are entirely zero are skipped in both passes (they add exact zeros).  O(N^3) worst case.
 */
int oracle_dft2_separable(const double *grid, int n_pix, double norm, double *img,
                          double *imag_max) {
  const int64_t N = n_pix;
  double *w = make_twiddles(n_pix);
  double *T = (double *)calloc((size_t)(2 * N * N), sizeof(double));
  char *rowhas = (char *)calloc((size_t)N, 1);
  if (!w || !T || !rowhas) { free(w); free(T); free(rowhas); return -1; }
  /* row pass: T[iy][x] = sum_ix G'[iy][ix] w^(ix * (x - N/2)) */
  for (int64_t iy = 0; iy < N; ++iy) {
    int any = 0;
    for (int64_t ix = 0; ix < N; ++ix)
      if (grid[2 * (iy * N + ix)] != 0.0 || grid[2 * (iy * N + ix) + 1] != 0.0) { any = 1; break; }
    rowhas[iy] = (char)any;
    if (!any) continue;
    for (int64_t x = 0; x < N; ++x) {
      int64_t xs = (x + N / 2) % N;
      double sr = 0.0, si = 0.0;
      for (int64_t ix = 0; ix < N; ++ix) {
        double gr = grid[2 * (iy * N + ix)], gi = grid[2 * (iy * N + ix) + 1];
        if (gr == 0.0 && gi == 0.0) continue;
        int64_t k = (ix * xs) % N;
        sr += gr * w[2 * k] - gi * w[2 * k + 1];
        si += gr * w[2 * k + 1] + gi * w[2 * k];
      }
      T[2 * (iy * N + x)] = sr;
      T[2 * (iy * N + x) + 1] = si;
    }
  }
  /* column pass: F[y][x] = sum_iy T[iy][x] w^(iy * (y - N/2)) */
  double imax = 0.0;
  for (int64_t y = 0; y < N; ++y) {
    int64_t ys = (y + N / 2) % N;
    for (int64_t x = 0; x < N; ++x) {
      double sr = 0.0, si = 0.0;
      for (int64_t iy = 0; iy < N; ++iy) {
        if (!rowhas[iy]) continue;
        int64_t k = (iy * ys) % N;
        double tr = T[2 * (iy * N + x)], ti = T[2 * (iy * N + x) + 1];
        sr += tr * w[2 * k] - ti * w[2 * k + 1];
        si += tr * w[2 * k + 1] + ti * w[2 * k];
      }
      img[y * N + x] = sr / norm;
      if (fabs(si / norm) > imax) imax = fabs(si / norm);
    }
  }
  if (imag_max) *imag_max = imax;
  free(w); free(T); free(rowhas);
  return 0;
}

/*
 * Step 6 for a list of pixels only (sampled parity at sizes where the whole image is too slow):
 * yx: int32 [n][2] = (y, x); out_re / out_im: fp64 [n].  Literal sum over the non-zero cells.
 */
int oracle_dft2_pixels(const double *grid, int n_pix, double norm, const int32_t *yx, int64_t n,
                       double *out_re, double *out_im) {
  const int64_t N = n_pix;
  double *w = make_twiddles(n_pix);
  if (!w) return -1;
  /* compact list of non-zero cells */
  int64_t nnz = 0;
  for (int64_t c = 0; c < N * N; ++c)
    if (grid[2 * c] != 0.0 || grid[2 * c + 1] != 0.0) ++nnz;
  int64_t *idx = (int64_t *)malloc(sizeof(int64_t) * (size_t)(nnz > 0 ? nnz : 1));
  if (!idx) { free(w); return -1; }
  nnz = 0;
  for (int64_t c = 0; c < N * N; ++c)
    if (grid[2 * c] != 0.0 || grid[2 * c + 1] != 0.0) idx[nnz++] = c;
  for (int64_t p = 0; p < n; ++p) {
    int64_t ys = (yx[2 * p] + N / 2) % N, xs = (yx[2 * p + 1] + N / 2) % N;
    double sr = 0.0, si = 0.0;
    for (int64_t q = 0; q < nnz; ++q) {
      int64_t c = idx[q], iy = c / N, ix = c % N;
      int64_t k = (ix * xs + iy * ys) % N;
      double gr = grid[2 * c], gi = grid[2 * c + 1];
      sr += gr * w[2 * k] - gi * w[2 * k + 1];
      si += gr * w[2 * k + 1] + gi * w[2 * k];
    }
    out_re[p] = sr / norm;
    if (out_im) out_im[p] = si / norm;
  }
  free(w); free(idx);
  return 0;
}

/*
 * Whole chain, batched over snapshots s = t*n_ch + ch (steps 1-6), for parity sampling and the
 * timed CPU baseline.  sel: int64 [n_sel] flat snapshot indices into vis [n_t][n_ch][n_bl]
 * (complex64 as float pairs).  grids_out: fp64 [n_sel][N*N][2] UNWEIGHTED grids or NULL;
 * imgs_out: fp64 [n_sel][N*N] or NULL.  n_threads <= 0: OpenMP default.  Returns threads used,
 * or -1 on error.
 */
int oracle_image_batch(const double *ant_enu_m, int n_ant, const double *freq_hz, int n_ch,
                       int n_pix, double pixscale, int weighting, const float *vis,
                       const int64_t *sel, int64_t n_sel, double *grids_out, double *imgs_out,
                       int n_threads) {
  const int64_t n_bl = oracle_n_baselines(n_ant);
  const int64_t NN = (int64_t)n_pix * n_pix;
  int used = 1, err = 0;
#ifdef _OPENMP
  if (n_threads > 0) omp_set_num_threads(n_threads);
  used = omp_get_max_threads();
  if (used > n_sel) used = (int)(n_sel > 0 ? n_sel : 1);
#endif
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t q = 0; q < n_sel; ++q) {
    int64_t s = sel[q];
    int ch = (int)(s % n_ch);
    int32_t *cell = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_bl);
    int32_t *cellc = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_bl);
    double *grid = (double *)malloc(sizeof(double) * 2 * (size_t)NN);
    uint32_t *count = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)NN);
    double *img = (double *)malloc(sizeof(double) * (size_t)NN);
    if (!cell || !cellc || !grid || !count || !img) {
      err = 1;
    } else if (oracle_uv_cells(ant_enu_m, n_ant, freq_hz[ch], n_pix, pixscale, NULL, NULL, cell,
                               cellc) < 0) {
      err = 1;
    } else {
      oracle_grid(cell, cellc, n_bl, vis + 2 * s * n_bl, n_pix, grid, count);
      if (grids_out) memcpy(grids_out + 2 * q * NN, grid, sizeof(double) * 2 * (size_t)NN);
      if (imgs_out) {
        double norm = oracle_weight(grid, count, n_pix, weighting);
        if (norm > 0.0) {
          if (oracle_dft2_separable(grid, n_pix, norm, img, NULL) != 0) err = 1;
        } else {
          memset(img, 0, sizeof(double) * (size_t)NN);
        }
        memcpy(imgs_out + q * NN, img, sizeof(double) * (size_t)NN);
      }
    }
    free(cell); free(cellc); free(grid); free(count); free(img);
  }
  return err ? -1 : used;
}
