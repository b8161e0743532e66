/*
 * oracle/nfs_oracle.c — CPU ORACLE. TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision statement of what the hot path of arxiv 1209.3362
 * ("Quasi-real-time analysis of dynamic near field scattering data using a GPU")
 * computes.  Only tests/, __graft_entry__.smoke() and the cpu_baseline / --impl reference
 * legs of bench.py may call it.  It shares no code, header, table or constant with the
 * CUDA path under paper_1209_3362_b200/csrc and neither includes the other.
 *
 * The method reaches exactly (up to rounding order) a result with a plain definition, so the
 * oracle IS that definition written out:
 *
 *   1. m_t = (1/WH) sum_x I_t(x);  i_t = I_t / m_t
 *        PAPER.md:L21 "images are normalized by their spatial average values"
 *   2. F_t(k) = (1/sqrt(WH)) sum_x i_t(x) exp(-2 pi i (kx x/W + ky y/H)), full plane
 *        PAPER.md:L25 "spatial Fourier transform"; L31 FFT of single images (linearity)
 *   3. D2d(k,tau) = 1/(N-tau) sum_{t=0}^{N-1-tau} |F_t(k) - F_{t+tau}(k)|^2
 *        PAPER.md:L21 (difference), L25 (power spectrum, average over measurement time),
 *        L31 (N(N-1)/2 pairs for N-1 lags => N-tau pairs at lag tau)
 *   4. I2d(k) = (1/N) sum_t |F_t(k)|^2            (reading R9)
 *   5. bin b(k) = isqrt( floor( 4 nb^2 (kx'^2 H^2 + ky'^2 W^2) / (W^2 H^2) ) ), kx',ky' signed
 *        FFT-order indices; DC and b >= nb excluded   ("azimuthally averaged";
 *        DESIGN.md readings R6, R7)
 *   6. D(b,tau) = mean of D2d over the bin, I(b) likewise, c_b = pixel count; empty => 0
 *
 * No blocking or fusion beyond a pixel-tiled loop order and OpenMP over pixel tiles in the
 * pair loop (it is still the explicit pair loop of step 3).  No -ffast-math.
 *
 *   7. V2d(k) = (1/N) sum_t |F_t(k) - <F(k)>_t|^2 and its azimuthal mean: see
 *        nfso_variance_spectrum below.
 *
 * nfso_structure_function_half is the same definition evaluated on the half plane kx <= W/2 only (the other
 * half is its Hermitian mirror, the image being real; SURVEY.md 8(c) "half-plane fast variant", pin P11: equal
 * to the full-plane function to 1e-12 on configs 0 and 1).  It exists so that the full-size parity tests of
 * BASELINE.json configs 1-4 finish in minutes; the timed cpu_baseline stays the full-plane function.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): brute-force DFT, numpy.fft, Parseval,
 * constant stack, gain invariance, travelling plane wave closed form, telegraph stack, ramp,
 * linearity (real-space difference then DFT), white noise D = 2 sigma^2 = 2 I, bin-count brute
 * force, all-pairs identity, golden vector tests/golden/p13_golden.txt.  Nothing here is
 * "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define NFSO_OK 0
#define NFSO_ERR_ARG -1
#define NFSO_ERR_MEM -2
#define NFSO_ERR_ZERO_MEAN -3

int nfso_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ---- step 1 ------------------------------------------------------------------------------ */

/* exact integer sum of the uint16 pixels (reading R3) */
uint64_t nfso_frame_sum(const uint16_t* frame, int W, int H) {
  uint64_t S = 0;
  for (long p = 0; p < (long)W * H; ++p) S += frame[p];
  return S;
}

/* i_t = I_t / m_t, m_t = S_t/(WH).  Returns NFSO_ERR_ZERO_MEAN if the frame sums to zero. */
int nfso_normalise(const uint16_t* frame, int W, int H, double* out) {
  uint64_t S = nfso_frame_sum(frame, W, H);
  if (S == 0) return NFSO_ERR_ZERO_MEAN;
  double m = (double)S / ((double)W * (double)H);
  for (long p = 0; p < (long)W * H; ++p) out[p] = (double)frame[p] / m;
  return NFSO_OK;
}

/* ---- step 2 ------------------------------------------------------------------------------ */

/* Brute-force unitary 2-D DFT straight from the definition, O((WH)^2); any W,H. */
void nfso_dft2_direct(const double* img, int W, int H, cplx* F) {
  const double two_pi = 2.0 * M_PI;
  const double scale = 1.0 / sqrt((double)W * (double)H);
  for (int ky = 0; ky < H; ++ky)
    for (int kx = 0; kx < W; ++kx) {
      cplx s = 0.0;
      for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
          /* reduce the phase index exactly before it becomes a float */
          double ph = -two_pi * ((double)(((long)kx * x) % W) / W + (double)(((long)ky * y) % H) / H);
          s += img[(long)y * W + x] * (cos(ph) + I * sin(ph));
        }
      F[(long)ky * W + kx] = s * scale;
    }
}

static int is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

/* Textbook in-place iterative radix-2 decimation-in-time FFT (bit reversal, then log2 n
 * butterfly stages); twiddles are evaluated directly per index, no recurrences. Unnormalised. */
static void fft1d_radix2(cplx* a, int n, int stride, const cplx* tw /* tw[k]=exp(-2 pi i k/n), k<n/2 */) {
  for (int i = 1, j = 0; i < n; ++i) {
    int bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) {
      cplx tmp = a[(long)i * stride];
      a[(long)i * stride] = a[(long)j * stride];
      a[(long)j * stride] = tmp;
    }
  }
  for (int len = 2; len <= n; len <<= 1) {
    int half = len >> 1, step = n / len;
    for (int i = 0; i < n; i += len)
      for (int k = 0; k < half; ++k) {
        cplx u = a[(long)(i + k) * stride];
        cplx v = a[(long)(i + k + half) * stride] * tw[(long)k * step];
        a[(long)(i + k) * stride] = u + v;
        a[(long)(i + k + half) * stride] = u - v;
      }
  }
}

static cplx* make_twiddles(int n) {
  cplx* tw = (cplx*)malloc(sizeof(cplx) * (size_t)(n / 2 + 1));
  if (!tw) return NULL;
  for (int k = 0; k < n / 2; ++k) {
    double ph = -2.0 * M_PI * (double)k / (double)n;
    tw[k] = cos(ph) + I * sin(ph);
  }
  return tw;
}

/* Unitary 2-D FFT of a real image on the FULL plane (rows, then columns); W,H powers of two. */
int nfso_fft2(const double* img, int W, int H, cplx* F) {
  if (!is_pow2(W) || !is_pow2(H)) return NFSO_ERR_ARG;
  cplx* twW = make_twiddles(W);
  cplx* twH = make_twiddles(H);
  if (!twW || !twH) { free(twW); free(twH); return NFSO_ERR_MEM; }
  for (long p = 0; p < (long)W * H; ++p) F[p] = img[p];
  for (int y = 0; y < H; ++y) fft1d_radix2(F + (long)y * W, W, 1, twW);
  for (int x = 0; x < W; ++x) fft1d_radix2(F + x, H, W, twH);
  const double scale = 1.0 / sqrt((double)W * (double)H);
  for (long p = 0; p < (long)W * H; ++p) F[p] *= scale;
  free(twW);
  free(twH);
  return NFSO_OK;
}

/* normalise + transform one frame; method 0 = radix-2 FFT, 1 = brute-force DFT */
static int transform_frame(const uint16_t* frame, int W, int H, int method, double* tmp, cplx* F) {
  int rc = nfso_normalise(frame, W, H, tmp);
  if (rc) return rc;
  if (method == 1) { nfso_dft2_direct(tmp, W, H, F); return NFSO_OK; }
  return nfso_fft2(tmp, W, H, F);
}

/* exported for the pins: unitary transform of one normalised uint16 frame, interleaved re,im */
int nfso_transform_u16(const uint16_t* frame, int W, int H, int method, double* F_out) {
  double* tmp = (double*)malloc(sizeof(double) * (size_t)W * H);
  if (!tmp) return NFSO_ERR_MEM;
  int rc = transform_frame(frame, W, H, method, tmp, (cplx*)F_out);
  free(tmp);
  return rc;
}

/* exported for the pins: unitary transform of a real fp64 image (no normalisation) */
int nfso_transform_f64(const double* img, int W, int H, int method, double* F_out) {
  if (method == 1) { nfso_dft2_direct(img, W, H, (cplx*)F_out); return NFSO_OK; }
  return nfso_fft2(img, W, H, (cplx*)F_out);
}

/* ---- step 5: exact-integer |q| bin -------------------------------------------------------- */

static uint64_t isqrt_u64(uint64_t v) {
  uint64_t r = (uint64_t)sqrt((double)v);
  while (r * r > v) --r;
  while ((r + 1) * (r + 1) <= v) ++r;
  return r;
}

/* bin of full-plane FFT-order pixel (kx,ky); -1 if excluded (DC, or |q| >= q_Nyquist) */
int nfso_qbin(int kx, int ky, int W, int H, int n_b) {
  long sx = kx < W / 2 ? kx : kx - W; /* Nyquist index W/2 -> -W/2 */
  long sy = ky < H / 2 ? ky : ky - H;
  if (sx == 0 && sy == 0) return -1;
  unsigned __int128 num = (unsigned __int128)(4ull * (uint64_t)n_b * (uint64_t)n_b) *
                          ((unsigned __int128)((uint64_t)(sx * sx) * (uint64_t)H * (uint64_t)H) +
                           (unsigned __int128)((uint64_t)(sy * sy) * (uint64_t)W * (uint64_t)W));
  unsigned __int128 den = (unsigned __int128)((uint64_t)W * (uint64_t)W) * ((uint64_t)H * (uint64_t)H);
  uint64_t q = (uint64_t)(num / den);
  uint64_t b = isqrt_u64(q);
  return b >= (uint64_t)n_b ? -1 : (int)b;
}

/* steps 5-6 applied to one full-plane map; out[b] = mean over the bin (0 if empty) */
static void azimuthal_mean(const double* map2d, int W, int H, int n_b, double* out, int64_t* counts) {
  for (int b = 0; b < n_b; ++b) { out[b] = 0.0; if (counts) counts[b] = 0; }
  int64_t* c = (int64_t*)calloc((size_t)n_b, sizeof(int64_t));
  for (int ky = 0; ky < H; ++ky)
    for (int kx = 0; kx < W; ++kx) {
      int b = nfso_qbin(kx, ky, W, H, n_b);
      if (b < 0) continue;
      out[b] += map2d[(long)ky * W + kx];
      c[b] += 1;
    }
  for (int b = 0; b < n_b; ++b) {
    if (c[b] > 0) out[b] /= (double)c[b];
    if (counts) counts[b] = c[b];
  }
  free(c);
}

/* exported for the pins */
void nfso_azimuthal_mean(const double* map2d, int W, int H, int n_b, double* out, int64_t* counts) {
  azimuthal_mean(map2d, W, H, n_b, out, counts);
}

/* ---- steps 1-6, everything in memory: THE definition --------------------------------------- */

#define PIX_TILE 256

/* wall-clock seconds of the two stages of the last nfso_structure_function call (bench.py's cpu_baseline
 * reports them): [0] steps 1-2 (normalise + transform), [1] steps 3-4 (pair loop, I2d). */
static double g_stage_seconds[2] = {0.0, 0.0};
static double now_seconds(void) {
#ifdef _OPENMP
  return omp_get_wtime();
#else
  return 0.0;
#endif
}
void nfso_last_stage_seconds(double* out2) { out2[0] = g_stage_seconds[0]; out2[1] = g_stage_seconds[1]; }

/*
 * frames  [N][H][W] uint16 row-major.        lags [n_lags] (>=1, strictly increasing).
 * D       [n_lags][n_b]   azimuthal means of D2d.    I_q [n_b].   counts [n_b].
 * n_pairs [n_lags]        N - tau, or 0 when tau >= N (row of zeros, reading R5).
 * D2d     optional [n_lags][H][W] full plane, FFT order.   I2d optional [H][W].
 * method  0 = radix-2 FFT, 1 = brute-force DFT (tiny inputs).
 */
int nfso_structure_function(const uint16_t* frames, int N, int W, int H, const int32_t* lags, int n_lags,
                            int n_b, int method, double* D, double* I_q, int64_t* counts, int64_t* n_pairs,
                            double* D2d_out, double* I2d_out) {
  if (!frames || !lags || N < 1 || W < 1 || H < 1 || n_lags < 1 || n_b < 1) return NFSO_ERR_ARG;
  for (int l = 0; l < n_lags; ++l)
    if (lags[l] < 1 || (l > 0 && lags[l] <= lags[l - 1])) return NFSO_ERR_ARG;
  const long P = (long)W * H;
  cplx* F = (cplx*)malloc(sizeof(cplx) * (size_t)N * P);
  double* D2d = D2d_out ? D2d_out : (double*)malloc(sizeof(double) * (size_t)n_lags * P);
  double* I2d = I2d_out ? I2d_out : (double*)malloc(sizeof(double) * (size_t)P);
  if (!F || !D2d || !I2d) {
    free(F);
    if (!D2d_out) free(D2d);
    if (!I2d_out) free(I2d);
    return NFSO_ERR_MEM;
  }
  int rc_all = NFSO_OK;
  const double t_start = now_seconds();

  /* steps 1-2: every frame is normalised and transformed exactly once (L31) */
#pragma omp parallel for schedule(dynamic, 1)
  for (int t = 0; t < N; ++t) {
    double* tmp = (double*)malloc(sizeof(double) * (size_t)P);
    int rc = tmp ? transform_frame(frames + (size_t)t * P, W, H, method, tmp, F + (size_t)t * P) : NFSO_ERR_MEM;
    if (rc) {
#pragma omp critical
      rc_all = rc;
    }
    free(tmp);
  }
  if (rc_all) { free(F); if (!D2d_out) free(D2d); if (!I2d_out) free(I2d); return rc_all; }
  const double t_fft = now_seconds();

  /* step 3: explicit pair loop, pixel-tiled */
  memset(D2d, 0, sizeof(double) * (size_t)n_lags * P);
#pragma omp parallel for schedule(dynamic, 1)
  for (long k0 = 0; k0 < P; k0 += PIX_TILE) {
    long k1 = k0 + PIX_TILE < P ? k0 + PIX_TILE : P;
    for (int l = 0; l < n_lags; ++l) {
      int tau = lags[l];
      if (tau >= N) continue;
      double* acc = D2d + (size_t)l * P;
      for (int t = 0; t + tau < N; ++t) {
        const cplx* a = F + (size_t)t * P;
        const cplx* b = F + (size_t)(t + tau) * P;
        for (long k = k0; k < k1; ++k) {
          cplx d = a[k] - b[k];
          acc[k] += creal(d) * creal(d) + cimag(d) * cimag(d);
        }
      }
      for (long k = k0; k < k1; ++k) acc[k] /= (double)(N - tau);
    }
  }
  for (int l = 0; l < n_lags; ++l) n_pairs[l] = lags[l] < N ? (int64_t)(N - lags[l]) : 0;

  /* step 4 */
#pragma omp parallel for schedule(static)
  for (long k = 0; k < P; ++k) {
    double s = 0.0;
    for (int t = 0; t < N; ++t) {
      cplx f = F[(size_t)t * P + k];
      s += creal(f) * creal(f) + cimag(f) * cimag(f);
    }
    I2d[k] = s / (double)N;
  }
  g_stage_seconds[0] = t_fft - t_start;
  g_stage_seconds[1] = now_seconds() - t_fft;

  /* steps 5-6 */
  for (int l = 0; l < n_lags; ++l) azimuthal_mean(D2d + (size_t)l * P, W, H, n_b, D + (size_t)l * n_b, NULL);
  azimuthal_mean(I2d, W, H, n_b, I_q, counts);

  free(F);
  if (!D2d_out) free(D2d);
  if (!I2d_out) free(I2d);
  return NFSO_OK;
}

/* ---- steps 1-6 on the half plane kx = 0..W/2 ("half-plane fast variant", pin P11) -------------
 *
 * The image is real, so F_t(W-kx, H-ky) = conj F_t(kx, ky): every full-plane pixel with kx > W/2 repeats the
 * value |.|^2 of its mirror with kx < W/2, which lies at the same |q| and therefore in the same bin.  The
 * definition is evaluated for kx <= W/2 only and a bin mean weights the columns 0 < kx < W/2 twice (columns 0
 * and W/2 map onto themselves): c_b and the sums are those of the full plane.
 * Every frame is still normalised and transformed in full (steps 1-2, the same transform_frame); the explicit
 * pair loop (step 3) runs pixel tile by pixel tile over a contiguous copy of the tile's time series (loop order
 * and memory management only).  Memory: N * H * (W/2+1) complex128.
 *
 * D [n_lags][n_b], I_q [n_b], counts [n_b], n_pairs [n_lags] as in nfso_structure_function.
 * D2d_out optional [n_lags][H][W/2+1], I2d_out optional [H][W/2+1]  (half plane, FFT order). */
int nfso_structure_function_half(const uint16_t* frames, int N, int W, int H, const int32_t* lags, int n_lags,
                                 int n_b, double* D, double* I_q, int64_t* counts, int64_t* n_pairs,
                                 double* D2d_out, double* I2d_out) {
  if (!frames || !lags || N < 1 || W < 2 || H < 1 || n_lags < 1 || n_b < 1) return NFSO_ERR_ARG;
  for (int l = 0; l < n_lags; ++l)
    if (lags[l] < 1 || (l > 0 && lags[l] <= lags[l - 1])) return NFSO_ERR_ARG;
  const long P = (long)W * H;
  const int Wh = W / 2 + 1;
  const long Ph = (long)Wh * H;
  cplx* F = (cplx*)malloc(sizeof(cplx) * (size_t)N * Ph); /* [t][ky][kx <= W/2] */
  double* D2d = D2d_out ? D2d_out : (double*)malloc(sizeof(double) * (size_t)n_lags * Ph);
  double* I2d = I2d_out ? I2d_out : (double*)malloc(sizeof(double) * (size_t)Ph);
  int rc_all = (F && D2d && I2d) ? NFSO_OK : NFSO_ERR_MEM;

  /* steps 1-2: every frame normalised and transformed exactly once, in full; the half plane is kept */
  if (!rc_all) {
#pragma omp parallel
    {
      double* tmp = (double*)malloc(sizeof(double) * (size_t)P);
      cplx* Ff = (cplx*)malloc(sizeof(cplx) * (size_t)P);
#pragma omp for schedule(dynamic, 1)
      for (int t = 0; t < N; ++t) {
        int rc = (tmp && Ff) ? transform_frame(frames + (size_t)t * P, W, H, 0, tmp, Ff) : NFSO_ERR_MEM;
        if (rc) {
#pragma omp critical
          rc_all = rc;
          continue;
        }
        for (int ky = 0; ky < H; ++ky)
          for (int kx = 0; kx < Wh; ++kx) F[(size_t)t * Ph + (long)ky * Wh + kx] = Ff[(long)ky * W + kx];
      }
      free(tmp);
      free(Ff);
    }
  }

  /* steps 3-4: explicit pair loop over a contiguous copy of each pixel tile's time series.  The tile is sized
   * so that the copy (N * tile complex128) stays in a core's cache. */
  if (!rc_all) {
    long tile = (long)(1 << 20) / (16L * N);
    if (tile > PIX_TILE) tile = PIX_TILE;
    if (tile < 4) tile = 4;
#pragma omp parallel
    {
      cplx* ts = (cplx*)malloc(sizeof(cplx) * (size_t)N * tile); /* [t][k - k0] */
      double* acc = (double*)malloc(sizeof(double) * (size_t)tile);
#pragma omp for schedule(dynamic, 1)
      for (long k0 = 0; k0 < Ph; k0 += tile) {
        if (!ts || !acc) {
#pragma omp critical
          rc_all = NFSO_ERR_MEM;
          continue;
        }
        const long nk = k0 + tile < Ph ? tile : Ph - k0;
        for (int t = 0; t < N; ++t)
          for (long k = 0; k < nk; ++k) ts[(size_t)t * tile + k] = F[(size_t)t * Ph + k0 + k];
        for (int l = 0; l < n_lags; ++l) {
          const int tau = lags[l];
          for (long k = 0; k < nk; ++k) acc[k] = 0.0;
          for (int t = 0; t + tau < N; ++t) {
            const cplx* a = ts + (size_t)t * tile;
            const cplx* b = ts + (size_t)(t + tau) * tile;
            for (long k = 0; k < nk; ++k) {
              cplx d = a[k] - b[k];
              acc[k] += creal(d) * creal(d) + cimag(d) * cimag(d);
            }
          }
          for (long k = 0; k < nk; ++k) D2d[(size_t)l * Ph + k0 + k] = tau < N ? acc[k] / (double)(N - tau) : 0.0;
        }
        for (long k = 0; k < nk; ++k) acc[k] = 0.0;
        for (int t = 0; t < N; ++t)
          for (long k = 0; k < nk; ++k) {
            cplx f = ts[(size_t)t * tile + k];
            acc[k] += creal(f) * creal(f) + cimag(f) * cimag(f);
          }
        for (long k = 0; k < nk; ++k) I2d[k0 + k] = acc[k] / (double)N;
      }
      free(ts);
      free(acc);
    }
  }

  /* steps 5-6 with the Hermitian weights: 2 for 0 < kx < W/2, 1 for kx = 0 and kx = W/2 */
  if (!rc_all) {
    for (int l = 0; l < n_lags; ++l) n_pairs[l] = lags[l] < N ? (int64_t)(N - lags[l]) : 0;
    for (int row = 0; row <= n_lags; ++row) {
      const double* map = row < n_lags ? D2d + (size_t)row * Ph : I2d;
      double* out = row < n_lags ? D + (size_t)row * n_b : I_q;
      for (int b = 0; b < n_b; ++b) { out[b] = 0.0; counts[b] = 0; }
      for (int ky = 0; ky < H; ++ky)
        for (int kx = 0; kx < Wh; ++kx) {
          int b = nfso_qbin(kx, ky, W, H, n_b);
          if (b < 0) continue;
          int w = (kx == 0 || 2 * kx == W) ? 1 : 2;
          out[b] += (double)w * map[(long)ky * Wh + kx];
          counts[b] += w;
        }
      for (int b = 0; b < n_b; ++b)
        if (counts[b] > 0) out[b] /= (double)counts[b];
    }
  }
  free(F);
  if (!D2d_out) free(D2d);
  if (!I2d_out) free(I2d);
  return rc_all;
}

/* ---- variance form of the static-free spectrum (reading R9b) ------------
 *
 *   7. M(k)   = (1/N) sum_t F_t(k)                       time-averaged field (the static image: beam, fringes)
 *      V2d(k) = (1/N) sum_t |F_t(k) - M(k)|^2            power of the fluctuations alone
 *      V(b)   = azimuthal mean of V2d (same bins as step 5-6)
 *
 * PAPER.md:L21-25, Eq. 1: the difference spectrum is 2a{T(q) I_s(q) [1 - f(q,tau)] + B(q)}; for lags beyond the
 * relaxation time (f -> 0) it reaches the plateau 2a{T I_s + B}, and the variance of the field in time is half
 * of that plateau: for all N(N-1)/2 pairs, sum_tau (N - tau) D2d(k,tau) = N^2 V2d(k) (pin P10).  Written as its
 * two-pass definition: pass 1 forms M, pass 2 transforms every frame again and sums |F_t - M|^2 (O(P) memory). */
int nfso_variance_spectrum(const uint16_t* frames, int N, int W, int H, int n_b, int method, double* V_q,
                           int64_t* counts, double* V2d_out) {
  if (!frames || N < 1 || W < 1 || H < 1 || n_b < 1 || !V_q) return NFSO_ERR_ARG;
  const long P = (long)W * H;
  cplx* M = (cplx*)calloc((size_t)P, sizeof(cplx));
  cplx* F = (cplx*)malloc(sizeof(cplx) * (size_t)P);
  double* tmp = (double*)malloc(sizeof(double) * (size_t)P);
  double* V2d = V2d_out ? V2d_out : (double*)malloc(sizeof(double) * (size_t)P);
  if (!M || !F || !tmp || !V2d) return NFSO_ERR_MEM;
  int rc = NFSO_OK;
  for (int t = 0; t < N && !rc; ++t) { /* pass 1: the mean field */
    rc = transform_frame(frames + (size_t)t * P, W, H, method, tmp, F);
    if (!rc)
      for (long k = 0; k < P; ++k) M[k] += F[k];
  }
  if (!rc) {
    for (long k = 0; k < P; ++k) M[k] /= (double)N;
    memset(V2d, 0, sizeof(double) * (size_t)P);
    for (int t = 0; t < N && !rc; ++t) { /* pass 2: squared deviations from it */
      rc = transform_frame(frames + (size_t)t * P, W, H, method, tmp, F);
      if (!rc)
        for (long k = 0; k < P; ++k) {
          cplx d = F[k] - M[k];
          V2d[k] += creal(d) * creal(d) + cimag(d) * cimag(d);
        }
    }
  }
  if (!rc) {
    for (long k = 0; k < P; ++k) V2d[k] /= (double)N;
    azimuthal_mean(V2d, W, H, n_b, V_q, counts);
  }
  free(M);
  free(F);
  free(tmp);
  if (!V2d_out) free(V2d);
  return rc;
}

/* ---- same definition, frames streamed through a window of Lmax+1 transforms ------------------
 * Memory management only (the paper's FIFO, L33): pair (t-tau, t) is formed when frame t
 * arrives.  Pinned against nfso_structure_function (pin P12). */
int nfso_structure_function_windowed(const uint16_t* frames, int N, int W, int H, const int32_t* lags,
                                     int n_lags, int n_b, double* D, double* I_q, int64_t* counts,
                                     int64_t* n_pairs, double* D2d_out, double* I2d_out) {
  if (!frames || !lags || N < 1 || n_lags < 1 || n_b < 1) return NFSO_ERR_ARG;
  for (int l = 0; l < n_lags; ++l)
    if (lags[l] < 1 || (l > 0 && lags[l] <= lags[l - 1])) return NFSO_ERR_ARG;
  const long P = (long)W * H;
  const int Lmax = lags[n_lags - 1];
  const int R = (Lmax < N ? Lmax : N - 1) + 1; /* window slots */
  cplx* ring = (cplx*)malloc(sizeof(cplx) * (size_t)R * P);
  double* tmp = (double*)malloc(sizeof(double) * (size_t)P);
  double* D2d = D2d_out ? D2d_out : (double*)malloc(sizeof(double) * (size_t)n_lags * P);
  double* I2d = I2d_out ? I2d_out : (double*)malloc(sizeof(double) * (size_t)P);
  if (!ring || !tmp || !D2d || !I2d) return NFSO_ERR_MEM;
  memset(D2d, 0, sizeof(double) * (size_t)n_lags * P);
  memset(I2d, 0, sizeof(double) * (size_t)P);
  for (int t = 0; t < N; ++t) {
    cplx* cur = ring + (size_t)(t % R) * P;
    int rc = transform_frame(frames + (size_t)t * P, W, H, 0, tmp, cur);
    if (rc) { free(ring); free(tmp); if (!D2d_out) free(D2d); if (!I2d_out) free(I2d); return rc; }
#pragma omp parallel for schedule(static)
    for (long k0 = 0; k0 < P; k0 += PIX_TILE) {
      long k1 = k0 + PIX_TILE < P ? k0 + PIX_TILE : P;
      for (long k = k0; k < k1; ++k) I2d[k] += creal(cur[k]) * creal(cur[k]) + cimag(cur[k]) * cimag(cur[k]);
      for (int l = 0; l < n_lags; ++l) {
        int tau = lags[l];
        if (tau > t) break;
        const cplx* old = ring + (size_t)((t - tau) % R) * P;
        double* acc = D2d + (size_t)l * P;
        for (long k = k0; k < k1; ++k) {
          cplx d = old[k] - cur[k];
          acc[k] += creal(d) * creal(d) + cimag(d) * cimag(d);
        }
      }
    }
  }
  for (int l = 0; l < n_lags; ++l) {
    n_pairs[l] = lags[l] < N ? (int64_t)(N - lags[l]) : 0;
    if (n_pairs[l] > 0)
      for (long k = 0; k < P; ++k) D2d[(size_t)l * P + k] /= (double)n_pairs[l];
  }
  for (long k = 0; k < P; ++k) I2d[k] /= (double)N;
  for (int l = 0; l < n_lags; ++l) azimuthal_mean(D2d + (size_t)l * P, W, H, n_b, D + (size_t)l * n_b, NULL);
  azimuthal_mean(I2d, W, H, n_b, I_q, counts);
  free(ring);
  free(tmp);
  if (!D2d_out) free(D2d);
  if (!I2d_out) free(I2d);
  return NFSO_OK;
}

/* ---- the definition restricted to a list of Fourier pixels ----------------------------------
 * For stacks too large to hold: every frame is still normalised and transformed in full
 * (steps 1-2), only the n_s sampled pixels (ky,kx) are kept, then steps 3-4 run on them.
 * D2d_s [n_lags][n_s], I2d_s [n_s].  Pinned against nfso_structure_function in the pins. */
int nfso_structure_function_sampled(const uint16_t* frames, int N, int W, int H, const int32_t* lags,
                                    int n_lags, const int32_t* sample_ky, const int32_t* sample_kx, int n_s,
                                    double* D2d_s, double* I2d_s, int64_t* n_pairs) {
  if (!frames || !lags || !sample_ky || !sample_kx || N < 1 || n_lags < 1 || n_s < 1) return NFSO_ERR_ARG;
  const long P = (long)W * H;
  cplx* Fs = (cplx*)malloc(sizeof(cplx) * (size_t)N * n_s); /* [t][s] */
  if (!Fs) return NFSO_ERR_MEM;
  int rc_all = NFSO_OK;
#pragma omp parallel
  {
    double* tmp = (double*)malloc(sizeof(double) * (size_t)P);
    cplx* F = (cplx*)malloc(sizeof(cplx) * (size_t)P);
#pragma omp for schedule(dynamic, 1)
    for (int t = 0; t < N; ++t) {
      int rc = transform_frame(frames + (size_t)t * P, W, H, 0, tmp, F);
      if (rc) {
#pragma omp critical
        rc_all = rc;
        continue;
      }
      for (int s = 0; s < n_s; ++s) Fs[(size_t)t * n_s + s] = F[(long)sample_ky[s] * W + sample_kx[s]];
    }
    free(tmp);
    free(F);
  }
  if (rc_all) { free(Fs); return rc_all; }
  for (int l = 0; l < n_lags; ++l) {
    int tau = lags[l];
    n_pairs[l] = tau < N ? (int64_t)(N - tau) : 0;
    for (int s = 0; s < n_s; ++s) {
      double acc = 0.0;
      for (int t = 0; t + tau < N; ++t) {
        cplx d = Fs[(size_t)t * n_s + s] - Fs[(size_t)(t + tau) * n_s + s];
        acc += creal(d) * creal(d) + cimag(d) * cimag(d);
      }
      D2d_s[(size_t)l * n_s + s] = tau < N ? acc / (double)(N - tau) : 0.0;
    }
  }
  for (int s = 0; s < n_s; ++s) {
    double acc = 0.0;
    for (int t = 0; t < N; ++t) {
      cplx f = Fs[(size_t)t * n_s + s];
      acc += creal(f) * creal(f) + cimag(f) * cimag(f);
    }
    I2d_s[s] = acc / (double)N;
  }
  free(Fs);
  return NFSO_OK;
}
