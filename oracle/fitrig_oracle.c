/* fitrig_oracle.c -- CPU fp64 ORACLE for the FITrig hot path (tLISI map + detection).
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code, header, table or constant with the CUDA path
 * (paper_2509_21754_b200/csrc) and neither includes the other.
 *
 * What it is: the plain definition of tLISI and of the detection rules, written
 * out in the paper's order and notation, evaluated in double precision on the same
 * fp32 input bits the GPU sees.  No blocking, fusion or reordering; the only
 * concession to run time is an OpenMP "parallel for" over independent (unit, tile-row)
 * pairs, which the paper itself states are independent.
 *
 * Citations are /root/reference/PAPER.md line numbers (+ equation).  Readings R1..R30
 * of silent / ambiguous passages are SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * Notation (0-based): snapshots x_0..x_{L-1}, each H x W row-major fp32.
 * Unit u = 0..L-3 uses x_u, x_{u+1}, x_{u+2}  (the paper's s = u+1).
 * Tiles: Ty = ceil(H/N_T), Tx = ceil(W/N_T); tile (ty,tx) covers rows
 * [ty*N_T, min(H,(ty+1)*N_T)), cols likewise (R5: partial edge tiles keep their own
 * pixel count n_t).
 *
 * Pins (tests/test_oracle_pins.py, tests/golden/): P1..P13 of SURVEY.md section 8(c).
 * Every function below is pinned; none is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_REF_ABS 0     /* R1 (default): x_hat = |x|, |x| == 0 -> C                      */
#define ORACLE_REF_LITERAL 1 /* Eq. 5 exactly as printed: x_hat = x, x == 0 -> C (signed)      */
#define ORACLE_REF_FLOOR 2   /* x_hat = max(x, C)                                             */

int fitrig_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void fitrig_oracle_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* O1.  M = max( max_{s=1..L} x^(s), C )  -- the signed maximum pixel value over ALL
 * pixels of ALL L snapshots, floored at C.  PAPER.md:153 (Eq. 2 denominator), 189
 * ("maximum pixel value across all snapshots"), 223 (M definition).  R2, R14. */
double fitrig_oracle_global_max(const float* const* snaps, int L, int64_t H, int64_t W, double C) {
  double m = C;
  for (int s = 0; s < L; ++s) {
    const float* x = snaps[s];
    double ms = C;
#pragma omp parallel for reduction(max : ms)
    for (int64_t i = 0; i < H * W; ++i) {
      double v = (double)x[i];
      if (v > ms) ms = v;
    }
    if (ms > m) m = ms;
  }
  return m;
}

/* Reference intensity x_hat^(s+1), Eq. 5 under reading R1. */
static double ref_intensity(double x, double C, int ref_mode) {
  if (ref_mode == ORACLE_REF_LITERAL) return (x == 0.0) ? C : x;
  if (ref_mode == ORACLE_REF_FLOOR) return (x > C) ? x : C;
  double a = fabs(x);
  return (a == 0.0) ? C : a;
}

/* O2..O5.  For every unit u and tile t:
 *   D^(s)   = |x^(s+1) - x^(s)|                                   Eq. 3
 *   Delta   = |D^(s) - D^(s+1)|
 *   r_i     = Delta_i / x_hat_i  if that is < 1, else 1           Eq. 4-5
 *   q       = mean(Delta) * max(Delta) * mean(r) / (M * M)        Eq. 2, PAPER.md:153 (R13: M^2)
 *   tLISI   = 1 - q
 * Outputs are [U][Ty][Tx]; any output pointer may be NULL.
 * argmax = y*W + x of the first (lowest row-major) pixel attaining max(Delta) in the tile (R20).
 * Returns 0, or -1 on bad arguments (R10: L < 3). */
/* Pixel p of image k: the images are either the fp32 snapshots themselves or fp64 accumulated snapshots
 * (fitrig_oracle_tlisi_f64, PAPER.md:497 / Fig. 16); widening fp32 -> fp64 is exact. */
static double px(const void* const* img, int is_f64, int k, int64_t p) {
  return is_f64 ? ((const double*)img[k])[p] : (double)((const float*)img[k])[p];
}

/* Number of windows of `tile` pixels placed every `stride` pixels along an axis of n pixels (stride divides tile).
 * stride == tile: the paper's non-overlapping tiles, ceil(n / tile) with a partial last tile (R5).  stride < tile
 * (overlapping windows, reading R27): the image is cut into cells of `stride` pixels, C = ceil(n / stride) of them,
 * and a window is tile / stride consecutive cells: C - tile/stride + 1 windows, at least one. */
static int n_windows(int n, int tile, int stride) {
  const int cells = (n + stride - 1) / stride, m = tile / stride;
  return (cells - m + 1 > 1) ? cells - m + 1 : 1;
}

static int tlisi_core(const void* const* snaps, int is_f64, int L, int H, int W, int tile, int stride, double C,
                      int ref_mode, double M, double* sumD, double* maxD, double* sumR, int64_t* argmax, double* q,
                      double* tlisi) {
  if (L < 3 || H < 1 || W < 1 || tile < 1 || stride < 1 || tile % stride != 0 || !snaps) return -1;
  const int U = L - 2;
  const int Ty = n_windows(H, tile, stride), Tx = n_windows(W, tile, stride);
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
  for (int u = 0; u < U; ++u) {
    for (int ty = 0; ty < Ty; ++ty) {
      /* images u, u+1, u+2 are x^(s), x^(s+1) (the reference image) and x^(s+2) */
      for (int tx = 0; tx < Tx; ++tx) {
        const int r0 = ty * stride, r1 = (r0 + tile < H) ? r0 + tile : H;
        const int c0 = tx * stride, c1 = (c0 + tile < W) ? c0 + tile : W;
        double s_delta = 0.0, m_delta = 0.0, s_r = 0.0;
        int64_t arg = (int64_t)r0 * W + c0;
        int first = 1;
        for (int i = r0; i < r1; ++i) {
          for (int j = c0; j < c1; ++j) {
            const int64_t p = (int64_t)i * W + j;
            const double a = px(snaps, is_f64, u, p), b = px(snaps, is_f64, u + 1, p), c = px(snaps, is_f64, u + 2, p);
            const double D1 = fabs(b - a);
            const double D2 = fabs(c - b);
            const double delta = fabs(D1 - D2);
            const double xh = ref_intensity(b, C, ref_mode);
            const double ratio = delta / xh;
            const double r = (ratio < 1.0) ? ratio : 1.0;
            s_delta += delta;
            s_r += r;
            if (first || delta > m_delta) {
              m_delta = delta;
              arg = p;
              first = 0;
            }
          }
        }
        const double n_t = (double)(r1 - r0) * (double)(c1 - c0);
        const double mean_delta = s_delta / n_t;
        const double mean_r = s_r / n_t;
        const double qv = mean_delta * m_delta * mean_r / (M * M);
        const int64_t o = ((int64_t)u * Ty + ty) * Tx + tx;
        if (sumD) sumD[o] = s_delta;
        if (maxD) maxD[o] = m_delta;
        if (sumR) sumR[o] = s_r;
        if (argmax) argmax[o] = arg;
        if (q) q[o] = qv;
        if (tlisi) tlisi[o] = 1.0 - qv;
      }
    }
  }
  return 0;
}

int fitrig_oracle_tlisi(const float* const* snaps, int L, int H, int W, int tile, double C, int ref_mode,
                        double M, double* sumD, double* maxD, double* sumR, int64_t* argmax, double* q,
                        double* tlisi) {
  return tlisi_core((const void* const*)snaps, 0, L, H, W, tile, tile, C, ref_mode, M, sumD, maxD, sumR, argmax, q, tlisi);
}

/* The same O2..O5 on fp64 images: used for ACCUMULATED snapshots (section 3.3.2, Fig. 16:
 * "FITrig can be applied after combining multiple snapshots"), whose sums are formed in fp64 by the caller. */
int fitrig_oracle_tlisi_f64(const double* const* imgs, int L, int H, int W, int tile, double C, int ref_mode,
                            double M, double* sumD, double* maxD, double* sumR, int64_t* argmax, double* q,
                            double* tlisi) {
  return tlisi_core((const void* const*)imgs, 1, L, H, W, tile, tile, C, ref_mode, M, sumD, maxD, sumR, argmax, q, tlisi);
}

/* Overlapping windows (an EXTENSION: the paper's tiles never overlap).  Reading
 * R27: the same Eq. 2-6 on windows of tile x tile pixels placed every `stride` pixels (stride divides tile) in both
 * directions; window (ty, tx) covers rows [ty*stride, min(H, ty*stride + tile)), columns likewise; outputs are
 * [U][Ty][Tx] with Ty, Tx = n_windows().  stride == tile is fitrig_oracle_tlisi.  fp32 snapshots only. */
int fitrig_oracle_tlisi_windows(const float* const* snaps, int L, int H, int W, int tile, int stride, double C,
                                int ref_mode, double M, double* sumD, double* maxD, double* sumR, int64_t* argmax,
                                double* q, double* tlisi) {
  return tlisi_core((const void* const*)snaps, 0, L, H, W, tile, stride, C, ref_mode, M, sumD, maxD, sumR, argmax, q,
                    tlisi);
}

int fitrig_oracle_n_windows(int n, int tile, int stride) { return n_windows(n, tile, stride); }

/* O6.  z-score of the tile matrix of each unit, Eq. 8:
 *   z_t = ((1 - tLISI_t) - (1 - mu)) / sigma = (q_t - mean(q)) / std(q)
 * with the population standard deviation (R3); sigma == 0 -> z = 0 everywhere (R4).
 * v is [U][n]; mu, sigma are [U]; z is [U][n]. */
void fitrig_oracle_zscore(const double* v, int U, int64_t n, double* mu, double* sigma, double* z) {
  for (int u = 0; u < U; ++u) {
    const double* a = v + (int64_t)u * n;
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i) s += a[i];
    const double m = s / (double)n;
    double ss = 0.0;
    for (int64_t i = 0; i < n; ++i) ss += (a[i] - m) * (a[i] - m);
    const double sd = sqrt(ss / (double)n);
    if (mu) mu[u] = m;
    if (sigma) sigma[u] = sd;
    if (z)
      for (int64_t i = 0; i < n; ++i) z[(int64_t)u * n + i] = (sd == 0.0) ? 0.0 : (a[i] - m) / sd;
  }
}

/* O7.  Candidate set { t | z_t^(s) > tau }, Eq. 9, strict '>' (R6),
 * listed in (u, ty, tx) order; (x, y) = column, row of the tile's first max-Delta pixel (R16, R20).
 * Returns the total number found; at most `capacity` are written. */
int64_t fitrig_oracle_select(const double* z, const int64_t* argmax, int U, int64_t n, int W, double tau,
                             int32_t* out_x, int32_t* out_y, int32_t* out_u, int64_t* out_tile, double* out_z,
                             int64_t capacity) {
  int64_t k = 0;
  for (int u = 0; u < U; ++u)
    for (int64_t t = 0; t < n; ++t) {
      const double zv = z[(int64_t)u * n + t];
      if (zv > tau) {
        if (k < capacity) {
          const int64_t p = argmax ? argmax[(int64_t)u * n + t] : 0;
          if (out_x) out_x[k] = (int32_t)(p % W);
          if (out_y) out_y[k] = (int32_t)(p / W);
          if (out_u) out_u[k] = u;
          if (out_tile) out_tile[k] = t;
          if (out_z) out_z[k] = zv;
        }
        ++k;
      }
    }
  return k;
}

/* O8.  Image-frequency branch, Eq. 10 with h = maximum spectral magnitude
 * (PAPER.md:503):  per tile t,
 *   a_u   = q_t(u) - mean_u q_t(u)                 (DC removed; |F[tLISI-mean]| == |F[q-mean]|)
 *   F_k   = sum_u a_u exp(-2 pi i k u / U)         unnormalised DFT of length U (any U, R17)
 *   eta_t = max_{1 <= k <= floor(U/2)} |F_k| ,  kstar = first k attaining it
 * q is [U][n]; eta, kstar are [n]. */
void fitrig_oracle_spectrum(const double* q, int U, int64_t n, double* eta, int32_t* kstar) {
  const double two_pi = 6.283185307179586476925286766559;
#pragma omp parallel for schedule(static)
  for (int64_t t = 0; t < n; ++t) {
    double mean = 0.0;
    for (int u = 0; u < U; ++u) mean += q[(int64_t)u * n + t];
    mean /= (double)U;
    double best = 0.0;
    int32_t kb = (U / 2 >= 1) ? 1 : 0;
    for (int k = 1; k <= U / 2; ++k) {
      double re = 0.0, im = 0.0;
      for (int u = 0; u < U; ++u) {
        const double a = q[(int64_t)u * n + t] - mean;
        const double ang = -two_pi * (double)k * (double)u / (double)U;
        re += a * cos(ang);
        im += a * sin(ang);
      }
      const double mag = sqrt(re * re + im * im);
      if (k == 1 || mag > best) {
        best = mag;
        kb = k;
      }
    }
    eta[t] = best;
    if (kstar) kstar[t] = kb;
  }
}

/* O8h.  Image-frequency branch, Eq. 10 with h = HARMONIC SUMMING ("a spectral refinement
 * function, such as harmonic summing (Adamek et al., 2022)"; used for the real-data result,
 * PAPER.md:389-393, Fig. 11).  The paper does not restate the rule; reading R26 is the standard
 * incoherent harmonic sum of pulsar searching on the one-sided magnitude spectrum m_k = |F_k|, k = 1..K,
 * K = floor(U/2):
 *     s_h(k) = (1 / sqrt(h)) * sum_{i=1..h} m_{i*k}      for h = 1, 2, 4, ..., H  with  h*k <= K
 *     eta    = max over (k, h) of s_h(k);   k* = the fundamental bin k of the first maximum
 *              (k ascending, then h ascending; strict > keeps the first)
 * H = 1 is exactly O8 (maximum magnitude).  mag_out (may be NULL) receives m_k as [K][n]. */
void fitrig_oracle_spectrum_hsum(const double* q, int U, int64_t n, int H, double* eta, int32_t* kstar,
                                 double* mag_out) {
  const double two_pi = 6.283185307179586476925286766559;
  const int K = U / 2;
#pragma omp parallel for schedule(static)
  for (int64_t t = 0; t < n; ++t) {
    double* m = (double*)malloc(sizeof(double) * (size_t)(K + 1));
    double mean = 0.0;
    for (int u = 0; u < U; ++u) mean += q[(int64_t)u * n + t];
    mean /= (double)U;
    for (int k = 1; k <= K; ++k) {
      double re = 0.0, im = 0.0;
      for (int u = 0; u < U; ++u) {
        const double a = q[(int64_t)u * n + t] - mean;
        const double ang = -two_pi * (double)k * (double)u / (double)U;
        re += a * cos(ang);
        im += a * sin(ang);
      }
      m[k] = sqrt(re * re + im * im);
      if (mag_out) mag_out[(int64_t)(k - 1) * n + t] = m[k];
    }
    double best = 0.0;
    int32_t kb = (K >= 1) ? 1 : 0;
    int first = 1;
    for (int k = 1; k <= K; ++k) {
      for (int h = 1; h <= H && h * k <= K; h *= 2) {
        double s = 0.0;
        for (int i = 1; i <= h; ++i) s += m[i * k];
        s /= sqrt((double)h);
        if (first || s > best) {
          best = s;
          kb = k;
          first = 0;
        }
      }
    }
    eta[t] = best;
    if (kstar) kstar[t] = kb;
    free(m);
  }
}

/* Eq. 11-12 are fitrig_oracle_zscore(eta, 1, n, ...) followed by the same
 * strict threshold; the candidate record for this branch is (tile centre, kstar, z), R18:
 *   x = tx*N_T + w_t/2, y = ty*N_T + h_t/2 (integer division; w_t, h_t the tile's extent). */
int64_t fitrig_oracle_select_spectrum(const double* z, const int32_t* kstar, int Ty, int Tx, int H, int W,
                                      int tile, double tau, int32_t* out_x, int32_t* out_y, int32_t* out_k,
                                      int64_t* out_tile, double* out_z, int64_t capacity) {
  int64_t k = 0;
  for (int ty = 0; ty < Ty; ++ty)
    for (int tx = 0; tx < Tx; ++tx) {
      const int64_t t = (int64_t)ty * Tx + tx;
      if (z[t] > tau) {
        if (k < capacity) {
          const int r0 = ty * tile, r1 = (r0 + tile < H) ? r0 + tile : H;
          const int c0 = tx * tile, c1 = (c0 + tile < W) ? c0 + tile : W;
          if (out_x) out_x[k] = c0 + (c1 - c0) / 2;
          if (out_y) out_y[k] = r0 + (r1 - r0) / 2;
          if (out_k) out_k[k] = kstar[t];
          if (out_tile) out_tile[k] = t;
          if (out_z) out_z[k] = z[t];
        }
        ++k;
      }
    }
  return k;
}

/* ---------------------------------------------------------------------------------------------
 * O9.  Sub-tile localisation by interpolating the spectrum matrix eta (section 2.4.2: "interpolation
 * methods are activated for precise pulsar localisation in the selected regions ... bilinear, spline, bicubic, or
 * Makima cubic interpolation"; section 3.1: "We apply spline interpolation to the spectrum matrix ...
 * the peak position, corresponding to the pulsar position").  The paper names the four schemes and gives no formula;
 * reading R28:
 *
 *   - eta_t is a sample of a surface at the CENTRE of tile t.  Index coordinates: tile column tx sits at u = tx, tile
 *     row ty at v = ty; pixel x (pixel centres at integers) is u = (x + 0.5) / N_T - 0.5, i.e. the centre of tile tx
 *     is x_c = (tx + 0.5) N_T - 0.5.  (A partial edge tile is placed at its nominal full-tile centre.)
 *   - the surface is the tensor-product interpolant of the Ty x Tx samples on that uniform grid: first along x
 *     (within every tile row), then along y, with one of the four named 1-D schemes -- the four methods of the
 *     usual gridded-interpolation routine ('linear', 'cubic', 'spline', 'makima'):
 *       0 BILINEAR  piecewise linear
 *       1 BICUBIC   cubic convolution, Keys (1981) kernel a = -1/2, with Keys' boundary samples
 *                   f_{-1} = 3 f_0 - 3 f_1 + f_2 and f_n = 3 f_{n-1} - 3 f_{n-2} + f_{n-3}
 *       2 SPLINE    cubic spline with not-a-knot end conditions (3 samples: the parabola through them)
 *       3 MAKIMA    modified Akima piecewise cubic Hermite: node slopes from the weights
 *                   w1 = |d_{i+1} - d_i| + |d_{i+1} + d_i| / 2, w2 = |d_{i-1} - d_{i-2}| + |d_{i-1} + d_{i-2}| / 2,
 *                   slope = (w1 d_{i-1} + w2 d_i) / (w1 + w2), 0 when w1 + w2 = 0; d extended by
 *                   d_{-1} = 2 d_0 - d_1, d_{-2} = 2 d_{-1} - d_0 and likewise at the far end
 *     (2 samples along an axis: every scheme is the straight line; 1 sample: the constant).
 *   - for a selected tile (ty, tx) the surface is evaluated on the lattice
 *         x = x_c + i / r,  y = y_c + j / r,   i, j = -N_T r .. +N_T r   (r = oversample >= 1)
 *     that is u = tx + i / (r N_T), v = ty + j / (r N_T): one tile either side of the tile's centre, which the
 *     centres of the neighbouring tiles bound exactly; lattice points outside the hull of the tile centres
 *     (u < 0, u > Tx - 1, v < 0, v > Ty - 1) are left out (no extrapolation);
 *   - the position is the lattice point with the largest value, the first in (j, i) row-major order on ties.
 *
 * Everything is evaluated literally: the spline solves its full linear system (n equations, the two not-a-knot rows
 * written out) by Gaussian elimination, row by row and then for every lattice column (built once per column: it does
 * not depend on v).
 * --------------------------------------------------------------------------------------------- */
#define ORACLE_INTERP_BILINEAR 0
#define ORACLE_INTERP_BICUBIC 1
#define ORACLE_INTERP_SPLINE 2
#define ORACLE_INTERP_MAKIMA 3

/* Gaussian elimination with partial pivoting: A is n x n row-major, b is overwritten with the solution. */
static void solve_dense(int n, double* A, double* b) {
  for (int c = 0; c < n; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r)
      if (fabs(A[(size_t)r * n + c]) > fabs(A[(size_t)piv * n + c])) piv = r;
    if (piv != c) {
      for (int k = 0; k < n; ++k) {
        const double t = A[(size_t)c * n + k];
        A[(size_t)c * n + k] = A[(size_t)piv * n + k];
        A[(size_t)piv * n + k] = t;
      }
      const double t = b[c];
      b[c] = b[piv];
      b[piv] = t;
    }
    for (int r = c + 1; r < n; ++r) {
      const double f = A[(size_t)r * n + c] / A[(size_t)c * n + c];
      if (f == 0.0) continue;
      for (int k = c; k < n; ++k) A[(size_t)r * n + k] -= f * A[(size_t)c * n + k];
      b[r] -= f * b[c];
    }
  }
  for (int r = n - 1; r >= 0; --r) {
    double s = b[r];
    for (int k = r + 1; k < n; ++k) s -= A[(size_t)r * n + k] * b[k];
    b[r] = s / A[(size_t)r * n + r];
  }
}

/* Second derivatives m_0..m_{n-1} of the not-a-knot cubic spline through (i, f_i), i = 0..n-1 (unit spacing), n >= 3:
 *   interior knots  m_{i-1} + 4 m_i + m_{i+1} = 6 (f_{i-1} - 2 f_i + f_{i+1}),  i = 1..n-2
 *   not-a-knot      m_0 - 2 m_1 + m_2 = 0  and  m_{n-3} - 2 m_{n-2} + m_{n-1} = 0   (continuous third derivative at
 *                   the second and the second-to-last knot)
 * n == 3: both end conditions are the same equation; the spline is the parabola, m_i = f_0 - 2 f_1 + f_2. */
static void spline_second_derivs(const double* f, int n, double* m) {
  if (n < 3) {
    for (int i = 0; i < n; ++i) m[i] = 0.0;
    return;
  }
  if (n == 3) {
    m[0] = m[1] = m[2] = f[0] - 2.0 * f[1] + f[2];
    return;
  }
  double* A = (double*)calloc((size_t)n * n, sizeof(double));
  A[0] = 1.0; A[1] = -2.0; A[2] = 1.0;
  m[0] = 0.0;
  for (int i = 1; i <= n - 2; ++i) {
    A[(size_t)i * n + i - 1] = 1.0;
    A[(size_t)i * n + i] = 4.0;
    A[(size_t)i * n + i + 1] = 1.0;
    m[i] = 6.0 * (f[i - 1] - 2.0 * f[i] + f[i + 1]);
  }
  A[(size_t)(n - 1) * n + n - 3] = 1.0; A[(size_t)(n - 1) * n + n - 2] = -2.0; A[(size_t)(n - 1) * n + n - 1] = 1.0;
  m[n - 1] = 0.0;
  solve_dense(n, A, m);
  free(A);
}

/* Keys' cubic convolution kernel, a = -1/2. */
static double keys_kernel(double s) {
  s = fabs(s);
  if (s <= 1.0) return (1.5 * s - 2.5) * s * s + 1.0;
  if (s < 2.0) return ((-0.5 * s + 2.5) * s - 4.0) * s + 2.0;
  return 0.0;
}

/* Sample f_i with Keys' boundary extension (two samples: the straight line through them). */
static double keys_sample(const double* f, int n, int i) {
  if (i >= 0 && i < n) return f[i];
  if (n == 2) return (i < 0) ? 2.0 * f[0] - f[1] : 2.0 * f[1] - f[0];
  return (i < 0) ? 3.0 * f[0] - 3.0 * f[1] + f[2] : 3.0 * f[n - 1] - 3.0 * f[n - 2] + f[n - 3];
}

/* Difference d_i = f_{i+1} - f_i, i = 0..n-2, extended linearly by two entries at either end (makima). */
static double makima_diff(const double* f, int n, int i) {
  if (i >= 0 && i <= n - 2) return f[i + 1] - f[i];
  if (n == 2) return f[1] - f[0];
  if (i < 0) {
    const double d0 = f[1] - f[0], d1 = f[2] - f[1];
    const double dm1 = 2.0 * d0 - d1;
    return (i == -1) ? dm1 : 2.0 * dm1 - d0;
  }
  const double e0 = f[n - 1] - f[n - 2], e1 = f[n - 2] - f[n - 3];
  const double ep1 = 2.0 * e0 - e1;
  return (i == n - 1) ? ep1 : 2.0 * ep1 - e0;
}

static double makima_slope(const double* f, int n, int i) {
  const double dm2 = makima_diff(f, n, i - 2), dm1 = makima_diff(f, n, i - 1);
  const double d0 = makima_diff(f, n, i), d1 = makima_diff(f, n, i + 1);
  const double w1 = fabs(d1 - d0) + fabs(d1 + d0) / 2.0;
  const double w2 = fabs(dm1 - dm2) + fabs(dm1 + dm2) / 2.0;
  return (w1 + w2 > 0.0) ? (w1 * dm1 + w2 * d0) / (w1 + w2) : 0.0;
}

/* Value at index coordinate u in [0, n-1] of the 1-D interpolant through (i, f_i).  m: the spline's second
 * derivatives (method SPLINE only). */
static double interp1_eval(const double* f, const double* m, int n, int method, double u) {
  if (n == 1) return f[0];
  int i = (int)floor(u);
  if (i < 0) i = 0;
  if (i > n - 2) i = n - 2;
  const double t = u - (double)i;
  if (method == ORACLE_INTERP_BILINEAR || n == 2) return (1.0 - t) * f[i] + t * f[i + 1];
  if (method == ORACLE_INTERP_BICUBIC) {
    double s = 0.0;
    for (int k = -1; k <= 2; ++k) s += keys_sample(f, n, i + k) * keys_kernel(t - (double)k);
    return s;
  }
  if (method == ORACLE_INTERP_SPLINE) {
    const double a = 1.0 - t;
    return a * f[i] + t * f[i + 1] + ((a * a * a - a) * m[i] + (t * t * t - t) * m[i + 1]) / 6.0;
  }
  /* makima: cubic Hermite with the modified Akima slopes */
  const double s0 = makima_slope(f, n, i), s1 = makima_slope(f, n, i + 1);
  const double t2 = t * t, t3 = t2 * t;
  return (2.0 * t3 - 3.0 * t2 + 1.0) * f[i] + (t3 - 2.0 * t2 + t) * s0 + (-2.0 * t3 + 3.0 * t2) * f[i + 1] +
         (t3 - t2) * s1;
}

/* Tensor-product surface at (u, v): along x in every row, then along y.  rowm: [Ty][Tx] second derivatives of the
 * row splines (SPLINE) or NULL.  col, colm: scratch of Ty doubles each. */
static double surface_eval(const double* eta, const double* rowm, int Ty, int Tx, int method, double u, double v,
                           double* col, double* colm) {
  for (int ty = 0; ty < Ty; ++ty)
    col[ty] = interp1_eval(eta + (size_t)ty * Tx, rowm ? rowm + (size_t)ty * Tx : NULL, Tx, method, u);
  if (method == ORACLE_INTERP_SPLINE) spline_second_derivs(col, Ty, colm);
  return interp1_eval(col, colm, Ty, method, v);
}

/* The surface at npts index coordinates (u_k, v_k), 0 <= u <= Tx-1, 0 <= v <= Ty-1 (for the pins).  Returns 0 or -1. */
int fitrig_oracle_interp_eval(const double* eta, int Ty, int Tx, int method, const double* u, const double* v,
                              int64_t npts, double* out) {
  if (!eta || Ty < 1 || Tx < 1 || method < 0 || method > 3) return -1;
  double* rowm = NULL;
  if (method == ORACLE_INTERP_SPLINE) {
    rowm = (double*)malloc(sizeof(double) * (size_t)Ty * Tx);
    for (int ty = 0; ty < Ty; ++ty) spline_second_derivs(eta + (size_t)ty * Tx, Tx, rowm + (size_t)ty * Tx);
  }
  double* col = (double*)malloc(sizeof(double) * (size_t)Ty * 2);
  for (int64_t k = 0; k < npts; ++k) out[k] = surface_eval(eta, rowm, Ty, Tx, method, u[k], v[k], col, col + Ty);
  free(col);
  free(rowm);
  return 0;
}

/* Position of the surface's maximum around each selected tile (R28).  cand_tile[k] = ty * Tx + tx.  Outputs per
 * candidate: x, y in pixels (pixel centres at integers) and the surface value there.  Returns 0 or -1. */
int fitrig_oracle_localise(const double* eta, int Ty, int Tx, int tile, int method, int oversample,
                           const int64_t* cand_tile, int64_t ncand, double* out_x, double* out_y, double* out_val) {
  if (!eta || Ty < 1 || Tx < 1 || tile < 1 || oversample < 1 || method < 0 || method > 3) return -1;
  double* rowm = NULL;
  if (method == ORACLE_INTERP_SPLINE) {
    rowm = (double*)malloc(sizeof(double) * (size_t)Ty * Tx);
    for (int ty = 0; ty < Ty; ++ty) spline_second_derivs(eta + (size_t)ty * Tx, Tx, rowm + (size_t)ty * Tx);
  }
  const int half = tile * oversample;  /* lattice offsets -half .. +half, spacing 1 / oversample pixels */
  const int side = 2 * half + 1;
  double* col = (double*)malloc(sizeof(double) * (size_t)Ty * 2);
  double* val = (double*)malloc(sizeof(double) * (size_t)side * side);  /* surface on the lattice, [j][i] */
  for (int64_t k = 0; k < ncand; ++k) {
    const int ty = (int)(cand_tile[k] / Tx), tx = (int)(cand_tile[k] % Tx);
    const double xc = ((double)tx + 0.5) * (double)tile - 0.5, yc = ((double)ty + 0.5) * (double)tile - 0.5;
    /* the column of row-interpolant values at u does not depend on v: built once per lattice column */
    for (int i = -half; i <= half; ++i) {
      const double u = (double)tx + (double)i / (double)half;
      if (u < 0.0 || u > (double)(Tx - 1)) continue;
      for (int r = 0; r < Ty; ++r)
        col[r] = interp1_eval(eta + (size_t)r * Tx, rowm ? rowm + (size_t)r * Tx : NULL, Tx, method, u);
      if (method == ORACLE_INTERP_SPLINE) spline_second_derivs(col, Ty, col + Ty);
      for (int j = -half; j <= half; ++j) {
        const double v = (double)ty + (double)j / (double)half;
        if (v < 0.0 || v > (double)(Ty - 1)) continue;
        val[(size_t)(j + half) * side + (i + half)] = interp1_eval(col, col + Ty, Ty, method, v);
      }
    }
    double best = 0.0, bx = xc, by = yc;
    int first = 1;
    for (int j = -half; j <= half; ++j) {
      const double v = (double)ty + (double)j / (double)half;
      if (v < 0.0 || v > (double)(Ty - 1)) continue;
      for (int i = -half; i <= half; ++i) {
        const double u = (double)tx + (double)i / (double)half;
        if (u < 0.0 || u > (double)(Tx - 1)) continue;
        const double w = val[(size_t)(j + half) * side + (i + half)];
        if (first || w > best) {
          best = w;
          bx = xc + (double)i / (double)oversample;
          by = yc + (double)j / (double)oversample;
          first = 0;
        }
      }
    }
    out_x[k] = bx;
    out_y[k] = by;
    if (out_val) out_val[k] = best;
  }
  free(val);
  free(col);
  free(rowm);
  return 0;
}
