/*
 * oracle/pyhst_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU statement of what the hot path of
 * arxiv/paper_1306_1392 (PyHST2) computes: ramp filter, parallel-beam
 * pixel-driven backprojection, its exact transpose (forward projection) and
 * FBP.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  It shares no code, header, table or
 * constant generator with paper_1306_1392_b200/ (the CUDA path) and neither
 * includes the other.
 *
 * What the paper fixes:
 *   L63-L65 (sec. 2.3)  FBP; backprojection reads the sinogram with linear
 *                       interpolation, one value per (pixel, projection).
 *   L35 (sec. 2.1)      projections span >= 180 deg; rotation-axis position and
 *                       angle may be given per projection; with a 360 deg scan
 *                       and the axis near the detector border the detector
 *                       "can be virtually doubled".
 *   L59 (sec. 2.3)      one sinogram per slice; slices are independent.
 *   L71-L73 (sec. 3.1, eq. 1)  P and P^T: projection and back-projection.
 * Everything the paper leaves open is taken from SURVEY.md sec. 8(c) readings
 * R1-R15 (listed in DESIGN.md); the R-number is quoted where it is used.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): K1 affine rows, K2 mass /
 * first moment, K3 adjoint identity, K4 dense brute force, K5 zero extension,
 * K6 kernel sums / DFT, K7 FFT vs direct sum, K9 Gaussian blob, K10 FBP ->
 * phantom, K11 half acquisition, K12 batch independence; for the TV-FISTA
 * part at the end of this file (tests/test_oracle_pins_fista.py): K13 TV closed
 * forms, K14 proximal step (limits, two-plateau closed form, optimality), K15
 * Lipschitz constant vs dense eigenvalue, K16 first iterates vs a dense matrix
 * and the O(1/k^2) bound, K17 energy value / regularisation / batch.
 * NOT pinned: the orientation conventions R1/R2 against PyHST2's own (no
 * reference output exists): "PyHST convention parity unpinned".
 *
 * No blocking, fusion or reordering: every sum runs in index order in double.
 * OpenMP only distributes independent outputs (pixels, rows) over threads.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_INVALID_ARG 1
#define ORACLE_ERR_NOMEM 3

static const double ORACLE_PI = 3.14159265358979323846264338327950288;

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* Tiny pin problems run faster on one thread than on a spinning team; results do not depend on
 * the thread count (OpenMP only distributes independent outputs). */
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ---- R8: spatial-domain band-limited ramp kernels, bin width 1 ------------
 * Ram-Lak     : h[0] = 1/4 ; h[n] = 0 (n even, n != 0) ; h[n] = -1/(pi^2 n^2) (n odd)
 * Shepp-Logan : h[n] = -2 / (pi^2 (4 n^2 - 1))
 * Hann (2), Hamming (3): the Ram-Lak ramp times the window a0 + 2 a1 cos(2 pi w), w in cycles per
 *   bin (|w| <= 1/2), (a0, a1) = (0.5, 0.25) resp. (0.54, 0.23); a cosine in frequency is a pair of
 *   unit shifts in space:  h_w[n] = a0 h[n] + a1 (h[n-1] + h[n+1])   (NEXT row N2: more windows)
 * (PAPER.md:L13, L63 only say "filtered back projection"; no formula given.) */
double oracle_ramp_kernel(int filter, int64_t n) {
  double dn = (double)n;
  if (filter == 2 || filter == 3) {
    const double a0 = filter == 2 ? 0.5 : 0.54, a1 = filter == 2 ? 0.25 : 0.23;
    return a0 * oracle_ramp_kernel(0, n) + a1 * (oracle_ramp_kernel(0, n - 1) + oracle_ramp_kernel(0, n + 1));
  }
  if (filter == 0) {
    if (n == 0) return 0.25;
    if ((n & 1) == 0) return 0.0;
    return -1.0 / (ORACLE_PI * ORACLE_PI * dn * dn);
  }
  return -2.0 / (ORACLE_PI * ORACLE_PI * (4.0 * dn * dn - 1.0));
}

/* ---- R10: half-acquisition overlap weights --------------------------------
 * s = b - cbar.  Axis right of the detector centre: omega = (B-1) - cbar,
 * w = 1 for s < -omega, w = (omega - s)/(2 omega) for |s| <= omega.
 * Axis left of centre: omega = cbar, mirrored.  w(s) + w(-s) = 1. */
int oracle_halfacq_weights(int32_t n_bins, double cbar, double* w) {
  double mid = 0.5 * (double)(n_bins - 1);
  int right = cbar >= mid;
  double omega = right ? (double)(n_bins - 1) - cbar : cbar;
  if (!(omega > 0.0)) return ORACLE_ERR_INVALID_ARG;
  for (int32_t b = 0; b < n_bins; ++b) {
    double s = (double)b - cbar;
    if (!right) s = -s;
    if (s < -omega) w[b] = 1.0;
    else if (s <= omega) w[b] = (omega - s) / (2.0 * omega);
    else w[b] = 0.0;
  }
  return ORACLE_OK;
}

/* Extended row length and left padding of the virtually doubled detector (R10):
 * far = max(cbar, B-1-cbar); B_ext = ceil(2 far) + 1 rounded up to a multiple
 * of 64; the physical row sits at pad_left = 0 (axis right of centre) or
 * pad_left = B_ext - B (axis left of centre). */
void oracle_halfacq_extent(int32_t n_bins, double cbar, int32_t* n_bins_ext, int32_t* pad_left) {
  double mid = 0.5 * (double)(n_bins - 1);
  double far = cbar >= mid ? cbar : (double)(n_bins - 1) - cbar;
  int64_t need = (int64_t)ceil(2.0 * far) + 1;
  if (need < n_bins) need = n_bins;
  int64_t ext = ((need + 63) / 64) * 64;
  *n_bins_ext = (int32_t)ext;
  *pad_left = cbar >= mid ? 0 : (int32_t)(ext - n_bins);
}

/* ---- FILTER (a1): direct linear convolution, O(B_in * B_out) per row -------
 * g[n] = sum_{m=0}^{B_in-1} h[n - pad_left - m] * w[m] * q[m],  0 <= n < B_out
 * in : float32 [n_rows][in_pitch], widened exactly.  w: float32 or NULL.
 * out: double [n_rows][n_bins_out]. */
int oracle_ramp_filter(const float* in, int64_t in_pitch, double* out, int64_t n_rows,
                       int32_t n_bins_in, int32_t n_bins_out, int32_t pad_left, int filter,
                       const float* col_weights) {
  if (!in || !out || n_rows < 0 || n_bins_in <= 0 || n_bins_out <= 0 || pad_left < 0 ||
      n_bins_out < n_bins_in + pad_left || filter < 0 || filter > 3)
    return ORACLE_ERR_INVALID_ARG;
  if (in_pitch == 0) in_pitch = n_bins_in;
  int64_t nh = (int64_t)n_bins_in + n_bins_out;         /* lags -(B_in-1) .. B_out-1 */
  double* h = (double*)malloc(sizeof(double) * (size_t)(2 * nh + 1));
  if (!h) return ORACLE_ERR_NOMEM;
  for (int64_t n = -nh; n <= nh; ++n) h[n + nh] = oracle_ramp_kernel(filter, n);
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < n_rows; ++r) {
    const float* q = in + r * in_pitch;
    double* g = out + r * (int64_t)n_bins_out;
    for (int32_t n = 0; n < n_bins_out; ++n) {
      double acc = 0.0;
      for (int32_t m = 0; m < n_bins_in; ++m) {
        double v = (double)q[m];
        if (col_weights) v = (double)col_weights[m] * v;
        acc += h[(int64_t)n - pad_left - m + nh] * v;
      }
      g[n] = acc;
    }
  }
  free(h);
  return ORACLE_OK;
}

/* ---- linear interpolation with per-tap zero extension (R5, R6, R7) --------
 * lerp(q,t) = (1-f) qz(k) + f qz(k+1), k = floor(t), f = t - k,
 * qz(b) = q[b] if 0 <= b < B else 0. */
static inline double lerp_zero_ext(const double* q, int32_t n_bins, double t) {
  double kf = floor(t);
  double f = t - kf;
  double a = 0.0, b = 0.0;
  if (kf >= 0.0 && kf < (double)n_bins) a = q[(int64_t)kf];
  if (kf + 1.0 >= 0.0 && kf + 1.0 < (double)n_bins) b = q[(int64_t)kf + 1];
  return (1.0 - f) * a + f * b;
}

/* Detector coordinate of pixel (i, j) in projection p (R1, R2, R3):
 * t = c_p + h * ((j - j0) cos(theta_p) + (i - i0) sin(theta_p)),
 * j0 = (nx-1)/2, i0 = (ny-1)/2; bin centres at integer coordinates. */
static inline double detector_coord(double c, double h, double ct, double st, double dj, double di) {
  return c + h * (dj * ct + di * st);
}

static int check_geom(int32_t n_slices, int32_t n_angles, int32_t n_bins, const double* angles,
                      const double* axis, int32_t nx, int32_t ny, double h) {
  if (n_slices <= 0 || n_angles <= 0 || n_bins <= 0 || nx <= 0 || ny <= 0 || !angles || !axis)
    return ORACLE_ERR_INVALID_ARG;
  if (!(h > 0.0) || !isfinite(h)) return ORACLE_ERR_INVALID_ARG;
  for (int32_t p = 0; p < n_angles; ++p)
    if (!isfinite(angles[p]) || !isfinite(axis[p])) return ORACLE_ERR_INVALID_ARG;
  return ORACLE_OK;
}

/* ---- BP (a2) on a double sinogram [S][P][pitch] ----------------------------
 * img[s,i,j] = scale * sum_{p=0}^{P-1} lerp(q[s,p,:], t_p(i,j)), sum in index order. */
int oracle_backproject_f64(const double* sino, int64_t pitch, double* img, int32_t n_slices,
                           int32_t n_angles, int32_t n_bins, const double* angles,
                           const double* axis, int32_t nx, int32_t ny, double h, double scale) {
  int rc = check_geom(n_slices, n_angles, n_bins, angles, axis, nx, ny, h);
  if (rc || !sino || !img) return rc ? rc : ORACLE_ERR_INVALID_ARG;
  if (pitch == 0) pitch = n_bins;
  double* ct = (double*)malloc(sizeof(double) * 2 * (size_t)n_angles);
  if (!ct) return ORACLE_ERR_NOMEM;
  double* st = ct + n_angles;
  for (int32_t p = 0; p < n_angles; ++p) { ct[p] = cos(angles[p]); st[p] = sin(angles[p]); }
  const double j0 = 0.5 * (double)(nx - 1), i0 = 0.5 * (double)(ny - 1);
#pragma omp parallel for collapse(2) schedule(static)
  for (int32_t s = 0; s < n_slices; ++s)
    for (int32_t i = 0; i < ny; ++i)
      for (int32_t j = 0; j < nx; ++j) {
        double acc = 0.0;
        for (int32_t p = 0; p < n_angles; ++p) {
          double t = detector_coord(axis[p], h, ct[p], st[p], (double)j - j0, (double)i - i0);
          acc += lerp_zero_ext(sino + ((int64_t)s * n_angles + p) * pitch, n_bins, t);
        }
        img[((int64_t)s * ny + i) * nx + j] = scale * acc;
      }
  free(ct);
  return ORACLE_OK;
}

/* Same definition evaluated only at the listed pixels (s,i,j); used for parity
 * at BASELINE.json's full sizes where the whole image would take hours. */
int oracle_backproject_points_f64(const double* sino, int64_t pitch, int32_t n_slices,
                                  int32_t n_angles, int32_t n_bins, const double* angles,
                                  const double* axis, int32_t nx, int32_t ny, double h,
                                  double scale, int64_t n_pts, const int32_t* ps,
                                  const int32_t* pi, const int32_t* pj, double* out) {
  int rc = check_geom(n_slices, n_angles, n_bins, angles, axis, nx, ny, h);
  if (rc || !sino || !out || n_pts < 0) return rc ? rc : ORACLE_ERR_INVALID_ARG;
  if (pitch == 0) pitch = n_bins;
  const double j0 = 0.5 * (double)(nx - 1), i0 = 0.5 * (double)(ny - 1);
  for (int64_t n = 0; n < n_pts; ++n)
    if (ps[n] < 0 || ps[n] >= n_slices || pi[n] < 0 || pi[n] >= ny || pj[n] < 0 || pj[n] >= nx)
      return ORACLE_ERR_INVALID_ARG;
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < n_pts; ++n) {
    double acc = 0.0;
    for (int32_t p = 0; p < n_angles; ++p) {
      double t = detector_coord(axis[p], h, cos(angles[p]), sin(angles[p]),
                                (double)pj[n] - j0, (double)pi[n] - i0);
      acc += lerp_zero_ext(sino + ((int64_t)ps[n] * n_angles + p) * pitch, n_bins, t);
    }
    out[n] = scale * acc;
  }
  return ORACLE_OK;
}

static double* widen_f32(const float* src, int64_t rows, int32_t cols, int64_t pitch) {
  double* d = (double*)malloc(sizeof(double) * (size_t)rows * (size_t)cols);
  if (!d) return NULL;
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < rows; ++r)
    for (int32_t c = 0; c < cols; ++c) d[r * cols + c] = (double)src[r * pitch + c];
  return d;
}

/* BP on the float32 sinogram the GPU gets, widened exactly. */
int oracle_backproject(const float* sino, int64_t pitch, double* img, int32_t n_slices,
                       int32_t n_angles, int32_t n_bins, const double* angles, const double* axis,
                       int32_t nx, int32_t ny, double h, double scale) {
  if (!sino || n_slices <= 0 || n_angles <= 0 || n_bins <= 0) return ORACLE_ERR_INVALID_ARG;
  if (pitch == 0) pitch = n_bins;
  double* d = widen_f32(sino, (int64_t)n_slices * n_angles, n_bins, pitch);
  if (!d) return ORACLE_ERR_NOMEM;
  int rc = oracle_backproject_f64(d, n_bins, img, n_slices, n_angles, n_bins, angles, axis, nx,
                                  ny, h, scale);
  free(d);
  return rc;
}

int oracle_backproject_points(const float* sino, int64_t pitch, int32_t n_slices, int32_t n_angles,
                              int32_t n_bins, const double* angles, const double* axis, int32_t nx,
                              int32_t ny, double h, double scale, int64_t n_pts, const int32_t* ps,
                              const int32_t* pi, const int32_t* pj, double* out) {
  if (!sino || n_slices <= 0 || n_angles <= 0 || n_bins <= 0) return ORACLE_ERR_INVALID_ARG;
  if (pitch == 0) pitch = n_bins;
  double* d = widen_f32(sino, (int64_t)n_slices * n_angles, n_bins, pitch);
  if (!d) return ORACLE_ERR_NOMEM;
  int rc = oracle_backproject_points_f64(d, n_bins, n_slices, n_angles, n_bins, angles, axis, nx,
                                         ny, h, scale, n_pts, ps, pi, pj, out);
  free(d);
  return rc;
}

/* ---- FP (a3): the exact transpose of BP, written as the scatter ------------
 * y[s,p,b] = scale * sum_{i,j} Lambda(t_p(i,j) - b) x[s,i,j], Lambda(u) = max(0, 1-|u|):
 * every pixel adds (1-f) x to y[k] and f x to y[k+1], bins outside [0,B) skipped (R6, R13).
 * Rows (s,p) are independent; within a row pixels are visited in (i,j) order. */
static void fp_row(const float* x, double* y, int32_t n_bins, double c, double h, double ct,
                   double st, int32_t nx, int32_t ny, double scale) {
  const double j0 = 0.5 * (double)(nx - 1), i0 = 0.5 * (double)(ny - 1);
  for (int32_t b = 0; b < n_bins; ++b) y[b] = 0.0;
  for (int32_t i = 0; i < ny; ++i)
    for (int32_t j = 0; j < nx; ++j) {
      double t = detector_coord(c, h, ct, st, (double)j - j0, (double)i - i0);
      double kf = floor(t);
      double f = t - kf;
      double v = (double)x[(int64_t)i * nx + j];
      if (kf >= 0.0 && kf < (double)n_bins) y[(int64_t)kf] += (1.0 - f) * v;
      if (kf + 1.0 >= 0.0 && kf + 1.0 < (double)n_bins) y[(int64_t)kf + 1] += f * v;
    }
  for (int32_t b = 0; b < n_bins; ++b) y[b] *= scale;
}

int oracle_forward_project(const float* img, double* sino, int32_t n_slices, int32_t n_angles,
                           int32_t n_bins, const double* angles, const double* axis, int32_t nx,
                           int32_t ny, double h, double scale) {
  int rc = check_geom(n_slices, n_angles, n_bins, angles, axis, nx, ny, h);
  if (rc || !img || !sino) return rc ? rc : ORACLE_ERR_INVALID_ARG;
#pragma omp parallel for collapse(2) schedule(static)
  for (int32_t s = 0; s < n_slices; ++s)
    for (int32_t p = 0; p < n_angles; ++p)
      fp_row(img + (int64_t)s * ny * nx, sino + ((int64_t)s * n_angles + p) * n_bins, n_bins,
             axis[p], h, cos(angles[p]), sin(angles[p]), nx, ny, scale);
  return ORACLE_OK;
}

/* Only the listed rows (s,p); out is [n_rows][n_bins]. */
int oracle_forward_project_rows(const float* img, int32_t n_slices, int32_t n_angles,
                                int32_t n_bins, const double* angles, const double* axis,
                                int32_t nx, int32_t ny, double h, double scale, int64_t n_rows,
                                const int32_t* rs, const int32_t* rp, double* out) {
  int rc = check_geom(n_slices, n_angles, n_bins, angles, axis, nx, ny, h);
  if (rc || !img || !out || n_rows < 0) return rc ? rc : ORACLE_ERR_INVALID_ARG;
  for (int64_t r = 0; r < n_rows; ++r)
    if (rs[r] < 0 || rs[r] >= n_slices || rp[r] < 0 || rp[r] >= n_angles)
      return ORACLE_ERR_INVALID_ARG;
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < n_rows; ++r)
    fp_row(img + (int64_t)rs[r] * ny * nx, out + r * n_bins, n_bins, axis[rp[r]], h,
           cos(angles[rp[r]]), sin(angles[rp[r]]), nx, ny, scale);
  return ORACLE_OK;
}

/* ---- FBP (a4) = FILTER then BP, all in double ------------------------------
 * mode 0 SCAN_180, 1 SCAN_360: scale = pi/P, rows filtered onto B_out = B.
 * mode 2 SCAN_360_HALF (R10): rows weighted by w (cbar = mean axis), filtered onto
 * the extended row (oracle_halfacq_extent), axis shifted by pad_left, scale = 2 pi/P.
 * If n_pts >= 0 only the listed pixels are evaluated into `out` (img may be NULL),
 * and only the slices that occur in ps[] are filtered. */
int oracle_fbp(const float* sino_raw, int64_t pitch, double* img, int32_t n_slices,
               int32_t n_angles, int32_t n_bins, const double* angles, const double* axis,
               int32_t nx, int32_t ny, double h, int filter, int mode, int64_t n_pts,
               const int32_t* ps, const int32_t* pi, const int32_t* pj, double* out) {
  int rc = check_geom(n_slices, n_angles, n_bins, angles, axis, nx, ny, h);
  if (rc || !sino_raw || mode < 0 || mode > 2) return rc ? rc : ORACLE_ERR_INVALID_ARG;
  if (pitch == 0) pitch = n_bins;
  int32_t b_out = n_bins, pad_left = 0;
  float* wf = NULL;
  double scale = ORACLE_PI / (double)n_angles;
  if (mode == 2) {
    double cbar = 0.0;
    for (int32_t p = 0; p < n_angles; ++p) cbar += axis[p];
    cbar /= (double)n_angles;
    double* w = (double*)malloc(sizeof(double) * (size_t)n_bins);
    wf = (float*)malloc(sizeof(float) * (size_t)n_bins);
    if (!w || !wf) { free(w); free(wf); return ORACLE_ERR_NOMEM; }
    rc = oracle_halfacq_weights(n_bins, cbar, w);
    if (rc) { free(w); free(wf); return rc; }
    /* the weights reach the filter as float32, as they do on the device */
    for (int32_t b = 0; b < n_bins; ++b) wf[b] = (float)w[b];
    free(w);
    oracle_halfacq_extent(n_bins, cbar, &b_out, &pad_left);
    scale = 2.0 * ORACLE_PI / (double)n_angles;
  }
  double* axis_out = (double*)malloc(sizeof(double) * (size_t)n_angles);
  double* filt = (double*)calloc((size_t)n_slices * (size_t)n_angles * (size_t)b_out, sizeof(double));
  if (!axis_out || !filt) { free(axis_out); free(filt); free(wf); return ORACLE_ERR_NOMEM; }
  for (int32_t p = 0; p < n_angles; ++p) axis_out[p] = axis[p] + (double)pad_left;
  for (int32_t s = 0; s < n_slices && !rc; ++s) {
    int used = n_pts < 0;
    for (int64_t n = 0; n < n_pts && !used; ++n) used = ps[n] == s;
    if (!used) continue;
    rc = oracle_ramp_filter(sino_raw + (int64_t)s * n_angles * pitch, pitch,
                            filt + (int64_t)s * n_angles * b_out, n_angles, n_bins, b_out,
                            pad_left, filter, wf);
  }
  if (!rc) {
    if (n_pts < 0)
      rc = oracle_backproject_f64(filt, b_out, img, n_slices, n_angles, b_out, angles, axis_out,
                                  nx, ny, h, scale);
    else
      rc = oracle_backproject_points_f64(filt, b_out, n_slices, n_angles, b_out, angles, axis_out,
                                         nx, ny, h, scale, n_pts, ps, pi, pj, out);
  }
  free(axis_out); free(filt); free(wf);
  return rc;
}

/* ============================================================================
 * NEXT row N1: TV-regularised FISTA
 * (sec. 3.1, eq. 1-3):  x = argmin 1/2 ||y - P x||^2 + beta TV(x),
 * TV(x) = sum_pixels sqrt((d1 x)^2 + (d2 x)^2)  (isotropic, eq. 2), solved by
 * FISTA (L84, ref. [18]); "the value of the energy in (3) is displayed" (L86).
 * The paper gives neither the discrete gradient, the inner solver of the TV
 * proximal step, the step size nor the starting point: readings R17-R20 of
 * DESIGN.md, quoted where used.  Everything below is double precision, index
 * order, no blocking; slices are independent (the operator is the same).
 * Pins: tests/test_oracle_pins.py K13-K17.
 * ========================================================================== */

/* FP of a double image (same scatter as fp_row; input not rounded to float). */
static void fp_row_f64(const double* x, double* y, int32_t n_bins, double c, double h, double ct,
                       double st, int32_t nx, int32_t ny, double scale) {
  const double j0 = 0.5 * (double)(nx - 1), i0 = 0.5 * (double)(ny - 1);
  for (int32_t b = 0; b < n_bins; ++b) y[b] = 0.0;
  for (int32_t i = 0; i < ny; ++i)
    for (int32_t j = 0; j < nx; ++j) {
      double t = detector_coord(c, h, ct, st, (double)j - j0, (double)i - i0);
      double kf = floor(t);
      double f = t - kf;
      double v = x[(int64_t)i * nx + j];
      if (kf >= 0.0 && kf < (double)n_bins) y[(int64_t)kf] += (1.0 - f) * v;
      if (kf + 1.0 >= 0.0 && kf + 1.0 < (double)n_bins) y[(int64_t)kf + 1] += f * v;
    }
  for (int32_t b = 0; b < n_bins; ++b) y[b] *= scale;
}

int oracle_forward_project_f64(const double* img, double* sino, int32_t n_slices, int32_t n_angles,
                               int32_t n_bins, const double* angles, const double* axis,
                               int32_t nx, int32_t ny, double h, double scale) {
  int rc = check_geom(n_slices, n_angles, n_bins, angles, axis, nx, ny, h);
  if (rc || !img || !sino) return rc ? rc : ORACLE_ERR_INVALID_ARG;
#pragma omp parallel for collapse(2) schedule(static)
  for (int32_t s = 0; s < n_slices; ++s)
    for (int32_t p = 0; p < n_angles; ++p)
      fp_row_f64(img + (int64_t)s * ny * nx, sino + ((int64_t)s * n_angles + p) * n_bins, n_bins,
                 axis[p], h, cos(angles[p]), sin(angles[p]), nx, ny, scale);
  return ORACLE_OK;
}

/* Discrete gradient (R18): forward differences, zero at the last column / row.
 *   (d1 x)[i,j] = x[i,j+1] - x[i,j] (j < nx-1), (d2 x)[i,j] = x[i+1,j] - x[i,j] (i < ny-1). */
static inline double d1_at(const double* x, int32_t nx, int32_t i, int32_t j) {
  return j + 1 < nx ? x[(int64_t)i * nx + j + 1] - x[(int64_t)i * nx + j] : 0.0;
}
static inline double d2_at(const double* x, int32_t nx, int32_t ny, int32_t i, int32_t j) {
  return i + 1 < ny ? x[(int64_t)(i + 1) * nx + j] - x[(int64_t)i * nx + j] : 0.0;
}

/* TV(x) of eq. 2, summed over all slices of the stack. */
double oracle_tv(const double* x, int32_t n_slices, int32_t ny, int32_t nx) {
  double tv = 0.0;
  for (int32_t s = 0; s < n_slices; ++s) {
    const double* xs = x + (int64_t)s * ny * nx;
    for (int32_t i = 0; i < ny; ++i)
      for (int32_t j = 0; j < nx; ++j) {
        double a = d1_at(xs, nx, i, j), b = d2_at(xs, nx, ny, i, j);
        tv += sqrt(a * a + b * b);
      }
  }
  return tv;
}

/* Adjoint of the gradient: (G^T p)[i,j] = p1[i,j-1] - p1[i,j] + p2[i-1,j] - p2[i,j]
 * with p1[i,-1] = p2[-1,j] = 0 and p1[i,nx-1] = p2[ny-1,j] = 0 (those components of
 * the gradient are identically zero). */
static inline double gt_at(const double* p1, const double* p2, int32_t nx, int32_t ny, int32_t i,
                           int32_t j) {
  double v = 0.0;
  if (j > 0) v += p1[(int64_t)i * nx + j - 1];
  if (j + 1 < nx) v -= p1[(int64_t)i * nx + j];
  if (i > 0) v += p2[(int64_t)(i - 1) * nx + j];
  if (i + 1 < ny) v -= p2[(int64_t)i * nx + j];
  return v;
}

/* Proximal operator of tau * TV (R18):  x = argmin_x 1/2 ||x - z||^2 + tau TV(x), per slice.
 * Dual form: x = z - tau G^T p with |p[i,j]| <= 1 (isotropic: the pair (p1, p2) of a pixel lies
 * in the unit disc).  n_inner projected-gradient steps on the dual (Chambolle 2004), step
 * 1 / (8 tau) (||G||^2 <= 8), started from p = 0:
 *     u = z - tau G^T p ;  q = p + G u / (8 tau) ;  p = q / max(1, |q|).
 * tau <= 0 or n_inner == 0 returns x = z. */
int oracle_prox_tv(const double* z, double* x, int32_t n_slices, int32_t ny, int32_t nx, double tau,
                   int32_t n_inner) {
  if (!z || !x || n_slices <= 0 || ny <= 0 || nx <= 0 || n_inner < 0) return ORACLE_ERR_INVALID_ARG;
  const int64_t n = (int64_t)ny * nx;
  if (!(tau > 0.0) || n_inner == 0) {
    memcpy(x, z, sizeof(double) * (size_t)(n * n_slices));
    return ORACLE_OK;
  }
  int rc = ORACLE_OK;
#pragma omp parallel for schedule(static)
  for (int32_t s = 0; s < n_slices; ++s) {
    const double* zs = z + s * n;
    double* u = x + s * n; /* the output doubles as u */
    double* p1 = (double*)calloc((size_t)(2 * n), sizeof(double));
    if (!p1) { rc = ORACLE_ERR_NOMEM; continue; }
    double* p2 = p1 + n;
    for (int32_t it = 0; it <= n_inner; ++it) {
      for (int32_t i = 0; i < ny; ++i)
        for (int32_t j = 0; j < nx; ++j)
          u[(int64_t)i * nx + j] = zs[(int64_t)i * nx + j] - tau * gt_at(p1, p2, nx, ny, i, j);
      if (it == n_inner) break; /* u = z - tau G^T p of the last dual iterate is the result */
      for (int32_t i = 0; i < ny; ++i)
        for (int32_t j = 0; j < nx; ++j) {
          double q1 = p1[(int64_t)i * nx + j] + d1_at(u, nx, i, j) / (8.0 * tau);
          double q2 = p2[(int64_t)i * nx + j] + d2_at(u, nx, ny, i, j) / (8.0 * tau);
          double m = sqrt(q1 * q1 + q2 * q2);
          if (m < 1.0) m = 1.0;
          p1[(int64_t)i * nx + j] = q1 / m;
          p2[(int64_t)i * nx + j] = q2 / m;
        }
    }
    free(p1);
  }
  return rc;
}

/* Lipschitz constant of the data term (R17): n_power iterations v <- P^T P v from v = 1 on ONE
 * slice (the operator is the same for every slice); returns 1.1 * ||v_n|| / ||v_{n-1}||
 * (the power iteration approaches lambda_max(P^T P) from below; FISTA needs L >= lambda_max). */
int oracle_lipschitz(int32_t n_angles, int32_t n_bins, const double* angles, const double* axis,
                     int32_t nx, int32_t ny, double h, int32_t n_power, double* L) {
  int rc = check_geom(1, n_angles, n_bins, angles, axis, nx, ny, h);
  if (rc || !L || n_power <= 0) return rc ? rc : ORACLE_ERR_INVALID_ARG;
  const int64_t n = (int64_t)ny * nx, m = (int64_t)n_angles * n_bins;
  double* v = (double*)malloc(sizeof(double) * (size_t)(2 * n + m));
  if (!v) return ORACLE_ERR_NOMEM;
  double* w = v + n;
  double* y = w + n;
  for (int64_t k = 0; k < n; ++k) v[k] = 1.0;
  double ratio = 0.0;
  for (int32_t it = 0; it < n_power && rc == ORACLE_OK; ++it) {
    double nv = 0.0, nw = 0.0;
    rc = oracle_forward_project_f64(v, y, 1, n_angles, n_bins, angles, axis, nx, ny, h, 1.0);
    if (!rc) rc = oracle_backproject_f64(y, n_bins, w, 1, n_angles, n_bins, angles, axis, nx, ny, h, 1.0);
    for (int64_t k = 0; k < n; ++k) { nv += v[k] * v[k]; nw += w[k] * w[k]; }
    ratio = sqrt(nw) / sqrt(nv);
    for (int64_t k = 0; k < n; ++k) v[k] = w[k] / sqrt(nw); /* normalised: no overflow */
  }
  *L = 1.1 * ratio;
  free(v);
  return rc;
}

/* FISTA for eq. 3 (Beck & Teboulle's scheme, ref. [18]; R19, R20):
 *   x_0 = y_0 = 0, t_0 = 1;   for k = 0 .. n_iter-1:
 *     r = P y_k - data ;  energy[k] = 1/2 ||r||^2 + beta TV(y_k)     (eq. 3 at the point where the
 *                                                                     gradient is taken: one P, P^T
 *                                                                     pair per iteration, R19)
 *     z = y_k - P^T r / L                                             (gradient of eq. 9's sign, R16)
 *     x_{k+1} = prox_{(beta/L) TV}(z)                                 (oracle_prox_tv, n_inner steps)
 *     t_{k+1} = (1 + sqrt(1 + 4 t_k^2)) / 2 ;  y_{k+1} = x_{k+1} + (t_k - 1)/t_{k+1} (x_{k+1} - x_k)
 * data: float32 [S][P][pitch] widened exactly; x_out = x_{n_iter} [S][ny][nx] in double; energy
 * (nullable) [n_iter], summed over the slices of the stack. */
int oracle_fista_tv(const float* data, int64_t pitch, double* x_out, int32_t n_slices,
                    int32_t n_angles, int32_t n_bins, const double* angles, const double* axis,
                    int32_t nx, int32_t ny, double h, double beta, double L, int32_t n_iter,
                    int32_t n_inner, double* energy) {
  int rc = check_geom(n_slices, n_angles, n_bins, angles, axis, nx, ny, h);
  if (rc || !data || !x_out || !(L > 0.0) || !(beta >= 0.0) || n_iter < 0 || n_inner < 0)
    return rc ? rc : ORACLE_ERR_INVALID_ARG;
  if (pitch == 0) pitch = n_bins;
  const int64_t n = (int64_t)n_slices * ny * nx, m = (int64_t)n_slices * n_angles * n_bins;
  double* xk = (double*)calloc((size_t)(4 * n + m), sizeof(double));
  if (!xk) return ORACLE_ERR_NOMEM;
  double* yk = xk + n;
  double* z = yk + n;
  double* g = z + n;
  double* r = g + n;
  double t = 1.0;
  for (int32_t k = 0; k < n_iter && rc == ORACLE_OK; ++k) {
    rc = oracle_forward_project_f64(yk, r, n_slices, n_angles, n_bins, angles, axis, nx, ny, h, 1.0);
    if (rc) break;
    double half = 0.0;
    for (int32_t s = 0; s < n_slices; ++s)
      for (int32_t p = 0; p < n_angles; ++p)
        for (int32_t b = 0; b < n_bins; ++b) {
          int64_t o = ((int64_t)s * n_angles + p) * n_bins + b;
          r[o] -= (double)data[((int64_t)s * n_angles + p) * pitch + b];
          half += r[o] * r[o];
        }
    if (energy) energy[k] = 0.5 * half + beta * oracle_tv(yk, n_slices, ny, nx);
    rc = oracle_backproject_f64(r, n_bins, g, n_slices, n_angles, n_bins, angles, axis, nx, ny, h, 1.0);
    if (rc) break;
    for (int64_t i = 0; i < n; ++i) z[i] = yk[i] - g[i] / L;
    rc = oracle_prox_tv(z, g, n_slices, ny, nx, beta / L, n_inner); /* g := x_{k+1} */
    if (rc) break;
    const double tn = 0.5 * (1.0 + sqrt(1.0 + 4.0 * t * t));
    const double mom = (t - 1.0) / tn;
    for (int64_t i = 0; i < n; ++i) {
      yk[i] = g[i] + mom * (g[i] - xk[i]);
      xk[i] = g[i];
    }
    t = tn;
  }
  memcpy(x_out, xk, sizeof(double) * (size_t)n);
  free(xk);
  return rc;
}
