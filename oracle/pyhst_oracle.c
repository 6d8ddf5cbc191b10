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
 * Cosine (4): the ramp times cos(pi w) = (e^{i pi w} + e^{-i pi w}) / 2, a pair of HALF-bin shifts of
 *   the continuous band-limited ramp  h(x) = int_{-1/2}^{1/2} |w| e^{2 pi i w x} dw
 *                                          = sin(pi x) / (2 pi x) + (cos(pi x) - 1) / (2 pi^2 x^2):
 *   h_c[n] = (h(n - 1/2) + h(n + 1/2)) / 2,  with  h(m + 1/2) = (-1)^m / (2 pi (m + 1/2)) - 1 / (2 pi^2 (m + 1/2)^2)
 * (PAPER.md:L13, L63 only say "filtered back projection"; no formula given.) */
static double ramp_at_half_integer(int64_t m) { /* h(m + 1/2) */
  double x = (double)m + 0.5;
  double sgn = (m & 1) ? -1.0 : 1.0;
  return sgn / (2.0 * ORACLE_PI * x) - 1.0 / (2.0 * ORACLE_PI * ORACLE_PI * x * x);
}

double oracle_ramp_kernel(int filter, int64_t n) {
  double dn = (double)n;
  if (filter == 4) return 0.5 * (ramp_at_half_integer(n - 1) + ramp_at_half_integer(n));
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
      n_bins_out < n_bins_in + pad_left || filter < 0 || filter > 4)
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
static int tv_solver(const float* data, int64_t pitch, double* x_out, int32_t n_slices,
                     int32_t n_angles, int32_t n_bins, const double* angles, const double* axis,
                     int32_t nx, int32_t ny, double h, double beta, double L, int32_t n_iter,
                     int32_t n_inner, double* energy, int accelerated) {
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
    const double mom = accelerated ? (t - 1.0) / tn : 0.0;   /* ISTA: y_{k+1} = x_{k+1} */
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

int oracle_fista_tv(const float* data, int64_t pitch, double* x_out, int32_t n_slices,
                    int32_t n_angles, int32_t n_bins, const double* angles, const double* axis,
                    int32_t nx, int32_t ny, double h, double beta, double L, int32_t n_iter,
                    int32_t n_inner, double* energy) {
  return tv_solver(data, pitch, x_out, n_slices, n_angles, n_bins, angles, axis, nx, ny, h, beta, L,
                   n_iter, n_inner, energy, 1);
}

/* ISTA ("ISTA ... or the accelerated FISTA ... can be used"): the same iteration
 * without the momentum, y_{k+1} = x_{k+1}; energy[k] is then eq. 3 at the iterate x_k itself and
 * does not increase from one iteration to the next (exact proximal step, L >= lambda_max). */
int oracle_ista_tv(const float* data, int64_t pitch, double* x_out, int32_t n_slices,
                   int32_t n_angles, int32_t n_bins, const double* angles, const double* axis,
                   int32_t nx, int32_t ny, double h, double beta, double L, int32_t n_iter,
                   int32_t n_inner, double* energy) {
  return tv_solver(data, pitch, x_out, n_slices, n_angles, n_bins, angles, axis, nx, ny, h, beta, L,
                   n_iter, n_inner, energy, 0);
}

/* ============================================================================
 * NEXT row N4: ring-artefact filter (sec. 2.3) and the
 * parameter-selection estimators of sec. 4 (L149-L162, eq. 10-11).
 * ========================================================================== */

/* Ring filter: "The filter reduces first the sinogram to a 1D signal by summing
 * over the projection-angles.  An high-frequencies filter is then applied in an attempt to
 * extract these features and the result is subtracted from the sinogram."  The optional model
 * (L61: "thresholding the bone in a first reconstructed slice.  The thresholded signal is then
 * subtracted to the data before application of the high-pass filter") is a sinogram of the same
 * shape -- the projection of the thresholded slice -- or NULL.  Readings R21, the
 * paper names neither the normalisation nor the high-pass filter:
 *   m[b]  = (1/P) sum_p (q[p,b] - model[p,b])          angular MEAN (a per-bin error e[b] that sits
 *                                                      in every row sums to P e[b])
 *   lp[b] = mean of m over the bins b-r .. b+r that exist (centred moving average, window
 *           clipped at the detector edges), r = half_width >= 1
 *   hp[b] = m[b] - lp[b] ;   out[p,b] = q[p,b] - hp[b]  for every projection p.
 * in: float32 [S][P][pitch]; out: double [S][P][B]. */
int oracle_ring_filter(const float* sino, const float* model, int64_t pitch, double* out,
                       int32_t n_slices, int32_t n_angles, int32_t n_bins, int32_t half_width) {
  if (!sino || !out || n_slices <= 0 || n_angles <= 0 || n_bins <= 0 || half_width < 1)
    return ORACLE_ERR_INVALID_ARG;
  if (pitch == 0) pitch = n_bins;
  int rc = ORACLE_OK;
#pragma omp parallel for schedule(static)
  for (int32_t s = 0; s < n_slices; ++s) {
    double* m = (double*)malloc(sizeof(double) * 2 * (size_t)n_bins);
    if (!m) { rc = ORACLE_ERR_NOMEM; continue; }
    double* hp = m + n_bins;
    for (int32_t b = 0; b < n_bins; ++b) {
      double acc = 0.0;
      for (int32_t p = 0; p < n_angles; ++p) {
        int64_t o = ((int64_t)s * n_angles + p) * pitch + b;
        acc += (double)sino[o] - (model ? (double)model[o] : 0.0);
      }
      m[b] = acc / (double)n_angles;
    }
    for (int32_t b = 0; b < n_bins; ++b) {
      int32_t lo = b - half_width < 0 ? 0 : b - half_width;
      int32_t hi = b + half_width > n_bins - 1 ? n_bins - 1 : b + half_width;
      double acc = 0.0;
      for (int32_t k = lo; k <= hi; ++k) acc += m[k];
      hp[b] = m[b] - acc / (double)(hi - lo + 1);
    }
    for (int32_t p = 0; p < n_angles; ++p)
      for (int32_t b = 0; b < n_bins; ++b)
        out[((int64_t)s * n_angles + p) * n_bins + b] =
            (double)sino[((int64_t)s * n_angles + p) * pitch + b] - hp[b];
    free(m);
  }
  return rc;
}

/* Decoherence estimator, eq. 11:
 *   E_cohe = Cos(I(beta) - I(0+), I(beta)) = <a - b, a> / (||a - b|| ||a||),  a = I(beta), b = I(0+),
 * one value per slice of the stacks a, b [S][n] (float32, widened exactly).  A zero norm gives 0. */
int oracle_ecohe(const float* a, const float* b, int32_t n_slices, int64_t n, double* out) {
  if (!a || !b || !out || n_slices <= 0 || n <= 0) return ORACLE_ERR_INVALID_ARG;
  for (int32_t s = 0; s < n_slices; ++s) {
    double dot = 0.0, nd = 0.0, na = 0.0;
    for (int64_t k = 0; k < n; ++k) {
      double av = (double)a[s * n + k], d = av - (double)b[s * n + k];
      dot += d * av;
      nd += d * d;
      na += av * av;
    }
    out[s] = (nd > 0.0 && na > 0.0) ? dot / (sqrt(nd) * sqrt(na)) : 0.0;
  }
  return ORACLE_OK;
}

/* Cross-validation estimator: "we reconstruct the slice using all the projections
 * except a selected one at a given angle.  Then we calculate the quadratic distance between the
 * reconstructed sample projection and the data for the excluded angle."  Given the reconstruction
 * x [S][ny][nx] (made without the excluded projections) and the excluded projections' geometry
 * (n_excl angles / axis positions) and data [S][n_excl][pitch]:
 *   out[s] = sum_{e < n_excl} sum_b ( (P x)[s,e,b] - data[s,e,b] )^2 . */
int oracle_cv_distance(const float* img, const float* data, int64_t pitch, int32_t n_slices,
                       int32_t n_excl, int32_t n_bins, const double* angles, const double* axis,
                       int32_t nx, int32_t ny, double h, double* out) {
  int rc = check_geom(n_slices, n_excl, n_bins, angles, axis, nx, ny, h);
  if (rc || !img || !data || !out) return rc ? rc : ORACLE_ERR_INVALID_ARG;
  if (pitch == 0) pitch = n_bins;
  double* y = (double*)malloc(sizeof(double) * (size_t)n_bins);
  if (!y) return ORACLE_ERR_NOMEM;
  for (int32_t s = 0; s < n_slices; ++s) {
    double acc = 0.0;
    for (int32_t e = 0; e < n_excl; ++e) {
      fp_row(img + (int64_t)s * ny * nx, y, n_bins, axis[e], h, cos(angles[e]), sin(angles[e]), nx, ny, 1.0);
      for (int32_t b = 0; b < n_bins; ++b) {
        double d = y[b] - (double)data[((int64_t)s * n_excl + e) * pitch + b];
        acc += d * d;
      }
    }
    out[s] = acc;
  }
  free(y);
  return ORACLE_OK;
}

/* ============================================================================
 * NEXT row N3: overlapping-patch dictionary reconstruction,
 * PAPER.md L102-L145 (sec. 3.2.1-3.2.2, eq. 4-9) and Algorithm 1 (L201-L228).
 *
 *   x_i = sum_p 1^c_p(i) sum_k w_kp phi_k(i - r_p)                                   (eq. 7)
 *   f(w) = || y - Pi x ||^2 + rho sum_{p,i} 1_p(i) (x_i - sum_k w_kp phi_k(i - r_p))^2   (eq. 8)
 *   F(w) = f(w) + beta ||w||_1, minimised by FISTA; "the L1 norm shrinking step is trivial" (L141)
 *
 * Matrices as in L145: D [Nc][m*m] (row k = basis function phi_k, row-major m x m), W [N][Nc],
 * P = W D [N][m*m] (row p = the patch p rebuilt from its coefficients), G [N][Nc].
 * Readings R16, R22-R24 of DESIGN.md (the paper gives no patch placement, tie-break, rho, m, Nc,
 * step size):
 *   R22 patches m x m on a regular grid of stride st (1 <= st <= m) that covers the image (eq. 4):
 *       origins oy[a] = min(a st, ny - m), a < na = ceil((ny - m)/st) + 1 (ox[b] likewise),
 *       patch index p = a nb + b, r_p = (oy[a], ox[b]), centre C_p = r_p + (m-1)/2;
 *       core map (eq. 5-6): C_j = the patch whose centre is closest to j in the L1 norm, the
 *       smallest p among equals; N_v(j) = number of patches that contain j.
 *   R16 the residual image is R = Pi^T (Pi x - y) (eq. 9), not Alg. 1's Bp(data - Fp(X));
 *       L226's garbled "P_{r_p+i}" is P_{p i}.
 *   R23 step 1/Lw, Lw = 1.1 x the power-iteration estimate of the largest eigenvalue of the
 *       Hessian of f (f is quadratic: grad f(w) = H w + g0; H v = grad f(v) evaluated with y = 0).
 *   R24 w_0 = 0, Beck-Teboulle momentum as R20; energy[k] = F(v_k) at the point v_k where the
 *       gradient of iteration k is taken.
 * One slice per call (slices are independent; the dictionary is shared).
 * ========================================================================== */

static int32_t patch_count_1d(int32_t n, int32_t m, int32_t st) {
  return n <= m ? 1 : (n - m + st - 1) / st + 1;
}
static int32_t patch_origin_1d(int32_t a, int32_t n, int32_t m, int32_t st) {
  int32_t o = a * st;
  return o > n - m ? n - m : o;
}

int oracle_patch_grid(int32_t ny, int32_t nx, int32_t m, int32_t st, int32_t* na, int32_t* nb) {
  if (ny < m || nx < m || m <= 0 || st <= 0 || st > m || !na || !nb) return ORACLE_ERR_INVALID_ARG;
  *na = patch_count_1d(ny, m, st);
  *nb = patch_count_1d(nx, m, st);
  return ORACLE_OK;
}

/* core[j] = C_j (eq. 5-6, brute force over all patches), cover[j] = N_v(j) (eq. 4). */
int oracle_patch_maps(int32_t ny, int32_t nx, int32_t m, int32_t st, int32_t* core, int32_t* cover) {
  int32_t na, nb;
  int rc = oracle_patch_grid(ny, nx, m, st, &na, &nb);
  if (rc || !core || !cover) return rc ? rc : ORACLE_ERR_INVALID_ARG;
  const double half = 0.5 * (double)(m - 1);
  for (int32_t iy = 0; iy < ny; ++iy)
    for (int32_t ix = 0; ix < nx; ++ix) {
      double best = 1e300;
      int32_t bestp = -1, nv = 0;
      for (int32_t a = 0; a < na; ++a)
        for (int32_t b = 0; b < nb; ++b) {
          int32_t oy = patch_origin_1d(a, ny, m, st), ox = patch_origin_1d(b, nx, m, st);
          if (iy >= oy && iy < oy + m && ix >= ox && ix < ox + m) ++nv;
          double d = fabs((double)iy - ((double)oy + half)) + fabs((double)ix - ((double)ox + half));
          if (d < best) { best = d; bestp = a * nb + b; }
        }
      core[(int64_t)iy * nx + ix] = bestp;
      cover[(int64_t)iy * nx + ix] = nv;
    }
  return ORACLE_OK;
}

/* Algorithm 1 in the paper's order.  W [N][Nc], D [Nc][m*m], data float32 [P][pitch] (one slice).
 * Outputs (each nullable): G [N][Nc] = grad f(W) (eq. 9), X [ny][nx] (eq. 7), *fval = f(W) (eq. 8). */
int oracle_patch_gradient(const double* W, const double* D, const float* data, int64_t pitch,
                          int32_t n_angles, int32_t n_bins, const double* angles, const double* axis,
                          int32_t nx, int32_t ny, double h, int32_t m, int32_t st, int32_t n_atoms,
                          double rho, double* G, double* X_out, double* fval) {
  int rc = check_geom(1, n_angles, n_bins, angles, axis, nx, ny, h);
  int32_t na, nb;
  if (!rc) rc = oracle_patch_grid(ny, nx, m, st, &na, &nb);
  if (rc || !W || !D || !data || n_atoms <= 0 || !(rho >= 0.0)) return rc ? rc : ORACLE_ERR_INVALID_ARG;
  if (pitch == 0) pitch = n_bins;
  const int64_t N = (int64_t)na * nb, mm = (int64_t)m * m, npix = (int64_t)ny * nx;
  const int64_t nsino = (int64_t)n_angles * n_bins;
  double* P = (double*)calloc((size_t)(2 * N * mm + 3 * npix + nsino), sizeof(double));
  int32_t* core = (int32_t*)malloc(sizeof(int32_t) * 2 * (size_t)npix);
  if (!P || !core) { free(P); free(core); return ORACLE_ERR_NOMEM; }
  double* Pp = P + N * mm;          /* P' */
  double* X = Pp + N * mm;
  double* R = X + npix;
  double* S = R + npix;
  double* r = S + npix;             /* residual sinogram */
  int32_t* cover = core + npix;
  oracle_patch_maps(ny, nx, m, st, core, cover);
  /* P <- W . D */
  for (int64_t p = 0; p < N; ++p)
    for (int64_t e = 0; e < mm; ++e) {
      double acc = 0.0;
      for (int32_t k = 0; k < n_atoms; ++k) acc += W[p * n_atoms + k] * D[(int64_t)k * mm + e];
      P[p * mm + e] = acc;
    }
  /* for all image positions j: p <- C_j; i <- j - r_p; X_j <- P_{p i} */
  for (int32_t jy = 0; jy < ny; ++jy)
    for (int32_t jx = 0; jx < nx; ++jx) {
      int32_t p = core[(int64_t)jy * nx + jx];
      int32_t oy = patch_origin_1d(p / nb, ny, m, st), ox = patch_origin_1d(p % nb, nx, m, st);
      X[(int64_t)jy * nx + jx] = P[(int64_t)p * mm + (int64_t)(jy - oy) * m + (jx - ox)];
    }
  /* R = Pi^T (Pi X - data)   (R16: the sign of eq. 9) */
  rc = oracle_forward_project_f64(X, r, 1, n_angles, n_bins, angles, axis, nx, ny, h, 1.0);
  double fid = 0.0;
  for (int32_t p = 0; p < n_angles && !rc; ++p)
    for (int32_t b = 0; b < n_bins; ++b) {
      r[(int64_t)p * n_bins + b] -= (double)data[(int64_t)p * pitch + b];
      fid += r[(int64_t)p * n_bins + b] * r[(int64_t)p * n_bins + b];
    }
  if (!rc) rc = oracle_backproject_f64(r, n_bins, R, 1, n_angles, n_bins, angles, axis, nx, ny, h, 1.0);
  /* S <- sum of all the patches covering each pixel; similarity term of eq. 8 */
  double sim = 0.0;
  for (int64_t p = 0; p < N; ++p) {
    int32_t oy = patch_origin_1d((int32_t)(p / nb), ny, m, st), ox = patch_origin_1d((int32_t)(p % nb), nx, m, st);
    for (int32_t iy = 0; iy < m; ++iy)
      for (int32_t ix = 0; ix < m; ++ix) {
        int64_t j = (int64_t)(oy + iy) * nx + (ox + ix);
        double v = P[p * mm + (int64_t)iy * m + ix];
        S[j] += v;
        sim += (X[j] - v) * (X[j] - v);
      }
  }
  /* P' per Algorithm 1 */
  for (int64_t p = 0; p < N; ++p) {
    int32_t oy = patch_origin_1d((int32_t)(p / nb), ny, m, st), ox = patch_origin_1d((int32_t)(p % nb), nx, m, st);
    for (int32_t iy = 0; iy < m; ++iy)
      for (int32_t ix = 0; ix < m; ++ix) {
        int64_t j = (int64_t)(oy + iy) * nx + (ox + ix), e = (int64_t)iy * m + ix;
        double v = 0.0;
        if (core[j] == (int32_t)p) v += R[j] + rho * ((double)cover[j] * X[j] - S[j]);
        v += rho * (P[p * mm + e] - X[j]);
        Pp[p * mm + e] = v;
      }
  }
  /* G <- 2 P' . D^T */
  if (G)
    for (int64_t p = 0; p < N; ++p)
      for (int32_t k = 0; k < n_atoms; ++k) {
        double acc = 0.0;
        for (int64_t e = 0; e < mm; ++e) acc += Pp[p * mm + e] * D[(int64_t)k * mm + e];
        G[p * n_atoms + k] = 2.0 * acc;
      }
  if (X_out) memcpy(X_out, X, sizeof(double) * (size_t)npix);
  if (fval) *fval = fid + rho * sim;
  free(P); free(core);
  return rc;
}

/* "the L1 norm shrinking step is trivial" (L141): soft threshold sign(v) max(|v| - t, 0). */
void oracle_soft_threshold(const double* v, int64_t n, double t, double* out) {
  for (int64_t k = 0; k < n; ++k) {
    double a = fabs(v[k]) - t;
    out[k] = a > 0.0 ? (v[k] > 0.0 ? a : -a) : 0.0;
  }
}

/* R23: Lw = 1.1 ||H v_n|| / ||v_n|| after n_power iterations v <- H v / ||H v|| from v = 1, where
 * H v = grad f(v) with zero data (f is quadratic in w). */
int oracle_patch_lipschitz(const double* D, int32_t n_angles, int32_t n_bins, const double* angles,
                           const double* axis, int32_t nx, int32_t ny, double h, int32_t m, int32_t st,
                           int32_t n_atoms, double rho, int32_t n_power, double* Lw) {
  int32_t na, nb;
  int rc = oracle_patch_grid(ny, nx, m, st, &na, &nb);
  if (rc || !Lw || n_power <= 0) return rc ? rc : ORACLE_ERR_INVALID_ARG;
  const int64_t n = (int64_t)na * nb * n_atoms;
  double* v = (double*)malloc(sizeof(double) * 2 * (size_t)n);
  float* zero = (float*)calloc((size_t)n_angles * (size_t)n_bins, sizeof(float));
  if (!v || !zero) { free(v); free(zero); return ORACLE_ERR_NOMEM; }
  double* g = v + n;
  for (int64_t k = 0; k < n; ++k) v[k] = 1.0;
  double ratio = 0.0;
  for (int32_t it = 0; it < n_power && !rc; ++it) {
    rc = oracle_patch_gradient(v, D, zero, n_bins, n_angles, n_bins, angles, axis, nx, ny, h, m, st,
                               n_atoms, rho, g, NULL, NULL);
    double nv = 0.0, ng = 0.0;
    for (int64_t k = 0; k < n; ++k) { nv += v[k] * v[k]; ng += g[k] * g[k]; }
    ratio = sqrt(ng) / sqrt(nv);
    for (int64_t k = 0; k < n; ++k) v[k] = g[k] / sqrt(ng);
  }
  *Lw = 1.1 * ratio;
  free(v); free(zero);
  return rc;
}

/* FISTA on the coefficients (L139-L141; R23, R24):
 *   w_0 = v_0 = 0, t_0 = 1;  for k < n_iter:
 *     G = grad f(v_k) (Algorithm 1);  energy[k] = f(v_k) + beta ||v_k||_1
 *     w_{k+1} = shrink(v_k - G / Lw, beta / Lw);  momentum as R20.
 * W_out [N][Nc] = w_{n_iter}; X_out [ny][nx] = the image of eq. 7 at w_{n_iter} (nullable). */
int oracle_patch_fista(const double* D, const float* data, int64_t pitch, int32_t n_angles,
                       int32_t n_bins, const double* angles, const double* axis, int32_t nx, int32_t ny,
                       double h, int32_t m, int32_t st, int32_t n_atoms, double rho, double beta,
                       double Lw, int32_t n_iter, double* W_out, double* X_out, double* energy) {
  int32_t na, nb;
  int rc = oracle_patch_grid(ny, nx, m, st, &na, &nb);
  if (rc || !D || !data || !W_out || !(Lw > 0.0) || !(beta >= 0.0) || n_iter < 0)
    return rc ? rc : ORACLE_ERR_INVALID_ARG;
  const int64_t n = (int64_t)na * nb * n_atoms;
  double* w = (double*)calloc((size_t)(4 * n), sizeof(double));
  if (!w) return ORACLE_ERR_NOMEM;
  double* v = w + n;
  double* g = v + n;
  double* wn = g + n;
  double t = 1.0;
  for (int32_t k = 0; k < n_iter && !rc; ++k) {
    double f = 0.0, l1 = 0.0;
    rc = oracle_patch_gradient(v, D, data, pitch, n_angles, n_bins, angles, axis, nx, ny, h, m, st,
                               n_atoms, rho, g, NULL, &f);
    if (rc) break;
    for (int64_t i = 0; i < n; ++i) l1 += fabs(v[i]);
    if (energy) energy[k] = f + beta * l1;
    for (int64_t i = 0; i < n; ++i) g[i] = v[i] - g[i] / Lw;
    oracle_soft_threshold(g, n, beta / Lw, wn);
    const double tn = 0.5 * (1.0 + sqrt(1.0 + 4.0 * t * t));
    const double mom = (t - 1.0) / tn;
    for (int64_t i = 0; i < n; ++i) {
      v[i] = wn[i] + mom * (wn[i] - w[i]);
      w[i] = wn[i];
    }
    t = tn;
  }
  memcpy(W_out, w, sizeof(double) * (size_t)n);
  if (!rc && X_out) {
    float* zero = (float*)calloc((size_t)n_angles * (size_t)n_bins, sizeof(float));
    if (!zero) rc = ORACLE_ERR_NOMEM;
    else rc = oracle_patch_gradient(w, D, zero, n_bins, n_angles, n_bins, angles, axis, nx, ny, h, m,
                                    st, n_atoms, rho, NULL, X_out, NULL);
    free(zero);
  }
  free(w);
  return rc;
}
