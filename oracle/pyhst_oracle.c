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
 * phantom, K11 half acquisition, K12 batch independence.
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

/* ---- R8: spatial-domain band-limited ramp kernels, bin width 1 ------------
 * Ram-Lak     : h[0] = 1/4 ; h[n] = 0 (n even, n != 0) ; h[n] = -1/(pi^2 n^2) (n odd)
 * Shepp-Logan : h[n] = -2 / (pi^2 (4 n^2 - 1))
 * (PAPER.md:L13, L63 only say "filtered back projection"; no formula given.) */
double oracle_ramp_kernel(int filter, int64_t n) {
  double dn = (double)n;
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
      n_bins_out < n_bins_in + pad_left || (filter != 0 && filter != 1))
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
