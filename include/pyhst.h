/*
 * pyhst.h -- C ABI of the B200-native (sm_100a) hot path of PyHST2 (arxiv/paper_1306_1392):
 * ramp filter -> parallel-beam pixel-driven backprojection (linear detector interpolation,
 * per-projection rotation-axis position, optional 360-degree half-acquisition field
 * doubling) and its exactly matched adjoint forward projector.
 *
 * Conventions shared by every entry point
 * ---------------------------------------
 * - extern "C", plain pointers and sizes, int status returned, never throws, never exits.
 * - `d_*` pointers are DEVICE pointers owned by the caller (4-byte aligned); `h_*` pointers
 *   and the arrays inside pyhst_geom_t are HOST pointers that need only live for the duration
 *   of the call (the library copies them).
 * - Work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = default stream) of the
 *   CURRENT device.  Errors detectable at enqueue time are returned, asynchronous faults surface
 *   at the caller's next sync.  The *_host entry points synchronise `stream` before returning.
 * - Concurrency rule: ONE CALL IN FLIGHT PER DEVICE.  All library state (workspace, plans, geometry
 *   tables) is kept per device and shared by that device's calls, so the library serialises them:
 *   entry points may be called from any thread and on any stream, but a call takes the device's
 *   lock while it enqueues, and a call on another stream than the previous one first makes its
 *   stream wait (cudaStreamWaitEvent, on the device, no host block) for the previous call's work.
 *   Calls on one stream cost nothing extra.  Different devices are independent.
 * - Synchronisation: in steady state (same shapes as an earlier call) the d_* entry points only
 *   enqueue.  The FIRST call with a new shape, filter or geometry builds plans and may grow the
 *   workspace: cudaMalloc / cudaFree of a grown block, one-time cuFFT plan creation and the
 *   one-time ramp-spectrum set-up synchronise the device or `stream`.  Warm the shapes up once
 *   (one call per shape) before a latency-critical loop or a CUDA-graph capture.
 * - Internal workspace (filtered sinogram, filter spectra, per-projection geometry tables)
 *   lives in a per-device cache keyed by shapes; pyhst_release_cache() frees it on every device.
 * - There is no CPU fallback: a missing/non-sm_100 device yields PYHST_ERR_UNSUPPORTED.
 * - On any error nothing is written to the output buffers and pyhst_last_error() describes it.
 *
 * Geometry (paper: sec. 2.1 "rotation axis displacement and the angular position
 * can be given in input, as a function of the projection"; L59 one sinogram per slice;
 * readings R1-R3, R14 of DESIGN.md):
 *   sinogram stack  q[s][p][b]   s < n_slices, p < n_angles, b < n_bins (C order, row pitch
 *                                sino_pitch floats), float32
 *   image stack     x[s][i][j]   i < ny (rows, y), j < nx (columns, x), C order, float32
 *   detector coordinate of pixel (i,j) in projection p (bin centres at integers):
 *     t_p(i,j) = axis_pos[p] + pixel_size * ((j - (nx-1)/2) cos(angles_rad[p])
 *                                          + (i - (ny-1)/2) sin(angles_rad[p]))
 */
#ifndef PYHST_H_
#define PYHST_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  PYHST_OK = 0,
  PYHST_ERR_INVALID_ARG = 1,
  PYHST_ERR_UNSUPPORTED = 2,
  PYHST_ERR_NOMEM = 3,
  PYHST_ERR_CUDA = 4
};

/* Band-limited ramp kernels, bin width 1 (reading R8; PAPER.md:L13, L63 give no formula):
 *   Ram-Lak     h[0] = 1/4, h[n odd] = -1/(pi^2 n^2), h[n even != 0] = 0
 *   Shepp-Logan h[n] = -2 / (pi^2 (4 n^2 - 1))
 *   Hann, Hamming (NEXT row N2): Ram-Lak times the window a0 + 2 a1 cos(2 pi w), w in cycles per
 *               bin, (a0, a1) = (0.5, 0.25) resp. (0.54, 0.23): h_w[n] = a0 h[n] + a1 (h[n-1] + h[n+1])
 *   Cosine      Ram-Lak times cos(pi w): a pair of half-bin shifts of the continuous band-limited ramp,
 *               h_c[n] = (h(n-1/2) + h(n+1/2)) / 2,  h(m+1/2) = (-1)^m / (2 pi (m+1/2)) - 1 / (2 pi^2 (m+1/2)^2)
 *               (reading R8c; h_c[0] = 1/pi - 2/pi^2) */
typedef enum { PYHST_FILTER_RAMLAK = 0, PYHST_FILTER_SHEPP_LOGAN = 1, PYHST_FILTER_HANN = 2,
               PYHST_FILTER_HAMMING = 3, PYHST_FILTER_COSINE = 4 } pyhst_filter_t;

/* >= 180 degrees; with 360 degrees and the axis near the detector border the
 * detector "can be virtually doubled" (PYHST_SCAN_360_HALF, reading R10). */
typedef enum { PYHST_SCAN_180 = 0, PYHST_SCAN_360 = 1, PYHST_SCAN_360_HALF = 2 } pyhst_scan_t;

typedef struct {
  int32_t n_slices, n_angles, n_bins; /* sinogram stack [n_slices][n_angles][n_bins], C order */
  int64_t sino_pitch;                 /* floats between rows; 0 => n_bins (contiguous)        */
  const double* angles_rad;           /* HOST, [n_angles]                                     */
  const double* axis_pos;             /* HOST, [n_angles], bin coordinate of the rotation axis */
  int32_t nx, ny;                     /* output slice size; image [n_slices][ny][nx], C order */
  double pixel_size;                  /* in detector-bin units, > 0                            */
} pyhst_geom_t;

/* a1 -- ramp filter ("filtered back projection"; readings R8, R9).
 * For each of n_rows rows:  out[n] = sum_{m<n_bins_in} h[n - pad_left - m] * w[m] * in[m],
 * 0 <= n < n_bins_out: the exact LINEAR convolution of the (optionally column-weighted) row,
 * zero-extended, with the kernel `f`; evaluated with a zero-padded FFT of length
 * >= n_bins_in + n_bins_out.
 *   d_in   [n_rows][n_bins_in]  float32, contiguous            (device, read)
 *   d_out  [n_rows][out_pitch]  float32; columns >= n_bins_out are not touched
 *                               (device, written; out_pitch 0 => n_bins_out; may not alias d_in)
 *   d_col_weights  [n_bins_in] float32 or NULL (= all ones)    (device, read)
 * Errors: null pointers, n_rows < 0, sizes <= 0, pad_left < 0, n_bins_out < n_bins_in +
 * pad_left, out_pitch < n_bins_out, n_bins_in + n_bins_out > 16384 -> INVALID_ARG /
 * UNSUPPORTED.  n_rows == 0 is a no-op. */
int pyhst_ramp_filter(const float* d_in, float* d_out, int64_t n_rows, int32_t n_bins_in,
                      int32_t n_bins_out, int32_t pad_left, int64_t out_pitch, pyhst_filter_t f,
                      const float* d_col_weights, void* stream);

/* a2 -- backprojection P^T ("Each tile is reconstructed by a block of threads.
 * The values to be back-projected are read ... using ... interpolation"; L71 P^T; R4-R7):
 *   d_img[s][i][j] = scale * sum_p lerp(q[s][p][:], t_p(i,j)),
 *   lerp(q,t) = (1-f) qz(k) + f qz(k+1), k = floor(t), f = t - k, qz = q zero-extended
 *   outside [0, n_bins) per tap.  FP32 FMA arithmetic, geometry bases in double.
 *   d_sino  [n_slices][n_angles][sino_pitch] float32 (device, read)
 *   d_img   [n_slices][ny][nx]               float32 (device, overwritten)
 * Errors: null pointers, sizes <= 0, pixel_size <= 0 or non-finite, non-finite angle/axis,
 * sino_pitch != 0 and < n_bins -> INVALID_ARG. */
int pyhst_backproject(const float* d_sino, float* d_img, const pyhst_geom_t* g, float scale,
                      void* stream);

/* a3 -- forward projection P, the exact transpose of a2 (eq. 1; L211
 * Alg. 1 "Fp"; reading R13):
 *   d_sino[s][p][b] = scale * sum_{i,j} Lambda(t_p(i,j) - b) * x[s][i][j],
 *   Lambda(u) = max(0, 1 - |u|).  Computed as a gather over detector bins (no atomics), so
 *   <P x, y> = <x, P^T y> holds up to FP32 rounding for the same `g`.
 *   d_img   [n_slices][ny][nx]               float32 (device, read)
 *   d_sino  [n_slices][n_angles][sino_pitch] float32 (device, columns < n_bins overwritten)
 * Workspace (cached per device, released by pyhst_release_cache): the diagonal-line kernel, which the library
 * chooses for dense angle lists, keeps two sheared copies of the image stack,
 *   2 * ceil(n_slices / 4) * (nx + ny + 7) lines * (nx + 392) * 16 bytes
 * -- about 4.8x the stack: 1.3 GB for 16 slices of 2048^2, 7.7 GB for 64 slices of 2560^2.  The banded kernel
 * (sparse lists, or when that block cannot be allocated: the library then falls back to it by itself) keeps
 * about 2x the stack.  Stacks too large for either are projected in slice chunks by the caller
 * (pyhst_forward_project_host does so). */
int pyhst_forward_project(const float* d_img, float* d_sino, const pyhst_geom_t* g, float scale,
                          void* stream);

/* a4 -- FBP = a1 then a2 (readings R8-R10):
 *   PYHST_SCAN_180 / PYHST_SCAN_360 : rows filtered onto n_bins, scale = pi / n_angles.
 *   PYHST_SCAN_360_HALF: rows weighted by the overlap ramp w (R10; cbar = mean axis position),
 *     filtered onto the virtually doubled row of pyhst_halfacq_extent(), axis shifted by
 *     pad_left, all projections backprojected with scale = 2 pi / n_angles.
 *   d_sino_raw [n_slices][n_angles][sino_pitch] float32 (device, read)
 *   d_img      [n_slices][ny][nx] float32 (device, overwritten)                            */
int pyhst_fbp(const float* d_sino_raw, float* d_img, const pyhst_geom_t* g, pyhst_filter_t f,
              pyhst_scan_t mode, void* stream);

/* Same as pyhst_fbp with HOST buffers (pinned or pageable): the stack is processed in slice
 * chunks, host->device copy of chunk n+1 and device->host copy of chunk n-1 overlapping the
 * kernels of chunk n (three internal streams, ordered after `stream`).  Synchronises before
 * returning.  max_slices_per_chunk <= 0 lets the library choose. */
int pyhst_fbp_host(const float* h_sino_raw, float* h_img, const pyhst_geom_t* g,
                   pyhst_filter_t f, pyhst_scan_t mode, int32_t max_slices_per_chunk,
                   void* stream);

/* a2 / a3 with HOST buffers, same chunked pipeline and synchronisation as pyhst_fbp_host.
 * With sino_pitch > n_bins the padding columns of h_sino travel too (forward projection leaves
 * them unspecified). */
int pyhst_backproject_host(const float* h_sino, float* h_img, const pyhst_geom_t* g, float scale,
                           int32_t max_slices_per_chunk, void* stream);
int pyhst_forward_project_host(const float* h_img, float* h_sino, const pyhst_geom_t* g, float scale,
                               int32_t max_slices_per_chunk, void* stream);

/* NEXT row N1: TV-regularised FISTA, PAPER.md L73-L86 (sec. 3.1, eq. 1-3):
 *     x = argmin 1/2 ||data - P x||^2 + beta TV(x),  TV = isotropic total variation (eq. 2),
 * solved by FISTA (L84, ref. [18]) with P = pyhst_forward_project and P^T = pyhst_backproject
 * (scale 1), one pair per iteration.  Readings R16-R20 of DESIGN.md: gradient P^T (P y - data);
 * step 1/L with L = 1.1 x the estimate of lambda_max(P^T P) after n_power power iterations from
 * v = 1 on one slice; TV proximal step by n_inner projected-gradient steps on the dual (forward
 * differences, zero at the last row / column, step 1/8, dual restarted at zero every outer
 * iteration); x0 = 0; energy[k] = eq. 3 evaluated at the point y_k where the gradient of
 * iteration k is taken, summed over the slices of the stack.
 *   d_data   DEVICE [n_slices][n_angles][sino_pitch] f32, read only
 *   d_img    DEVICE [n_slices][ny][nx] f32, overwritten with x after n_iter iterations
 *   energy   HOST [n_iter] or NULL;  lipschitz HOST scalar or NULL.  If either is given the call
 *            copies them back and synchronises `stream` before returning; otherwise it only enqueues.
 * Errors: null pointers, beta < 0 or not finite, n_iter < 0, n_inner < 0, n_power <= 0 ->
 * PYHST_ERR_INVALID_ARG; no sm_100 device -> PYHST_ERR_UNSUPPORTED.  Workspace (7 image stacks +
 * one sinogram stack) is owned by the library and freed by pyhst_release_cache(). */
int pyhst_fista_tv(const float* d_data, float* d_img, const pyhst_geom_t* g, float beta,
                   int32_t n_iter, int32_t n_inner, int32_t n_power, double* energy,
                   double* lipschitz, void* stream);

/* ISTA ("ISTA ... or the accelerated FISTA ... can be used"): pyhst_fista_tv without
 * the momentum (y_{k+1} = x_{k+1}); same arguments, workspace and errors.  energy[k] is then eq. 3
 * at the iterate x_k itself and does not increase from one iteration to the next. */
int pyhst_ista_tv(const float* d_data, float* d_img, const pyhst_geom_t* g, float beta,
                  int32_t n_iter, int32_t n_inner, int32_t n_power, double* energy,
                  double* lipschitz, void* stream);

/* NEXT row N4 -- ring-artefact filter (sec. 2.3: "The filter reduces first the sinogram
 * to a 1D signal by summing over the projection-angles.  An high-frequencies filter is then applied in
 * an attempt to extract these features and the result is subtracted from the sinogram"; reading R21):
 *   m[s][b]  = (1/P) sum_p (sino[s][p][b] - model[s][p][b])       angular mean, per slice
 *   hp[s][b] = m[s][b] - mean of m[s] over the bins b-r .. b+r that exist    (r = half_width >= 1)
 *   out[s][p][b] = sino[s][p][b] - hp[s][b]                        for every projection p
 *   d_sino   DEVICE [n_slices][n_angles][pitch] f32, read
 *   d_model  DEVICE, same layout, or NULL (= 0): the projection of the thresholded first reconstruction
 *            (L61: "thresholding the bone ... The thresholded signal is then subtracted to the data
 *            before application of the high-pass filter")
 *   d_out    DEVICE, same layout, written; may be d_sino itself (in place)
 * pitch 0 => n_bins.  Errors: null pointers, sizes <= 0, half_width < 1, pitch < n_bins -> INVALID_ARG. */
int pyhst_ring_filter(const float* d_sino, const float* d_model, float* d_out, int32_t n_slices,
                      int32_t n_angles, int32_t n_bins, int64_t pitch, int32_t half_width, void* stream);

/* The same ring filter for callers that cannot let the library allocate device memory.
 *
 * pyhst_ring_filter keeps two intermediates in the library's grow-on-demand workspace: the per-chunk
 * column sums (double [n_slices][<= 32][n_bins]) and the high-pass row (float [n_slices][n_bins]).  Its first
 * call with a new shape therefore runs cudaMalloc (and cudaFree of the outgrown block), which synchronises
 * the device and can fail.  That rules it out for code running where allocation is forbidden or impossible:
 * a host application that has carved the whole device memory up in advance into pools of its own (nothing
 * is left for a library to claim), a latency-bound acquisition loop in which the device-wide
 * synchronisation of cudaMalloc / cudaFree is not acceptable, or a process that has to keep correcting
 * sinograms after the device ran out of memory.
 *
 * pyhst_ring_filter_static computes exactly the same result with exactly the same kernels, in the same
 * summation order (bit-identical output), but keeps the two intermediates in a fixed array compiled into
 * the library.  It calls no cudaMalloc / cudaFree / cudaMallocAsync, creates no stream, event or plan, and
 * uses none of the library's cached workspace; the caller supplies the input and output buffers as before.
 *
 * Limit and cost: n_slices * n_bins <= PYHST_RING_STATIC_MAX_CELLS (32768 -- e.g. 16 slices of 2048 bins,
 * any number of projections).  Larger requests are refused with PYHST_ERR_UNSUPPORTED and an explanatory
 * pyhst_last_error(); split the stack by slices (slices are independent).  The array takes
 * 32768 * (32 * 8 + 4) = 8 519 680 bytes of device memory on EVERY GPU on which this library is loaded,
 * from load until the process exits, whether or not this entry point is ever called.
 *
 * First call on a device: it looks the array's device address up (cudaGetSymbolAddress) and raises the
 * shared-memory limit of one kernel (cudaFuncSetAttribute), with that device current.  Neither allocates,
 * but make this first call once per device during set-up, and before any stream capture is started.  Every
 * later call only enqueues three kernels on `stream`.
 *
 * Sharing: all calls on one device use the same array, and it is NOT covered by the library's
 * one-call-in-flight serialisation.  Two calls whose kernels can overlap on the GPU (different streams
 * without an ordering between them, or different host threads on different streams) race on it and give
 * wrong results; order them on one stream or with events.  The array keeps whatever the last call wrote;
 * nothing in it needs to start at zero, because each call writes every element before reading it.
 * Arguments, layouts and the remaining errors are those of pyhst_ring_filter (d_out may be d_sino). */
#define PYHST_RING_STATIC_MAX_CELLS 32768
int pyhst_ring_filter_static(const float* d_sino, const float* d_model, float* d_out, int32_t n_slices,
                             int32_t n_angles, int32_t n_bins, int64_t pitch, int32_t half_width, void* stream);

/* NEXT row N4 -- decoherence-maximising estimator, eq. 11:
 *   E_cohe[s] = Cos(I(beta) - I(0+), I(beta)) = <a - b, a> / (||a - b|| ||a||),  a = d_img_beta[s], b = d_img_0[s]
 * one fused pass over the two stacks, sums in double, fixed summation order (deterministic).
 *   d_img_beta, d_img_0  DEVICE [n_slices][n_per_slice] f32, read
 *   h_out                HOST [n_slices]; the call synchronises `stream`.  A zero norm gives 0. */
int pyhst_ecohe(const float* d_img_beta, const float* d_img_0, int32_t n_slices, int64_t n_per_slice,
                double* h_out, void* stream);

/* NEXT row N4 -- cross-validation estimator ("we reconstruct the slice using all the
 * projections except a selected one at a given angle.  Then we calculate the quadratic distance between
 * the reconstructed sample projection and the data for the excluded angle"):
 *   h_out[s] = sum_{e < g_excl->n_angles} sum_b ( (P x)[s][e][b] - d_data_excl[s][e][b] )^2
 * g_excl describes ONLY the excluded projections (their angles / axis positions; n_slices, n_bins, nx,
 * ny, pixel_size as in the reconstruction; sino_pitch = row pitch of d_data_excl).  The reconstruction
 * d_img is made by the caller from the remaining projections (e.g. pyhst_fista_tv with the reduced
 * angle list).  P = pyhst_forward_project (scale 1); the call synchronises `stream`. */
int pyhst_cv_distance(const float* d_img, const float* d_data_excl, const pyhst_geom_t* g_excl,
                      double* h_out, void* stream);

/* NEXT row N3 -- overlapping-patch dictionary reconstruction, PAPER.md L102-L145 (sec. 3.2, eq. 4-9)
 * and Algorithm 1 (L201-L228); readings R16, R22-R24 of DESIGN.md.
 *   x_i = sum_p 1^c_p(i) sum_k w_kp phi_k(i - r_p)                                       (eq. 7)
 *   f(w) = ||y - P x||^2 + rho sum_{p,i} 1_p(i) (x_i - sum_k w_kp phi_k(i - r_p))^2       (eq. 8)
 *   F(w) = f(w) + beta ||w||_1, minimised by FISTA with the soft-threshold step (L139-L141).
 * Patches are m x m on a regular grid of stride `stride` (1 <= stride <= m): origins
 * min(a * stride, n - m), a < na (pyhst_patch_grid), patch index p = a * nb + b; the core of a patch
 * (eq. 5-6) is the set of pixels whose L1-closest patch centre is its own (smallest p among equals).
 * Matrices as in L145: D [n_atoms][m*m] (row k = basis function phi_k, row-major m x m, shared by
 * all slices), W [n_slices][N][n_atoms] with N = na * nb, G like W.  All DEVICE, float32. */
typedef struct {
  int32_t m, stride, n_atoms;
  float rho;                        /* weight of the similarity term of eq. 8, >= 0 */
} pyhst_patch_t;

/* Pure host function: number of patch rows / columns that cover an ny x nx image (eq. 4). */
int pyhst_patch_grid(int32_t ny, int32_t nx, int32_t m, int32_t stride, int32_t* na, int32_t* nb);

/* Algorithm 1: P <- W D; X from the patch cores (eq. 7); R <- P^T (P X - data) (eq. 9's sign, R16);
 * S <- sum of the covering patches; P' per Algorithm 1; G <- 2 P' D^T  (= grad f(W), eq. 9).
 *   d_data [n_slices][n_angles][sino_pitch]  read;   g as for pyhst_forward_project
 *   d_G    [n_slices][N][n_atoms]  written, or NULL (then only X / f are computed)
 *   d_X    [n_slices][ny][nx]      written, or NULL
 *   h_fval HOST scalar = f(W) of eq. 8 summed over the slices, or NULL; if given the call synchronises.
 * Errors: null pointers, stride > m or < 1, m < 1, image smaller than a patch, rho < 0 -> INVALID_ARG. */
int pyhst_patch_gradient(const float* d_W, const float* d_D, const float* d_data, const pyhst_geom_t* g,
                         const pyhst_patch_t* pp, float* d_G, float* d_X, double* h_fval, void* stream);

/* FISTA on the coefficients (R23, R24): w_0 = 0; step 1/Lw with Lw = 1.1 x the power-iteration estimate
 * (n_power iterations from w = 1) of the largest eigenvalue of the Hessian of f; w_{k+1} =
 * shrink(v_k - grad f(v_k)/Lw, beta/Lw); Beck-Teboulle momentum.  energy[k] = f(v_k) + beta ||v_k||_1.
 *   d_W [n_slices][N][n_atoms] written (w after n_iter iterations); d_X [n_slices][ny][nx] = eq. 7 at the
 *   result, or NULL; energy HOST [n_iter] or NULL; lipschitz HOST scalar or NULL (either one: the call
 *   synchronises). */
int pyhst_patch_fista(const float* d_D, const float* d_data, const pyhst_geom_t* g, const pyhst_patch_t* pp,
                      float beta, int32_t n_iter, int32_t n_power, float* d_W, float* d_X, double* energy,
                      double* lipschitz, void* stream);

/* Extended row length / left padding of the virtually doubled detector (R10):
 * far = max(cbar, n_bins-1-cbar); *n_bins_ext = ceil(2 far) + 1 rounded up to a multiple of
 * 64; *pad_left = 0 if the axis is right of the detector centre else n_bins_ext - n_bins. */
int pyhst_halfacq_extent(int32_t n_bins, double cbar, int32_t* n_bins_ext, int32_t* pad_left);

/* Stage accounting for bench.py / tests.  Stages of the hot path, in call order: */
enum {
  PYHST_STAGE_FILTER = 0,      /* a1: pad/weight + cuFFT R2C + x H + cuFFT C2R + crop/interleave */
  PYHST_STAGE_REPACK = 1,      /* a2: [S][P][B] -> slice-interleaved layout (pyhst_backproject only) */
  PYHST_STAGE_BACKPROJECT = 2, /* a2: the backprojection kernel                                  */
  PYHST_STAGE_TRANSPOSE = 3,   /* a3: image transpose for the column walk                        */
  PYHST_STAGE_FORWARD = 4,     /* a3: the forward-projection kernel                              */
  PYHST_STAGE_TV = 5,          /* N1: the solver's own kernels (residual, gradient step, dual steps, momentum) */
  PYHST_N_STAGES = 6
};
/* pyhst_profile_enable(1): from now on every stage is bracketed by a pair of CUDA events recorded
 * on the stream the stage is launched on (no synchronisation is added).  Returns the previous
 * setting.  pyhst_profile_read() synchronises the recorded events and returns, accumulated since
 * the last reset, per stage: device milliseconds (ms, nullable), number of the library's own
 * kernel launches (kernels, nullable; counted whether or not profiling is enabled) and number of
 * cuFFT executions (fft_execs, nullable).  Arrays are HOST, [PYHST_N_STAGES]. */
int pyhst_profile_enable(int enable);
int pyhst_profile_read(double* ms, int64_t* kernels, int64_t* fft_execs, int32_t reset);

const char* pyhst_last_error(void); /* thread-local, static storage; "" if none */
void pyhst_release_cache(void);     /* frees cached plans / workspace (synchronises the device) */

#ifdef __cplusplus
}
#endif
#endif /* PYHST_H_ */
