// Ramp filter (include/pyhst.h a1; "filtered back projection"; readings R8-R10
// of DESIGN.md): exact linear convolution of every (optionally column-weighted) sinogram row with
// the band-limited ramp kernel h, evaluated as a zero-padded batched FFT multiply:
//
//   pad/weight kernel -> cuFFT R2C (in place) -> x H[k]/M -> cuFFT C2R (in place) -> crop kernel
//
// The row is embedded at offset pad_left in a length-M buffer, M >= 2 n_bins_out, so that every
// lag the output needs, -(pad_left + n_bins_in - 1) .. n_bins_out - 1, lies inside (-M/2, M/2)
// and the circular convolution with hc[l mod M] = h[l] (|l| <= M/2) equals the linear one.
// H = DFT_M(hc) is real and even; it is computed once per (filter, M) in DOUBLE on the device
// (closed-form h in double, cuFFT D2Z) and stored as float already divided by M.
#include <cufft.h>

#include <map>
#include <mutex>
#include <tuple>

#include "common.h"

namespace pyhst {

namespace {

#define PYHST_CUFFT_TRY(expr)                                                                  \
  do {                                                                                         \
    cufftResult _r = (expr);                                                                   \
    if (_r != CUFFT_SUCCESS)                                                                   \
      return set_error(_r == CUFFT_ALLOC_FAILED ? PYHST_ERR_NOMEM : PYHST_ERR_CUDA,            \
                       "%s failed: cufftResult %d (%s:%d)", #expr, (int)_r, __FILE__, __LINE__); \
  } while (0)

std::mutex g_mu;
struct Spectrum { float* d_H = nullptr; };                    // [M/2 + 1], H[k] / M
std::map<std::tuple<int, int, int>, Spectrum> g_spectra;      // (device, filter, M)
struct FftPlans { cufftHandle r2c = 0, c2r = 0; };
std::map<std::tuple<int, int, int>, FftPlans> g_plans;        // (device, M, batch)

// smallest M = 2^a * {1, 3, 5} with M >= n (cuFFT is efficient for these radices)
int fft_length(int64_t n) {
  int64_t best = INT64_MAX;
  for (int64_t m : {1, 3, 5})
    for (int64_t v = m; v < (int64_t)1 << 30; v *= 2)
      if (v >= n && v >= 16) { if (v < best) best = v; break; }
  return (int)best;
}

// hc[l mod M] = h[l] for -M/2 < l <= M/2, in double (R8)
__global__ void ramp_kernel_table(double* hc, int M, int filter) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= M) return;
  const int l = n <= M / 2 ? n : n - M;
  const double PI = 3.14159265358979323846264338327950288;
  const double dl = (double)l;
  auto ramlak = [PI](int m) {
    const double dm = (double)m;
    return m == 0 ? 0.25 : ((m & 1) ? -1.0 / (PI * PI * dm * dm) : 0.0);
  };
  double h;
  if (filter == PYHST_FILTER_RAMLAK)
    h = ramlak(l);
  else if (filter == PYHST_FILTER_SHEPP_LOGAN)
    h = -2.0 / (PI * PI * (4.0 * dl * dl - 1.0));
  else if (filter == PYHST_FILTER_COSINE) {
    // window cos(pi w) = half-bin shifts of the continuous band-limited ramp (R8c):
    // ramp(m + 1/2) = (-1)^m / (2 pi (m + 1/2)) - 1 / (2 pi^2 (m + 1/2)^2)
    auto half_shifted = [PI](int m) {
      const double x = (double)m + 0.5;
      return ((m & 1) ? -1.0 : 1.0) / (2.0 * PI * x) - 1.0 / (2.0 * PI * PI * x * x);
    };
    h = 0.5 * (half_shifted(l - 1) + half_shifted(l));
  } else {  // Hann / Hamming window a0 + 2 a1 cos(2 pi w) on the Ram-Lak ramp = unit shifts in space
    const double a0 = filter == PYHST_FILTER_HANN ? 0.5 : 0.54, a1 = filter == PYHST_FILTER_HANN ? 0.25 : 0.23;
    h = a0 * ramlak(l) + a1 * (ramlak(l - 1) + ramlak(l + 1));
  }
  hc[n] = h;
}

__global__ void spectrum_to_float(const cufftDoubleComplex* Hd, float* H, int nk, double inv_m) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k < nk) H[k] = (float)(Hd[k].x * inv_m);
}

int get_spectrum(int filter, int M, cudaStream_t stream, const float** out) {
  auto key = std::make_tuple(current_device(), filter, M);
  auto it = g_spectra.find(key);
  if (it != g_spectra.end()) { *out = it->second.d_H; return PYHST_OK; }
  const int nk = M / 2 + 1;
  double* d_hc = nullptr;
  cufftDoubleComplex* d_Hd = nullptr;
  float* d_H = nullptr;
  struct Cleanup {   // the temporaries always, the spectrum itself unless it reached the cache
    double*& hc; cufftDoubleComplex*& Hd; float*& H; bool keep = false; cufftHandle* plan = nullptr;
    ~Cleanup() { if (plan) cufftDestroy(*plan); cudaFree(hc); cudaFree(Hd); if (!keep) cudaFree(H); }
  } cleanup{d_hc, d_Hd, d_H};
  PYHST_CUDA_TRY(cudaMalloc(&d_hc, sizeof(double) * M));
  PYHST_CUDA_TRY(cudaMalloc(&d_Hd, sizeof(cufftDoubleComplex) * nk));
  PYHST_CUDA_TRY(cudaMalloc(&d_H, sizeof(float) * nk));
  cufftHandle plan;
  PYHST_CUFFT_TRY(cufftPlan1d(&plan, M, CUFFT_D2Z, 1));
  cleanup.plan = &plan;
  PYHST_CUFFT_TRY(cufftSetStream(plan, stream));
  ramp_kernel_table<<<(M + 255) / 256, 256, 0, stream>>>(d_hc, M, filter);
  PYHST_CUFFT_TRY(cufftExecD2Z(plan, d_hc, d_Hd));
  spectrum_to_float<<<(nk + 255) / 256, 256, 0, stream>>>(d_Hd, d_H, nk, 1.0 / (double)M);
  PYHST_CUDA_TRY(cudaGetLastError());
  PYHST_CUDA_TRY(cudaStreamSynchronize(stream));  // one-time set-up; temporaries freed below
  cleanup.keep = true;   // (the plan and the temporaries go with `cleanup`)
  g_spectra[key].d_H = d_H;
  *out = d_H;
  return PYHST_OK;
}

int get_plans(int M, int batch, FftPlans* out) {
  auto key = std::make_tuple(current_device(), M, batch);
  auto it = g_plans.find(key);
  if (it != g_plans.end()) { *out = it->second; return PYHST_OK; }
  FftPlans pl;
  int n[1] = {M};
  int rembed[1] = {M + 2}, cembed[1] = {M / 2 + 1};
  PYHST_CUFFT_TRY(cufftPlanMany(&pl.r2c, 1, n, rembed, 1, M + 2, cembed, 1, M / 2 + 1, CUFFT_R2C, batch));
  PYHST_CUFFT_TRY(cufftPlanMany(&pl.c2r, 1, n, cembed, 1, M / 2 + 1, rembed, 1, M + 2, CUFFT_C2R, batch));
  g_plans[key] = pl;
  *out = pl;
  return PYHST_OK;
}

// buf[r][n] = w[n - pad] in[r][n - pad] inside the embedded row, 0 elsewhere; n < M + 2
__global__ void pad_weight_kernel(const float* __restrict__ in, int64_t in_pitch,
                                  const float* __restrict__ w, float* __restrict__ buf, int Mp,
                                  int n_bins_in, int pad_left) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t r = blockIdx.y;
  if (n >= Mp) return;
  const int m = n - pad_left;
  float v = 0.f;
  if (m >= 0 && m < n_bins_in) {
    v = in[r * in_pitch + m];
    if (w) v *= w[m];
  }
  buf[r * Mp + n] = v;
}

__global__ void multiply_spectrum_kernel(float2* __restrict__ spec, const float* __restrict__ H,
                                         int nk) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t r = blockIdx.y;
  if (k >= nk) return;
  float2 v = spec[r * nk + k];
  const float h = H[k];
  v.x *= h;
  v.y *= h;
  spec[r * nk + k] = v;
}

__global__ void crop_rows_kernel(const float* __restrict__ buf, int Mp, float* __restrict__ out,
                                 int64_t out_pitch, int n_bins_out) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t r = blockIdx.y;
  if (n < n_bins_out) out[r * out_pitch + n] = buf[r * Mp + n];
}

// rows r = sl * P + p of one slice group -> QI[p][zpad + b][sl], pads and missing slices zero
__global__ void crop_interleave_kernel(const float* __restrict__ buf, int Mp, float4* __restrict__ qi,
                                       int P, int n_bins_out, int zpad, int n_slices_in,
                                       const uint8_t* __restrict__ flip) {
  const int64_t row_f4 = (int64_t)n_bins_out + 2 * zpad;
  const int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (x >= row_f4) return;
  int64_t b = x - zpad;
  float v[4] = {0.f, 0.f, 0.f, 0.f};
  if (b >= 0 && b < n_bins_out) {
    if (flip && flip[p]) b = n_bins_out - 1 - b;  // reversed row, see bp_run_kernel
#pragma unroll
    for (int sl = 0; sl < 4; ++sl)
      if (sl < n_slices_in) v[sl] = buf[((int64_t)sl * P + p) * Mp + b];
  }
  qi[(int64_t)p * row_f4 + x] = make_float4(v[0], v[1], v[2], v[3]);
}

__global__ void halfacq_weights_kernel(float* w, int n_bins, double cbar) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= n_bins) return;
  // R10: s = b - cbar; axis right of centre: omega = (B-1) - cbar, w = 1 (s < -omega),
  // (omega - s) / (2 omega) (|s| <= omega), 0 beyond; mirrored when the axis is left of centre
  const double mid = 0.5 * (double)(n_bins - 1);
  const bool right = cbar >= mid;
  const double omega = right ? (double)(n_bins - 1) - cbar : cbar;
  double s = (double)b - cbar;
  if (!right) s = -s;
  double v;
  if (s < -omega) v = 1.0;
  else if (s <= omega) v = (omega - s) / (2.0 * omega);
  else v = 0.0;
  w[b] = (float)v;
}

}  // namespace

int launch_halfacq_weights(float* d_w, int32_t n_bins, double cbar, cudaStream_t stream) {
  halfacq_weights_kernel<<<(n_bins + 255) / 256, 256, 0, stream>>>(d_w, n_bins, cbar);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

int launch_ramp_filter(const float* d_in, int64_t in_pitch, int64_t n_rows, int32_t n_bins_in,
                       int32_t n_bins_out, int32_t pad_left, int filter,
                       const float* d_col_weights, float* d_out, int64_t out_pitch,
                       float4* d_qi, const QiLayout* L, int32_t n_slices_in, const uint8_t* d_flip,
                       cudaStream_t stream) {
  if (n_rows == 0) return PYHST_OK;
  {
    // product path: the fused shared-memory FFT kernel (one read, one write); cuFFT for longer rows
    const int variant = filter_variant();
    const bool fused_ok = ramp_fused_log2m(n_bins_out) != 0;
    if (variant == 2 && !fused_ok)
      return set_error(PYHST_ERR_UNSUPPORTED, "fused ramp filter does not cover rows of %d bins", n_bins_out);
    if (variant != 1 && fused_ok)
      return launch_ramp_filter_fused(d_in, in_pitch, n_rows, n_bins_in, n_bins_out, pad_left, filter, d_col_weights,
                                      d_out, out_pitch, d_qi, L, n_slices_in, d_flip, stream);
  }
  std::lock_guard<std::mutex> lock(g_mu);
  const int M = fft_length(2 * (int64_t)n_bins_out);
  const int Mp = M + 2, nk = M / 2 + 1;
  const float* d_H = nullptr;
  PYHST_TRY(get_spectrum(filter, M, stream, &d_H));

  // rows per FFT batch: a whole slice group when interleaving, else bounded by ~256 MB
  int64_t batch_rows = n_rows;
  if (!d_qi) {
    const int64_t cap = std::max<int64_t>(1, ((int64_t)256 << 20) / ((int64_t)Mp * 4));
    batch_rows = std::min<int64_t>(n_rows, std::min<int64_t>(cap, 65535));
  } else if (n_rows > 65535 * 4) {
    return set_error(PYHST_ERR_UNSUPPORTED, "ramp filter: slice group has too many rows");
  }
  void* ws = nullptr;
  PYHST_TRY(get_workspace(WS_FFT, (size_t)batch_rows * Mp * 4, &ws));
  float* buf = static_cast<float*>(ws);
  StageScope scope(ST_FILTER, stream);

  for (int64_t r0 = 0; r0 < n_rows; r0 += batch_rows) {
    const int nb = (int)std::min<int64_t>(batch_rows, n_rows - r0);
    FftPlans pl;
    PYHST_TRY(get_plans(M, nb, &pl));
    PYHST_CUFFT_TRY(cufftSetStream(pl.r2c, stream));
    PYHST_CUFFT_TRY(cufftSetStream(pl.c2r, stream));
    // gridDim.y <= 65535: split the row range of the elementwise kernels
    for (int y0 = 0; y0 < nb; y0 += 65535) {
      const int ny = std::min(65535, nb - y0);
      scope.kernels();
      pad_weight_kernel<<<dim3((Mp + 255) / 256, ny), 256, 0, stream>>>(
          d_in + (r0 + y0) * in_pitch, in_pitch, d_col_weights, buf + (int64_t)y0 * Mp, Mp,
          n_bins_in, pad_left);
    }
    scope.library(2);
    PYHST_CUFFT_TRY(cufftExecR2C(pl.r2c, buf, reinterpret_cast<cufftComplex*>(buf)));
    for (int y0 = 0; y0 < nb; y0 += 65535) {
      const int ny = std::min(65535, nb - y0);
      scope.kernels();
      multiply_spectrum_kernel<<<dim3((nk + 255) / 256, ny), 256, 0, stream>>>(
          reinterpret_cast<float2*>(buf) + (int64_t)y0 * nk, d_H, nk);
    }
    PYHST_CUFFT_TRY(cufftExecC2R(pl.c2r, reinterpret_cast<cufftComplex*>(buf), buf));
    if (d_qi) {
      const int64_t row_f4 = L->row_f4();
      scope.kernels();
      crop_interleave_kernel<<<dim3((unsigned)((row_f4 + 255) / 256), L->n_angles), 256, 0, stream>>>(
          buf, Mp, d_qi, L->n_angles, n_bins_out, L->zpad, n_slices_in, d_flip);
    } else {
      for (int y0 = 0; y0 < nb; y0 += 65535) {
        const int ny = std::min(65535, nb - y0);
        scope.kernels();
        crop_rows_kernel<<<dim3((n_bins_out + 255) / 256, ny), 256, 0, stream>>>(
            buf + (int64_t)y0 * Mp, Mp, d_out + (r0 + y0) * out_pitch, out_pitch, n_bins_out);
      }
    }
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  return PYHST_OK;
}

void release_filter_plans(int device) {
  release_fused_filter_tables(device);
  std::lock_guard<std::mutex> lock(g_mu);
  for (auto it = g_plans.begin(); it != g_plans.end();) {
    if (std::get<0>(it->first) != device) { ++it; continue; }
    cufftDestroy(it->second.r2c);
    cufftDestroy(it->second.c2r);
    it = g_plans.erase(it);
  }
  for (auto it = g_spectra.begin(); it != g_spectra.end();) {
    if (std::get<0>(it->first) != device) { ++it; continue; }
    cudaFree(it->second.d_H);
    it = g_spectra.erase(it);
  }
}

// ---- stitched half acquisition (NEXT row N2; reading R10) -------------------------
// A 360-degree half-acquisition scan whose projections pair up (theta_{p+P/2} = theta_p + pi, same
// axis c, 2c integer) folds into a 180-degree scan of P/2 full-width rows: the opposite projection
// sees the pixel at 2c - t, and lerp is symmetric, so
//     lerp(g_p, t) + lerp(g_{p+P/2}, 2c - t) = lerp(g_p + flip(g_{p+P/2}), t),  flip(g)[b] = g[2c - b].
// out[s][p][j], j in [0, b_st): bin b = j - off of the filtered rows' coordinate.
__global__ void halfacq_fold_kernel(const float* __restrict__ rows, float* __restrict__ out, int P2,
                                    int b_out, int b_st, int off, const int* __restrict__ two_c) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y, s = blockIdx.z;
  if (j >= b_st) return;
  const int b = j - off, bf = two_c[p] - b;
  const float* ra = rows + ((int64_t)s * 2 * P2 + p) * b_out;
  const float* rb = rows + ((int64_t)s * 2 * P2 + p + P2) * b_out;
  float v = 0.f;
  if (b >= 0 && b < b_out) v = ra[b];
  if (bf >= 0 && bf < b_out) v += rb[bf];
  out[((int64_t)s * P2 + p) * b_st + j] = v;
}

int launch_halfacq_fold(const float* d_rows, float* d_out, int32_t n_slices, int32_t half_angles,
                        int32_t b_out, int32_t b_st, int32_t off, const int* d_two_c, cudaStream_t stream) {
  dim3 grid((b_st + 255) / 256, half_angles, n_slices);
  if (grid.y > 65535 || grid.z > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "half-acquisition fold: grid too large");
  StageScope scope(ST_FILTER, stream);
  scope.kernels();
  halfacq_fold_kernel<<<grid, 256, 0, stream>>>(d_rows, d_out, half_angles, b_out, b_st, off, d_two_c);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

}  // namespace pyhst
