// NEXT row N4: ring-artefact filter (sec. 2.3; reading R21 of
// DESIGN.md) and the parameter-selection estimators of sec. 4 (L149-L162, eq. 10-11): the
// decoherence estimator E_cohe and the cross-validation distance.  All three are HBM-bound
// reductions / element-wise passes: one read of each operand, sums in double, two-stage
// reductions in a fixed order (no atomics: results are bit-reproducible).
#include <algorithm>
#include <cmath>
#include <mutex>
#include <vector>

#include "common.h"

namespace pyhst {

namespace {

constexpr int RG_BX = 128;   // bins per block of the column-sum kernel
constexpr int RG_PY = 32;    // projection chunks per slice (blockIdx.y): partial sums, then a fixed-order add

// part[s][c][b] = sum over the projections of chunk c of (sino - model)[s][p][b]   (double)
__global__ void __launch_bounds__(RG_BX)
ring_colsum_kernel(const float* __restrict__ sino, const float* __restrict__ model, int64_t pitch, int P,
                   int B, int rows_per_chunk, double* __restrict__ part) {
  const int b = blockIdx.x * RG_BX + threadIdx.x;
  const int c = blockIdx.y, s = blockIdx.z;
  if (b >= B) return;
  const int p0 = c * rows_per_chunk, p1 = min(P, p0 + rows_per_chunk);
  const int64_t base = (int64_t)s * P * pitch + b;
  double acc = 0.0;
  if (model) {
    for (int p = p0; p < p1; ++p) acc += (double)sino[base + (int64_t)p * pitch] - (double)model[base + (int64_t)p * pitch];
  } else {
    for (int p = p0; p < p1; ++p) acc += (double)sino[base + (int64_t)p * pitch];
  }
  part[((int64_t)s * gridDim.y + c) * B + b] = acc;
}

// hp[s][b] = m[b] - mean(m[b-r .. b+r] clipped), m = (sum_c part[s][c][.]) / P ; one block per slice,
// m staged in shared memory (B <= 16384 doubles = 128 KB)
__global__ void __launch_bounds__(256)
ring_highpass_kernel(const double* __restrict__ part, int n_chunks, int P, int B, int r, float* __restrict__ hp) {
  extern __shared__ double m[];
  const int s = blockIdx.x;
  for (int b = threadIdx.x; b < B; b += blockDim.x) {
    double acc = 0.0;
    for (int c = 0; c < n_chunks; ++c) acc += part[((int64_t)s * n_chunks + c) * B + b];
    m[b] = acc / (double)P;
  }
  __syncthreads();
  for (int b = threadIdx.x; b < B; b += blockDim.x) {
    const int lo = max(0, b - r), hi = min(B - 1, b + r);
    double acc = 0.0;
    for (int k = lo; k <= hi; ++k) acc += m[k];
    hp[(int64_t)s * B + b] = (float)(m[b] - acc / (double)(hi - lo + 1));
  }
}

__global__ void __launch_bounds__(256)
ring_subtract_kernel(const float* __restrict__ sino, const float* __restrict__ hp, float* __restrict__ out,
                     int64_t pitch, int P, int B) {
  const int b = blockIdx.x * 256 + threadIdx.x;
  const int s = blockIdx.z;
  if (b >= B) return;
  const float h = hp[(int64_t)s * B + b];
  for (int p = blockIdx.y; p < P; p += gridDim.y) {
    const int64_t o = ((int64_t)s * P + p) * pitch + b;
    out[o] = sino[o] - h;
  }
}

// ---- E_cohe: per block three partial sums (<a-b, a>, ||a-b||^2, ||a||^2) of one slice's chunk
constexpr int EC_NT = 256;
constexpr int EC_BLOCKS = 256;   // blocks per slice

__device__ __forceinline__ double block_sum(double v, double* sh) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
  if (threadIdx.x == 0)
    for (int w = 0; w < EC_NT / 32; ++w) s += sh[w];
  return s;   // valid in thread 0
}

__global__ void __launch_bounds__(EC_NT)
ecohe_partial_kernel(const float* __restrict__ a, const float* __restrict__ b, int64_t n, double* __restrict__ part) {
  __shared__ double sh[EC_NT / 32];
  const int s = blockIdx.y;
  const float* as = a + (int64_t)s * n;
  const float* bs = b + (int64_t)s * n;
  double dot = 0.0, nd = 0.0, na = 0.0;
  for (int64_t k = (int64_t)blockIdx.x * EC_NT + threadIdx.x; k < n; k += (int64_t)gridDim.x * EC_NT) {
    const double av = (double)as[k], d = av - (double)bs[k];
    dot += d * av;
    nd += d * d;
    na += av * av;
  }
  const double s0 = block_sum(dot, sh), s1 = block_sum(nd, sh), s2 = block_sum(na, sh);
  if (threadIdx.x == 0) {
    double* o = part + ((int64_t)s * gridDim.x + blockIdx.x) * 3;
    o[0] = s0; o[1] = s1; o[2] = s2;
  }
}

__global__ void ecohe_final_kernel(const double* __restrict__ part, int n_blocks, double* __restrict__ out) {
  const int s = blockIdx.x;
  if (threadIdx.x != 0) return;
  double dot = 0.0, nd = 0.0, na = 0.0;
  for (int k = 0; k < n_blocks; ++k) {
    const double* o = part + ((int64_t)s * n_blocks + k) * 3;
    dot += o[0]; nd += o[1]; na += o[2];
  }
  out[s] = (nd > 0.0 && na > 0.0) ? dot / (sqrt(nd) * sqrt(na)) : 0.0;
}

// ---- cross-validation: part[s][block] = sum over the block's rows of (y - d)^2
__global__ void __launch_bounds__(EC_NT)
cv_partial_kernel(const float* __restrict__ y, const float* __restrict__ d, int64_t d_pitch, int n_excl, int B,
                  double* __restrict__ part) {
  __shared__ double sh[EC_NT / 32];
  const int s = blockIdx.y;
  double acc = 0.0;
  const int64_t n = (int64_t)n_excl * B;
  for (int64_t k = (int64_t)blockIdx.x * EC_NT + threadIdx.x; k < n; k += (int64_t)gridDim.x * EC_NT) {
    const int64_t e = k / B, b = k - e * B;
    const double v = (double)y[((int64_t)s * n_excl + e) * B + b] - (double)d[((int64_t)s * n_excl + e) * d_pitch + b];
    acc += v * v;
  }
  const double t = block_sum(acc, sh);
  if (threadIdx.x == 0) part[(int64_t)s * gridDim.x + blockIdx.x] = t;
}

__global__ void cv_final_kernel(const double* __restrict__ part, int n_blocks, double* __restrict__ out) {
  if (threadIdx.x != 0) return;
  double acc = 0.0;
  for (int k = 0; k < n_blocks; ++k) acc += part[(int64_t)blockIdx.x * n_blocks + k];
  out[blockIdx.x] = acc;
}

}  // namespace

}  // namespace pyhst

using namespace pyhst;

extern "C" int pyhst_ring_filter(const float* d_sino, const float* d_model, float* d_out, int32_t n_slices,
                                 int32_t n_angles, int32_t n_bins, int64_t pitch, int32_t half_width,
                                 void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!d_sino || !d_out) return set_error(PYHST_ERR_INVALID_ARG, "pyhst_ring_filter: null pointer");
  if (n_slices <= 0 || n_angles <= 0 || n_bins <= 0 || half_width < 1)
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_ring_filter: S=%d P=%d B=%d half_width=%d", n_slices, n_angles,
                     n_bins, half_width);
  if (pitch == 0) pitch = n_bins;
  if (pitch < n_bins) return set_error(PYHST_ERR_INVALID_ARG, "pyhst_ring_filter: pitch %lld < n_bins %d",
                                       (long long)pitch, n_bins);
  if (n_bins > 16384 || n_slices > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "pyhst_ring_filter: more than 16384 bins or 65535 slices");
  PYHST_TRY(require_sm100(nullptr));
  PYHST_CALL_SCOPE(stream);
  const int n_chunks = std::min(RG_PY, n_angles);
  const int rows_per_chunk = (n_angles + n_chunks - 1) / n_chunks;
  const size_t part_bytes = (size_t)n_slices * n_chunks * n_bins * sizeof(double);
  void* ws = nullptr;
  PYHST_TRY(get_workspace(WS_FPL, part_bytes + (size_t)n_slices * n_bins * 4, &ws));
  double* part = static_cast<double*>(ws);
  float* hp = reinterpret_cast<float*>(static_cast<char*>(ws) + part_bytes);
  static DeviceMask configured{0};
  if (first_use_on_device(&configured))
    PYHST_CUDA_TRY(cudaFuncSetAttribute(ring_highpass_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 16384 * 8));
  StageScope scope(ST_FILTER, stream);
  scope.kernels(3);
  ring_colsum_kernel<<<dim3((n_bins + RG_BX - 1) / RG_BX, n_chunks, n_slices), RG_BX, 0, stream>>>(
      d_sino, d_model, pitch, n_angles, n_bins, rows_per_chunk, part);
  ring_highpass_kernel<<<n_slices, 256, (size_t)n_bins * 8, stream>>>(part, n_chunks, n_angles, n_bins, half_width, hp);
  ring_subtract_kernel<<<dim3((n_bins + 255) / 256, std::min(n_angles, 64), n_slices), 256, 0, stream>>>(
      d_sino, hp, d_out, pitch, n_angles, n_bins);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

extern "C" int pyhst_ecohe(const float* d_img_beta, const float* d_img_0, int32_t n_slices, int64_t n_per_slice,
                           double* h_out, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!d_img_beta || !d_img_0 || !h_out) return set_error(PYHST_ERR_INVALID_ARG, "pyhst_ecohe: null pointer");
  if (n_slices <= 0 || n_per_slice <= 0 || n_slices > 65535)
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_ecohe: n_slices %d, n_per_slice %lld", n_slices,
                     (long long)n_per_slice);
  PYHST_TRY(require_sm100(nullptr));
  PYHST_CALL_SCOPE(stream);
  const int nb = (int)std::min<int64_t>(EC_BLOCKS, (n_per_slice + EC_NT - 1) / EC_NT);
  void* ws = nullptr;
  PYHST_TRY(get_workspace(WS_FPL, (size_t)n_slices * nb * 3 * 8 + (size_t)n_slices * 8, &ws));
  double* part = static_cast<double*>(ws);
  double* d_out = part + (size_t)n_slices * nb * 3;
  ecohe_partial_kernel<<<dim3(nb, n_slices), EC_NT, 0, stream>>>(d_img_beta, d_img_0, n_per_slice, part);
  ecohe_final_kernel<<<n_slices, 32, 0, stream>>>(part, nb, d_out);
  PYHST_CUDA_TRY(cudaGetLastError());
  PYHST_CUDA_TRY(cudaMemcpyAsync(h_out, d_out, (size_t)n_slices * 8, cudaMemcpyDeviceToHost, stream));
  PYHST_CUDA_TRY(cudaStreamSynchronize(stream));
  return PYHST_OK;
}

extern "C" int pyhst_cv_distance(const float* d_img, const float* d_data_excl, const pyhst_geom_t* g_excl,
                                 double* h_out, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!d_img || !d_data_excl || !g_excl || !h_out)
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_cv_distance: null pointer");
  if (g_excl->n_slices <= 0 || g_excl->n_angles <= 0 || g_excl->n_bins <= 0 || g_excl->n_slices > 65535)
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_cv_distance: non-positive size");
  const int64_t d_pitch = g_excl->sino_pitch ? g_excl->sino_pitch : g_excl->n_bins;
  if (d_pitch < g_excl->n_bins) return set_error(PYHST_ERR_INVALID_ARG, "pyhst_cv_distance: sino_pitch < n_bins");
  PYHST_TRY(require_sm100(nullptr));
  PYHST_CALL_SCOPE(stream);
  const int S = g_excl->n_slices, E = g_excl->n_angles, B = g_excl->n_bins;
  const int64_t n = (int64_t)E * B;
  const int nb = (int)std::min<int64_t>(EC_BLOCKS, (n + EC_NT - 1) / EC_NT);
  const size_t y_bytes = (((size_t)S * n * 4) + 255) & ~(size_t)255;
  void* ws = nullptr;
  PYHST_TRY(get_workspace(WS_STITCH, y_bytes + (size_t)S * nb * 8 + (size_t)S * 8, &ws));
  float* y = static_cast<float*>(ws);
  double* part = reinterpret_cast<double*>(static_cast<char*>(ws) + y_bytes);
  double* d_out = part + (size_t)S * nb;
  pyhst_geom_t g = *g_excl;
  g.sino_pitch = 0;   // the projection of the reconstruction is written contiguously
  PYHST_TRY(pyhst_forward_project(d_img, y, &g, 1.f, stream));
  cv_partial_kernel<<<dim3(nb, S), EC_NT, 0, stream>>>(y, d_data_excl, d_pitch, E, B, part);
  cv_final_kernel<<<S, 32, 0, stream>>>(part, nb, d_out);
  PYHST_CUDA_TRY(cudaGetLastError());
  PYHST_CUDA_TRY(cudaMemcpyAsync(h_out, d_out, (size_t)S * 8, cudaMemcpyDeviceToHost, stream));
  PYHST_CUDA_TRY(cudaStreamSynchronize(stream));
  return PYHST_OK;
}

// ---- pyhst_ring_filter_static: the ring filter for callers that must not allocate -----------------
// Same three kernels as pyhst_ring_filter, but the column sums `part` and the high-pass row `hp` live in
// a fixed array that is part of the library image instead of the grow-on-demand workspace.  See
// include/pyhst.h for who needs this and what it costs.
namespace pyhst {
namespace {

// bytes per (slice, bin) cell: RG_PY partial column sums in double + one float of hp
constexpr size_t RG_STATIC_CELL_BYTES = (size_t)RG_PY * sizeof(double) + sizeof(float);
constexpr size_t RG_STATIC_BYTES = (size_t)PYHST_RING_STATIC_MAX_CELLS * RG_STATIC_CELL_BYTES;   // 8 519 680

// One copy per GPU that loads the library, resident from module load until the process exits.
// In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device address and
// must never be handed to a kernel as a pointer.
static __device__ __align__(256) unsigned char g_ring_static_scratch[RG_STATIC_BYTES];

constexpr int RG_STATIC_MAX_DEVICES = 64;
std::mutex g_ring_static_mu;
void* g_ring_static_ptr[RG_STATIC_MAX_DEVICES] = {nullptr};   // device address of the array, per device

// First call on the current device: look the array's device address up and raise the shared-memory limit
// of the high-pass kernel.  Neither step allocates.  Later calls return the remembered address.
int ring_static_setup(void** scratch) {
  const int dev = current_device();
  if (dev < 0 || dev >= RG_STATIC_MAX_DEVICES)
    return set_error(PYHST_ERR_UNSUPPORTED, "pyhst_ring_filter_static: device index %d outside 0..%d", dev,
                     RG_STATIC_MAX_DEVICES - 1);
  std::lock_guard<std::mutex> lock(g_ring_static_mu);
  if (!g_ring_static_ptr[dev]) {
    void* p = nullptr;
    PYHST_CUDA_TRY(cudaGetSymbolAddress(&p, g_ring_static_scratch));
    PYHST_CUDA_TRY(cudaFuncSetAttribute(ring_highpass_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 16384 * 8));
    g_ring_static_ptr[dev] = p;
  }
  *scratch = g_ring_static_ptr[dev];
  return PYHST_OK;
}

}  // namespace
}  // namespace pyhst

extern "C" int pyhst_ring_filter_static(const float* d_sino, const float* d_model, float* d_out, int32_t n_slices,
                                        int32_t n_angles, int32_t n_bins, int64_t pitch, int32_t half_width,
                                        void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!d_sino || !d_out) return set_error(PYHST_ERR_INVALID_ARG, "pyhst_ring_filter_static: null pointer");
  if (n_slices <= 0 || n_angles <= 0 || n_bins <= 0 || half_width < 1)
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_ring_filter_static: S=%d P=%d B=%d half_width=%d", n_slices,
                     n_angles, n_bins, half_width);
  if (pitch == 0) pitch = n_bins;
  if (pitch < n_bins) return set_error(PYHST_ERR_INVALID_ARG, "pyhst_ring_filter_static: pitch %lld < n_bins %d",
                                       (long long)pitch, n_bins);
  if (n_bins > 16384 || n_slices > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "pyhst_ring_filter_static: more than 16384 bins or 65535 slices");
  if ((int64_t)n_slices * n_bins > PYHST_RING_STATIC_MAX_CELLS)
    return set_error(PYHST_ERR_UNSUPPORTED,
                     "pyhst_ring_filter_static: n_slices * n_bins = %lld exceeds the fixed scratch of %d cells "
                     "(PYHST_RING_STATIC_MAX_CELLS); filter fewer slices per call or use pyhst_ring_filter",
                     (long long)n_slices * n_bins, (int)PYHST_RING_STATIC_MAX_CELLS);
  PYHST_TRY(require_sm100(nullptr));
  void* scratch = nullptr;
  PYHST_TRY(ring_static_setup(&scratch));
  const int n_chunks = std::min(RG_PY, n_angles);
  const int rows_per_chunk = (n_angles + n_chunks - 1) / n_chunks;
  const size_t part_bytes = (size_t)n_slices * n_chunks * n_bins * sizeof(double);
  double* part = static_cast<double*>(scratch);
  float* hp = reinterpret_cast<float*>(static_cast<char*>(scratch) + part_bytes);
  // Nothing has to be cleared: ring_colsum_kernel writes every part[s][c][b] (an empty chunk writes 0) and
  // ring_highpass_kernel every hp[s][b] before the next kernel reads them; what the previous call left in
  // the array is never read.
  ring_colsum_kernel<<<dim3((n_bins + RG_BX - 1) / RG_BX, n_chunks, n_slices), RG_BX, 0, stream>>>(
      d_sino, d_model, pitch, n_angles, n_bins, rows_per_chunk, part);
  ring_highpass_kernel<<<n_slices, 256, (size_t)n_bins * 8, stream>>>(part, n_chunks, n_angles, n_bins, half_width, hp);
  ring_subtract_kernel<<<dim3((n_bins + 255) / 256, std::min(n_angles, 64), n_slices), 256, 0, stream>>>(
      d_sino, hp, d_out, pitch, n_angles, n_bins);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}
