// Forward projection P = (P^T)^T, gather form (include/pyhst.h a3; eq. 1,
// L211 Alg. 1 "Fp"; readings R6, R13 of DESIGN.md):
//
//   y[s,p,b] = scale * sum_{i,j} Lambda(t_p(i,j) - b) x[s,i,j],  Lambda(u) = max(0, 1 - |u|)
//
// One thread per detector bin (p, b): it walks the image lines that cross the 2-bin-wide strip
// |t - b| < 1 and gathers the few pixels of each line that fall inside it -- no atomics, every
// output written once.  The walk runs along rows when |ch| >= |sh| (then at most ceil(2/|ch|)
// pixels of a row lie in the strip) and along columns otherwise; the column walk reads a
// transposed copy of the image so that neighbouring bins read neighbouring addresses.
// The position of the strip centre on each line is evaluated in double and only the small
// offset (pixel - centre) is carried in FP32 (R11), so the weights are the same function of
// (pixel, bin) as the backprojector's.
#include "common.h"

namespace pyhst {

// ---- [S][ny][nx] -> [S][nx][ny] ----------------------------------------------------------
__global__ void transpose_images_kernel(const float* __restrict__ src, float* __restrict__ dst,
                                        int ny, int nx) {
  __shared__ float tile[32][33];
  const int s = blockIdx.z;
  const float* in = src + (int64_t)s * ny * nx;
  float* out = dst + (int64_t)s * ny * nx;
  const int bx = blockIdx.x * 32, by = blockIdx.y * 32;
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    const int y = by + r, x = bx + threadIdx.x;
    tile[r][threadIdx.x] = (y < ny && x < nx) ? in[(int64_t)y * nx + x] : 0.f;
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    const int x = bx + r, y = by + threadIdx.x;
    if (x < nx && y < ny) out[(int64_t)x * ny + y] = tile[threadIdx.x][r];
  }
}

int launch_transpose_images(const float* d_img, float* d_img_t, int32_t n_slices, int32_t ny,
                            int32_t nx, cudaStream_t stream) {
  dim3 block(32, 8, 1);
  dim3 grid((nx + 31) / 32, (ny + 31) / 32, n_slices);
  if (grid.y > 65535 || grid.z > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "transpose: grid too large");
  StageScope scope(ST_TRANSPOSE, stream);
  scope.kernels();
  transpose_images_kernel<<<grid, block, 0, stream>>>(d_img, d_img_t, ny, nx);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

// ---- gather kernel -----------------------------------------------------------------------
// Generic line walk.  `u` = coordinate along the line (fast axis, length nu, centre u0),
// `v` = line index (slow axis, length nv, centre v0):  t = c + cu (u - u0) + cv (v - v0) with
// |cu| >= |cv|.  Row walk: u = j, v = i, image [nv][nu] = x.  Column walk: u = i, v = j,
// image = x transposed.
constexpr int FP_NT = 128;

__global__ void __launch_bounds__(FP_NT)
fp_gather_kernel(const float* __restrict__ img, const float* __restrict__ img_t,
                 float* __restrict__ sino, int64_t pitch, int P, int B, int nx, int ny, float scale,
                 const ProjGeom* __restrict__ proj) {
  const int b = blockIdx.x * FP_NT + threadIdx.x;
  const int p = blockIdx.y, s = blockIdx.z;
  if (b >= B) return;
  const ProjGeom pg = proj[p];
  const bool row_walk = fabs(pg.ch) >= fabs(pg.sh);
  const double cu = row_walk ? pg.ch : pg.sh;
  const double cv = row_walk ? pg.sh : pg.ch;
  const int nu = row_walk ? nx : ny;
  const int nv = row_walk ? ny : nx;
  const double u0 = 0.5 * (double)(nu - 1), v0 = 0.5 * (double)(nv - 1);
  const float* x = (row_walk ? img : img_t) + (int64_t)s * nx * ny;

  // centre of the strip on line v:  u*(v) = u0 + (b - c - cv (v - v0)) / cu = a0 + a1 v
  const double inv = 1.0 / cu;
  const double a1 = -cv * inv;
  const double a0 = u0 + ((double)b - pg.c + cv * v0) * inv;
  const double hw = fabs(inv);                 // half-width of the strip in pixels
  const int nc = (int)ceil(2.0 * hw);          // pixels of one line that can lie inside it
  const float cuf = (float)cu;

  float acc = 0.f;
  for (int v = 0; v < nv; ++v) {
    const double us = fma(a1, (double)v, a0);
    const double lo = floor(us - hw);          // first candidate is lo + 1
    if (lo >= (double)(nu - 1) || lo + (double)nc < 0.0) continue;
    const int u_first = (int)lo + 1;
    const float d0 = (float)((lo + 1.0) - us); // in (-hw, -hw + 1]
    const float* line = x + (int64_t)v * nu;
    for (int c = 0; c < nc; ++c) {
      const int u = u_first + c;
      const float w = 1.f - fabsf(cuf * (d0 + (float)c));
      if (u >= 0 && u < nu && w > 0.f) acc = fmaf(w, line[u], acc);
    }
  }
  sino[((int64_t)s * P + p) * pitch + b] = scale * acc;
}

int launch_forward_project(const FpArgs& a, cudaStream_t stream) {
  dim3 grid((a.n_bins + FP_NT - 1) / FP_NT, a.n_angles, a.n_slices);
  if (grid.y > 65535 || grid.z > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "forward projector: grid too large");
  StageScope scope(ST_FORWARD, stream);
  scope.kernels();
  fp_gather_kernel<<<grid, FP_NT, 0, stream>>>(a.d_img, a.d_img_t, a.d_sino, a.pitch, a.n_angles,
                                               a.n_bins, a.nx, a.ny, a.scale, a.d_proj);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

}  // namespace pyhst
