// TV-regularised FISTA (include/pyhst.h pyhst_fista_tv; NEXT row N1 of SURVEY.md sec. 8(f);
// PAPER.md L73-L86, sec. 3.1, eq. 1-3; readings R16-R20 of DESIGN.md):
//
//   x = argmin 1/2 ||data - P x||^2 + beta TV(x),  TV(x) = sum_pixels sqrt((d1 x)^2 + (d2 x)^2)
//
// Every iteration calls the projector pair once (pyhst_forward_project, pyhst_backproject of this
// library) and a handful of element-wise / 5-point-stencil kernels over the image stack:
//   r = P y - data, 1/2 ||r||^2            ftv_residual_kernel
//   z = y - P^T r / L, TV(y)               ftv_step_kernel
//   n_inner dual projected-gradient steps  ftv_dual_fused_kernel (5 steps per launch on a shared-memory tile)
//   x+ = z - tau G^T p, momentum           ftv_finish_kernel
// All scalars (L, the energies) stay on the device: the loop enqueues without a host sync.
#include <algorithm>
#include <cmath>
#include <vector>

#include "common.h"

namespace pyhst {

namespace {

constexpr int FT_BX = 32, FT_BY = 8;

// Deterministic two-stage sum: every block stores the sum of its threads' values (fixed shuffle /
// warp order) into part[linear block index]; ftv_reduce_kernel then adds the partials to the
// accumulator in a fixed order.  (Round 1 used atomicAdd(double): the order of the additions, hence
// the last bits of L, of the energies and of every iterate, changed from run to run.)
__device__ __forceinline__ void block_sum_to(double v, double* part) {
  __shared__ double wsum[FT_BX * FT_BY / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int t = threadIdx.y * blockDim.x + threadIdx.x;
  if ((t & 31) == 0) wsum[t >> 5] = v;
  __syncthreads();
  if (t == 0) {
    double s = 0.0;
    for (int w = 0; w < (int)(blockDim.x * blockDim.y) / 32; ++w) s += wsum[w];
    part[((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = s;
  }
}

// *dst += sum_k part[k], k < n: thread t adds part[t], part[t + 1024], ... in that order, then a
// fixed binary tree over the 1024 threads
__global__ void __launch_bounds__(1024) ftv_reduce_kernel(const double* __restrict__ part, int n, double* dst) {
  __shared__ double sh[1024];
  double s = 0.0;
  for (int k = threadIdx.x; k < n; k += 1024) s += part[k];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) *dst += sh[0];
}

// forward differences, zero at the last column / row (R18)
__device__ __forceinline__ float d1f(const float* x, int nx, int i, int j) {
  return j + 1 < nx ? x[(int64_t)i * nx + j + 1] - x[(int64_t)i * nx + j] : 0.f;
}
__device__ __forceinline__ float d2f(const float* x, int nx, int ny, int i, int j) {
  return i + 1 < ny ? x[(int64_t)(i + 1) * nx + j] - x[(int64_t)i * nx + j] : 0.f;
}
// (G^T p)[i,j] = p1[i,j-1] - p1[i,j] + p2[i-1,j] - p2[i,j]; p1 of the last column and p2 of the
// last row are identically zero (they are never made non-zero by the dual steps)
__device__ __forceinline__ float gtf(const float* p1, const float* p2, int nx, int ny, int i, int j) {
  float v = 0.f;
  if (j > 0) v += p1[(int64_t)i * nx + j - 1];
  if (j + 1 < nx) v -= p1[(int64_t)i * nx + j];
  if (i > 0) v += p2[(int64_t)(i - 1) * nx + j];
  if (i + 1 < ny) v -= p2[(int64_t)i * nx + j];
  return v;
}

// r[s,p,b] -= data[s,p,b] (r contiguous, data pitched); *half_acc += 1/2 sum r^2
__global__ void ftv_residual_kernel(float* __restrict__ r, const float* __restrict__ data,
                                    int64_t data_pitch, int n_bins, int64_t n_rows, double* half_acc) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  double acc = 0.0;
  for (int64_t row = (int64_t)blockIdx.y * blockDim.y + threadIdx.y; row < n_rows;
       row += (int64_t)gridDim.y * blockDim.y) {
    if (b < n_bins) {
      const float v = r[row * n_bins + b] - data[row * data_pitch + b];
      r[row * n_bins + b] = v;
      acc += 0.5 * (double)v * (double)v;
    }
  }
  block_sum_to(acc, half_acc);   // half_acc = partials [gridDim.x * gridDim.y]
}

// z = y - g * (1/L);  *tv_acc += beta * TV(y)   (energy of eq. 3 at y, R19)
__global__ void ftv_step_kernel(const float* __restrict__ y, const float* __restrict__ g,
                                float* __restrict__ z, int nx, int ny, const float* __restrict__ fs, double beta,
                                double* tv_acc) {
  const int j = blockIdx.x * FT_BX + threadIdx.x, i = blockIdx.y * FT_BY + threadIdx.y;
  const int64_t o = (int64_t)blockIdx.z * ny * nx;
  double tv = 0.0;
  if (i < ny && j < nx) {
    const float inv_l = fs[0];
    const int64_t k = o + (int64_t)i * nx + j;
    z[k] = fmaf(-g[k], inv_l, y[k]);
    const float a = d1f(y + o, nx, i, j), b = d2f(y + o, nx, ny, i, j);
    tv = beta * (double)sqrtf(a * a + b * b);
  }
  if (tv_acc) block_sum_to(tv, tv_acc);
}

// Dual projected-gradient steps (R18):  u = z - tau G^T p ;  q = p + G u / (8 tau) ;  p' = q / max(1, |q|)
// -- p is read from (p1, p2) and written to (q1, q2) (Jacobi: ping-pong between two buffer pairs).
// K dual steps per launch (temporal blocking): the block owns a 64 x 32 tile of the image plus a halo of K
// cells and iterates the Jacobi step K times on it.  A cell's value after one step depends on its neighbours
// at distance 1, so what enters from the edge of the staged region spoils one more ring per step and never
// reaches the tile; every cell of the tile goes through exactly the arithmetic of K single steps.  HBM traffic
// per step falls from 5 arrays to (3 x 1.5 + 2) / K arrays.
// Register blocking: a thread owns a column segment of FD_SEG = 14 cells (3 segments x (64 + 2K) columns <= 222
// threads) and keeps their z, p1, p2 and u in registers for all K steps; only what a NEIGHBOUR needs goes
// through shared memory: p1 (read by the cell to the right), u (read by the cell to the left) and, at the
// segment ends, p2 of the last row / u of the first row.  Two block barriers per step.
// Cells outside the image hold p = z = 0 and are never updated (p1 of the last column and p2 of the last row
// stay zero by construction: their differences are 0).
constexpr int FD_TX = 64, FD_TY = 32, FD_KMAX = 5, FD_NT = 256, FD_SEG = 14, FD_NSEG = 3;
constexpr int FD_RW = FD_TX + 2 * FD_KMAX, FD_RH = FD_TY + 2 * FD_KMAX;
static_assert(FD_SEG * FD_NSEG >= FD_RH && FD_RW * FD_NSEG <= FD_NT, "thread map of the fused dual kernel");

// FAST: the block's staged region lies strictly inside the image and K = FD_KMAX -- every bounds test on image
// coordinates is dropped and the region's extent is a compile-time constant (the common case: all blocks but
// those on the image border); the arithmetic per cell is the same.
template <bool FAST>
__device__ __forceinline__ void ftv_dual_fused_body(const float* __restrict__ z, const float* __restrict__ p1,
                                                    const float* __restrict__ p2, float* __restrict__ q1,
                                                    float* __restrict__ q2, int nx, int ny, float tau, float step, int Kr,
                                                    int p_is_zero, float (*S1)[FD_RW], float (*SU)[FD_RW],
                                                    float (*E2)[FD_RW]) {
  const int K = FAST ? FD_KMAX : Kr;
  const int rw = FD_TX + 2 * K, rh = FD_TY + 2 * K;
  const int col = (int)threadIdx.x % rw, seg = (int)threadIdx.x / rw;
  const bool active = seg < FD_NSEG;
  const int row0 = seg * FD_SEG;
  const int64_t o = (int64_t)blockIdx.z * ny * nx;
  const int gx = blockIdx.x * FD_TX - K + col, gy0 = blockIdx.y * FD_TY - K + row0;
  const bool x_in = FAST || (gx >= 0 && gx < nx);
  const bool right_ok = (FAST || gx + 1 < nx) && col + 1 < rw;

  float vz[FD_SEG], v1[FD_SEG], v2[FD_SEG], vu[FD_SEG];
  if (active) {
#pragma unroll
    for (int r = 0; r < FD_SEG; ++r) {
      const int gy = gy0 + r;
      const bool in = row0 + r < rh && (FAST || (x_in && gy >= 0 && gy < ny));
      const int64_t k = o + (int64_t)gy * nx + gx;
      vz[r] = in ? z[k] : 0.f;
      v1[r] = (in && !p_is_zero) ? p1[k] : 0.f;
      v2[r] = (in && !p_is_zero) ? p2[k] : 0.f;
      if (row0 + r < rh) S1[row0 + r][col] = v1[r];
    }
    E2[seg][col] = v2[FD_SEG - 1];
  }
  __syncthreads();
  for (int it = 0; it < K; ++it) {
    if (active) {
      float above = seg > 0 ? E2[seg - 1][col] : 0.f;    // p2 of the cell above the segment
#pragma unroll
      for (int r = 0; r < FD_SEG; ++r) {
        if (row0 + r < rh) {
          const float l1 = col > 0 ? S1[row0 + r][col - 1] : 0.f;
          vu[r] = fmaf(-tau, (l1 - v1[r]) + (above - v2[r]), vz[r]);
          SU[row0 + r][col] = vu[r];
        }
        above = v2[r];
      }
    }
    __syncthreads();
    if (active) {
#pragma unroll
      for (int r = 0; r < FD_SEG; ++r) {
        const int gy = gy0 + r, row = row0 + r;
        if (row < rh && (FAST || (x_in && gy >= 0 && gy < ny))) {
          const float u = vu[r];
          const float ur = right_ok ? SU[row][col + 1] - u : 0.f;
          float ub = 0.f;
          if ((FAST || gy + 1 < ny) && row + 1 < rh) ub = (r + 1 < FD_SEG ? vu[r + 1] : SU[row + 1][col]) - u;
          const float n1 = fmaf(ur, step, v1[r]), n2 = fmaf(ub, step, v2[r]);
          // p = q / max(1, |q|) = q * min(1, 1/|q|)
          const float inv = fminf(1.f, rsqrtf(fmaf(n1, n1, n2 * n2)));
          v1[r] = n1 * inv;
          v2[r] = n2 * inv;
          S1[row][col] = v1[r];
        }
      }
      E2[seg][col] = v2[FD_SEG - 1];
    }
    __syncthreads();
  }
  if (active && col >= K && col < K + FD_TX && x_in) {
#pragma unroll
    for (int r = 0; r < FD_SEG; ++r) {
      const int row = row0 + r, gy = gy0 + r;
      if (row >= K && row < K + FD_TY && (FAST || gy < ny)) {
        const int64_t k = o + (int64_t)gy * nx + gx;
        q1[k] = v1[r];
        q2[k] = v2[r];
      }
    }
  }
}

__global__ void __launch_bounds__(FD_NT)
ftv_dual_fused_kernel(const float* __restrict__ z, const float* __restrict__ p1, const float* __restrict__ p2,
                      float* __restrict__ q1, float* __restrict__ q2, int nx, int ny,
                      const float* __restrict__ fs, int K, int p_is_zero) {
  __shared__ float S1[FD_RH][FD_RW];          // p1 as of the last completed step
  __shared__ float SU[FD_RH][FD_RW];          // u of the current step
  __shared__ float E2[FD_NSEG][FD_RW];        // p2 of the last row of every segment
  const float tau = fs[1], step = fs[2];
  // the staged region [x0 - K, x0 + TX + K) x [y0 - K, y0 + TY + K) and its right / lower neighbours inside the image?
  const int x0 = blockIdx.x * FD_TX, y0 = blockIdx.y * FD_TY;
  const bool fast = K == FD_KMAX && x0 - K >= 0 && y0 - K >= 0 && x0 + FD_TX + K < nx && y0 + FD_TY + K < ny;
  if (fast)
    ftv_dual_fused_body<true>(z, p1, p2, q1, q2, nx, ny, tau, step, K, p_is_zero, S1, SU, E2);
  else
    ftv_dual_fused_body<false>(z, p1, p2, q1, q2, nx, ny, tau, step, K, p_is_zero, S1, SU, E2);
}

// x+ = z - tau G^T p (tau = 0: x+ = z);  y = x+ + mom (x+ - x);  x = x+
__global__ void ftv_finish_kernel(const float* __restrict__ z, const float* __restrict__ p1,
                                  const float* __restrict__ p2, float* __restrict__ x,
                                  float* __restrict__ y, int nx, int ny, const float* __restrict__ fs, float mom,
                                  int use_p) {
  const int j = blockIdx.x * FT_BX + threadIdx.x, i = blockIdx.y * FT_BY + threadIdx.y;
  if (i >= ny || j >= nx) return;
  const int64_t o = (int64_t)blockIdx.z * ny * nx, k = o + (int64_t)i * nx + j;
  float xn = z[k];
  if (use_p) xn = fmaf(-fs[1], gtf(p1 + o, p2 + o, nx, ny, i, j), xn);
  const float xo = x[k];
  y[k] = fmaf(mom, xn - xo, xn);
  x[k] = xn;
}

// power iteration helpers: *acc += sum v^2 ;  v = w / sqrt(*nw), L = 1.1 sqrt(*nw / *nv)
__global__ void ftv_sumsq_kernel(const float* __restrict__ v, int64_t n, double* acc) {
  double s = 0.0;
  for (int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.y * 32 + threadIdx.x; k < n;
       k += (int64_t)gridDim.x * 256)
    s += (double)v[k] * (double)v[k];
  block_sum_to(s, acc);
}
__global__ void ftv_normalise_kernel(const float* __restrict__ w, float* __restrict__ v, int64_t n,
                                     const double* nv, const double* nw, double* L) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const double s = sqrt(*nw);
  if (k < n) v[k] = (float)((double)w[k] / s);
  if (k == 0) *L = 1.1 * s / sqrt(*nv);
}
// fs[0] = 1/L, fs[1] = tau = beta/L, fs[2] = 1/(8 tau): the per-thread constants of the loop, once
__global__ void ftv_scalars_kernel(const double* L, double beta, float* fs) {
  fs[0] = (float)(1.0 / *L);
  const float tau = (float)(beta / *L);
  fs[1] = tau;
  fs[2] = 1.f / (8.f * tau);
}
__global__ void ftv_fill_kernel(float* v, int64_t n, float value) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) v[k] = value;
}

}  // namespace

}  // namespace pyhst

using namespace pyhst;

static int tv_solver(const float* d_data, float* d_img, const pyhst_geom_t* g, float beta,
                     int32_t n_iter, int32_t n_inner, int32_t n_power, double* energy,
                     double* lipschitz, void* stream_, bool accelerated) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!d_data || !d_img || !g)
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_fista_tv: null pointer");
  if (!(beta >= 0.f) || n_iter < 0 || n_inner < 0 || n_power <= 0 || n_iter > (1 << 20))
    return set_error(PYHST_ERR_INVALID_ARG,
                     "pyhst_fista_tv: beta %g, n_iter %d, n_inner %d, n_power %d", (double)beta,
                     n_iter, n_inner, n_power);
  if (g->n_slices <= 0 || g->n_angles <= 0 || g->n_bins <= 0 || g->nx <= 0 || g->ny <= 0)
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_fista_tv: non-positive size");
  PYHST_TRY(require_sm100(nullptr));
  PYHST_CALL_SCOPE(stream);
  const int S = g->n_slices, nx = g->nx, ny = g->ny;
  const int64_t n_img = (int64_t)S * ny * nx, n1 = (int64_t)ny * nx;
  const int64_t n_rows = (int64_t)S * g->n_angles, n_sino = n_rows * g->n_bins;
  const int64_t data_pitch = g->sino_pitch ? g->sino_pitch : g->n_bins;
  if ((S + 0) > 65535) return set_error(PYHST_ERR_UNSUPPORTED, "pyhst_fista_tv: more than 65535 slices");

  // workspace: y, z, grad, 4 dual stacks, residual sinogram, scalars (nv, nw, L, energy[n_iter])
  const size_t img_bytes = ((size_t)n_img * 4 + 255) & ~(size_t)255;
  const size_t sino_bytes = ((size_t)n_sino * 4 + 255) & ~(size_t)255;
  const size_t sc_bytes = (size_t)(3 + n_iter) * 8;   // doubles: nv, nw, L, energy[n_iter]; then 4 floats
  // per-block partial sums of the reductions (deterministic two-stage sums)
  const int64_t n_part_img = (int64_t)((nx + FT_BX - 1) / FT_BX) * ((ny + FT_BY - 1) / FT_BY) * S;
  const int64_t res_gy = std::min<int64_t>((n_rows + FT_BY - 1) / FT_BY, 4096);
  const int64_t n_part_res = (int64_t)((g->n_bins + FT_BX - 1) / FT_BX) * res_gy;
  const int64_t n_part = std::max<int64_t>(std::max(n_part_img, n_part_res), 148 * 4);
  if (n_part > (1 << 30)) return set_error(PYHST_ERR_UNSUPPORTED, "pyhst_fista_tv: stack too large");
  const size_t part_off = (7 * img_bytes + sino_bytes + sc_bytes + 16 + 255) & ~(size_t)255;
  void* ws = nullptr;
  PYHST_TRY(get_workspace(WS_FISTA, part_off + (size_t)n_part * 8, &ws));
  char* base = static_cast<char*>(ws);
  float* y = reinterpret_cast<float*>(base);
  float* z = reinterpret_cast<float*>(base + img_bytes);
  float* gr = reinterpret_cast<float*>(base + 2 * img_bytes);
  float* p[4];
  for (int k = 0; k < 4; ++k) p[k] = reinterpret_cast<float*>(base + (3 + k) * img_bytes);
  float* r = reinterpret_cast<float*>(base + 7 * img_bytes);
  double* sc = reinterpret_cast<double*>(base + 7 * img_bytes + sino_bytes);
  double *d_nv = sc, *d_nw = sc + 1, *d_L = sc + 2, *d_e = sc + 3;
  float* d_fs = reinterpret_cast<float*>(sc + 3 + n_iter);
  double* d_part = reinterpret_cast<double*>(base + part_off);

  pyhst_geom_t g1 = *g, gs = *g;
  g1.n_slices = 1;
  g1.sino_pitch = 0;
  gs.sino_pitch = 0;
  const dim3 blk(FT_BX, FT_BY, 1);
  const dim3 grid_img((nx + FT_BX - 1) / FT_BX, (ny + FT_BY - 1) / FT_BY, S);
  const unsigned red_blocks = 148 * 4;

  // ---- L = 1.1 ||P^T P v|| / ||v|| after n_power iterations from v = 1, one slice (R17)
  PYHST_CUDA_TRY(cudaMemsetAsync(sc, 0, sc_bytes, stream));
  ftv_fill_kernel<<<(unsigned)((n1 + 255) / 256), 256, 0, stream>>>(y, n1, 1.f);
  for (int it = 0; it < n_power; ++it) {
    PYHST_CUDA_TRY(cudaMemsetAsync(sc, 0, 16, stream));
    ftv_sumsq_kernel<<<red_blocks, blk, 0, stream>>>(y, n1, d_part);
    ftv_reduce_kernel<<<1, 1024, 0, stream>>>(d_part, (int)red_blocks, d_nv);
    PYHST_TRY(pyhst_forward_project(y, r, &g1, 1.f, stream));
    PYHST_TRY(pyhst_backproject(r, gr, &g1, 1.f, stream));
    ftv_sumsq_kernel<<<red_blocks, blk, 0, stream>>>(gr, n1, d_part);
    ftv_reduce_kernel<<<1, 1024, 0, stream>>>(d_part, (int)red_blocks, d_nw);
    ftv_normalise_kernel<<<(unsigned)((n1 + 255) / 256), 256, 0, stream>>>(gr, y, n1, d_nv, d_nw, d_L);
  }
  ftv_scalars_kernel<<<1, 1, 0, stream>>>(d_L, (double)beta, d_fs);
  PYHST_CUDA_TRY(cudaGetLastError());

  // ---- FISTA (R19, R20): x0 = y0 = 0, t0 = 1
  PYHST_CUDA_TRY(cudaMemsetAsync(d_img, 0, (size_t)n_img * 4, stream));
  PYHST_CUDA_TRY(cudaMemsetAsync(y, 0, (size_t)n_img * 4, stream));
  const bool use_p = beta > 0.f && n_inner > 0;
  double t = 1.0;
  for (int k = 0; k < n_iter; ++k) {
    PYHST_TRY(pyhst_forward_project(y, r, &gs, 1.f, stream));
    {
      StageScope scope(ST_TV, stream);
      scope.kernels(2);
      dim3 grid((g->n_bins + FT_BX - 1) / FT_BX, (unsigned)res_gy, 1);
      ftv_residual_kernel<<<grid, blk, 0, stream>>>(r, d_data, data_pitch, g->n_bins, n_rows, d_part);
      ftv_reduce_kernel<<<1, 1024, 0, stream>>>(d_part, (int)n_part_res, d_e + k);
    }
    PYHST_TRY(pyhst_backproject(r, gr, &gs, 1.f, stream));
    StageScope scope(ST_TV, stream);
    scope.kernels(3 + (use_p ? (n_inner + FD_KMAX - 1) / FD_KMAX : 0));
    ftv_step_kernel<<<grid_img, blk, 0, stream>>>(y, gr, z, nx, ny, d_fs, (double)beta, d_part);
    ftv_reduce_kernel<<<1, 1024, 0, stream>>>(d_part, (int)n_part_img, d_e + k);
    int cur = 0;
    if (use_p) {
      // n_inner dual steps, FD_KMAX per launch; the first launch starts from p = 0 without reading it
      const dim3 grid_d((nx + FD_TX - 1) / FD_TX, (ny + FD_TY - 1) / FD_TY, S);
      for (int done = 0; done < n_inner;) {
        const int kk = std::min(FD_KMAX, n_inner - done);
        ftv_dual_fused_kernel<<<grid_d, FD_NT, 0, stream>>>(z, p[cur], p[cur + 1], p[2 - cur], p[3 - cur], nx,
                                                                 ny, d_fs, kk, done == 0 ? 1 : 0);
        cur = 2 - cur;
        done += kk;
      }
    }
    const double tn = 0.5 * (1.0 + std::sqrt(1.0 + 4.0 * t * t));
    ftv_finish_kernel<<<grid_img, blk, 0, stream>>>(z, p[cur], p[cur + 1], d_img, y, nx, ny, d_fs,
                                                    accelerated ? (float)((t - 1.0) / tn) : 0.f, use_p ? 1 : 0);
    t = tn;
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  if (energy || lipschitz) {
    std::vector<double> h((size_t)(3 + n_iter));
    PYHST_CUDA_TRY(cudaMemcpyAsync(h.data(), sc, sc_bytes, cudaMemcpyDeviceToHost, stream));
    PYHST_CUDA_TRY(cudaStreamSynchronize(stream));
    if (lipschitz) *lipschitz = h[2];
    if (energy)
      for (int k = 0; k < n_iter; ++k) energy[k] = h[(size_t)3 + k];
  }
  return PYHST_OK;
}

extern "C" int pyhst_fista_tv(const float* d_data, float* d_img, const pyhst_geom_t* g, float beta,
                              int32_t n_iter, int32_t n_inner, int32_t n_power, double* energy,
                              double* lipschitz, void* stream) {
  return tv_solver(d_data, d_img, g, beta, n_iter, n_inner, n_power, energy, lipschitz, stream, true);
}

// ISTA: no momentum, y_{k+1} = x_{k+1}
extern "C" int pyhst_ista_tv(const float* d_data, float* d_img, const pyhst_geom_t* g, float beta,
                             int32_t n_iter, int32_t n_inner, int32_t n_power, double* energy,
                             double* lipschitz, void* stream) {
  return tv_solver(d_data, d_img, g, beta, n_iter, n_inner, n_power, energy, lipschitz, stream, false);
}
