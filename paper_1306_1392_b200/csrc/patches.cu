// NEXT row N3: overlapping-patch dictionary reconstruction
// (sec. 3.2, eq. 4-9) and Algorithm 1 (L201-L228); readings R16, R22-R24 of DESIGN.md.
//
//   x_i = sum_p 1^c_p(i) sum_k w_kp phi_k(i - r_p)                                          (eq. 7)
//   f(w) = ||y - Pi x||^2 + rho sum_{p,i} 1_p(i) (x_i - sum_k w_kp phi_k(i - r_p))^2         (eq. 8)
//
// Algorithm 1 on the device, one stack of independent slices per call:
//   P  <- W D                     patch_gemm_kernel<false>   ([N x Nc] [Nc x m^2], the paper's first GEMM)
//   X, S, similarity sum          patch_compose_kernel       (per pixel: core patch (eq. 5-6), the patches
//                                                             that cover it -- a gather, no atomics)
//   R  <- Pi^T (Pi X - y)         pyhst_forward_project, patch_residual_kernel, pyhst_backproject  (R16)
//   P' <- Algorithm 1's update    patch_pprime_kernel
//   G  <- 2 P' D^T                patch_gemm_kernel<true>    (the second GEMM)
// The core map C_j and the cover count N_v(j) are evaluated per pixel in integer arithmetic (the
// doubled L1 distance |2i - 2o - (m-1)| is exact), never stored.
// The two GEMMs are tall and skinny (N ~ 1e5 patches, K and the other side 64..256): the tcgen05
// 3xTF32 tensor-core kernel of patch_gemm_tc.cu when the shapes allow it, else the FP32 SIMT tiles
// here; both keep the gradient's parity bar (rel-L2 2e-5).
#include <algorithm>
#include <cmath>
#include <vector>

#include "common.h"

namespace pyhst {

namespace {

struct PatchGrid {
  int ny, nx, m, st, na, nb;
};

__host__ __device__ inline int pg_count(int n, int m, int st) { return n <= m ? 1 : (n - m + st - 1) / st + 1; }
__host__ __device__ inline int pg_origin(int a, int n, int m, int st) {
  const int o = a * st;
  return o > n - m ? n - m : o;
}
// patch (along one axis) whose centre o + (m-1)/2 is closest to pixel i; smallest index among equals (R22)
__device__ __forceinline__ int pg_core_1d(int i, int n, int m, int st, int cnt) {
  int a0 = (2 * i - (m - 1) + st) / (2 * st);   // ~ round((i - (m-1)/2) / st)
  a0 = max(0, min(cnt - 1, a0));
  int best = 0x7fffffff, besta = 0;
#pragma unroll
  for (int d = -2; d <= 2; ++d) {
    const int a = a0 + d;
    if (a < 0 || a >= cnt) continue;
    const int dist = abs(2 * i - 2 * pg_origin(a, n, m, st) - (m - 1));
    if (dist < best) { best = dist; besta = a; }
  }
  // the clamped last patch may sit closer than its index suggests
  {
    const int a = cnt - 1;
    const int dist = abs(2 * i - 2 * pg_origin(a, n, m, st) - (m - 1));
    if (dist < best || (dist == best && a < besta)) { best = dist; besta = a; }
  }
  return besta;
}
// range [lo, hi] of patches (along one axis) that contain pixel i
__device__ __forceinline__ void pg_cover_1d(int i, int n, int m, int st, int cnt, int* lo, int* hi) {
  int l = (i - m + 1 + st - 1) / st;
  if (i - m + 1 < 0) l = 0;
  int h = i / st;
  l = max(0, l - 1);
  h = min(cnt - 1, h + 1);
  while (l <= h && !(pg_origin(l, n, m, st) <= i && i < pg_origin(l, n, m, st) + m)) ++l;
  while (h >= l && !(pg_origin(h, n, m, st) <= i && i < pg_origin(h, n, m, st) + m)) --h;
  *lo = l;
  *hi = h;
}

// ---- C[M x N] = alpha * A[M x K] * B, B = Bm[K x N] (TRANS_B = false) or Bm[N x K]^T (true); row-major,
// FP32 FMA, 64 x 64 tile per block, 4 x 4 outputs per thread, K in steps of 16 through shared memory
constexpr int GM_BM = 64, GM_BN = 64, GM_BK = 16, GM_NT = 256;

template <bool TRANS_B>
__global__ void __launch_bounds__(GM_NT)
patch_gemm_kernel(const float* __restrict__ A, const float* __restrict__ Bm, float* __restrict__ C, int64_t M,
                  int N, int K, float alpha) {
  __shared__ float As[GM_BK][GM_BM + 4];
  __shared__ float Bs[GM_BK][GM_BN + 4];
  const int64_t m0 = (int64_t)blockIdx.x * GM_BM;
  const int n0 = blockIdx.y * GM_BN;
  const int64_t z = blockIdx.z;
  A += z * M * K;
  C += z * M * N;
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  float acc[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;
  for (int k0 = 0; k0 < K; k0 += GM_BK) {
    // A tile: 64 rows x 16 k
#pragma unroll
    for (int e = tid; e < GM_BM * GM_BK; e += GM_NT) {
      const int r = e / GM_BK, k = e - r * GM_BK;
      const int64_t gr = m0 + r;
      As[k][r] = (gr < M && k0 + k < K) ? A[gr * K + k0 + k] : 0.f;
    }
#pragma unroll
    for (int e = tid; e < GM_BN * GM_BK; e += GM_NT) {
      int k, c;
      if (TRANS_B) { c = e / GM_BK; k = e - c * GM_BK; } else { k = e / GM_BN; c = e - k * GM_BN; }
      float v = 0.f;
      if (n0 + c < N && k0 + k < K) v = TRANS_B ? Bm[(int64_t)(n0 + c) * K + k0 + k] : Bm[(int64_t)(k0 + k) * N + n0 + c];
      Bs[k][c] = v;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < GM_BK; ++k) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[k][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[k][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int64_t gr = m0 + ty * 4 + i;
    if (gr >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int gc = n0 + tx * 4 + j;
      if (gc < N) C[gr * N + gc] = alpha * acc[i][j];
    }
  }
}

// block-wide sum into part[linear block id] (fixed order)
__device__ __forceinline__ void block_store_sum(double v, double* part) {
  __shared__ double wsum[8];
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

__global__ void __launch_bounds__(1024) sum_partials_kernel(const double* __restrict__ part, int n, double scale,
                                                            double* dst) {
  __shared__ double sh[1024];
  double s = 0.0;
  for (int k = threadIdx.x; k < n; k += 1024) s += part[k];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) *dst += scale * sh[0];
}

// per pixel j: X_j = P[C_j][j - r_C] (eq. 7), S_j = sum of the covering patches' values at j,
// part = sum_j sum_{p covers j} (X_j - P_p(j))^2   (the similarity term of eq. 8)
__global__ void __launch_bounds__(256)
patch_compose_kernel(const float* __restrict__ Pm, PatchGrid pg, float* __restrict__ X, float* __restrict__ S,
                     double* __restrict__ part, const short4* __restrict__ pix) {
  const int jx = blockIdx.x * 32 + threadIdx.x, jy = blockIdx.y * 8 + threadIdx.y;
  const int64_t s = blockIdx.z;
  const int mm = pg.m * pg.m;
  const float* Ps = Pm + s * (int64_t)pg.na * pg.nb * mm;
  double sim = 0.0;
  if (jx < pg.nx && jy < pg.ny) {
    // per-axis pixel tables (patch_axis_tables_kernel): x = core patch, y / z = first / last covering patch
    const short4 ty = pix[jy], tx = pix[pg.ny + jx];
    const int ca = ty.x, cb = tx.x;
    const int coy = pg_origin(ca, pg.ny, pg.m, pg.st), cox = pg_origin(cb, pg.nx, pg.m, pg.st);
    const float x = Ps[(int64_t)(ca * pg.nb + cb) * mm + (jy - coy) * pg.m + (jx - cox)];
    float sum = 0.f;
    for (int a = ty.y; a <= ty.z; ++a) {
      const int oy = pg_origin(a, pg.ny, pg.m, pg.st);
      for (int b = tx.y; b <= tx.z; ++b) {
        const int ox = pg_origin(b, pg.nx, pg.m, pg.st);
        const float v = Ps[(int64_t)(a * pg.nb + b) * mm + (jy - oy) * pg.m + (jx - ox)];
        sum += v;
        sim += (double)(x - v) * (double)(x - v);
      }
    }
    const int64_t j = s * (int64_t)pg.ny * pg.nx + (int64_t)jy * pg.nx + jx;
    X[j] = x;
    S[j] = sum;
  }
  if (part) block_store_sum(sim, part);
}

// r -= data (r contiguous, data pitched); part = sum r^2
__global__ void __launch_bounds__(256)
patch_residual_kernel(float* __restrict__ r, const float* __restrict__ data, int64_t data_pitch, int n_bins,
                      int64_t n_rows, double* __restrict__ part) {
  const int b = blockIdx.x * 32 + threadIdx.x;
  double acc = 0.0;
  for (int64_t row = (int64_t)blockIdx.y * 8 + threadIdx.y; row < n_rows; row += (int64_t)gridDim.y * 8) {
    if (b < n_bins) {
      const float v = r[row * n_bins + b] - data[row * data_pitch + b];
      r[row * n_bins + b] = v;
      acc += (double)v * (double)v;
    }
  }
  if (part) block_store_sum(acc, part);
}

// Whether a pixel of a patch is a core pixel of that patch, and how many patches cover it, factorises over the two
// axes.  tab[axis][idx][off] (32 offsets per patch index; axis 0: rows, na entries; axis 1: columns, nb entries):
// bit 7 = "the pixel at offset off of patch idx has idx as its core patch along this axis", bits 0..6 = patches
// that contain it along this axis.  (na + nb) * 32 bytes, rebuilt per call by one small kernel.
__global__ void patch_axis_tables_kernel(PatchGrid pg, unsigned char* __restrict__ tab, short4* __restrict__ pix) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int total = (pg.na + pg.nb) * 32;
  if (t < pg.ny + pg.nx) {   // per pixel and axis: core patch, first and last covering patch (patch_compose_kernel)
    const int axis = t >= pg.ny ? 1 : 0, j = axis ? t - pg.ny : t;
    const int n = axis ? pg.nx : pg.ny, cnt = axis ? pg.nb : pg.na;
    int lo, hi;
    pg_cover_1d(j, n, pg.m, pg.st, cnt, &lo, &hi);
    pix[t] = make_short4((short)pg_core_1d(j, n, pg.m, pg.st, cnt), (short)lo, (short)hi, 0);
  }
  if (t >= total) return;
  const int idx_all = t >> 5, off = t & 31;
  const int axis = idx_all >= pg.na ? 1 : 0, idx = axis ? idx_all - pg.na : idx_all;
  unsigned char v = 0;
  if (off < pg.m) {
    const int n = axis ? pg.nx : pg.ny, cnt = axis ? pg.nb : pg.na;
    const int j = pg_origin(idx, n, pg.m, pg.st) + off;
    int lo, hi;
    pg_cover_1d(j, n, pg.m, pg.st, cnt, &lo, &hi);
    v = (unsigned char)((hi - lo + 1) | (pg_core_1d(j, n, pg.m, pg.st, cnt) == idx ? 0x80 : 0));
  }
  tab[t] = v;
}

// Algorithm 1: P'_{p i} = [p == C_j] (R_j + rho (N_v X_j - S_j)) + rho (P_{p i} - X_j), j = r_p + i
// One thread per element, patches of one slice along blockIdx.x; the core / cover logic comes from the axis tables
// (2 byte loads instead of 2 m^2-fold evaluated integer routines): the kernel runs at the speed of its two streams
// (P in, P' out).
__global__ void __launch_bounds__(256)
patch_pprime_kernel(const float* __restrict__ Pm, const float* __restrict__ X, const float* __restrict__ S,
                    const float* __restrict__ R, PatchGrid pg, float rho, float* __restrict__ Pp,
                    const unsigned char* __restrict__ tab) {
  const int m = pg.m, mm = m * m;
  const int N = pg.na * pg.nb;
  const int64_t s = blockIdx.y;
  const uint32_t e = blockIdx.x * 256u + threadIdx.x;       // element of the slice: patch * mm + i  (< 2^32)
  if (e >= (uint32_t)N * (uint32_t)mm) return;
  const uint32_t p = e / (uint32_t)mm, i = e - p * (uint32_t)mm;
  const uint32_t a = p / (uint32_t)pg.nb, b = p - a * (uint32_t)pg.nb;
  const uint32_t iy = i / (uint32_t)m, ix = i - iy * (uint32_t)m;
  const int jy = pg_origin((int)a, pg.ny, m, pg.st) + (int)iy, jx = pg_origin((int)b, pg.nx, m, pg.st) + (int)ix;
  const int64_t j = s * (int64_t)pg.ny * pg.nx + (int64_t)jy * pg.nx + jx;
  const int64_t k = s * (int64_t)N * mm + e;
  const float x = X[j];
  float v = rho * (Pm[k] - x);
  const unsigned ty = tab[a * 32u + iy], tx = tab[(pg.na + b) * 32u + ix];
  if (ty & tx & 0x80u) {
    const float nv = (float)((ty & 0x7fu) * (tx & 0x7fu));
    v += R[j] + rho * fmaf(nv, x, -S[j]);
  }
  Pp[k] = v;
}

// FISTA on the coefficients: u = v - g / Lw; w+ = shrink(u, beta / Lw); v = w+ + mom (w+ - w); w = w+
__global__ void __launch_bounds__(256)
patch_update_kernel(float* __restrict__ w, float* __restrict__ v, const float* __restrict__ g, int64_t n,
                    const float* __restrict__ fs, float mom) {
  const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (k >= n) return;
  const float inv_l = fs[0], thr = fs[1];
  const float u = fmaf(-g[k], inv_l, v[k]);
  const float a = fabsf(u) - thr;
  const float wn = a > 0.f ? copysignf(a, u) : 0.f;
  const float wo = w[k];
  v[k] = fmaf(mom, wn - wo, wn);
  w[k] = wn;
}

__global__ void __launch_bounds__(256) abs_sum_kernel(const float* __restrict__ v, int64_t n, double* __restrict__ part) {
  double s = 0.0;
  for (int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x; k < n; k += (int64_t)gridDim.x * 256) s += fabs((double)v[k]);
  block_store_sum(s, part);
}
__global__ void __launch_bounds__(256) sq_sum_kernel(const float* __restrict__ v, int64_t n, double* __restrict__ part) {
  double s = 0.0;
  for (int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x; k < n; k += (int64_t)gridDim.x * 256) s += (double)v[k] * (double)v[k];
  block_store_sum(s, part);
}
__global__ void fill_kernel(float* v, int64_t n, float value) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) v[k] = value;
}
// v = g / sqrt(*ng); *L = 1.1 sqrt(*ng / *nv)
__global__ void normalise_kernel(const float* __restrict__ g, float* __restrict__ v, int64_t n, const double* nv,
                                 const double* ng, double* L) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const double s = sqrt(*ng);
  if (k < n) v[k] = (float)((double)g[k] / s);
  if (k == 0) *L = 1.1 * s / sqrt(*nv);
}
__global__ void scalars_kernel(const double* L, double beta, float* fs) {
  fs[0] = (float)(1.0 / *L);
  fs[1] = (float)(beta / *L);
}

// C[z][M x N] = alpha A[z][M x K] B for every slice z; B = Bm[K x N] or, trans_b, Bm[N x K]^T
int patch_gemm(const float* A, const float* Bm, float* C, int64_t M, int N, int K, float alpha, bool trans_b, int S,
               cudaStream_t stream) {
  const int variant = patch_gemm_variant();
  const bool aligned = ((reinterpret_cast<uintptr_t>(A) | reinterpret_cast<uintptr_t>(Bm) |
                         reinterpret_cast<uintptr_t>(C)) & 15) == 0 && (M * K) % 4 == 0 && (M * N) % 4 == 0;
  const bool tc_ok = aligned && patch_gemm_tc_covers(N, K);
  if (variant == 2 && !tc_ok)
    return set_error(PYHST_ERR_UNSUPPORTED, "tensor-core patch GEMM does not cover N = %d, K = %d", N, K);
  if (variant != 1 && tc_ok) return launch_patch_gemm_tc(A, Bm, C, M, N, K, alpha, trans_b, S, stream);
  const dim3 grid((unsigned)((M + GM_BM - 1) / GM_BM), (N + GM_BN - 1) / GM_BN, S);
  if (trans_b) patch_gemm_kernel<true><<<grid, GM_NT, 0, stream>>>(A, Bm, C, M, N, K, alpha);
  else patch_gemm_kernel<false><<<grid, GM_NT, 0, stream>>>(A, Bm, C, M, N, K, alpha);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

struct PatchWs {
  float *P, *Pp, *X, *S, *R, *r;
  double* part;
  unsigned char* tab;   // axis tables of patch_pprime_kernel, (na + nb) * 32 bytes
  short4* pix;          // per-pixel axis tables of patch_compose_kernel, ny + nx entries
  int64_t n_part;
  size_t bytes;
};

size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }

// lays the gradient's scratch arrays out in one block starting at `base` (base may be NULL to size it)
PatchWs carve(char* base, int S, const PatchGrid& pg, int n_angles, int n_bins) {
  PatchWs w{};
  const int64_t N = (int64_t)pg.na * pg.nb, mm = (int64_t)pg.m * pg.m, npix = (int64_t)pg.ny * pg.nx;
  size_t off = 0;
  auto take = [&](size_t bytes) { char* p = base ? base + off : nullptr; off += align256(bytes); return p; };
  w.P = reinterpret_cast<float*>(take((size_t)S * N * mm * 4));
  w.Pp = reinterpret_cast<float*>(take((size_t)S * N * mm * 4));
  w.X = reinterpret_cast<float*>(take((size_t)S * npix * 4));
  w.S = reinterpret_cast<float*>(take((size_t)S * npix * 4));
  w.R = reinterpret_cast<float*>(take((size_t)S * npix * 4));
  w.r = reinterpret_cast<float*>(take((size_t)S * n_angles * n_bins * 4));
  const int64_t g_img = (int64_t)((pg.nx + 31) / 32) * ((pg.ny + 7) / 8) * S;
  const int64_t g_res = (int64_t)((n_bins + 31) / 32) * std::min<int64_t>(((int64_t)S * n_angles + 7) / 8, 4096);
  w.n_part = std::max<int64_t>(std::max(g_img, g_res), 1024);
  w.part = reinterpret_cast<double*>(take((size_t)w.n_part * 8));
  w.tab = reinterpret_cast<unsigned char*>(take((size_t)(pg.na + pg.nb) * 32));
  w.pix = reinterpret_cast<short4*>(take((size_t)(pg.ny + pg.nx) * sizeof(short4)));
  w.bytes = off;
  return w;
}

// One evaluation of Algorithm 1 for the whole stack.  d_f (device double, nullable) receives
// f(W) = ||y - Pi X||^2 + rho * similarity, accumulated with += (zero it first).
int patch_gradient_device(const float* d_W, const float* d_D, const float* d_data, const pyhst_geom_t* g,
                          const PatchGrid& pg, int n_atoms, float rho, const PatchWs& w, float* d_G, double* d_f,
                          cudaStream_t stream) {
  const int S = g->n_slices;
  const int64_t N = (int64_t)pg.na * pg.nb;
  const int mm = pg.m * pg.m;
  const int64_t data_pitch = g->sino_pitch ? g->sino_pitch : g->n_bins;
  const int64_t n_rows = (int64_t)S * g->n_angles;
  // P <- W D
  PYHST_TRY(patch_gemm(d_W, d_D, w.P, N, mm, n_atoms, 1.f, false, S, stream));
  // X, S, similarity
  const dim3 blk(32, 8, 1), grid_img((pg.nx + 31) / 32, (pg.ny + 7) / 8, S);
  {
    const int n_tab = std::max((pg.na + pg.nb) * 32, pg.ny + pg.nx);
    patch_axis_tables_kernel<<<(n_tab + 255) / 256, 256, 0, stream>>>(pg, w.tab, w.pix);
  }
  patch_compose_kernel<<<grid_img, blk, 0, stream>>>(w.P, pg, w.X, w.S, d_f ? w.part : nullptr, w.pix);
  if (d_f) sum_partials_kernel<<<1, 1024, 0, stream>>>(w.part, (int)(grid_img.x * grid_img.y * grid_img.z), (double)rho, d_f);
  PYHST_CUDA_TRY(cudaGetLastError());
  // R <- Pi^T (Pi X - y)
  pyhst_geom_t gs = *g;
  gs.sino_pitch = 0;
  PYHST_TRY(pyhst_forward_project(w.X, w.r, &gs, 1.f, stream));
  const dim3 grid_res((g->n_bins + 31) / 32, (unsigned)std::min<int64_t>((n_rows + 7) / 8, 4096), 1);
  patch_residual_kernel<<<grid_res, blk, 0, stream>>>(w.r, d_data, data_pitch, g->n_bins, n_rows, d_f ? w.part : nullptr);
  if (d_f) sum_partials_kernel<<<1, 1024, 0, stream>>>(w.part, (int)(grid_res.x * grid_res.y), 1.0, d_f);
  PYHST_CUDA_TRY(cudaGetLastError());
  if (!d_G) return PYHST_OK;
  PYHST_TRY(pyhst_backproject(w.r, w.R, &gs, 1.f, stream));
  // P' and G <- 2 P' D^T
  if (N * mm >= ((int64_t)1 << 32) || N >= ((int64_t)1 << 31))
    return set_error(PYHST_ERR_UNSUPPORTED, "patch: more than 2^32 patch elements per slice");
  patch_pprime_kernel<<<dim3((unsigned)((N * mm + 255) / 256), (unsigned)S), 256, 0, stream>>>(w.P, w.X, w.S, w.R, pg, rho, w.Pp, w.tab);
  PYHST_TRY(patch_gemm(w.Pp, d_D, d_G, N, n_atoms, mm, 2.f, true, S, stream));
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

int check_patch_args(const pyhst_geom_t* g, const pyhst_patch_t* pp, PatchGrid* pg) {
  if (!g || !pp) return set_error(PYHST_ERR_INVALID_ARG, "patch: geometry / patch parameters are NULL");
  if (g->n_slices <= 0 || g->n_angles <= 0 || g->n_bins <= 0 || g->nx <= 0 || g->ny <= 0)
    return set_error(PYHST_ERR_INVALID_ARG, "patch: non-positive size");
  if (pp->m <= 0 || pp->stride <= 0 || pp->stride > pp->m || pp->n_atoms <= 0 || !(pp->rho >= 0.f))
    return set_error(PYHST_ERR_INVALID_ARG, "patch: m %d, stride %d, n_atoms %d, rho %g", pp->m, pp->stride,
                     pp->n_atoms, (double)pp->rho);
  if (g->ny < pp->m || g->nx < pp->m) return set_error(PYHST_ERR_INVALID_ARG, "patch: image smaller than a patch");
  if (pp->m > 32 || g->n_slices > 65535) return set_error(PYHST_ERR_UNSUPPORTED, "patch: m > 32 or more than 65535 slices");
  pg->ny = g->ny; pg->nx = g->nx; pg->m = pp->m; pg->st = pp->stride;
  pg->na = pg_count(g->ny, pp->m, pp->stride);
  pg->nb = pg_count(g->nx, pp->m, pp->stride);
  return PYHST_OK;
}

}  // namespace

}  // namespace pyhst

using namespace pyhst;

extern "C" int pyhst_patch_grid(int32_t ny, int32_t nx, int32_t m, int32_t stride, int32_t* na, int32_t* nb) {
  if (m <= 0 || stride <= 0 || stride > m || ny < m || nx < m || !na || !nb)
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_patch_grid: bad argument");
  *na = pg_count(ny, m, stride);
  *nb = pg_count(nx, m, stride);
  return PYHST_OK;
}

extern "C" int pyhst_patch_gradient(const float* d_W, const float* d_D, const float* d_data, const pyhst_geom_t* g,
                                    const pyhst_patch_t* pp, float* d_G, float* d_X, double* h_fval, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!d_W || !d_D || !d_data) return set_error(PYHST_ERR_INVALID_ARG, "pyhst_patch_gradient: null pointer");
  PatchGrid pg;
  PYHST_TRY(check_patch_args(g, pp, &pg));
  PYHST_TRY(require_sm100(nullptr));
  PYHST_CALL_SCOPE(stream);
  PatchWs w = carve(nullptr, g->n_slices, pg, g->n_angles, g->n_bins);
  void* ws = nullptr;
  PYHST_TRY(get_workspace(WS_FISTA, w.bytes + 64, &ws));
  w = carve(static_cast<char*>(ws), g->n_slices, pg, g->n_angles, g->n_bins);
  double* d_f = reinterpret_cast<double*>(static_cast<char*>(ws) + w.bytes);
  if (h_fval) PYHST_CUDA_TRY(cudaMemsetAsync(d_f, 0, 8, stream));
  PYHST_TRY(patch_gradient_device(d_W, d_D, d_data, g, pg, pp->n_atoms, pp->rho, w, d_G, h_fval ? d_f : nullptr, stream));
  if (d_X)
    PYHST_CUDA_TRY(cudaMemcpyAsync(d_X, w.X, (size_t)g->n_slices * g->ny * g->nx * 4, cudaMemcpyDeviceToDevice, stream));
  if (h_fval) {
    PYHST_CUDA_TRY(cudaMemcpyAsync(h_fval, d_f, 8, cudaMemcpyDeviceToHost, stream));
    PYHST_CUDA_TRY(cudaStreamSynchronize(stream));
  }
  return PYHST_OK;
}

extern "C" int pyhst_patch_fista(const float* d_D, const float* d_data, const pyhst_geom_t* g, const pyhst_patch_t* pp,
                                 float beta, int32_t n_iter, int32_t n_power, float* d_W, float* d_X, double* energy,
                                 double* lipschitz, void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  if (!d_D || !d_data || !d_W) return set_error(PYHST_ERR_INVALID_ARG, "pyhst_patch_fista: null pointer");
  if (!(beta >= 0.f) || n_iter < 0 || n_power <= 0 || n_iter > (1 << 20))
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_patch_fista: beta %g, n_iter %d, n_power %d", (double)beta, n_iter,
                     n_power);
  PatchGrid pg;
  PYHST_TRY(check_patch_args(g, pp, &pg));
  PYHST_TRY(require_sm100(nullptr));
  PYHST_CALL_SCOPE(stream);
  const int S = g->n_slices;
  const int64_t n_w = (int64_t)S * pg.na * pg.nb * pp->n_atoms;
  PatchWs w = carve(nullptr, S, pg, g->n_angles, g->n_bins);
  const size_t w_bytes = align256((size_t)n_w * 4);
  const size_t zero_bytes = align256((size_t)S * g->n_angles * g->n_bins * 4);
  const size_t sc_bytes = align256((size_t)(3 + n_iter) * 8 + 16);
  void* ws = nullptr;
  PYHST_TRY(get_workspace(WS_FISTA, w.bytes + 2 * w_bytes + zero_bytes + sc_bytes, &ws));
  char* base = static_cast<char*>(ws);
  w = carve(base, S, pg, g->n_angles, g->n_bins);
  float* v = reinterpret_cast<float*>(base + w.bytes);
  float* G = reinterpret_cast<float*>(base + w.bytes + w_bytes);
  float* zero = reinterpret_cast<float*>(base + w.bytes + 2 * w_bytes);
  double* sc = reinterpret_cast<double*>(base + w.bytes + 2 * w_bytes + zero_bytes);
  double *d_nv = sc, *d_ng = sc + 1, *d_L = sc + 2, *d_e = sc + 3;
  float* d_fs = reinterpret_cast<float*>(sc + 3 + n_iter);
  const unsigned red_blocks = 1024;
  const unsigned ew_blocks = (unsigned)((n_w + 255) / 256);
  pyhst_geom_t gz = *g;
  gz.sino_pitch = 0;

  // ---- R23: Lw = 1.1 ||H v|| / ||v|| after n_power iterations from v = 1 (H v = grad f(v), zero data)
  PYHST_CUDA_TRY(cudaMemsetAsync(sc, 0, sc_bytes, stream));
  PYHST_CUDA_TRY(cudaMemsetAsync(zero, 0, zero_bytes, stream));
  fill_kernel<<<ew_blocks, 256, 0, stream>>>(v, n_w, 1.f);
  for (int it = 0; it < n_power; ++it) {
    PYHST_CUDA_TRY(cudaMemsetAsync(sc, 0, 16, stream));
    sq_sum_kernel<<<red_blocks, 256, 0, stream>>>(v, n_w, w.part);
    sum_partials_kernel<<<1, 1024, 0, stream>>>(w.part, (int)red_blocks, 1.0, d_nv);
    PYHST_TRY(patch_gradient_device(v, d_D, zero, &gz, pg, pp->n_atoms, pp->rho, w, G, nullptr, stream));
    sq_sum_kernel<<<red_blocks, 256, 0, stream>>>(G, n_w, w.part);
    sum_partials_kernel<<<1, 1024, 0, stream>>>(w.part, (int)red_blocks, 1.0, d_ng);
    normalise_kernel<<<ew_blocks, 256, 0, stream>>>(G, v, n_w, d_nv, d_ng, d_L);
  }
  scalars_kernel<<<1, 1, 0, stream>>>(d_L, (double)beta, d_fs);
  PYHST_CUDA_TRY(cudaGetLastError());

  // ---- FISTA (R24): w0 = v0 = 0, t0 = 1
  PYHST_CUDA_TRY(cudaMemsetAsync(d_W, 0, (size_t)n_w * 4, stream));
  PYHST_CUDA_TRY(cudaMemsetAsync(v, 0, (size_t)n_w * 4, stream));
  double t = 1.0;
  for (int k = 0; k < n_iter; ++k) {
    PYHST_TRY(patch_gradient_device(v, d_D, d_data, g, pg, pp->n_atoms, pp->rho, w, G, d_e + k, stream));
    abs_sum_kernel<<<red_blocks, 256, 0, stream>>>(v, n_w, w.part);
    sum_partials_kernel<<<1, 1024, 0, stream>>>(w.part, (int)red_blocks, (double)beta, d_e + k);
    const double tn = 0.5 * (1.0 + std::sqrt(1.0 + 4.0 * t * t));
    patch_update_kernel<<<ew_blocks, 256, 0, stream>>>(d_W, v, G, n_w, d_fs, (float)((t - 1.0) / tn));
    t = tn;
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  if (d_X) {  // the image of eq. 7 at the final coefficients
    PYHST_TRY(patch_gemm(d_W, d_D, w.P, (int64_t)pg.na * pg.nb, pg.m * pg.m, pp->n_atoms, 1.f, false, S, stream));
    {
      const int n_tab = std::max((pg.na + pg.nb) * 32, pg.ny + pg.nx);
      patch_axis_tables_kernel<<<(n_tab + 255) / 256, 256, 0, stream>>>(pg, w.tab, w.pix);
    }
    patch_compose_kernel<<<dim3((pg.nx + 31) / 32, (pg.ny + 7) / 8, S), dim3(32, 8, 1), 0, stream>>>(w.P, pg, d_X, w.S,
                                                                                                    nullptr, w.pix);
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  if (energy || lipschitz) {
    std::vector<double> h((size_t)(3 + n_iter));
    PYHST_CUDA_TRY(cudaMemcpyAsync(h.data(), sc, (size_t)(3 + n_iter) * 8, cudaMemcpyDeviceToHost, stream));
    PYHST_CUDA_TRY(cudaStreamSynchronize(stream));
    if (lipschitz) *lipschitz = h[2];
    if (energy)
      for (int k = 0; k < n_iter; ++k) energy[k] = h[(size_t)3 + k];
  }
  return PYHST_OK;
}
