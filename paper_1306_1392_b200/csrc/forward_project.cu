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
#include <algorithm>
#include <cmath>
#include <cstring>

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


// ==========================================================================================
// Banded forward projector (the product path).
//
// A block owns NB consecutive detector bins of up to NPJ projections of one walk class and one
// slice group (4 slices interleaved as float4).  It walks the image lines in bands of RB lines:
// per band the window of the interleaved image that the block's strips cross is staged into
// shared memory with one TMA bulk copy per line (mbarrier-signalled, double-buffered); every
// thread then gathers, for each of its (bin, projection) pairs and each line of the band, the NC
// pixels that can lie inside the strip |t - b| < 1, with weights 1 - |cu| |u - u*| (FP32 FMA),
// and accumulates 4 slices in registers.  No atomics: each output is written once.
// The strip centre u* is evaluated in double once per (pair, band) relative to the window and
// split into an integer and a fraction in [-1/2, 1/2]; only the fraction is carried in FP32 (R11).
// ==========================================================================================
namespace {

constexpr int FB_NB = 128;    // bins per block
constexpr int FB_NPJ = 16;    // projections per block (at most)
constexpr int FB_RB = 8;      // lines per band
constexpr int FB_NT = 256;    // threads: 8 warps x (16 bins x 2 projection parities), 8 pairs per thread
constexpr int FB_PAIRS = FB_NB * FB_NPJ / FB_NT;
constexpr int FB_HDR = 1024;  // 2 mbarriers, 2 origins, NPJ x FpProjD
constexpr int FB_WMAX = 416;  // window capacity (float4 per line): 2 x 8 x 416 x 16 B = 104 KB

struct XiDims { int32_t nv, nu, zpad; };

// MINB = blocks per SM the register budget is cut for (3: 80 registers; 4: 64, for windows small
// enough that four blocks fit in shared memory).  n_split > 1: blockIdx.z = group * n_split + h and
// the block walks only the h-th part of the bands; part h > 0 writes its sums to part[h - 1] (same
// layout as sino, pitch part_pitch), fp_split_combine_kernel adds them -- small scans then fill the GPU.
template <int NC, int MINB, bool SPLIT>
__global__ void __launch_bounds__(FB_NT, MINB)
fp_band_kernel(const float4* __restrict__ xi_rows, const float4* __restrict__ xi_cols, XiDims dr,
               XiDims dc, float* __restrict__ sino, int64_t pitch, int S, int P, int B, float scale,
               const FpProjD* __restrict__ projs, const FpChunk* __restrict__ chunks, int W,
               int n_split, float* __restrict__ part, int64_t part_pitch, int64_t part_stride, int n_tab) {
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);        // [2]
  int* sorigin = reinterpret_cast<int*>(smem + 16);          // [2]
  FpProjD* sproj = reinterpret_cast<FpProjD*>(smem + 64);    // [FB_NPJ]
  float4* buf = reinterpret_cast<float4*>(smem + FB_HDR);    // [2][FB_RB][W]

  const int tid = threadIdx.x, lane = tid & 31;
  const FpChunk ck = chunks[blockIdx.y];
  const int g = SPLIT ? blockIdx.z / n_split : blockIdx.z, hs = SPLIT ? blockIdx.z - g * n_split : 0;
  const int b0 = blockIdx.x * FB_NB;
  const XiDims d = ck.cls ? dc : dr;
  const int64_t line_f4 = (int64_t)d.nu + 2 * d.zpad;
  const float4* xi = (ck.cls ? xi_cols : xi_rows) + (int64_t)g * d.nv * line_f4;
  const int n_bands_all = (d.nv + FB_RB - 1) / FB_RB;
  const int k0 = SPLIT ? (int)((int64_t)hs * n_bands_all / n_split) : 0;
  const int n_bands = SPLIT ? (int)((int64_t)(hs + 1) * n_bands_all / n_split) : n_bands_all;
  const uint32_t row_bytes = (uint32_t)W * 16u;

  if (tid < ck.count) sproj[tid] = projs[ck.first + tid];
  if (tid == 0) {
    mbar_init(&full[0], FB_RB);
    mbar_init(&full[1], FB_RB);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // warp 0: window origin of band k (min over the chunk's strips at the band's four corners, in
  // double), then one bulk copy per line of the band
  auto produce = [&](int k) {
    const int vb = k * FB_RB;
    const int rows = min(FB_RB, d.nv - vb);
    double lo = 1e300;
    if (lane < ck.count) {
      const FpProjD pj = sproj[lane];
      const double ua = fma((double)b0, pj.inv_cu, pj.k0);
      const double ub = fma((double)(b0 + FB_NB - 1), pj.inv_cu, pj.k0);
      const double va = pj.sD * (double)vb, vz = pj.sD * (double)(vb + rows - 1);
      lo = fmin(fmin(ua, ub) + fmin(va, vz), lo) - (double)pj.hw;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    double of = floor(lo) - 1.0;
    of = fmax(of, -(double)d.zpad);
    of = fmin(of, (double)(d.nu + d.zpad - W));
    const int origin = (int)of;
    uint64_t* bar = &full[(k - k0) & 1];
    if (lane == 0) sorigin[(k - k0) & 1] = origin;
    if (lane < FB_RB) {
      if (lane < rows) {
        mbar_arrive_expect_tx(bar, row_bytes);
        bulk_g2s(buf + (((k - k0) & 1) * FB_RB + lane) * W,
                 xi + (int64_t)(vb + lane) * line_f4 + (origin + d.zpad), row_bytes, bar);
      } else {
        mbar_arrive(bar);
      }
    }
  };

  if (tid < 32 && k0 < n_bands) produce(k0);

  float acc[FB_PAIRS][4];
#pragma unroll
  for (int m = 0; m < FB_PAIRS; ++m)
#pragma unroll
    for (int sl = 0; sl < 4; ++sl) acc[m][sl] = 0.f;

  // lane pairs hold the same bin of two neighbouring projections: a quarter-warp (the unit of a
  // 128-bit shared load) then spans 4 bins x 2 projections, i.e. < 8 consecutive float4 -> no
  // bank conflict, where 8 consecutive bins at 45 degrees would span 10
  const int bl = (tid >> 5) * 16 + (lane >> 1);
  const int par = lane & 1;
  const double bd = (double)(b0 + bl);
  const int idx_hi = W - NC;
  float4 vlast = make_float4(0.f, 0.f, 0.f, 0.f);

  for (int k = k0; k < n_bands; ++k) {
    __syncthreads();  // everyone is done with band k-1: its stage may be overwritten
    if (k + 1 < n_bands && tid < 32) produce(k + 1);
    mbar_wait(&full[(k - k0) & 1], (uint32_t)(((k - k0) >> 1) & 1));
    const int origin = sorigin[(k - k0) & 1];
    const int vb = k * FB_RB;
    const int rows = min(FB_RB, d.nv - vb);
    const float4* stage = buf + ((k - k0) & 1) * FB_RB * W;
#pragma unroll
    for (int m = 0; m < FB_PAIRS; ++m) {
      const int pj = par + 2 * m;
      if (pj >= ck.count) break;
      const FpProjD* sp = &sproj[pj];
      // strip centre on the band's first line, relative to the window (double), split (R11)
      const double A = fma(sp->sD, (double)vb, fma(bd, sp->inv_cu, sp->k0)) - (double)origin;
      const int ai = __double2int_rn(A);
      const float afr = (float)(A - (double)ai);
      const float s = sp->s, hw = sp->hw, cuabs = sp->cuabs;
#pragma unroll 4
      for (int r = 0; r < rows; ++r) {
        const float dfr = fmaf(s, (float)r, afr);
        // first pixel that can lie inside the strip: ceil(dfr - hw) by a round-up add of
        // 1.5 * 2^23 (|dfr - hw| < 2^22), integer part read from the mantissa -- no XU-pipe F2I
        const float jm = __fadd_ru(dfr - hw, 12582912.f);
        const float jf = jm - 12582912.f;
        const float d0 = jf - dfr;               // in [-hw, -hw + 1)
        int idx = ai + (__float_as_int(jm) - 0x4b400000);
        idx = min(max(idx, 0), idx_hi);          // only acts where the strip is off the image
        const float4* wp = stage + r * W + idx;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
          const float w = fmaxf(0.f, fmaf(-cuabs, fabsf(d0 + (float)c), 1.f));
          // the last candidate lies outside the strip for most bins of a steep projection: its load
          // is predicated on the weight (a quarter-warp with no taker costs no shared-memory
          // wavefront); the register then keeps an older, finite pixel that is multiplied by 0
          if (c < NC - 1 || w > 0.f) vlast = wp[c];
          const float4 v = vlast;
          ffma2_bcast(acc[m][0], acc[m][1], v.x, v.y, w);
          ffma2_bcast(acc[m][2], acc[m][3], v.z, v.w, w);
        }
      }
    }
  }

  const int b = b0 + bl;
  if (b < B) {
#pragma unroll
    for (int m = 0; m < FB_PAIRS; ++m) {
      const int pj = par + 2 * m;
      if (pj >= ck.count) break;
      const int p = sproj[pj].p;
#pragma unroll
      for (int sl = 0; sl < 4; ++sl) {
        const int s = g * 4 + sl;
        if (s < S) {
          if (!SPLIT || hs == 0) sino[((int64_t)s * P + p) * pitch + b] = scale * acc[m][sl];
          else part[(int64_t)(hs - 1) * part_stride + ((int64_t)s * n_tab + (ck.first + pj)) * part_pitch + b] = scale * acc[m][sl];
        }
      }
    }
  }
}

// y[row][b] += sum_h part[h][row][b] for the rows (slice, projection) of the projections in the plan's table
// (all of them, or the few the diagonal-line kernel leaves to this one)
__global__ void fp_split_combine_kernel(float* __restrict__ y, int64_t pitch_y, const float* __restrict__ part,
                                        int64_t part_pitch, int64_t part_stride, int n_parts, int B,
                                        int64_t n_rows_tab, const FpProjD* __restrict__ projs, int n_tab, int P) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t rt = blockIdx.y + (int64_t)blockIdx.z * gridDim.y;
  if (b >= B || rt >= n_rows_tab) return;
  const int64_t sl = rt / n_tab;
  const int64_t row = sl * P + projs[rt - sl * n_tab].p;
  float v = y[row * pitch_y + b];
  for (int h = 0; h < n_parts; ++h) v += part[(int64_t)h * part_stride + rt * part_pitch + b];
  y[row * pitch_y + b] = v;
}

// ------------------------------------------------------------------------------------------
// Interval form of the banded gather (variant 3; measured alternative, NOT the default).
//
// fp_band_kernel above loads, for every (bin, line), the up to NC = 3 pixels inside the 2-bin-wide
// hat of the bin -- three LDS.128 per 4 slices, and the kernel is bound by shared-memory
// wavefronts.  Here a thread owns the unit INTERVAL [b-1, b) of the detector axis instead: on a
// line at most NCI = ceil(1/|cu|) pixels have their coordinate t in it, each is loaded once and
// used twice: with weight f = t - (b-1) for bin b (accumulator U, the thread's own bin) and with
// 1 - f for bin b-1 (accumulator L, the neighbour's).  Two loads and four FFMA-quads per
// (interval, line) instead of three and three.  A second kernel adds L of interval b+1 to U of
// interval b (fp_ivl_combine_kernel).
// Measured on config 2 (r01c): shared-memory wavefronts drop from 0.90 to 0.46 per clk per SM, but the
// two boundary evaluations, the membership masks and the second accumulator set raise the count to
// 60 warp instructions per (interval, line) against 43 for fp_band_kernel; the kernel becomes issue-
// bound (80 %) and takes 67.5 ms against 49.7 ms.  With 8 slices per thread (NG = 2, variant 4: the
// per-line logic is shared by twice the FMAs; bands of 4 lines so that both windows fit) and a
// three-stage mbarrier ring instead of the per-band block barrier it reaches 49.2 ms against the
// banded kernel's 47.8 ms: fewer instructions (42.6e9 vs 46.4e9) but two blocks per SM and ~11
// instructions per line of double-precision boundary set-up per 4-line band.  Kept selectable.
// Which pixels belong to an interval must be decided identically by the two threads that share a
// boundary, or a pixel at t ~ b would be counted twice or not at all: both evaluate the SAME
// expression for the boundary -- the position u*(b, v) of t = b on the line, in double per
// (thread, band), split into an integer (exact) and a float fraction independent of the window
// origin, then fmaf(s, r, fraction) per line -- so the pixel sets [ceil(u*(b-1)), ceil(u*(b))) are
// an exact partition of the line whatever the rounding.  The weights use the continuous f (a
// pixel assigned to the "wrong" side of a boundary by rounding gets f = 1 + eps or -eps: the two
// contributions still add up to the pixel value placed at the right coordinate).
// For cu < 0 the line is walked in the mirrored coordinate -u, so that t always grows with it.
// ------------------------------------------------------------------------------------------
constexpr int IV_NB = 64;     // intervals per block: 4 warps x 16, the other 4 warps take projections 8..15
constexpr int IV_PAIRS = IV_NB * FB_NPJ / FB_NT;   // (interval, projection) pairs per thread = 4

// NG = slice groups per block (1: 4 slices per thread, bands of RB = 8 lines; 2: 8 slices per thread --
// the boundary / membership / weight logic of a line is shared by twice the FMA work -- bands of RB = 4
// lines so that both groups' windows fit in shared memory).
template <int NCI, int NG, int RB>
__global__ void __launch_bounds__(FB_NT, NG == 2 ? 2 : 3)
fp_ivl_kernel(const float4* __restrict__ xi_rows, const float4* __restrict__ xi_cols, XiDims dr,
              XiDims dc, float* __restrict__ out_u, int64_t pitch_u, float* __restrict__ out_l,
              int64_t pitch_l, int S, int P, int B, float scale, const FpProjD* __restrict__ projs,
              const FpChunk* __restrict__ chunks, int W) {
  extern __shared__ __align__(128) unsigned char smem[];
  constexpr int NSTG = 3;                                    // stages of the band ring
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);        // [NSTG]
  uint64_t* empty = reinterpret_cast<uint64_t*>(smem + 24);  // [NSTG]
  int* sorigin = reinterpret_cast<int*>(smem + 48);          // [NSTG]
  FpProjD* sproj = reinterpret_cast<FpProjD*>(smem + 64);    // [FB_NPJ]
  float4* buf = reinterpret_cast<float4*>(smem + FB_HDR);    // [NSTG][RB][NG][W]

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const FpChunk ck = chunks[blockIdx.y];
  const int gA = blockIdx.z * NG;
  const int b0 = blockIdx.x * IV_NB;                         // interval b = [b-1, b), b in [b0, b0 + NB)
  const XiDims d = ck.cls ? dc : dr;
  const int64_t line_f4 = (int64_t)d.nu + 2 * d.zpad;
  const float4* xi = (ck.cls ? xi_cols : xi_rows) + (int64_t)gA * d.nv * line_f4;
  const int64_t group_f4 = (int64_t)d.nv * line_f4;
  const int n_bands = (d.nv + RB - 1) / RB;
  const uint32_t row_bytes = (uint32_t)W * 16u;

  if (tid < ck.count) sproj[tid] = projs[ck.first + tid];
  if (tid == 0) {
#pragma unroll
    for (int q = 0; q < NSTG; ++q) {
      mbar_init(&full[q], RB);
      mbar_init(&empty[q], FB_NT / 32);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // one warp (the role rotates): waits until the stage of band k - NSTG has been read by every warp,
  // then window origin of band k (the intervals lie inside the hats of bins b0-1 .. b0+NB-1),
  // then one bulk copy per line of the band
  auto produce = [&](int k) {
    const int st = k % NSTG;
    if (k >= NSTG) mbar_wait(&empty[st], (uint32_t)(((k / NSTG) - 1) & 1));
    const int vb = k * RB;
    const int rows = min(RB, d.nv - vb);
    double lo = 1e300;
    if (lane < ck.count) {
      const FpProjD pj = sproj[lane];
      const double ua = fma((double)(b0 - 1), pj.inv_cu, pj.k0);
      const double ub = fma((double)(b0 + IV_NB - 1), pj.inv_cu, pj.k0);
      const double va = pj.sD * (double)vb, vz = pj.sD * (double)(vb + rows - 1);
      lo = fmin(fmin(ua, ub) + fmin(va, vz), lo) - (double)pj.hw;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    double of = floor(lo) - 1.0;
    of = fmax(of, -(double)d.zpad);
    of = fmin(of, (double)(d.nu + d.zpad - W));
    const int origin = (int)of;
    uint64_t* bar = &full[st];
    if (lane == 0) sorigin[st] = origin;
    if (lane < RB) {
      if (lane < rows) {
        mbar_arrive_expect_tx(bar, NG * row_bytes);
#pragma unroll
        for (int q = 0; q < NG; ++q)
          bulk_g2s(buf + ((st * RB + lane) * NG + q) * W,
                   xi + q * group_f4 + (int64_t)(vb + lane) * line_f4 + (origin + d.zpad), row_bytes, bar);
      } else {
        mbar_arrive(bar);
      }
    }
  };

  if (tid < 32) produce(0);   // bands are issued one ahead of the one being read

  float accu[IV_PAIRS][4 * NG], accl[IV_PAIRS][4 * NG];
#pragma unroll
  for (int m = 0; m < IV_PAIRS; ++m)
#pragma unroll
    for (int sl = 0; sl < 4 * NG; ++sl) accu[m][sl] = accl[m][sl] = 0.f;

  // lane pairs hold the same interval of two neighbouring projections (see fp_band_kernel)
  const int bl = (warp & 3) * 16 + (lane >> 1);
  const int pj0 = (lane & 1) + 8 * (warp >> 2);
  const double bd = (double)(b0 + bl);

  for (int k = 0; k < n_bands; ++k) {
    if (k + 1 < n_bands && warp == ((k + 1) & 7)) produce(k + 1);
    const int st = k % NSTG;
    mbar_wait(&full[st], (uint32_t)((k / NSTG) & 1));
    const int origin = sorigin[st];
    const int vb = k * RB;
    const int rows = min(RB, d.nv - vb);
    const float4* stage = buf + st * RB * NG * W;
#pragma unroll
    for (int m = 0; m < IV_PAIRS; ++m) {
      const int pj = pj0 + 2 * m;
      if (pj >= ck.count) break;
      const FpProjD* sp = &sproj[pj];
      const double inv_cu = sp->inv_cu, k0 = sp->k0, sD = sp->sD;
      const double sigma = inv_cu >= 0.0 ? 1.0 : -1.0;
      const int sg = inv_cu >= 0.0 ? 1 : -1;
      // boundaries t = b-1 and t = b on the band's first line, mirrored pixel coordinate (double);
      // the neighbour's thread evaluates the shared boundary with the identical expression
      const double As = sigma * fma(sD, (double)vb, fma(bd - 1.0, inv_cu, k0));
      const double Ae = sigma * fma(sD, (double)vb, fma(bd, inv_cu, k0));
      const double aiS = rint(As), aiE = rint(Ae);
      const float afrS = (float)(As - aiS), afrE = (float)(Ae - aiE);
      const int dn = (int)(aiE - aiS);
      const int base_m = sg * (int)aiS - origin;      // window index of mirrored pixel aiS
      const float ss = (float)(sigma * sD), cuabs = sp->cuabs;
      const int m_lo = sg > 0 ? 0 : NCI - 1, m_hi = sg > 0 ? W - NCI : W - 1;
#pragma unroll
      for (int r = 0; r < RB; ++r) {
        if (r >= rows) break;
        const float rf = (float)r;
        // ceil by a round-up add of 1.5 * 2^23, integer part read from the mantissa
        const float dS = fmaf(ss, rf, afrS), dE = fmaf(ss, rf, afrE);
        const float jmS = __fadd_ru(dS, 12582912.f), jmE = __fadd_ru(dE, 12582912.f);
        const int kS = __float_as_int(jmS) - 0x4b400000;
        const int n = dn + (__float_as_int(jmE) - __float_as_int(jmS));   // pixels in the interval
        const float f0 = cuabs * ((jmS - 12582912.f) - dS);                // t - (b-1) of the first one
        int idx = base_m + sg * kS;
        idx = min(max(idx, m_lo), m_hi);              // only acts where the interval is off the image
        const float4* wp = stage + r * NG * W + idx;
#pragma unroll
        for (int c = 0; c < NCI; ++c) {
          const float f = fmaf((float)c, cuabs, f0);
          const bool in = c < n;
          const float wu = in ? f : 0.f, wl = in ? 1.f - f : 0.f;
#pragma unroll
          for (int q = 0; q < NG; ++q) {
            const float4 v = wp[q * W + sg * c];
            accu[m][4 * q + 0] = fmaf(wu, v.x, accu[m][4 * q + 0]);
            accu[m][4 * q + 1] = fmaf(wu, v.y, accu[m][4 * q + 1]);
            accu[m][4 * q + 2] = fmaf(wu, v.z, accu[m][4 * q + 2]);
            accu[m][4 * q + 3] = fmaf(wu, v.w, accu[m][4 * q + 3]);
            accl[m][4 * q + 0] = fmaf(wl, v.x, accl[m][4 * q + 0]);
            accl[m][4 * q + 1] = fmaf(wl, v.y, accl[m][4 * q + 1]);
            accl[m][4 * q + 2] = fmaf(wl, v.z, accl[m][4 * q + 2]);
            accl[m][4 * q + 3] = fmaf(wl, v.w, accl[m][4 * q + 3]);
          }
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[st]);
  }

  // U of interval b is bin b's share, L is bin b-1's (stored at index b of out_l, b in [0, B])
  const int b = b0 + bl;
  if (b <= B) {
#pragma unroll
    for (int m = 0; m < IV_PAIRS; ++m) {
      const int pj = pj0 + 2 * m;
      if (pj >= ck.count) break;
      const int p = sproj[pj].p;
#pragma unroll
      for (int sl = 0; sl < 4 * NG; ++sl) {
        const int s = gA * 4 + sl;
        if (s < S) {
          if (b < B) out_u[((int64_t)s * P + p) * pitch_u + b] = scale * accu[m][sl];
          out_l[((int64_t)s * P + p) * pitch_l + b] = scale * accl[m][sl];
        }
      }
    }
  }
}

// y[row][b] += l[row][b + 1], b in [0, B)
__global__ void fp_ivl_combine_kernel(float* __restrict__ y, int64_t pitch_y, const float* __restrict__ l,
                                      int64_t pitch_l, int B, int64_t n_rows) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t row = blockIdx.y + (int64_t)blockIdx.z * gridDim.y;
  if (b < B && row < n_rows) y[row * pitch_y + b] += l[row * pitch_l + b + 1];
}

// [S][ny][nx] -> XI rows copy [g][ny][zr + nx + zr] and XI columns copy [g][nx][zc + ny + zc]
__global__ void repack_image_kernel(const float* __restrict__ img, int S, int ny, int nx,
                                    float4* __restrict__ xi_rows, int zr, float4* __restrict__ xi_cols,
                                    int zc) {
  __shared__ float tile[4][32][33];
  const int g = blockIdx.z;
  const int bx = blockIdx.x * 32, by = blockIdx.y * 32;
#pragma unroll
  for (int sl = 0; sl < 4; ++sl) {
    const int s = g * 4 + sl;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      const int y = by + r, x = bx + threadIdx.x;
      tile[sl][r][threadIdx.x] = (s < S && y < ny && x < nx) ? img[((int64_t)s * ny + y) * nx + x] : 0.f;
    }
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    if (xi_rows) {
      const int y = by + r, x = bx + threadIdx.x;
      if (y < ny && x < nx)
        xi_rows[((int64_t)g * ny + y) * (nx + 2 * zr) + zr + x] =
            make_float4(tile[0][r][threadIdx.x], tile[1][r][threadIdx.x], tile[2][r][threadIdx.x],
                        tile[3][r][threadIdx.x]);
    }
    if (xi_cols) {
      const int x = bx + r, y = by + threadIdx.x;
      if (y < ny && x < nx)
        xi_cols[((int64_t)g * nx + x) * (ny + 2 * zc) + zc + y] =
            make_float4(tile[0][threadIdx.x][r], tile[1][threadIdx.x][r], tile[2][threadIdx.x][r],
                        tile[3][threadIdx.x][r]);
    }
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------
// host: walk classes, chunks of projections and the window width (all in double)
// ------------------------------------------------------------------------------------------
namespace {

struct Extent { double lo[4], hi[4]; };  // of u* - hw over a block's corners, at the 4 extreme (segment, band) places

// u*(b, v) - hw is affine in (b, v): over a block (NB bins x RB lines) its extremes sit at the
// block's corners; the window width max - min is convex in the block position, so its maximum
// over all blocks is attained at the four extreme (segment, band) positions.
Extent proj_extent(const FpProjD& pj, int n_bins, int nv) {
  Extent e;
  const int seg_last = ((n_bins + FB_NB - 1) / FB_NB - 1) * FB_NB;
  const int band_last = ((nv + FB_RB - 1) / FB_RB - 1) * FB_RB;
  int q = 0;
  for (int b0 : {0, seg_last})
    for (int vb : {0, band_last}) {
      const int rows = std::min(FB_RB, nv - vb);
      double lo = 1e300, hi = -1e300;
      for (int b : {b0, b0 + FB_NB - 1})
        for (int v : {vb, vb + rows - 1}) {
          const double u = (double)b * pj.inv_cu + pj.k0 + pj.sD * (double)v - (double)pj.hw;
          lo = std::min(lo, u);
          hi = std::max(hi, u);
        }
      e.lo[q] = lo;
      e.hi[q] = hi;
      ++q;
    }
  return e;
}

int width_of(const Extent& e, int nc) {
  int w = 0;
  for (int q = 0; q < 4; ++q) {
    const double origin = std::floor(e.lo[q]) - 1.0;
    w = std::max(w, (int)(std::ceil(e.hi[q]) - origin) + nc + 2);  // + 2: slack for the convexity bound
  }
  return w;
}

Extent merge(const Extent& a, const Extent& b) {
  Extent e;
  for (int q = 0; q < 4; ++q) {
    e.lo[q] = std::min(a.lo[q], b.lo[q]);
    e.hi[q] = std::max(a.hi[q], b.hi[q]);
  }
  return e;
}

}  // namespace

bool build_fp_tables(const pyhst_geom_t* g, FpPlan* plan, std::vector<FpProjD>* projs,
                     std::vector<FpChunk>* chunks, const std::vector<int32_t>* subset) {
  const int P = g->n_angles;
  const double h = g->pixel_size;
  // candidates per line: the open strip of width 2 / |cu| <= 2 sqrt(2) / h holds at most nc pixels
  const int nc = (int)std::ceil(2.0 * std::sqrt(2.0) / h - 1e-9);
  if (nc > 6) return false;
  plan->nc = nc <= 3 ? 3 : (nc <= 4 ? 4 : 6);
  // projections per chunk (<= FB_NPJ): picked below, once the two walk classes are known, so that
  // the grid fills whole waves of the GPU's block slots (3 blocks per SM)
  std::vector<int> order[2];
  std::vector<FpProjD> all(P);
  std::vector<char> wanted(P, subset ? 0 : 1);
  if (subset)
    for (int32_t p : *subset) wanted[p] = 1;
  for (int p = 0; p < P; ++p) {
    if (!wanted[p]) continue;
    const double ch = h * std::cos(g->angles_rad[p]), sh = h * std::sin(g->angles_rad[p]);
    const int cls = std::fabs(ch) >= std::fabs(sh) ? 0 : 1;
    const double cu = cls ? sh : ch, cv = cls ? ch : sh;
    const int nu = cls ? g->ny : g->nx, nv = cls ? g->nx : g->ny;
    const double u0 = 0.5 * (double)(nu - 1), v0 = 0.5 * (double)(nv - 1);
    FpProjD& d = all[p];
    d.inv_cu = 1.0 / cu;
    d.k0 = u0 + (cv * v0 - g->axis_pos[p]) * d.inv_cu;
    d.sD = -cv * d.inv_cu;
    d.s = (float)d.sD;
    d.hw = (float)std::fabs(d.inv_cu);
    d.cuabs = (float)std::fabs(cu);
    d.p = p;
    order[cls].push_back(p);
  }
  projs->clear();
  chunks->clear();
  plan->any_rows = !order[0].empty();
  plan->any_cols = !order[1].empty();
  // neighbours in angle have neighbouring strips: sort each class by angle (stable: the caller's
  // order is kept for the usual monotone lists)
  for (int cls = 0; cls < 2; ++cls)
    std::stable_sort(order[cls].begin(), order[cls].end(),
                     [&](int a, int b) { return g->angles_rad[a] < g->angles_rad[b]; });
  std::vector<Extent> ext(P);
  int w_single = 0;
  for (int cls = 0; cls < 2; ++cls) {
    const int nv = cls ? g->nx : g->ny;
    for (int p : order[cls]) {
      ext[p] = proj_extent(all[p], g->n_bins, nv);
      w_single = std::max(w_single, width_of(ext[p], plan->nc));
    }
  }
  // window width for chunks of c neighbours: wide enough for ~all of them (the 90th percentile of
  // their widths: a chunk that straddles a jump in angle, e.g. 45 -> 135 degrees inside a walk
  // class, is simply split below) and for every single projection; at most the capacity
  auto window_for = [&](int c) {
    std::vector<int> widths;
    for (int cls = 0; cls < 2; ++cls)
      for (size_t i = 0; i < order[cls].size(); i += c) {
        Extent e = ext[order[cls][i]];
        for (size_t j = i + 1; j < std::min(order[cls].size(), i + c); ++j) e = merge(e, ext[order[cls][j]]);
        widths.push_back(width_of(e, plan->nc));
      }
    std::sort(widths.begin(), widths.end());
    const int w_most = widths.empty() ? 0 : widths[(widths.size() - 1) * 9 / 10];
    return std::min(std::max(std::max(w_most, w_single), plan->nc + 4), FB_WMAX);
  };
  // projections per chunk: 16, 8 or 4.  Many neighbours share one staged window (good for dense
  // angle lists), but their strips fan out (sparse lists: config 4's 16 neighbours span 14 degrees
  // and need the full 416-pixel window, two blocks per SM).  Cost model, calibrated on configs 2 and 4:
  // waves of the GPU's block slots (fractional above one) x (projections + fixed part + window
  // staging) of one block.
  int npj = FB_NPJ, W = window_for(FB_NPJ);
  {
    int n_sm = 148, dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    const int64_t segs = (g->n_bins + FB_NB - 1) / FB_NB, groups = (g->n_slices + 3) / 4;
    double best = 1e300;
    for (int c = FB_NPJ; c >= 4; c /= 2) {
      const int w = window_for(c);
      const size_t smem = FB_HDR + (size_t)2 * FB_RB * w * 16;
      const int64_t per_sm = std::max<int64_t>(1, std::min<int64_t>(3, (int64_t)(227 * 1024) / (int64_t)(smem + 1024)));
      // (+ 10 %: chunks that straddle a jump in angle are split)
      const int64_t blocks = segs * groups * (int64_t)((order[0].size() + c - 1) / c + (order[1].size() + c - 1) / c) * 11 / 10;
      const int64_t slots = per_sm * n_sm;
      const double cost = std::max(1.0, (double)blocks / (double)slots) * ((double)c + 1.0 + (double)w / 64.0);
      if (std::getenv("PYHST_DEBUG"))
        std::fprintf(stderr, "[pyhst] fp chunk size %d: W %d, %lld blocks, %lld slots, cost %.1f\n", c, w,
                     (long long)blocks, (long long)slots, cost);
      if (cost < best * 0.999) { best = cost; npj = c; W = w; }
    }
  }
  plan->W = W;
  plan->npj = npj;
  // greedy chunks: add neighbours while the window still fits
  for (int cls = 0; cls < 2; ++cls) {
    size_t i = 0;
    while (i < order[cls].size()) {
      Extent e = ext[order[cls][i]];
      if (width_of(e, plan->nc) > W) return false;  // one projection alone does not fit
      FpChunk ck{(int32_t)projs->size(), 1, cls, 0};
      projs->push_back(all[order[cls][i]]);
      size_t j = i + 1;
      for (; j < order[cls].size() && ck.count < npj; ++j) {
        const Extent m = merge(e, ext[order[cls][j]]);
        if (width_of(m, plan->nc) > W) break;
        e = m;
        projs->push_back(all[order[cls][j]]);
        ++ck.count;
      }
      chunks->push_back(ck);
      i = j;
    }
  }
  plan->n_chunks = (int32_t)chunks->size();
  plan->n_tab = (int32_t)projs->size();
  return plan->n_chunks <= 65535;
}

// pixels that can fall into one unit interval of the detector axis on a line: floor(sqrt2/h) + 1
int forward_project_interval_candidates(double pixel_size) {
  return (int)std::floor(std::sqrt(2.0) / pixel_size) + 1;
}

int launch_forward_project_banded(const float* d_img, float* d_sino, int64_t pitch,
                                  const pyhst_geom_t* g, float scale, const FpPlan& plan,
                                  int interval_groups, cudaStream_t stream) {
  const bool interval = interval_groups > 0;
  const int n_groups = (g->n_slices + 3) / 4;
  const int W = plan.W;
  XiLayout Lr{n_groups, g->ny, g->nx, W}, Lc{n_groups, g->nx, g->ny, W};
  size_t bytes_r = plan.any_rows ? Lr.bytes() : 0, bytes_c = plan.any_cols ? Lc.bytes() : 0;
  void* ws = nullptr;
  PYHST_TRY(get_workspace(WS_XI, bytes_r + bytes_c, &ws));
  // the zero pads are written once per (block, layout); the repack only touches the interior
  // ("this very block": device + the slot's allocation generation, so that a block freed by
  // pyhst_release_cache or regrown and handed back at the same address is zeroed again).
  // A stack of FEWER slice groups than the one the block was zeroed for (the last chunk of a host
  // pipeline) is laid out as that larger stack -- the column copy keeps its place -- so that it finds
  // the pads already zero instead of clearing the block on every call; groups >= n_groups are not read.
  struct PadsKey { size_t k[8]; };
  static PadsKey pads[PYHST_MAX_DEVICES];
  PadsKey key = {{(size_t)plan.any_rows, (size_t)plan.any_cols, (size_t)g->nx, (size_t)g->ny, (size_t)W,
                  (size_t)n_groups, (size_t)workspace_generation(WS_XI), (size_t)reinterpret_cast<uintptr_t>(ws)}};
  PadsKey& seen = pads[std::max(0, current_device()) % PYHST_MAX_DEVICES];
  const size_t seen_groups = seen.k[5];
  key.k[5] = seen_groups;
  const bool pads_zero = std::memcmp(&seen, &key, sizeof(key)) == 0 && seen_groups >= (size_t)n_groups;
  key.k[5] = (size_t)n_groups;
  if (pads_zero && plan.any_rows) bytes_r = XiLayout{(int32_t)seen_groups, g->ny, g->nx, W}.bytes();
  float4* xi_r = plan.any_rows ? static_cast<float4*>(ws) : nullptr;
  float4* xi_c = plan.any_cols ? reinterpret_cast<float4*>(static_cast<char*>(ws) + bytes_r) : nullptr;
  {
    StageScope scope(ST_TRANSPOSE, stream);
    if (!pads_zero) {
      PYHST_CUDA_TRY(cudaMemsetAsync(ws, 0, bytes_r + bytes_c, stream));
      seen = key;
    }
    dim3 block(32, 8, 1);
    dim3 grid((g->nx + 31) / 32, (g->ny + 31) / 32, n_groups);
    if (grid.y > 65535 || grid.z > 65535)
      return set_error(PYHST_ERR_UNSUPPORTED, "image repack: grid too large");
    scope.kernels();
    repack_image_kernel<<<grid, block, 0, stream>>>(d_img, g->n_slices, g->ny, g->nx, xi_r, W, xi_c, W);
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  const size_t smem = FB_HDR + (size_t)2 * FB_RB * W * 16;
  const XiDims dr{g->ny, g->nx, W}, dc{g->nx, g->ny, W};
  const int nci = forward_project_interval_candidates(g->pixel_size);
  if (interval && (nci == 2 || nci == 3)) {
    // interval kernel: U -> d_sino, L -> workspace [S P][B + 1 pitched]; then d_sino[b] += L[b + 1]
    const int64_t n_rows = (int64_t)g->n_slices * g->n_angles;
    const int64_t pitch_l = ((int64_t)g->n_bins + 1 + 3) & ~(int64_t)3;
    void* wl = nullptr;
    PYHST_TRY(get_workspace(WS_FPL, (size_t)n_rows * pitch_l * 4, &wl));
    // 8 slices per thread (two groups per block, bands of 4 lines) when the stack has an even number
    // of slice groups and full 16-projection chunks (the thread map gives projections 8..15 to warps 4..7)
    const bool two = nci == 2 && n_groups % 2 == 0 && plan.npj == FB_NPJ && interval_groups == 2;
    static PerDeviceSize configured_i[3];
    auto kern_i = two ? fp_ivl_kernel<2, 2, 4> : (nci == 2 ? fp_ivl_kernel<2, 1, 8> : fp_ivl_kernel<3, 1, 8>);
    const int ci = two ? 2 : nci - 2;
    if (smem > configured_i[ci].here()) {
      PYHST_CUDA_TRY(cudaFuncSetAttribute(kern_i, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(FB_HDR + (size_t)3 * FB_RB * W * 16)));
      configured_i[ci].here() = smem;
    }
    const size_t smem_i = FB_HDR + (size_t)3 * FB_RB * W * 16;   // three stages of RB x NG = 8 lines
    dim3 grid((g->n_bins + 1 + IV_NB - 1) / IV_NB, plan.n_chunks, two ? n_groups / 2 : n_groups);
    if (grid.z > 65535) return set_error(PYHST_ERR_UNSUPPORTED, "forward projector: too many slice groups");
    StageScope scope(ST_FORWARD, stream);
    scope.kernels(2);
    kern_i<<<grid, FB_NT, smem_i, stream>>>(xi_r, xi_c, dr, dc, d_sino, pitch, static_cast<float*>(wl), pitch_l,
                                          g->n_slices, g->n_angles, g->n_bins, scale, plan.d_projs,
                                          plan.d_chunks, W);
    PYHST_CUDA_TRY(cudaGetLastError());
    const unsigned gy = (unsigned)std::min<int64_t>(n_rows, 32768);
    dim3 grid_c((g->n_bins + 255) / 256, gy, (unsigned)((n_rows + gy - 1) / gy));
    fp_ivl_combine_kernel<<<grid_c, 256, 0, stream>>>(d_sino, pitch, static_cast<const float*>(wl), pitch_l,
                                                      g->n_bins, n_rows);
    PYHST_CUDA_TRY(cudaGetLastError());
    return PYHST_OK;
  }
  // blocks per SM: 3 (80 registers), or 4 (64 registers) when four windows fit in shared memory;
  // small grids are split along the lines so that they fill the block slots (deterministic:
  // partial sums go to a workspace and are added by a second kernel)
  int n_sm = 148, dev = 0;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  const bool four = plan.nc == 3 && smem <= 56 * 1024;
  const int64_t blocks = (int64_t)((g->n_bins + FB_NB - 1) / FB_NB) * plan.n_chunks * n_groups;
  const int64_t slots = (int64_t)n_sm * (four ? 4 : 3);
  const int n_bands_min = (std::min(g->nx, g->ny) + FB_RB - 1) / FB_RB;
  int n_split = (int)std::max<int64_t>(1, std::min<int64_t>(plan.diag ? 8 : 4, slots / std::max<int64_t>(blocks, 1)));
  n_split = std::max(1, std::min(n_split, n_bands_min / 8));
  static PerDeviceSize configured[5];
  const int vi = four ? 3 : (plan.nc == 3 ? (n_split > 1 ? 4 : 0) : (plan.nc == 4 ? 1 : 2));
  auto kern = four ? fp_band_kernel<3, 4, true>
                   : (plan.nc == 3 ? (n_split > 1 ? fp_band_kernel<3, 3, true> : fp_band_kernel<3, 3, false>)
                                   : (plan.nc == 4 ? fp_band_kernel<4, 3, true> : fp_band_kernel<6, 3, true>));
  if (smem > configured[vi].here()) {
    PYHST_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured[vi].here() = smem;
  }
  const int64_t n_rows = (int64_t)g->n_slices * g->n_angles;
  float* part = nullptr;
  const int64_t part_pitch = g->n_bins, part_stride = (int64_t)g->n_slices * plan.n_tab * part_pitch;
  if (n_split > 1) {
    void* wp = nullptr;
    PYHST_TRY(get_workspace(WS_FPL, (size_t)(n_split - 1) * part_stride * 4, &wp));
    part = static_cast<float*>(wp);
  }
  dim3 grid((g->n_bins + FB_NB - 1) / FB_NB, plan.n_chunks, n_groups * n_split);
  if (grid.z > 65535) return set_error(PYHST_ERR_UNSUPPORTED, "forward projector: too many slice groups");
  StageScope scope(ST_FORWARD, stream);
  scope.kernels(n_split > 1 ? 2 : 1);
  kern<<<grid, FB_NT, smem, stream>>>(xi_r, xi_c, dr, dc, d_sino, pitch, g->n_slices, g->n_angles,
                                      g->n_bins, scale, plan.d_projs, plan.d_chunks, W, n_split, part,
                                      part_pitch, part_stride, plan.n_tab);
  PYHST_CUDA_TRY(cudaGetLastError());
  if (n_split > 1) {
    const int64_t n_rows_tab = (int64_t)g->n_slices * plan.n_tab;
    const unsigned gy = (unsigned)std::min<int64_t>(n_rows_tab, 32768);
    dim3 grid_c((g->n_bins + 255) / 256, gy, (unsigned)((n_rows_tab + gy - 1) / gy));
    fp_split_combine_kernel<<<grid_c, 256, 0, stream>>>(d_sino, pitch, part, part_pitch, part_stride,
                                                        n_split - 1, g->n_bins, n_rows_tab, plan.d_projs, plan.n_tab,
                                                        g->n_angles);
  }
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

}  // namespace pyhst
