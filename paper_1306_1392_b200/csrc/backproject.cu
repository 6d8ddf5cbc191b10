// Backprojection P^T (include/pyhst.h a2; readings R1-R7, R11 of DESIGN.md).
//
//   img[s,i,j] = scale * sum_p lerp(q[s,p,:], t_p(i,j)),   t_p(i,j) = c_p + ch_p (j-j0) + sh_p (i-i0)
//
// Two kernels:
//   bp_reference_kernel  one thread per pixel, global loads, t in double.  Cross-check and the
//                        path for geometries the tiled kernel does not cover (huge pixel size).
//   bp_tiled_kernel      the product path: a block owns a 64x64 output tile of one slice group
//                        (4 slices interleaved as float4), stages per chunk of 16 projections
//                        the detector window its tile touches with cp.async.bulk (TMA bulk
//                        copy, mbarrier-signalled, double-buffered), interpolates with FP32
//                        FMAs out of shared memory and accumulates 16 pixels x 4 slices per
//                        thread in registers.
#include "common.h"

namespace pyhst {

// ------------------------------------------------------------------------------------------
// reference kernel
// ------------------------------------------------------------------------------------------
__global__ void bp_reference_kernel(const float* __restrict__ sino, int64_t pitch,
                                    float* __restrict__ img, int P, int B, int nx, int ny,
                                    float scale, const ProjGeom* __restrict__ proj) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int i = blockIdx.y * blockDim.y + threadIdx.y;
  const int s = blockIdx.z;
  if (i >= ny || j >= nx) return;
  const double dj = (double)j - 0.5 * (double)(nx - 1);
  const double di = (double)i - 0.5 * (double)(ny - 1);
  const float* q = sino + (int64_t)s * P * pitch;
  float acc = 0.f;
  for (int p = 0; p < P; ++p) {
    const ProjGeom g = proj[p];
    const double t = g.c + g.ch * dj + g.sh * di;
    if (!(t > -1.0 && t < (double)B)) continue;  // both taps off the detector (R6)
    const double kf = floor(t);
    const float f = (float)(t - kf);
    const int k = (int)kf;
    const float* row = q + (int64_t)p * pitch;
    const float a = (k >= 0) ? row[k] : 0.f;
    const float b = (k + 1 < B) ? row[k + 1] : 0.f;
    acc = fmaf(f, b, fmaf(1.f - f, a, acc));
  }
  img[((int64_t)s * ny + i) * nx + j] = scale * acc;
}

int launch_backproject_reference(const float* d_sino, int64_t pitch, const BpArgs& a,
                                 cudaStream_t stream) {
  dim3 block(32, 8, 1);
  dim3 grid((a.nx + 31) / 32, (a.ny + 7) / 8, a.n_slices);
  if (grid.y > 65535 || grid.z > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "reference backprojector: grid too large");
  StageScope scope(ST_BACKPROJECT, stream);
  scope.kernels();
  bp_reference_kernel<<<grid, block, 0, stream>>>(d_sino, pitch, a.d_img, a.n_angles, a.n_bins,
                                                  a.nx, a.ny, a.scale, a.d_proj);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

// ------------------------------------------------------------------------------------------
// repack [S][P][pitch] -> QI[g][p][zpad + b][4]
// ------------------------------------------------------------------------------------------
__global__ void repack_to_qi_kernel(const float* __restrict__ sino, int64_t pitch, int S, int P,
                                    int B, int zpad, float4* __restrict__ qi) {
  const int64_t row_f4 = (int64_t)B + 2 * zpad;
  const int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;  // padded bin index
  const int p = blockIdx.y, g = blockIdx.z;
  if (x >= row_f4) return;
  const int64_t b = x - zpad;
  float v[4] = {0.f, 0.f, 0.f, 0.f};
  if (b >= 0 && b < B) {
#pragma unroll
    for (int sl = 0; sl < 4; ++sl) {
      const int s = g * 4 + sl;
      if (s < S) v[sl] = sino[((int64_t)s * P + p) * pitch + b];
    }
  }
  qi[((int64_t)g * P + p) * row_f4 + x] = make_float4(v[0], v[1], v[2], v[3]);
}

int launch_repack_to_qi(const float* d_sino, int64_t pitch, int32_t n_slices, float4* d_qi,
                        const QiLayout& L, cudaStream_t stream) {
  dim3 block(256, 1, 1);
  dim3 grid((unsigned)((L.row_f4() + 255) / 256), L.n_angles, L.n_groups);
  if (grid.y > 65535 || grid.z > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "repack: more than 65535 projections or slice groups");
  StageScope scope(ST_REPACK, stream);
  scope.kernels();
  repack_to_qi_kernel<<<grid, block, 0, stream>>>(d_sino, pitch, n_slices, L.n_angles, L.n_bins,
                                                  L.zpad, d_qi);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

// ------------------------------------------------------------------------------------------
// tiled kernel
// ------------------------------------------------------------------------------------------
namespace {

constexpr int TX = 64, TY = 64;   // output tile (pixels)
constexpr int NT = 256;           // threads per block: 8 warps, each an 8(x) x 4(y) lane patch
constexpr int NA = 16;            // projections per staged chunk
constexpr int MX = 4, MY = 4;     // pixels per thread: MX x MY, strided by the lane patch
constexpr int SMEM_HDR = 1024;    // mbarriers + geometry ring, keeps the windows 128-B aligned

}  // namespace

// W = window width in bins (float4 per projection), chosen by the host for the pixel size.
__global__ void __launch_bounds__(NT, 2)
bp_tiled_kernel(const float4* __restrict__ qi, int64_t row_f4, int zpad, float* __restrict__ img,
                int S, int P, int B, int nx, int ny, float scale,
                const ProjGeom* __restrict__ proj, int W) {
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);                 // [2]
  float4* geo = reinterpret_cast<float4*>(smem + 64);                 // [3][NA] (ch, sh, base, -)
  float4* buf = reinterpret_cast<float4*>(smem + SMEM_HDR);           // [2][NA][W]

  const int tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, g = blockIdx.z;
  // lane patch 8 x 4; warps tile the block as 2 (x) x 4 (y) regions of 32 x 16 pixels
  const int jl = (warp & 1) * 32 + (lane & 7);
  const int il = (warp >> 1) * 16 + (lane >> 3);
  const float fjl = (float)jl, fil = (float)il;

  const float4* qg = qi + (int64_t)g * P * row_f4;
  const int n_chunks = (P + NA - 1) / NA;
  const uint32_t win_bytes = (uint32_t)W * 16u;

  if (tid == 0) {
    mbar_init(&full[0], NA);
    mbar_init(&full[1], NA);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }

  // Per-(tile, projection) window origin and local base, in double (R11).  Thread a < NA owns
  // projection c*NA + a of chunk c: it writes geo[c % 3][a] and returns the global origin.
  const double dx0 = (double)x0 - 0.5 * (double)(nx - 1);
  const double dy0 = (double)y0 - 0.5 * (double)(ny - 1);
  auto chunk_geometry = [&](int c) -> int64_t {
    const int p = c * NA + tid;
    if (p >= P) return 0;
    const ProjGeom pg = proj[p];
    const double base = pg.c + pg.ch * dx0 + pg.sh * dy0;  // t of the tile's pixel (0,0)
    const double tmin = base + fmin(0.0, pg.ch * (TX - 1)) + fmin(0.0, pg.sh * (TY - 1));
    double o = floor(tmin) - 1.0;                           // one bin of slack for FP32 rounding
    o = fmax(o, -(double)zpad);
    o = fmin(o, (double)(B + zpad - W));
    geo[(c % 3) * NA + tid] = make_float4((float)pg.ch, (float)pg.sh, (float)(base - o), 0.f);
    return (int64_t)o + zpad;
  };
  auto issue_chunk = [&](int c, int64_t origin) {  // threads tid < NA, after the block barrier
    uint64_t* bar = &full[c & 1];
    const int p = c * NA + tid;
    if (p < P) {
      mbar_arrive_expect_tx(bar, win_bytes);
      bulk_g2s(buf + ((c & 1) * NA + tid) * W, qg + (int64_t)p * row_f4 + origin, win_bytes, bar);
    } else {
      mbar_arrive(bar);
    }
  };

  int64_t origin = 0;
  if (tid < NA) origin = chunk_geometry(0);
  __syncthreads();  // barrier init + geometry of chunk 0 visible
  if (tid < NA) issue_chunk(0, origin);

  float acc[MY][MX][4];
#pragma unroll
  for (int my = 0; my < MY; ++my)
#pragma unroll
    for (int mx = 0; mx < MX; ++mx)
#pragma unroll
      for (int sl = 0; sl < 4; ++sl) acc[my][mx][sl] = 0.f;

  const float t_hi = (float)(W - 2);
  const float MAGIC = 8388608.f;  // 2^23: t + 2^23 rounded down keeps floor(t) in the mantissa

  for (int c = 0; c < n_chunks; ++c) {
    if (c + 1 < n_chunks && tid < NA) origin = chunk_geometry(c + 1);
    __syncthreads();  // everyone is done with chunk c-1 (its buffer is free); geometry c+1 visible
    if (c + 1 < n_chunks && tid < NA) issue_chunk(c + 1, origin);
    mbar_wait(&full[c & 1], (uint32_t)((c >> 1) & 1));

    const int na = min(NA, P - c * NA);
    const float4* gch = geo + (c % 3) * NA;
    const float4* wb = buf + (c & 1) * NA * W;
#pragma unroll 2
    for (int a = 0; a < na; ++a) {
      const float4 gg = gch[a];
      const float4* win = wb + a * W;
      const float t0 = fmaf(fjl, gg.x, fmaf(fil, gg.y, gg.z));
#pragma unroll
      for (int my = 0; my < MY; ++my) {
        const float trow = fmaf((float)(my * 4), gg.y, t0);
#pragma unroll
        for (int mx = 0; mx < MX; ++mx) {
          float t = fmaf((float)(mx * 8), gg.x, trow);
          t = fminf(fmaxf(t, 0.f), t_hi);       // only acts in windows clamped at a row end
          const float tm = __fadd_rd(t, MAGIC);
          const int k = __float_as_int(tm) - __float_as_int(MAGIC);
          const float f = t - (tm - MAGIC);
          const float w0 = 1.f - f;
          const float4 q0 = win[k];
          const float4 q1 = win[k + 1];
          acc[my][mx][0] = fmaf(q1.x, f, fmaf(q0.x, w0, acc[my][mx][0]));
          acc[my][mx][1] = fmaf(q1.y, f, fmaf(q0.y, w0, acc[my][mx][1]));
          acc[my][mx][2] = fmaf(q1.z, f, fmaf(q0.z, w0, acc[my][mx][2]));
          acc[my][mx][3] = fmaf(q1.w, f, fmaf(q0.w, w0, acc[my][mx][3]));
        }
      }
    }
  }

  // 8 consecutive pixels of a lane-patch row are 32 contiguous bytes per slice
#pragma unroll
  for (int my = 0; my < MY; ++my) {
    const int y = y0 + il + my * 4;
    if (y >= ny) continue;
#pragma unroll
    for (int mx = 0; mx < MX; ++mx) {
      const int x = x0 + jl + mx * 8;
      if (x >= nx) continue;
#pragma unroll
      for (int sl = 0; sl < 4; ++sl) {
        const int s = g * 4 + sl;
        if (s < S) img[((int64_t)s * ny + y) * nx + x] = scale * acc[my][mx][sl];
      }
    }
  }
}

int backproject_tiled_window(double pixel_size) {
  // span of t over a tile <= h * sqrt((TX-1)^2 + (TY-1)^2); + floor, second tap and slack
  const double span = pixel_size * sqrt((double)((TX - 1) * (TX - 1) + (TY - 1) * (TY - 1)));
  const double w = ceil(span) + 5.0;
  if (w > 1024.0) return 0;
  return ((int)w + 3) & ~3;
}

int launch_backproject_tiled(const float4* d_qi, const QiLayout& L, const BpArgs& a,
                             cudaStream_t stream) {
  const int W = backproject_tiled_window(a.pixel_size);
  if (W == 0 || W > L.n_bins + 2 * L.zpad || L.zpad < 2)
    return set_error(PYHST_ERR_UNSUPPORTED, "tiled backprojector: window %d does not fit", W);
  const size_t smem = SMEM_HDR + (size_t)2 * NA * W * 16;
  if (smem > 200 * 1024)
    return set_error(PYHST_ERR_UNSUPPORTED, "tiled backprojector: pixel size too large");
  static size_t configured = 0;
  if (smem > configured) {
    PYHST_CUDA_TRY(cudaFuncSetAttribute(bp_tiled_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)smem));
    configured = smem;
  }
  dim3 grid((a.nx + TX - 1) / TX, (a.ny + TY - 1) / TY, L.n_groups);
  if (grid.y > 65535 || grid.z > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "tiled backprojector: grid too large");
  StageScope scope(ST_BACKPROJECT, stream);
  scope.kernels();
  bp_tiled_kernel<<<grid, NT, smem, stream>>>(d_qi, L.row_f4(), L.zpad, a.d_img, a.n_slices,
                                              a.n_angles, a.n_bins, a.nx, a.ny, a.scale, a.d_proj,
                                              W);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

}  // namespace pyhst
