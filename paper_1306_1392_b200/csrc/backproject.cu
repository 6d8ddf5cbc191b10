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
// flip (nullable): flip[p] != 0 stores row p reversed (bin b at position B-1-b), see bp_run_kernel
__global__ void repack_to_qi_kernel(const float* __restrict__ sino, int64_t pitch, int S, int P,
                                    int B, int zpad, float4* __restrict__ qi,
                                    const uint8_t* __restrict__ flip) {
  const int64_t row_f4 = (int64_t)B + 2 * zpad;
  const int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;  // padded bin index
  const int p = blockIdx.y, g = blockIdx.z;
  if (x >= row_f4) return;
  int64_t b = x - zpad;
  float v[4] = {0.f, 0.f, 0.f, 0.f};
  if (b >= 0 && b < B) {
    if (flip && flip[p]) b = B - 1 - b;
#pragma unroll
    for (int sl = 0; sl < 4; ++sl) {
      const int s = g * 4 + sl;
      if (s < S) v[sl] = sino[((int64_t)s * P + p) * pitch + b];
    }
  }
  qi[((int64_t)g * P + p) * row_f4 + x] = make_float4(v[0], v[1], v[2], v[3]);
}

int launch_repack_to_qi(const float* d_sino, int64_t pitch, int32_t n_slices, float4* d_qi,
                        const QiLayout& L, const uint8_t* d_flip, cudaStream_t stream) {
  dim3 block(256, 1, 1);
  dim3 grid((unsigned)((L.row_f4() + 255) / 256), L.n_angles, L.n_groups);
  if (grid.y > 65535 || grid.z > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "repack: more than 65535 projections or slice groups");
  StageScope scope(ST_REPACK, stream);
  scope.kernels();
  repack_to_qi_kernel<<<grid, block, 0, stream>>>(d_sino, pitch, n_slices, L.n_angles, L.n_bins,
                                                  L.zpad, d_qi, d_flip);
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

// ------------------------------------------------------------------------------------------
// run kernel (the product path)
//
// The tiled kernel above is bound by shared-memory bandwidth: two 128-bit loads per (pixel,
// projection) and thread = 2 words per update per lane = 16 updates/clk/SM (ncu: l1tex 96 %).
// Here a thread walks a RUN of 16 pixels along the image axis on which the detector coordinate
// moves slowest (step dl = h min(|cos|, |sin|) < 1 bin) and keeps the two taps of 4 slices in
// registers: a step either stays between the same two bins or moves on by exactly one, in which
// case the upper tap becomes the lower one and ONE new float4 is loaded.  Shared-memory traffic
// drops to <= 1 load per update-quad, and the interpolation runs as packed FFMA2.
//   class A projections (|sh| <= |ch|): lanes along x, runs along y
//   class B projections (|ch| <  |sh|): lanes along y, runs along x
// Rows are stored reversed where needed so that the run step is always >= 0 (lerp is symmetric:
// reversing the row maps t -> B-1-t, i.e. flips the signs of ch and sh).  A block first
// accumulates all class-A projections, writes its tile, then accumulates class B in the
// transposed thread mapping and adds it to the tile (same block, so no race).
// ------------------------------------------------------------------------------------------
namespace {

constexpr int RN = 16;        // pixels per run
constexpr int RMAGIC_I = 0x4b000000;

__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
  unsigned long long r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(unsigned long long v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
// d = a * b + d on two packed floats (SASS: FFMA2)
__device__ __forceinline__ void ffma2(unsigned long long& d, unsigned long long a, unsigned long long b) {
  asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
}
__device__ __forceinline__ unsigned long long fadd2(unsigned long long a, unsigned long long b) {
  unsigned long long r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b,
                                                   unsigned long long c) {
  unsigned long long r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}

}  // namespace

// One pass (PASS 0: class A, PASS 1: class B) over entries [e0, e0 + ne) of the run table.
template <int PASS>
__device__ __forceinline__ void bp_run_pass(const float4* __restrict__ qg, int64_t row_f4, int zpad,
                                            float* __restrict__ img, int S, int B, int nx, int ny,
                                            float scale, const RunProj* __restrict__ run, int e0, int ne,
                                            bool add, int W, uint64_t* full, float4* geo, float4* buf,
                                            int& n_issued) {
  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, g = blockIdx.z;
  const int fl = tid & 63;          // position along the fast axis of the class
  const int rn = (tid >> 6) * RN;   // first pixel of the run along the slow axis
  const float ffl = (float)fl, frn = (float)rn;
  const uint32_t win_bytes = (uint32_t)W * 16u;
  const double dx0 = (double)x0 - 0.5 * (double)(nx - 1);
  const double dy0 = (double)y0 - 0.5 * (double)(ny - 1);
  const int n_chunks = (ne + NA - 1) / NA;

  // thread a < NA owns entry c*NA + a of chunk c: window origin and local base in double (R11)
  auto chunk_geometry = [&](int c, int slot) -> int64_t {
    const int e = c * NA + tid;
    if (e >= ne) return -1;
    const RunProj pg = run[e0 + e];
    const double base = pg.c + pg.ch * dx0 + pg.sh * dy0;  // t of the tile's pixel (0,0)
    const double tmin = base + fmin(0.0, pg.ch * (TX - 1)) + fmin(0.0, pg.sh * (TY - 1));
    double o = floor(tmin) - 1.0;                           // one bin of slack for FP32 rounding
    o = fmax(o, -(double)zpad);
    o = fmin(o, (double)(B + zpad - W));
    const float cf = (float)(PASS ? pg.sh : pg.ch), dl = (float)(PASS ? pg.ch : pg.sh);
    // runs that would leave the window (only possible where the window is clamped onto the zero
    // pads, i.e. where every tap is zero) are moved inside it
    geo[slot * NA + tid] = make_float4(cf, dl, (float)(base - o), (float)(W - 3) - (float)(RN - 1) * dl);
    return ((int64_t)pg.p * row_f4 + (int64_t)o + zpad);
  };
  auto issue_chunk = [&](int64_t src, int q) {  // threads tid < NA, after the block barrier
    uint64_t* bar = &full[q & 1];
    if (src >= 0) {
      mbar_arrive_expect_tx(bar, win_bytes);
      bulk_g2s(buf + ((q & 1) * NA + tid) * W, qg + src, win_bytes, bar);
    } else {
      mbar_arrive(bar);
    }
  };

  unsigned long long acc[RN][2];
#pragma unroll
  for (int n = 0; n < RN; ++n) acc[n][0] = acc[n][1] = 0ull;

  int64_t src = -1;
  __syncthreads();  // the previous pass is done with both buffers, the geometry ring and its stores
  if (tid < NA) src = chunk_geometry(0, n_issued % 3);
  __syncthreads();
  if (tid < NA) issue_chunk(src, n_issued);

  for (int c = 0; c < n_chunks; ++c) {
    const int q = n_issued + c;
    if (c + 1 < n_chunks && tid < NA) src = chunk_geometry(c + 1, (q + 1) % 3);
    __syncthreads();  // chunk c-1 is consumed (its buffer is free); geometry of c+1 visible
    if (c + 1 < n_chunks && tid < NA) issue_chunk(src, q + 1);
    mbar_wait(&full[q & 1], (uint32_t)((q >> 1) & 1));

    const int na = min(NA, ne - c * NA);
    const float4* gch = geo + (q % 3) * NA;
    const uint32_t wb = smem_u32(buf + (q & 1) * NA * W);
    for (int a = 0; a < na; ++a) {
      const float4 gg = gch[a];
      float t = fmaf(ffl, gg.x, fmaf(frn, gg.y, gg.z));
      t = fminf(fmaxf(t, 0.f), gg.w);
      const float tm = __fadd_rd(t, 8388608.f);
      const int k = __float_as_int(tm) - RMAGIC_I;
      const float f0 = t - (tm - 8388608.f);
      uint32_t addr = wb + (uint32_t)(a * W + k) * 16u;
      float4 qa, qb;  // lower / upper tap of 4 slices
      asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                   : "=f"(qa.x), "=f"(qa.y), "=f"(qa.z), "=f"(qa.w) : "r"(addr));
      asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+16];"
                   : "=f"(qb.x), "=f"(qb.y), "=f"(qb.z), "=f"(qb.w) : "r"(addr));
      float f = f0;
      const float dl = gg.y;
#pragma unroll
      for (int n = 0; n < RN; ++n) {
        const float w = 1.f - f;
        const unsigned long long w2 = pack2(w, w), f2 = pack2(f, f);  // scalar-broadcast operands
        ffma2(acc[n][0], pack2(qa.x, qa.y), w2);
        ffma2(acc[n][1], pack2(qa.z, qa.w), w2);
        ffma2(acc[n][0], pack2(qb.x, qb.y), f2);
        ffma2(acc[n][1], pack2(qb.z, qb.w), f2);
        if (n + 1 < RN) {
          // f += dl; if f >= 1 the run moved on by one bin: f -= 1, the upper tap becomes the
          // lower one and one new float4 is loaded -- all predicated, registers updated in place.
          // Two of the four register moves are written as x + (-0) so that they issue on the FMA
          // pipe instead of the half-rate ALU pipe that FSEL/MOV use.
          asm volatile(
              "{\n\t"
              ".reg .pred p;\n\t"
              "add.rn.f32 %9, %9, %10;\n\t"
              "setp.ge.f32 p, %9, 0f3F800000;\n\t"
              "@p add.rn.f32 %9, %9, 0fBF800000;\n\t"
              "@p mov.f32 %0, %4;\n\t"
              "@p add.rn.f32 %1, %5, 0f80000000;\n\t"
              "@p mov.f32 %2, %6;\n\t"
              "@p add.rn.f32 %3, %7, 0f80000000;\n\t"
              "@p add.u32 %8, %8, 16;\n\t"
              "@p ld.shared.v4.f32 {%4, %5, %6, %7}, [%8+16];\n\t"
              "}"
              : "+f"(qa.x), "+f"(qa.y), "+f"(qa.z), "+f"(qa.w), "+f"(qb.x), "+f"(qb.y), "+f"(qb.z),
                "+f"(qb.w), "+r"(addr), "+f"(f)
              : "f"(dl));
        }
      }
    }
  }
  n_issued += n_chunks;

  // ---- write the tile
  if (PASS == 0) {  // pixel (x0 + fl, y0 + rn + n): lanes along x, coalesced
    const int x = x0 + fl;
    if (x < nx) {
#pragma unroll
      for (int n = 0; n < RN; ++n) {
        const int y = y0 + rn + n;
        float v[4];
        unpack2(acc[n][0], v[0], v[1]);
        unpack2(acc[n][1], v[2], v[3]);
        if (y < ny) {
#pragma unroll
          for (int sl = 0; sl < 4; ++sl) {
            const int s = g * 4 + sl;
            if (s < S) img[((int64_t)s * ny + y) * nx + x] = scale * v[sl];
          }
        }
      }
    }
  } else {  // pixel (x0 + rn + n, y0 + fl): 16 consecutive x per thread, added to what pass 0 wrote
    const int y = y0 + fl;
    if (y < ny) {
      float v[RN][4];
#pragma unroll
      for (int n = 0; n < RN; ++n) {
        unpack2(acc[n][0], v[n][0], v[n][1]);
        unpack2(acc[n][1], v[n][2], v[n][3]);
      }
#pragma unroll
      for (int sl = 0; sl < 4; ++sl) {
        const int s = g * 4 + sl;
        if (s < S) {
          float* row = img + ((int64_t)s * ny + y) * nx + x0 + rn;
          const bool vec = ((reinterpret_cast<uintptr_t>(row) & 15) == 0) && (x0 + rn + RN <= nx);
#pragma unroll
          for (int n4 = 0; n4 < RN; n4 += 4) {
            if (vec) {
              float4 o = add ? *reinterpret_cast<const float4*>(row + n4) : make_float4(0.f, 0.f, 0.f, 0.f);
              o.x = fmaf(scale, v[n4][sl], o.x);
              o.y = fmaf(scale, v[n4 + 1][sl], o.y);
              o.z = fmaf(scale, v[n4 + 2][sl], o.z);
              o.w = fmaf(scale, v[n4 + 3][sl], o.w);
              *reinterpret_cast<float4*>(row + n4) = o;
            } else {
#pragma unroll
              for (int j = 0; j < 4; ++j)
                if (x0 + rn + n4 + j < nx)
                  row[n4 + j] = fmaf(scale, v[n4 + j][sl], add ? row[n4 + j] : 0.f);
            }
          }
        }
      }
    }
  }
}

__global__ void __launch_bounds__(NT, 2)
bp_run_kernel(const float4* __restrict__ qi, int64_t row_f4, int zpad, float* img, int S, int B,
              int nx, int ny, float scale, const RunProj* __restrict__ run, int n_a, int n_b, int W) {
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);                 // [2]
  float4* geo = reinterpret_cast<float4*>(smem + 64);                 // [3][NA] (c_fast, dl, base, t_hi)
  float4* buf = reinterpret_cast<float4*>(smem + SMEM_HDR);           // [2][NA][W]
  const float4* qg = qi + (int64_t)blockIdx.z * (n_a + n_b) * row_f4;
  if (threadIdx.x == 0) {
    mbar_init(&full[0], NA);
    mbar_init(&full[1], NA);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  int n_issued = 0;  // chunks issued so far (both passes): buffer / mbarrier-parity bookkeeping
  if (n_a > 0)
    bp_run_pass<0>(qg, row_f4, zpad, img, S, B, nx, ny, scale, run, 0, n_a, false, W, full, geo, buf, n_issued);
  if (n_b > 0)
    bp_run_pass<1>(qg, row_f4, zpad, img, S, B, nx, ny, scale, run, n_a, n_b, n_a > 0, W, full, geo, buf,
                   n_issued);
}

int backproject_run_window(double pixel_size) {
  // the run step h min(|cos|, |sin|) <= h / sqrt(2) must stay below one bin
  if (!(pixel_size * 0.70710678118654757 < 0.999)) return 0;
  return backproject_tiled_window(pixel_size);
}

int launch_backproject_run(const float4* d_qi, const QiLayout& L, const BpArgs& a,
                           const RunProj* d_run, int32_t n_a, int32_t n_b, cudaStream_t stream) {
  const int W = backproject_run_window(a.pixel_size);
  if (W == 0 || W > L.n_bins + 2 * L.zpad || L.zpad < W + 2)
    return set_error(PYHST_ERR_UNSUPPORTED, "run backprojector: window %d does not fit", W);
  const size_t smem = SMEM_HDR + (size_t)2 * NA * W * 16;
  if (smem > 200 * 1024)
    return set_error(PYHST_ERR_UNSUPPORTED, "run backprojector: pixel size too large");
  static PerDeviceSize configured;
  if (smem > configured.here()) {
    PYHST_CUDA_TRY(cudaFuncSetAttribute(bp_run_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)smem));
    configured.here() = smem;
  }
  dim3 grid((a.nx + TX - 1) / TX, (a.ny + TY - 1) / TY, L.n_groups);
  if (grid.y > 65535 || grid.z > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "run backprojector: grid too large");
  StageScope scope(ST_BACKPROJECT, stream);
  scope.kernels();
  bp_run_kernel<<<grid, NT, smem, stream>>>(d_qi, L.row_f4(), L.zpad, a.d_img, a.n_slices, a.n_bins,
                                            a.nx, a.ny, a.scale, d_run, n_a, n_b, W);
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

int backproject_tiled_window(double pixel_size) {
  // span of t over a tile <= h * sqrt((TX-1)^2 + (TY-1)^2); + floor, second tap and slack
  const double span = pixel_size * sqrt((double)((TX - 1) * (TX - 1) + (TY - 1) * (TY - 1)));
  const double w = ceil(span) + 5.0;
  if (w > 1024.0) return 0;
  const int W = ((int)w + 3) & ~3;
  // same limit as launch_backproject_tiled: beyond it pick_bp_kernel falls back to the reference kernel
  if (SMEM_HDR + (size_t)2 * NA * W * 16 > 200 * 1024) return 0;
  return W;
}

int launch_backproject_tiled(const float4* d_qi, const QiLayout& L, const BpArgs& a,
                             cudaStream_t stream) {
  const int W = backproject_tiled_window(a.pixel_size);
  if (W == 0 || W > L.n_bins + 2 * L.zpad || L.zpad < 2)
    return set_error(PYHST_ERR_UNSUPPORTED, "tiled backprojector: window %d does not fit", W);
  const size_t smem = SMEM_HDR + (size_t)2 * NA * W * 16;
  if (smem > 200 * 1024)
    return set_error(PYHST_ERR_UNSUPPORTED, "tiled backprojector: pixel size too large");
  static PerDeviceSize configured;
  if (smem > configured.here()) {
    PYHST_CUDA_TRY(cudaFuncSetAttribute(bp_tiled_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)smem));
    configured.here() = smem;
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
