// Backprojection P^T for stacks of >= 13 slices (include/pyhst.h a2; readings R1-R7,
// R11 of DESIGN.md):   img[s,i,j] = scale * sum_p lerp(q[s,p,:], c_p + ch_p (j-j0) + sh_p (i-i0))
//
// bp_run16_kernel<PASS>: the run scheme of bp_run8_kernel (backproject_run8.cu) with SIXTEEN slices (four
// interleaved slice groups) per thread.  Every instruction of the run loop costs one issue slot
// (profiles/r02_micro.md); per step of one pixel the 5 instructions of weight logic (f += dl, compare, wrap,
// w = 1 - f, address) are shared by 32 FFMAs instead of 16.  Registers: 16 slices x 4 pixels of a run = 64
// accumulators + 32 taps, so runs are 4 pixels long and a block is 512 threads (64 lanes x 8 runs x 4 pixels
// = the 64 x 32 tile of bp_run8_kernel), one block per SM.  Staging, producer rotation and the two passes
// (class A: lanes along x, runs along y; class B: transposed, through shared memory) are those of
// bp_run8_kernel.  Taps are held as 64-bit register pairs so that the step fits one asm statement.
#include "common.h"

namespace pyhst {

namespace {

constexpr int R16_LANES = 64;   // tile extent along the fast axis of the class (one lane each)
constexpr int R16_RN = 4;       // pixels per run
constexpr int R16_RG = 8;       // runs per lane column: extent along the slow axis = RG * RN = 32
constexpr int R16_SLOW = R16_RG * R16_RN;
constexpr int R16_NT = R16_LANES * R16_RG;   // 512
constexpr int R16_NG = 4;       // slice groups per block
constexpr int R16_NA = 8;       // projections per staged chunk
constexpr int R16_HDR = 1024;   // mbarriers + geometry ring

__device__ __forceinline__ float lo32(uint64_t v) { return __uint_as_float((uint32_t)v); }
__device__ __forceinline__ float hi32(uint64_t v) { return __uint_as_float((uint32_t)(v >> 32)); }

#define R16_LD2(d0, d1, a) asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(d0), "=l"(d1) : "r"(a))

// One run of R16_RN pixels of one projection, 16 slices.  qa[g][0..1] / qb[g][0..1]: lower / upper taps of
// slice group g (two 64-bit pairs = 4 slices).  f += dl; when f >= 1 the run has moved on by one bin: f -= 1,
// the upper taps become the lower ones and one new 16-byte tap per group is loaded -- all predicated.
template <int GOFF>
__device__ __forceinline__ void r16_run(float (&acc)[R16_RN][16], uint32_t addr, float f, const float dl) {
  uint64_t qa[R16_NG][2], qb[R16_NG][2];
#pragma unroll
  for (int g = 0; g < R16_NG; ++g) {
    R16_LD2(qa[g][0], qa[g][1], addr + g * GOFF);
    R16_LD2(qb[g][0], qb[g][1], addr + g * GOFF + 16);
  }
#pragma unroll
  for (int n = 0; n < R16_RN; ++n) {
    const float w = 1.f - f;
#pragma unroll
    for (int g = 0; g < R16_NG; ++g) {
      acc[n][4 * g + 0] = fmaf(lo32(qb[g][0]), f, fmaf(lo32(qa[g][0]), w, acc[n][4 * g + 0]));
      acc[n][4 * g + 1] = fmaf(hi32(qb[g][0]), f, fmaf(hi32(qa[g][0]), w, acc[n][4 * g + 1]));
      acc[n][4 * g + 2] = fmaf(lo32(qb[g][1]), f, fmaf(lo32(qa[g][1]), w, acc[n][4 * g + 2]));
      acc[n][4 * g + 3] = fmaf(hi32(qb[g][1]), f, fmaf(hi32(qa[g][1]), w, acc[n][4 * g + 3]));
    }
    if (n + 1 < R16_RN) {
      asm volatile(
          "{\n\t"
          ".reg .pred p;\n\t"
          "add.rn.f32 %17, %17, %18;\n\t"
          "setp.ge.f32 p, %17, 0f3F800000;\n\t"
          "@p add.rn.f32 %17, %17, 0fBF800000;\n\t"
          "@p mov.b64 %0, %8;\n\t"
          "@p mov.b64 %1, %9;\n\t"
          "@p mov.b64 %2, %10;\n\t"
          "@p mov.b64 %3, %11;\n\t"
          "@p mov.b64 %4, %12;\n\t"
          "@p mov.b64 %5, %13;\n\t"
          "@p mov.b64 %6, %14;\n\t"
          "@p mov.b64 %7, %15;\n\t"
          "@p add.u32 %16, %16, 16;\n\t"
          "@p ld.shared.v2.b64 {%8, %9}, [%16+16];\n\t"
          "@p ld.shared.v2.b64 {%10, %11}, [%16+%19];\n\t"
          "@p ld.shared.v2.b64 {%12, %13}, [%16+%20];\n\t"
          "@p ld.shared.v2.b64 {%14, %15}, [%16+%21];\n\t"
          "}"
          : "+l"(qa[0][0]), "+l"(qa[0][1]), "+l"(qa[1][0]), "+l"(qa[1][1]), "+l"(qa[2][0]), "+l"(qa[2][1]),
            "+l"(qa[3][0]), "+l"(qa[3][1]), "+l"(qb[0][0]), "+l"(qb[0][1]), "+l"(qb[1][0]), "+l"(qb[1][1]),
            "+l"(qb[2][0]), "+l"(qb[2][1]), "+l"(qb[3][0]), "+l"(qb[3][1]), "+r"(addr), "+f"(f)
          : "f"(dl), "n"(GOFF + 16), "n"(2 * GOFF + 16), "n"(3 * GOFF + 16));
    }
  }
}

}  // namespace

// PASS 0: entries [e0, e0 + ne) are class A (lanes along x, runs along y), tile 64 (x) x 32 (y).
// PASS 1: class B (lanes along y, runs along x), tile 32 (x) x 64 (y); add != 0: added to img.
// WS = window slot stride in float4; NS = stages; chunks are issued NS - 2 ahead.
template <int PASS, int WS, int NS>
__global__ void __launch_bounds__(R16_NT, 1)
bp_run16_kernel(const float4* __restrict__ qi, int64_t row_f4, int zpad, float* img, int S, int n_groups, int P,
                int B, int nx, int ny, float scale, const RunProj* __restrict__ run, int e0, int ne, int add,
                int W) {
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);         // [NS]
  uint64_t* empty = reinterpret_cast<uint64_t*>(smem + 64);   // [NS]
  float4* geo = reinterpret_cast<float4*>(smem + 128);        // [NS][NA] (c_fast, dl, base, t_hi)
  float4* buf = reinterpret_cast<float4*>(smem + R16_HDR);    // [NS][NA][NG][WS]

  constexpr int EX = PASS ? R16_SLOW : R16_LANES, EY = PASS ? R16_LANES : R16_SLOW;
  constexpr int NWARP = R16_NT / 32;
  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * EX, y0 = blockIdx.y * EY;
  const int gA = blockIdx.z * R16_NG;
  const int n_chunks = (ne + R16_NA - 1) / R16_NA;
  const uint32_t win_bytes = (uint32_t)W * 16u;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full[s], R16_NA);
      mbar_init(&empty[s], NWARP);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // producer role (one warp, lanes < NA): window geometry in double (R11) + TMA bulk copies of chunk c
  const double dx0 = (double)x0 - 0.5 * (double)(nx - 1);
  const double dy0 = (double)y0 - 0.5 * (double)(ny - 1);
  auto produce = [&](int c) {
    const int st = c % NS;
    if (c >= NS) mbar_wait(&empty[st], (uint32_t)(((c / NS) - 1) & 1));
    const int pl = tid & 31;
    if (pl < R16_NA) {
      const int e = c * R16_NA + pl;
      uint64_t* bar = &full[st];
      if (e < ne) {
        const RunProj pg = run[e0 + e];
        const double base = pg.c + pg.ch * dx0 + pg.sh * dy0;  // t of the tile's pixel (0,0)
        const double tmin = base + fmin(0.0, pg.ch * (EX - 1)) + fmin(0.0, pg.sh * (EY - 1));
        double o = floor(tmin) - 1.0;                           // one bin of slack for FP32 rounding
        o = fmax(o, -(double)zpad);
        o = fmin(o, (double)(B + zpad - W));
        const float cf = (float)(PASS ? pg.sh : pg.ch), dl = (float)(PASS ? pg.ch : pg.sh);
        // runs that would leave the window (only where it is clamped onto the zero pads) are moved inside it
        geo[st * R16_NA + pl] =
            make_float4(cf, dl, (float)(base - o), (float)(W - 3) - (float)(R16_RN - 1) * dl);
        const int64_t src = (int64_t)pg.p * row_f4 + (int64_t)o + zpad;
        float4* dst = buf + (size_t)(st * R16_NA + pl) * R16_NG * WS;
        mbar_arrive_expect_tx(bar, R16_NG * win_bytes);
#pragma unroll
        for (int g = 0; g < R16_NG; ++g) {
          const int gg = min(gA + g, n_groups - 1);   // ragged stacks: a duplicate group, never stored
          bulk_g2s(dst + g * WS, qi + (int64_t)gg * P * row_f4 + src, win_bytes, bar);
        }
      } else {
        mbar_arrive(bar);
      }
    }
    __syncwarp();
  };
  if (tid < 32) {
#pragma unroll 1
    for (int c = 0; c < (NS - 2) && c < n_chunks; ++c) produce(c);
  }

  // consumers
  const int fl = tid & (R16_LANES - 1);       // position along the fast axis of the class
  const int rn = (tid >> 6) * R16_RN;         // first pixel of the run along the slow axis
  const float ffl = (float)fl, frn = (float)rn;
  const uint32_t wb = smem_u32(buf);

  float acc[R16_RN][16];
#pragma unroll
  for (int n = 0; n < R16_RN; ++n)
#pragma unroll
    for (int j = 0; j < 16; ++j) acc[n][j] = 0.f;

  for (int c = 0; c < n_chunks; ++c) {
    // the producer role rotates over the warps, so that no warp is the slowest one
    if ((tid >> 5) == ((c + (NS - 2)) % NWARP) && c + (NS - 2) < n_chunks) produce(c + (NS - 2));
    const int st = c % NS;
    mbar_wait(&full[st], (uint32_t)((c / NS) & 1));
    const int na = min(R16_NA, ne - c * R16_NA);
    const float4* gch = geo + st * R16_NA;
    const uint32_t sb = wb + (uint32_t)(st * R16_NA) * (uint32_t)(R16_NG * WS * 16);
#pragma unroll 2
    for (int a = 0; a < na; ++a) {
      const float4 gg = gch[a];
      float t = fmaf(ffl, gg.x, fmaf(frn, gg.y, gg.z));
      t = fminf(fmaxf(t, 0.f), gg.w);
      const float tm = __fadd_rd(t, 8388608.f);
      const int k = __float_as_int(tm) - 0x4b000000;
      const float f0 = t - (tm - 8388608.f);
      const uint32_t addr = sb + (uint32_t)a * (uint32_t)(R16_NG * WS * 16) + (uint32_t)k * 16u;
      r16_run<WS * 16>(acc, addr, f0, gg.y);
    }
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(&empty[st]);
  }

  // write the tile: acc[n][4 g + j] = slice 4 (gA + g) + j
  if (PASS == 0) {  // pixel (x0 + fl, y0 + rn + n): lanes along x, coalesced
    const int x = x0 + fl;
    if (x < nx) {
#pragma unroll
      for (int n = 0; n < R16_RN; ++n) {
        const int y = y0 + rn + n;
        if (y >= ny) continue;
#pragma unroll
        for (int sl = 0; sl < 16; ++sl) {
          const int s = gA * 4 + sl;
          if (s < S) {
            float* dst = img + ((int64_t)s * ny + y) * nx + x;
            *dst = add ? fmaf(scale, acc[n][sl], *dst) : scale * acc[n][sl];
          }
        }
      }
    }
  } else {
    // pixel (x0 + rn + n, y0 + fl): lanes run along y, so the tile goes through shared memory (the window ring is
    // free: every chunk has been consumed) and is written / added row by row
    constexpr int TP = R16_SLOW + 1;                     // padded row of the transposed tile
    float* ts = reinterpret_cast<float*>(buf);           // [16 slices][64 rows][TP]
    __syncthreads();
#pragma unroll
    for (int n = 0; n < R16_RN; ++n)
#pragma unroll
      for (int sl = 0; sl < 16; ++sl) ts[(sl * R16_LANES + fl) * TP + rn + n] = acc[n][sl];
    __syncthreads();
    const bool vec_ok = (nx % 4 == 0) && ((reinterpret_cast<uintptr_t>(img) & 15) == 0);
#pragma unroll 1
    for (int sl = 0; sl < 16; ++sl) {
      const int s = gA * 4 + sl;
      if (s >= S) break;
      const int yl = tid >> 3, xl = (tid & 7) * 4;     // 512 threads = 64 rows x 8 quads
      const int y = y0 + yl, x = x0 + xl;
      if (y >= ny || x >= nx) continue;
      const float* t4 = ts + (sl * R16_LANES + yl) * TP + xl;
      float* row = img + ((int64_t)s * ny + y) * nx + x;
      if (vec_ok && x + 4 <= nx) {
        float4 o = add ? *reinterpret_cast<const float4*>(row) : make_float4(0.f, 0.f, 0.f, 0.f);
        o.x = fmaf(scale, t4[0], o.x);
        o.y = fmaf(scale, t4[1], o.y);
        o.z = fmaf(scale, t4[2], o.z);
        o.w = fmaf(scale, t4[3], o.w);
        *reinterpret_cast<float4*>(row) = o;
      } else {
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (x + j < nx) row[j] = fmaf(scale, t4[j], add ? row[j] : 0.f);
      }
    }
  }
}

namespace {

template <int WS, int NS>
int launch_run16(const float4* d_qi, const QiLayout& L, const BpArgs& a, const RunProj* d_run, int32_t n_a,
                 int32_t n_b, int W, cudaStream_t stream) {
  const size_t smem = R16_HDR + (size_t)NS * R16_NA * R16_NG * WS * 16;
  static DeviceMask configured{0};   // one bit per device (cudaFuncSetAttribute is per device)
  if (first_use_on_device(&configured)) {
    PYHST_CUDA_TRY(cudaFuncSetAttribute(bp_run16_kernel<0, WS, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)smem));
    PYHST_CUDA_TRY(cudaFuncSetAttribute(bp_run16_kernel<1, WS, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)smem));
  }
  const unsigned gz = (unsigned)((L.n_groups + R16_NG - 1) / R16_NG);
  dim3 grid_a((a.nx + R16_LANES - 1) / R16_LANES, (a.ny + R16_SLOW - 1) / R16_SLOW, gz);
  dim3 grid_b((a.nx + R16_SLOW - 1) / R16_SLOW, (a.ny + R16_LANES - 1) / R16_LANES, gz);
  if (grid_a.y > 65535 || grid_b.y > 65535 || gz > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "run16 backprojector: grid too large");
  StageScope scope(ST_BACKPROJECT, stream);
  if (n_a > 0 || n_b == 0) {
    scope.kernels();
    bp_run16_kernel<0, WS, NS><<<grid_a, R16_NT, smem, stream>>>(d_qi, L.row_f4(), L.zpad, a.d_img, a.n_slices,
                                                                 L.n_groups, L.n_angles, a.n_bins, a.nx, a.ny,
                                                                 a.scale, d_run, 0, n_a, 0, W);
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  if (n_b > 0) {
    scope.kernels();
    bp_run16_kernel<1, WS, NS><<<grid_b, R16_NT, smem, stream>>>(d_qi, L.row_f4(), L.zpad, a.d_img, a.n_slices,
                                                                 L.n_groups, L.n_angles, a.n_bins, a.nx, a.ny,
                                                                 a.scale, d_run, n_a, n_b, n_a > 0 ? 1 : 0, W);
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  return PYHST_OK;
}

}  // namespace

// 16-slice form of the run backprojector: covers the same geometries as run8 with windows of <= 80 bins
bool backproject_run16_covers(double pixel_size, int n_groups) {
  const int W = backproject_run8_window(pixel_size);
  return W > 0 && W <= 80 && n_groups >= 4;
}

int launch_backproject_run16(const float4* d_qi, const QiLayout& L, const BpArgs& a, const RunProj* d_run,
                             int32_t n_a, int32_t n_b, cudaStream_t stream) {
  const int W = backproject_run8_window(a.pixel_size);
  if (W == 0 || W > 80 || W > L.n_bins + 2 * L.zpad || L.zpad < W + 2)
    return set_error(PYHST_ERR_UNSUPPORTED, "run16 backprojector: window %d does not fit", W);
  return launch_run16<80, 4>(d_qi, L, a, d_run, n_a, n_b, W, stream);   // 4 x 8 x 4 x 80 x 16 B = 160 KB
}

}  // namespace pyhst
