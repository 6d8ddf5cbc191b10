// Backprojection P^T, the product kernel (include/pyhst.h a2; readings R1-R7,
// R11 of DESIGN.md):   img[s,i,j] = scale * sum_p lerp(q[s,p,:], c_p + ch_p (j-j0) + sh_p (i-i0))
//
// bp_run8_kernel<PASS>: the run scheme of bp_run_kernel (backproject.cu) with the measured cost
// model of sm_100a applied.  On B200 an FFMA2 occupies the issue port for two cycles, so every
// instruction of the run loop costs as much as one FFMA: a warp-step (32 lanes x 4 slices x one
// pixel x one projection = 128 updates) is 8 slots of algorithmic FMA work plus one slot per
// overhead instruction.  Hence:
//   * a thread owns EIGHT slices (two interleaved slice groups): the weight logic (f += dl, wrap,
//     w = 1 - f, predicate, address) is shared by twice the FMA work;
//   * runs are 8 pixels long (64 accumulator registers), four independent projections are kept in
//     flight per thread (the loop is latency-sensitive at 4 warps per scheduler);
//   * the producer role rotates over the warps: the producing warp computes the window geometry
//     in double (R11) and issues the TMA bulk copies two chunks ahead; warps meet only through
//     full/empty mbarriers -- no block-wide barrier in the projection loop;
//   * class A (|sh| <= |ch|, lanes along x, runs along y) and class B (lanes along y, runs along
//     x) are two launches: pass 0 writes the image, pass 1 adds to it.
#include "common.h"

#ifndef R8_RELOAD
#define R8_RELOAD 0
#endif
namespace pyhst {

namespace {

constexpr int R8_LANES = 64;   // tile extent along the fast axis of the class (one lane each)
constexpr int R8_RN = 8;       // pixels per run
constexpr int R8_RG = 4;       // runs per lane column: extent along the slow axis = RG * RN = 32
constexpr int R8_SLOW = R8_RG * R8_RN;
constexpr int R8_NC = 256;     // consumer threads (8 warps)
constexpr int R8_NT = R8_NC;
constexpr int R8_NA = 8;       // projections per staged chunk
constexpr int R8_HDR = 1024;   // mbarriers + geometry ring; keeps the windows 128-B aligned

#define R8_LD4(q, a)                                                                      \
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"                                 \
               : "=f"(q.x), "=f"(q.y), "=f"(q.z), "=f"(q.w)                               \
               : "r"(a))

}  // namespace

namespace {

// One run of R8_RN pixels of one projection, 8 slices: (qa, qb) / (ra, rb) are the lower / upper
// taps of the two slice groups, kept in registers.  f += dl; when f >= 1 the run has moved on by
// one bin: f -= 1, the upper taps become the lower ones and one new float4 per group is loaded --
// all predicated, registers updated in place.  Half of the register moves are written as x + (-0)
// (FMA pipe), half as FSEL (ALU pipe).  The interpolation is scalar FFMA: an FFMA2 holds the issue
// port for two cycles on sm_100a, so packing saves nothing and costs pair-alignment MOVs.
// GOFF = byte offset of the second group's window (compile-time: one address register).
template <int GOFF>
__device__ __forceinline__ void r8_run(float (&acc)[R8_RN][8], uint32_t addr, float f,
                                       const float dl) {
  float4 qa, qb, ra, rb;
  R8_LD4(qa, addr);
  R8_LD4(qb, addr + 16);
  R8_LD4(ra, addr + GOFF);
  R8_LD4(rb, addr + GOFF + 16);
#pragma unroll
  for (int n = 0; n < R8_RN; ++n) {
    const float w = 1.f - f;
    acc[n][0] = fmaf(qb.x, f, fmaf(qa.x, w, acc[n][0]));
    acc[n][1] = fmaf(qb.y, f, fmaf(qa.y, w, acc[n][1]));
    acc[n][2] = fmaf(qb.z, f, fmaf(qa.z, w, acc[n][2]));
    acc[n][3] = fmaf(qb.w, f, fmaf(qa.w, w, acc[n][3]));
    acc[n][4] = fmaf(rb.x, f, fmaf(ra.x, w, acc[n][4]));
    acc[n][5] = fmaf(rb.y, f, fmaf(ra.y, w, acc[n][5]));
    acc[n][6] = fmaf(rb.z, f, fmaf(ra.z, w, acc[n][6]));
    acc[n][7] = fmaf(rb.w, f, fmaf(ra.w, w, acc[n][7]));
    if (n + 1 < R8_RN) {
      asm volatile(
          "{\n\t"
          ".reg .pred p;\n\t"
          "add.rn.f32 %17, %17, %18;\n\t"
          "setp.ge.f32 p, %17, 0f3F800000;\n\t"
          "@p add.rn.f32 %17, %17, 0fBF800000;\n\t"
#if R8_RELOAD
          "@p add.u32 %16, %16, 16;\n\t"
          "@p ld.shared.v4.f32 {%0, %1, %2, %3}, [%16];\n\t"
          "@p ld.shared.v4.f32 {%4, %5, %6, %7}, [%16+16];\n\t"
          "@p ld.shared.v4.f32 {%8, %9, %10, %11}, [%16+%20];\n\t"
          "@p ld.shared.v4.f32 {%12, %13, %14, %15}, [%16+%19];\n\t"
          "}"
#else
          "@p mov.f32 %0, %4;\n\t"
          "@p add.rn.f32 %1, %5, 0f80000000;\n\t"
          "@p mov.f32 %2, %6;\n\t"
          "@p add.rn.f32 %3, %7, 0f80000000;\n\t"
          "@p mov.f32 %8, %12;\n\t"
          "@p add.rn.f32 %9, %13, 0f80000000;\n\t"
          "@p mov.f32 %10, %14;\n\t"
          "@p add.rn.f32 %11, %15, 0f80000000;\n\t"
          "@p add.u32 %16, %16, 16;\n\t"
          "@p ld.shared.v4.f32 {%4, %5, %6, %7}, [%16+16];\n\t"
          "@p ld.shared.v4.f32 {%12, %13, %14, %15}, [%16+%19];\n\t"
          "}"
#endif
          : "+f"(qa.x), "+f"(qa.y), "+f"(qa.z), "+f"(qa.w), "+f"(qb.x), "+f"(qb.y), "+f"(qb.z),
            "+f"(qb.w), "+f"(ra.x), "+f"(ra.y), "+f"(ra.z), "+f"(ra.w), "+f"(rb.x), "+f"(rb.y),
            "+f"(rb.z), "+f"(rb.w), "+r"(addr), "+f"(f)
          : "f"(dl), "n"(GOFF + 16), "n"(GOFF));
    }
  }
}


// (c0, c1) += (a0, a1) * (s, s): one packed FFMA2.  Measured (profiles/r03_micro.md, counters): an FFMA2 occupies
// BOTH 16-lane FMA pipes of the scheduler (fmaheavy and fmalite) for two cycles and blocks the dispatch port for
// those two cycles; ALU-pipe (FSEL, LOP3) and FMA-pipe (FADD) instructions do NOT issue in its shadow (8 FFMA2 +
// 8 FSEL = 27.9 cycles against 26.7 for 16 FFMA + 8 FSEL).  Packing saves instructions, not time.
__device__ __forceinline__ uint64_t r8_pair(float s) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %1};" : "=l"(r) : "f"(s));
  return r;
}
__device__ __forceinline__ void r8_ffma2(float& c0, float& c1, float a0, float a1, uint64_t s2) {
  asm("{\n\t.reg .b64 ra, rc;\n\t"
      "mov.b64 ra, {%2, %3};\n\t"
      "mov.b64 rc, {%0, %1};\n\t"
      "fma.rn.f32x2 rc, ra, %4, rc;\n\t"
      "mov.b64 {%0, %1}, rc;\n\t}"
      : "+f"(c0), "+f"(c1)
      : "f"(a0), "f"(a1), "l"(s2));
}

// r8_run with the interpolation written as packed FFMA2 (two slices per instruction); the tap moves are
// all FSEL-class (ALU pipe), so that the FMA pipe only carries the FFMA2s and the three weight FADDs.
template <int GOFF>
__device__ __forceinline__ void r8_run_packed(float (&acc)[R8_RN][8], uint32_t addr, float f, const float dl) {
  float4 qa, qb, ra, rb;
  R8_LD4(qa, addr);
  R8_LD4(qb, addr + 16);
  R8_LD4(ra, addr + GOFF);
  R8_LD4(rb, addr + GOFF + 16);
#pragma unroll
  for (int n = 0; n < R8_RN; ++n) {
    const uint64_t w2 = r8_pair(1.f - f), f2 = r8_pair(f);
    r8_ffma2(acc[n][0], acc[n][1], qa.x, qa.y, w2);
    r8_ffma2(acc[n][2], acc[n][3], qa.z, qa.w, w2);
    r8_ffma2(acc[n][4], acc[n][5], ra.x, ra.y, w2);
    r8_ffma2(acc[n][6], acc[n][7], ra.z, ra.w, w2);
    r8_ffma2(acc[n][0], acc[n][1], qb.x, qb.y, f2);
    r8_ffma2(acc[n][2], acc[n][3], qb.z, qb.w, f2);
    r8_ffma2(acc[n][4], acc[n][5], rb.x, rb.y, f2);
    r8_ffma2(acc[n][6], acc[n][7], rb.z, rb.w, f2);
    if (n + 1 < R8_RN) {
      asm volatile(
          "{\n\t"
          ".reg .pred p;\n\t"
          "add.rn.f32 %17, %17, %18;\n\t"
          "setp.ge.f32 p, %17, 0f3F800000;\n\t"
          "@p add.rn.f32 %17, %17, 0fBF800000;\n\t"
          "@p mov.f32 %0, %4;\n\t"
          "@p mov.f32 %1, %5;\n\t"
          "@p mov.f32 %2, %6;\n\t"
          "@p mov.f32 %3, %7;\n\t"
          "@p mov.f32 %8, %12;\n\t"
          "@p mov.f32 %9, %13;\n\t"
          "@p mov.f32 %10, %14;\n\t"
          "@p mov.f32 %11, %15;\n\t"
          "@p add.u32 %16, %16, 16;\n\t"
          "@p ld.shared.v4.f32 {%4, %5, %6, %7}, [%16+16];\n\t"
          "@p ld.shared.v4.f32 {%12, %13, %14, %15}, [%16+%19];\n\t"
          "}"
          : "+f"(qa.x), "+f"(qa.y), "+f"(qa.z), "+f"(qa.w), "+f"(qb.x), "+f"(qb.y), "+f"(qb.z),
            "+f"(qb.w), "+f"(ra.x), "+f"(ra.y), "+f"(ra.z), "+f"(ra.w), "+f"(rb.x), "+f"(rb.y),
            "+f"(rb.z), "+f"(rb.w), "+r"(addr), "+f"(f)
          : "f"(dl), "n"(GOFF + 16));
    }
  }
}

}  // namespace

// PASS 0: entries [e0, e0 + ne) are class A (lanes along x, runs along y), tile 64 (x) x 32 (y).
// PASS 1: class B (lanes along y, runs along x), tile 32 (x) x 64 (y).
// add != 0: the tile is added to what is already in img (pass 1 after pass 0).
// WS = window slot stride in float4 (compile-time, so that the second slice group's taps sit at a
// constant offset from the first one's); W <= WS bins are staged.  NS = stages; chunks are issued
// NS - 2 ahead of the one being consumed (the producing warp may then run ahead of the slowest
// warp by up to two chunks without waiting).
template <int PASS, int WS, int NS, bool PACKED>
__global__ void __launch_bounds__(R8_NT, 2)
bp_run8_kernel(const float4* __restrict__ qi, int64_t row_f4, int zpad, float* img, int S,
               int n_groups, int P, int B, int nx, int ny, float scale,
               const RunProj* __restrict__ run, int e0, int ne, int add, int W) {
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);         // [NS]
  uint64_t* empty = reinterpret_cast<uint64_t*>(smem + 64);   // [NS]
  float4* geo = reinterpret_cast<float4*>(smem + 128);        // [NS][NA] (c_fast, dl, base, t_hi)
  float4* buf = reinterpret_cast<float4*>(smem + R8_HDR);     // [NS][NA][2][WS]

  constexpr int EX = PASS ? R8_SLOW : R8_LANES, EY = PASS ? R8_LANES : R8_SLOW;
  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * EX, y0 = blockIdx.y * EY;
  const int gA = blockIdx.z * 2, gB = min(gA + 1, n_groups - 1);
  const int n_chunks = (ne + R8_NA - 1) / R8_NA;
  const uint32_t win_bytes = (uint32_t)W * 16u;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full[s], R8_NA);
      mbar_init(&empty[s], R8_NC / 32);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // ---------------- producer role (one warp, lanes < NA): window geometry in double (R11) + TMA
  // bulk copies of chunk c into stage c % NS; the stage was last read as chunk c - NS
  const double dx0 = (double)x0 - 0.5 * (double)(nx - 1);
  const double dy0 = (double)y0 - 0.5 * (double)(ny - 1);
  const float4* qA = qi + (int64_t)gA * P * row_f4;
  const float4* qB = qi + (int64_t)gB * P * row_f4;
  auto produce = [&](int c) {
    const int st = c % NS;
    if (c >= NS) mbar_wait(&empty[st], (uint32_t)(((c / NS) - 1) & 1));
    const int pl = tid & 31;
    if (pl < R8_NA) {
      const int e = c * R8_NA + pl;
      uint64_t* bar = &full[st];
      if (e < ne) {
        const RunProj pg = run[e0 + e];
        const double base = pg.c + pg.ch * dx0 + pg.sh * dy0;  // t of the tile's pixel (0,0)
        const double tmin = base + fmin(0.0, pg.ch * (EX - 1)) + fmin(0.0, pg.sh * (EY - 1));
        double o = floor(tmin) - 1.0;                           // one bin of slack for FP32 rounding
        o = fmax(o, -(double)zpad);
        o = fmin(o, (double)(B + zpad - W));
        const float cf = (float)(PASS ? pg.sh : pg.ch), dl = (float)(PASS ? pg.ch : pg.sh);
        // runs that would leave the window (only possible where the window is clamped onto the
        // zero pads, i.e. where every tap is zero) are moved inside it
        geo[st * R8_NA + pl] =
            make_float4(cf, dl, (float)(base - o), (float)(W - 3) - (float)(R8_RN - 1) * dl);
        const int64_t src = (int64_t)pg.p * row_f4 + (int64_t)o + zpad;
        float4* dst = buf + (size_t)(st * R8_NA + pl) * 2 * WS;
        mbar_arrive_expect_tx(bar, 2 * win_bytes);
        bulk_g2s(dst, qA + src, win_bytes, bar);
        bulk_g2s(dst + WS, qB + src, win_bytes, bar);
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

  // ---------------- consumers
  const int fl = tid & (R8_LANES - 1);       // position along the fast axis of the class
  const int rn = (tid >> 6) * R8_RN;         // first pixel of the run along the slow axis
  const float ffl = (float)fl, frn = (float)rn;
  const uint32_t wb = smem_u32(buf);

  float acc[R8_RN][8];
#pragma unroll
  for (int n = 0; n < R8_RN; ++n)
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[n][j] = 0.f;

  for (int c = 0; c < n_chunks; ++c) {
    // the producer role rotates over the warps, so that no warp is the slowest one
    if ((tid >> 5) == ((c + (NS - 2)) & 7) && c + (NS - 2) < n_chunks) produce(c + (NS - 2));
    const int st = c % NS;
    mbar_wait(&full[st], (uint32_t)((c / NS) & 1));
    const int na = min(R8_NA, ne - c * R8_NA);
    const float4* gch = geo + st * R8_NA;
    const uint32_t sb = wb + (uint32_t)(st * R8_NA) * (2u * WS * 16u);
#pragma unroll 4
    for (int a = 0; a < na; ++a) {
      const float4 gg = gch[a];
      float t = fmaf(ffl, gg.x, fmaf(frn, gg.y, gg.z));
      t = fminf(fmaxf(t, 0.f), gg.w);
      const float tm = __fadd_rd(t, 8388608.f);
      const int k = __float_as_int(tm) - 0x4b000000;
      const float f0 = t - (tm - 8388608.f);
      const uint32_t addr = sb + (uint32_t)a * (2u * WS * 16u) + (uint32_t)k * 16u;
      if (PACKED) r8_run_packed<WS * 16>(acc, addr, f0, gg.y);
      else r8_run<WS * 16>(acc, addr, f0, gg.y);
    }
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(&empty[st]);
  }

  // ---------------- write the tile: acc[n][0..1] = slices of group gA, acc[n][2..3] = group gA + 1
  if (PASS == 0) {  // pixel (x0 + fl, y0 + rn + n): lanes along x, coalesced
    const int x = x0 + fl;
    if (x < nx) {
#pragma unroll
      for (int n = 0; n < R8_RN; ++n) {
        const int y = y0 + rn + n;
        if (y >= ny) continue;
        float v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = acc[n][j];
#pragma unroll
        for (int sl = 0; sl < 8; ++sl) {
          const int s = gA * 4 + sl;
          if (s < S) {
            float* dst = img + ((int64_t)s * ny + y) * nx + x;
            *dst = add ? fmaf(scale, v[sl], *dst) : scale * v[sl];
          }
        }
      }
    }
  } else {
    // pixel (x0 + rn + n, y0 + fl): lanes run along y, so the tile goes through shared memory (the
    // window ring is free: every chunk has been consumed) and is written / added row by row
    constexpr int TP = R8_SLOW + 1;                      // padded row of the transposed tile
    float* ts = reinterpret_cast<float*>(buf);           // [8 slices][64 rows][TP]
    __syncthreads();
#pragma unroll
    for (int n = 0; n < R8_RN; ++n)
#pragma unroll
      for (int sl = 0; sl < 8; ++sl) ts[(sl * R8_LANES + fl) * TP + rn + n] = acc[n][sl];
    __syncthreads();
    const bool vec_ok = (nx % 4 == 0) && ((reinterpret_cast<uintptr_t>(img) & 15) == 0);
#pragma unroll 1
    for (int sl = 0; sl < 8; ++sl) {
      const int s = gA * 4 + sl;
      if (s >= S) break;
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const int e = tid + R8_NC * q;
        const int yl = e >> 3, xl = (e & 7) * 4;
        const int y = y0 + yl, x = x0 + xl;
        if (y >= ny || x >= nx) continue;
        const float* t4 = ts + (sl * R8_LANES + yl) * TP + xl;
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
}

// window (bins) a 64 x 32 tile touches: span <= h sqrt(63^2 + 31^2), + floor, second tap, slack
int backproject_run8_window(double pixel_size) {
  if (!(pixel_size * 0.70710678118654757 < 0.999)) return 0;  // run step must stay below one bin
  const double span = pixel_size * sqrt((double)((R8_LANES - 1) * (R8_LANES - 1) +
                                                 (R8_SLOW - 1) * (R8_SLOW - 1)));
  const double w = ceil(span) + 5.0;
  if (w > 112.0) return 0;
  return ((int)w + 3) & ~3;
}

namespace {

template <int WS, int NS, bool PACKED>
int launch_run8(const float4* d_qi, const QiLayout& L, const BpArgs& a, const RunProj* d_run,
                int32_t n_a, int32_t n_b, int W, cudaStream_t stream) {
  const size_t smem = R8_HDR + (size_t)NS * R8_NA * 2 * WS * 16;
  static DeviceMask configured{0};   // one bit per device (cudaFuncSetAttribute is per device)
  if (first_use_on_device(&configured)) {
    PYHST_CUDA_TRY(cudaFuncSetAttribute(bp_run8_kernel<0, WS, NS, PACKED>,
                                        cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    PYHST_CUDA_TRY(cudaFuncSetAttribute(bp_run8_kernel<1, WS, NS, PACKED>,
                                        cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  }
  const unsigned gz = (unsigned)((L.n_groups + 1) / 2);
  dim3 grid_a((a.nx + R8_LANES - 1) / R8_LANES, (a.ny + R8_SLOW - 1) / R8_SLOW, gz);
  dim3 grid_b((a.nx + R8_SLOW - 1) / R8_SLOW, (a.ny + R8_LANES - 1) / R8_LANES, gz);
  if (grid_a.y > 65535 || grid_b.y > 65535 || gz > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "run8 backprojector: grid too large");
  StageScope scope(ST_BACKPROJECT, stream);
  if (n_a > 0 || n_b == 0) {  // n_a == n_b == 0 cannot happen (n_angles > 0)
    scope.kernels();
    bp_run8_kernel<0, WS, NS, PACKED><<<grid_a, R8_NT, smem, stream>>>(
        d_qi, L.row_f4(), L.zpad, a.d_img, a.n_slices, L.n_groups, L.n_angles, a.n_bins, a.nx, a.ny,
        a.scale, d_run, 0, n_a, 0, W);
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  if (n_b > 0) {
    scope.kernels();
    bp_run8_kernel<1, WS, NS, PACKED><<<grid_b, R8_NT, smem, stream>>>(
        d_qi, L.row_f4(), L.zpad, a.d_img, a.n_slices, L.n_groups, L.n_angles, a.n_bins, a.nx, a.ny,
        a.scale, d_run, n_a, n_b, n_a > 0 ? 1 : 0, W);
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  return PYHST_OK;
}

}  // namespace

int launch_backproject_run8(const float4* d_qi, const QiLayout& L, const BpArgs& a,
                            const RunProj* d_run, int32_t n_a, int32_t n_b, cudaStream_t stream) {
  const int W = backproject_run8_window(a.pixel_size);
  if (W == 0 || W > L.n_bins + 2 * L.zpad || L.zpad < W + 2)
    return set_error(PYHST_ERR_UNSUPPORTED, "run8 backprojector: window %d does not fit", W);
  // variant 7: 16 slices per thread where the stack has >= 13 slices (backproject_run16.cu) -- measured slower
  // (config 2: 19.2 vs 17.9 ms: 11 % fewer instructions, but one run in flight per thread instead of four leaves
  // the LDS -> FFMA latency exposed: issue slots 71 % instead of 86 %), so not the default
  if (bp_variant() == 7 && backproject_run16_covers(a.pixel_size, L.n_groups))
    return launch_backproject_run16(d_qi, L, a, d_run, n_a, n_b, stream);
  // two instantiations: slots of 80 bins, 4 stages (pixel size <= 1.03), or 112 bins, 3 stages
  const bool packed = run8_packed();
  if (W <= 80)
    return packed ? launch_run8<80, 4, true>(d_qi, L, a, d_run, n_a, n_b, W, stream)
                  : launch_run8<80, 4, false>(d_qi, L, a, d_run, n_a, n_b, W, stream);
  return packed ? launch_run8<112, 3, true>(d_qi, L, a, d_run, n_a, n_b, W, stream)
                : launch_run8<112, 3, false>(d_qi, L, a, d_run, n_a, n_b, W, stream);
}

}  // namespace pyhst
