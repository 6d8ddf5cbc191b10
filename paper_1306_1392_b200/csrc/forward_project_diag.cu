// Forward projection P = (P^T)^T, the product kernel (include/pyhst.h a3; PAPER.md:L65, L71-L73
// eq. 1, L211 Alg. 1 "Fp"; readings R6, R11, R13 of DESIGN.md):
//
//   y[s,p,b] = scale * sum_{i,j} Lambda(t_p(i,j) - b) x[s,i,j],   Lambda(u) = max(0, 1 - |u|)
//
// fp_diag_kernel: interval form of the gather on DIAGONAL image lines.
//
//   * Interval form: a thread owns unit intervals [m, m+1) of the detector axis.  A pixel whose
//     coordinate t falls into the interval is loaded once from shared memory and used twice, with
//     weight f = t - m for bin m+1 and 1 - f for bin m.  No atomics; each bin is the sum of the
//     upper share of the interval below it and the lower share of the interval above it.
//   * Diagonal lines: along a line of pixels (j + k, i +- k) the coordinate t moves by
//     |sigma| = h (|cos| + |sin|) >= 1 bin per pixel, so an interval holds AT MOST ONE pixel of a
//     line -- one candidate, one predicate, no second-candidate logic (on image rows or columns
//     the step is h max(|cos|, |sin|) <= 1: up to two pixels per interval and line, and half of
//     the executed FMAs carry weight zero).  The image is stored sheared (XD, below), so that a
//     diagonal is a contiguous run of float4 (4 slices) and a band of diagonals is staged by TMA
//     bulk copies like the rows of the banded kernel.
//   * A thread owns FD_M = 2 neighbouring intervals of one projection and 4 NG slices: three
//     boundaries serve two intervals, the middle bin has one accumulator.
//   * Which pixel belongs to which interval is decided identically by the two threads that share
//     a boundary: both evaluate the SAME expression for it -- ks(m, w) = K0 + m inv + sD w in
//     double per (boundary, band), split into an integer and a float fraction, then
//     fmaf(s, r, fraction) per line and a round-up add of 1.5 * 2^23 + integer -- so the sets
//     [ceil(ks(m)), ceil(ks(m+1))) partition the line whatever the rounding.  With
//     |sigma| >= 1 + 2^-12 such a set has at most one element.  Projections on or next to an image
//     axis (1 - 1e-6 <= |sigma| < 1 + 2^-12 at pixel size 1: theta = 0, pi/2 of every scan) may
//     get two: they form chunks of their own, run by the TWO form of the kernel, which also takes
//     the next pixel of the line when the computed boundaries enclose it.  Pixel sizes with
//     |sigma| < 1 - 1e-6 go to the banded kernel (forward_project.cu).
//   * The weight f = |sigma| (ceil(ks) - ks) uses the continuous position (R11: double per band,
//     FP32 only for the in-band offset).
#include <algorithm>
#include <cmath>
#include <cstring>

#include "common.h"

namespace pyhst {

namespace {

#ifndef FD_PACKED
#define FD_PACKED 0
#endif
#ifndef FD_NG4
#define FD_NG4 1
#endif
#ifndef FD_CHECK
#define FD_CHECK 0
#endif
// block order: chunk index fastest (1) -- the blocks resident together are the same detector range at neighbouring
// angles, whose staged bands overlap: L2 hit rate 29 % -> 74 %, DRAM reads 42 -> 10.6 GB per config-2 call -- or
// detector block fastest (0)
#ifndef FD_M1
#define FD_M1 0
#endif
// intervals per thread of the 8-slice dense form (NG = 2, 16 projections per block): 4 -- five boundaries serve four
// intervals and the per-band set-up is shared by twice the work (256-thread blocks, two per SM): config 2 run on this
// form 24.3 -> 23.3 ms, the 8-slice chunks of pyhst_forward_project_host 29.6 -> 28.6 ms
#ifndef FD_M2
#define FD_M2 4
#endif
#ifndef FD_SWAP
#define FD_SWAP 1
#endif
constexpr int FD_NB = 64;      // intervals per block (FD_NB - 1 complete bins)
constexpr int FD_NPJ = 16;     // projections per block (at most)
constexpr int FD_M = 2;        // neighbouring intervals per thread
constexpr int FD_NT = FD_NB / FD_M * FD_NPJ;   // 512 threads, one (interval pair, projection) each
constexpr int FD_RB = 8;       // lines per band
#ifndef FD_UNR_
#define FD_UNR_ 4
#endif
constexpr int FD_UNR = FD_UNR_;   // lines unrolled together (register budget)
constexpr int FD_SB = 4;       // bands per double-precision evaluation of the boundaries
constexpr int FD_LP = 4;       // projections per warp (lanes of a warp = FD_PPW interval pairs x FD_LP projections)
constexpr int FD_PPW = 32 / FD_LP;
constexpr int FD_NSTG = 4;     // stages of the band ring
constexpr int FD_WMAX = 100;   // window capacity (float4 per line): four stages of two blocks per SM fit in 227 KB
constexpr int FD_PW = FD_WMAX + FD_RB;   // row pitch of a stage (float4): room for the per-line skew
constexpr int FD_HDR = 1024;   // mbarriers, origins, FdProj table
constexpr float FD_MAGIC = 12582912.f;   // 1.5 * 2^23

// smem bytes of one launch
constexpr int fd_hdr(int npj) { return npj == 8 ? 512 : FD_HDR; }   // 128 B of barriers / origins + npj x 40 B
constexpr size_t fd_smem(int ng, int rb, int npj) { return fd_hdr(npj) + (size_t)FD_NSTG * rb * ng * FD_PW * 16; }

struct FdParams {
  const float4* xd[2];     // sheared image, layout 0 (diagonals i - j) and 1 (anti-diagonals i + j)
  int64_t line_f4;         // float4 per stored line (nx + 2 zpad)
  int64_t group_f4;        // float4 per slice group (line_f4 * stored lines)
  int32_t zpad;
  float* sino;
  int64_t pitch;
  int32_t S, P, B;
  float scale;
  const FdProj* projs;
  const FdChunk* chunks;
  const int2* ranges;      // [n_chunks][n_bx]: lines [x, y) the block walks
  int32_t n_bx, W;
  // n_seg > 1: blockIdx.z = group block * n_seg + seg; the block walks the seg-th part of its bands and writes its
  // sums to part[seg] (same row layout, pitch part_pitch); fd_combine_kernel adds the parts (small scans fill the GPU)
  int32_t n_seg;
  int32_t chunk_off;       // first chunk of this launch
  int32_t g_off;           // first slice group of this launch (a stack is covered by launches of 4, 2 and 1 groups per block)
  float* part;             // [n_seg][S][part_nt][part_pitch]: rows of the pass's projections only
  int64_t part_pitch, part_stride;
  int32_t part_t0, part_nt;   // the pass's range of the projection table
};

// One line of one interval, NG slice groups: two LDS.128 and 4 NG packed FFMA2 (two slices each).  The
// accumulators are kept as 64-bit register pairs.  f / g are the weights of the pixel ceil(ks_lo) for
// bins m + 1 / m, already zeroed when the interval does not hold that pixel (packed instructions cannot
// be predicated).  An FFMA2 occupies both 16-lane FMA pipes and the dispatch port for two cycles: nothing
// issues in its shadow, so the packed form costs what two scalar FFMAs cost (profiles/r03_micro.md).
template <int NG, int PLANE>
__device__ __forceinline__ void fd_line(uint64_t* al, uint64_t* au, float f, float g, uint32_t addr) {
  if constexpr (NG >= 2) {
    asm volatile("{\n\t"
        ".reg .b64 v<4>, wf, wg;\n\t"
        "ld.shared.v2.b64 {v0, v1}, [%10];\n\t"
        "ld.shared.v2.b64 {v2, v3}, [%10+%11];\n\t"
        "mov.b64 wf, {%8, %8};\n\t"
        "mov.b64 wg, {%9, %9};\n\t"
        "fma.rn.f32x2 %0, v0, wg, %0;\n\t"
        "fma.rn.f32x2 %1, v1, wg, %1;\n\t"
        "fma.rn.f32x2 %4, v0, wf, %4;\n\t"
        "fma.rn.f32x2 %5, v1, wf, %5;\n\t"
        "fma.rn.f32x2 %2, v2, wg, %2;\n\t"
        "fma.rn.f32x2 %3, v3, wg, %3;\n\t"
        "fma.rn.f32x2 %6, v2, wf, %6;\n\t"
        "fma.rn.f32x2 %7, v3, wf, %7;\n\t"
        "}"
        : "+l"(al[0]), "+l"(al[1]), "+l"(al[2]), "+l"(al[3]), "+l"(au[0]), "+l"(au[1]), "+l"(au[2]), "+l"(au[3])
        : "f"(f), "f"(g), "r"(addr), "n"(PLANE));
  } else {
    asm volatile("{\n\t"
        ".reg .b64 v<2>, wf, wg;\n\t"
        "ld.shared.v2.b64 {v0, v1}, [%6];\n\t"
        "mov.b64 wf, {%4, %4};\n\t"
        "mov.b64 wg, {%5, %5};\n\t"
        "fma.rn.f32x2 %0, v0, wg, %0;\n\t"
        "fma.rn.f32x2 %1, v1, wg, %1;\n\t"
        "fma.rn.f32x2 %2, v0, wf, %2;\n\t"
        "fma.rn.f32x2 %3, v1, wf, %3;\n\t"
        "}"
        : "+l"(al[0]), "+l"(al[1]), "+l"(au[0]), "+l"(au[1])
        : "f"(f), "f"(g), "r"(addr));
  }
}

#if !FD_PACKED
__device__ __forceinline__ void fd_line_s1(float (&al)[4], float (&au)[4], float f, float g, uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  al[0] = fmaf(g, v.x, al[0]); al[1] = fmaf(g, v.y, al[1]); al[2] = fmaf(g, v.z, al[2]); al[3] = fmaf(g, v.w, al[3]);
  au[0] = fmaf(f, v.x, au[0]); au[1] = fmaf(f, v.y, au[1]); au[2] = fmaf(f, v.z, au[2]); au[3] = fmaf(f, v.w, au[3]);
}
// scalar form: predicated FFMA on float accumulators (one issue slot each; the kernel is then bound by
// issue slots instead of the FMA pipe -- measured within 2 % of the packed form)
template <int PLANE>
__device__ __forceinline__ void fd_line_s(float* al, float* au, float jlo, float jhi, float f, float g,
                                          uint32_t addr) {
  asm volatile("{\n\t"
      ".reg .pred p;\n\t"
      ".reg .f32 v<8>;\n\t"
      "setp.lt.f32 p, %16, %17;\n\t"
      "ld.shared.v4.f32 {v0, v1, v2, v3}, [%20];\n\t"
      "ld.shared.v4.f32 {v4, v5, v6, v7}, [%20+%21];\n\t"
      "@p fma.rn.f32 %0, %19, v0, %0;\n\t"
      "@p fma.rn.f32 %1, %19, v1, %1;\n\t"
      "@p fma.rn.f32 %2, %19, v2, %2;\n\t"
      "@p fma.rn.f32 %3, %19, v3, %3;\n\t"
      "@p fma.rn.f32 %8, %18, v0, %8;\n\t"
      "@p fma.rn.f32 %9, %18, v1, %9;\n\t"
      "@p fma.rn.f32 %10, %18, v2, %10;\n\t"
      "@p fma.rn.f32 %11, %18, v3, %11;\n\t"
      "@p fma.rn.f32 %4, %19, v4, %4;\n\t"
      "@p fma.rn.f32 %5, %19, v5, %5;\n\t"
      "@p fma.rn.f32 %6, %19, v6, %6;\n\t"
      "@p fma.rn.f32 %7, %19, v7, %7;\n\t"
      "@p fma.rn.f32 %12, %18, v4, %12;\n\t"
      "@p fma.rn.f32 %13, %18, v5, %13;\n\t"
      "@p fma.rn.f32 %14, %18, v6, %14;\n\t"
      "@p fma.rn.f32 %15, %18, v7, %15;\n\t"
      "}"
      : "+f"(al[0]), "+f"(al[1]), "+f"(al[2]), "+f"(al[3]), "+f"(al[4]), "+f"(al[5]), "+f"(al[6]), "+f"(al[7]),
        "+f"(au[0]), "+f"(au[1]), "+f"(au[2]), "+f"(au[3]), "+f"(au[4]), "+f"(au[5]), "+f"(au[6]), "+f"(au[7])
      : "f"(jlo), "f"(jhi), "f"(f), "f"(g), "r"(addr), "n"(PLANE));
}
#endif

__device__ __forceinline__ float fd_lo(uint64_t v) { return __uint_as_float((uint32_t)v); }
__device__ __forceinline__ float fd_hi(uint64_t v) { return __uint_as_float((uint32_t)(v >> 32)); }

// NPJ = projections per block (16: dense angle lists; 8: sparse ones, whose strips fan out so that fewer fit one staged
// window -- 256-thread blocks with bands of RB = 4 lines, four blocks per SM), NT = 32 NPJ threads.
// TWO: chunks of projections with 1 - 1e-6 <= |sigma| < 1 + 2^-12 (on or next to an image axis at pixel size 1): the
// computed boundaries of an interval may then enclose two pixels of a line, and the second one is taken as well.
// M = neighbouring intervals per thread (2; 1 is a measured alternative for NG = 4: 1024 threads per block).
template <int NG, int NPJ, int RB, bool TWO, int M>
__global__ void __launch_bounds__(FD_NB / M * NPJ, NG == 4 ? 1 : (NPJ == 16 ? 2 : 4)) fp_diag_kernel(const FdParams prm) {
  constexpr int NT = FD_NB / M * NPJ, NWARP = NT / 32, PLANE = RB * FD_PW * 16;
  constexpr int WPG = FD_NB / M / FD_PPW;   // warps that share a group of FD_LP projections
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);              // [NSTG]
  uint64_t* empty = reinterpret_cast<uint64_t*>(smem + 32);        // [NSTG]
  int* sorigin = reinterpret_cast<int*>(smem + 64);                // [NSTG]
  FdProj* sproj = reinterpret_cast<FdProj*>(smem + 128);           // [NPJ] x 48 B
  float4* buf = reinterpret_cast<float4*>(smem + (NPJ == 8 ? 512 : FD_HDR));          // [NSTG][NG][RB][PW]
  constexpr int STAGE_F4 = NG * RB * FD_PW;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
#if FD_SWAP
  const int bxi = blockIdx.y, cki = blockIdx.x;
#else
  const int bxi = blockIdx.x, cki = blockIdx.y;
#endif
  const int chunk = prm.chunk_off + cki;
  const FdChunk ck = prm.chunks[chunk];
  const int seg = blockIdx.z % prm.n_seg;
  const int gA = prm.g_off + (blockIdx.z / prm.n_seg) * NG;
  const int mB = bxi * (FD_NB - 1) - 1;      // intervals [m, m+1), m in [mB, mB + NB)
  int2 rg = prm.ranges[(int64_t)chunk * prm.n_bx + bxi];
  if (prm.n_seg > 1) {
    const int nb_all = (rg.y - rg.x + RB - 1) / RB;
    const int k0 = seg * nb_all / prm.n_seg, k1 = (seg + 1) * nb_all / prm.n_seg;
    rg.y = min(rg.y, rg.x + k1 * RB);
    rg.x = rg.x + k0 * RB;
    if (rg.y < rg.x) rg.y = rg.x;
  }
  const int n_bands = (rg.y - rg.x + RB - 1) / RB;
  const int W = prm.W;
  const uint32_t row_bytes = (uint32_t)W * 16u;
  const float4* xd = (ck.layout ? prm.xd[1] : prm.xd[0]) + (int64_t)gA * prm.group_f4;
  const int sgn = ck.sgn, skew = ck.skew;
  const int bias = skew < 0 ? RB - 1 : 0;

  if (tid < ck.count) sproj[tid] = prm.projs[ck.first + tid];
  if (tid == 0) {
#pragma unroll
    for (int q = 0; q < FD_NSTG; ++q) {
      mbar_init(&full[q], RB);
      mbar_init(&empty[q], NT / 32);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // one warp (the role rotates): waits until the stage of band k - NSTG has been read by every
  // warp, computes the window origin of band k in double (the lowest stored position, over the
  // chunk's projections, of the block's outer boundaries on the band's first and last line, the
  // per-line skew taken off), then issues one bulk copy per line and slice group.  Line r of the
  // band is staged from stored position origin + skew * r.
  auto produce = [&](int k) {
    const int st = k % FD_NSTG;
    if (k >= FD_NSTG) mbar_wait(&empty[st], (uint32_t)(((k / FD_NSTG) - 1) & 1));
    const int w0 = rg.x + k * RB;
    double lo = 1e300;
    if (lane < ck.count) {
      const FdProj pj = sproj[lane];
      // stored position of t = m on line w: sgn * ks(m, w); the block's pixels lie between the two
      // outer boundaries
      const double e0 = fma((double)mB, pj.inv, pj.K0), e1 = fma((double)(mB + FD_NB), pj.inv, pj.K0);
      const double ea = sgn > 0 ? e0 : -e1;                      // lowest stored position on line 0
      const double da = (double)sgn * pj.sD;                     // its change per line
      const double a0 = fma(da, (double)w0, ea);
      const double a1 = fma(da, (double)(w0 + RB - 1), ea) - (double)(skew * (RB - 1));
      lo = fmin(a0, a1);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    const int origin = (int)floor(lo) - 2;
    uint64_t* bar = &full[st];
    if (lane == 0) sorigin[st] = origin;
    if (lane < RB) {
      mbar_arrive_expect_tx(bar, NG * row_bytes);
      const float4* src = xd + (int64_t)(w0 + lane) * prm.line_f4 + (prm.zpad + origin + skew * lane);
      float4* dst = buf + st * STAGE_F4 + lane * FD_PW + bias + skew * lane;
#pragma unroll
      for (int q = 0; q < NG; ++q) bulk_g2s(dst + q * RB * FD_PW, src + q * prm.group_f4, row_bytes, bar);
    }
  };

  if (warp == 0 && n_bands > 0) produce(0);
  if (warp == 1 && n_bands > 1) produce(1);
  if (warp == 2 && n_bands > 2) produce(2);

  // bins mB + 2 jp + {0, 1, 2}: lower share of the first interval, both shares of the middle bin,
  // upper share of the second interval
#if FD_PACKED
  uint64_t acc[M + 1][2 * NG];       // pairs of slices
#pragma unroll
  for (int q = 0; q <= M; ++q)
#pragma unroll
    for (int sl = 0; sl < 2 * NG; ++sl) acc[q][sl] = 0ull;
#else
  float acc[M + 1][4 * NG];
#pragma unroll
  for (int q = 0; q <= M; ++q)
#pragma unroll
    for (int sl = 0; sl < 4 * NG; ++sl) acc[q][sl] = 0.f;
#endif

  // a warp = 8 interval pairs x 4 projections: its 32 pixels of a line lie within ~16 stored
  // positions, i.e. the LDS.128 touches <= 256 B (2.4 cycles instead of 4, profiles/r02_micro.md)
  const int jp = (warp % WPG) * FD_PPW + lane / FD_LP;
  const int pj = (warp / WPG) * FD_LP + lane % FD_LP;
  const bool active = pj < ck.count;
  const int m0 = mB + M * jp;
  const float s = active ? sproj[pj].s : 0.f;
  const float sig = active ? sproj[pj].sig : 1.f;
  const int mul = ck.mul16;                    // sgn * 16 (from the table: one IMAD per address)

  float afr[M + 1], mg[M + 1];
#pragma unroll
  for (int q = 0; q <= M; ++q) afr[q] = mg[q] = 0.f;
  const uint32_t buf_u32 = smem_u32(buf);
  const uint32_t magic_off = (uint32_t)mul * 0x4b400000u;

  for (int k = 0; k < n_bands; ++k) {
    const int st = k % FD_NSTG;
    mbar_wait(&full[st], (uint32_t)((k / FD_NSTG) & 1));
    if (active) {
      const int origin = sorigin[st];
      if ((k % FD_SB) == 0) {
        // every FD_SB bands: the boundaries' positions on the band's first line (double), split into an
        // integer and a fraction; the thread that shares a boundary evaluates the identical expression
        const double w0 = (double)(rg.x + k * RB);
        const FdProj* sp = &sproj[pj];
        const double K0 = sp->K0, inv = sp->inv, sD = sp->sD;
#pragma unroll
        for (int q = 0; q <= M; ++q) {
          const double ks = fma(sD, w0, fma((double)(m0 + q), inv, K0));
          const double ai = rint(ks);
          afr[q] = (float)(ks - ai);
          mg[q] = (float)ai + FD_MAGIC;     // exact: |ai| < 2^22
        }
      }
      // byte address of stored position k = sgn * kappa on line 0:  (bias + k - origin) * 16, with
      // kappa = float_as_int(jm) - 0x4b400000
      const uint32_t cbase = buf_u32 + (uint32_t)(st * STAGE_F4 * 16) + (uint32_t)((bias - origin) * 16) - magic_off;
#pragma unroll 1
      for (int r0 = 0; r0 < RB; r0 += FD_UNR) {
        const uint32_t cb = cbase + (uint32_t)(r0 * FD_PW * 16);
        {
#pragma unroll
        for (int r = 0; r < FD_UNR; ++r) {
          float ksf[M + 1], jm[M + 1];
#pragma unroll
          for (int q = 0; q <= M; ++q) {
            ksf[q] = fmaf(s, (float)r, afr[q]);
            jm[q] = __fadd_ru(ksf[q], mg[q]);      // ceil(ks) + magic, integer part in the mantissa
          }
#pragma unroll
          for (int q = 0; q < M; ++q) {
            const float f = sig * ((jm[q] - mg[q]) - ksf[q]);   // t - m of the pixel ceil(ks), in [0, sigma)
            const float g = 1.f - f;
            const bool in = jm[q] < jm[q + 1];                  // the interval holds that pixel
            uint32_t addr;
            asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(addr) : "r"(__float_as_int(jm[q])), "r"(mul), "r"(cb + r * FD_PW * 16));
#if FD_CHECK
            // debug build (-DFD_CHECK=1): a claimed pixel must lie inside the window staged for its line
            {
              const int col = (int)(addr - (buf_u32 + (uint32_t)(st * STAGE_F4 * 16) + (uint32_t)((r0 + r) * FD_PW * 16))) / 16;
              const int lo = bias + skew * (r0 + r);
              if (in && (col < lo || col >= lo + W)) __trap();
            }
#endif
#if FD_PACKED
            const float fz = in ? f : 0.f, gz = in ? g : 0.f;
            fd_line<NG, PLANE>(acc[q], acc[q + 1], fz, gz, addr);
            if constexpr (NG == 4) fd_line<NG, PLANE>(acc[q] + 4, acc[q + 1] + 4, fz, gz, addr + 2 * PLANE);
#else
            if constexpr (NG >= 2) {
              fd_line_s<PLANE>(acc[q], acc[q + 1], jm[q], jm[q + 1], f, g, addr);
              if constexpr (NG == 4) fd_line_s<PLANE>(acc[q] + 8, acc[q + 1] + 8, jm[q], jm[q + 1], f, g, addr + 2 * PLANE);
            } else {
              fd_line_s1(acc[q], acc[q + 1], in ? f : 0.f, in ? g : 0.f, addr);
            }
#endif
            if constexpr (TWO) {   // the next pixel of the line, if the interval's computed boundaries enclose it too
              const float j2 = jm[q] + 1.f, f2 = f + sig, g2 = 1.f - f2;
              const uint32_t addr2 = addr + (uint32_t)mul;
#if FD_PACKED
              const bool in2 = j2 < jm[q + 1];
              const float fz2 = in2 ? f2 : 0.f, gz2 = in2 ? g2 : 0.f;
              fd_line<NG, PLANE>(acc[q], acc[q + 1], fz2, gz2, addr2);
              if constexpr (NG == 4) fd_line<NG, PLANE>(acc[q] + 4, acc[q + 1] + 4, fz2, gz2, addr2 + 2 * PLANE);
#else
              if constexpr (NG >= 2) {
                fd_line_s<PLANE>(acc[q], acc[q + 1], j2, jm[q + 1], f2, g2, addr2);
                if constexpr (NG == 4) fd_line_s<PLANE>(acc[q] + 8, acc[q + 1] + 8, j2, jm[q + 1], f2, g2, addr2 + 2 * PLANE);
              } else {
                const bool in2 = j2 < jm[q + 1];
                fd_line_s1(acc[q], acc[q + 1], in2 ? f2 : 0.f, in2 ? g2 : 0.f, addr2);
              }
#endif
            }
          }
        }
        }
        // the fractions move on by FD_UNR lines (the same FP32 operation in both threads that share a
        // boundary; re-based in double every FD_SB bands)
#pragma unroll
        for (int q = 0; q <= M; ++q) afr[q] = fmaf(s, (float)FD_UNR, afr[q]);
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[st]);
    // the producer role rotates; a warp produces AFTER its own share of band k, into the stage of band
    // k - 1, which the other warps have normally left by then: it does not become the straggler
    if (k + FD_NSTG - 1 < n_bands && warp == (k % NWARP)) produce(k + FD_NSTG - 1);
  }

  // ---- combine the shares through shared memory (the stages are free now) and store -------------
  __syncthreads();
  float* out = prm.n_seg > 1 ? prm.part + (int64_t)seg * prm.part_stride : prm.sino;
  const int64_t opitch = prm.n_seg > 1 ? prm.part_pitch : prm.pitch;
  float* lo_s = reinterpret_cast<float*>(buf);                 // [NPJ][NB + 1] lower shares (and complete middle bins)
  float* up_s = lo_s + NPJ * (FD_NB + 1);                   // [NPJ][NB + 1] upper shares
#pragma unroll
  for (int sl = 0; sl < 4 * NG; ++sl) {
    const int sidx = gA * 4 + sl;
    if (sidx >= prm.S) break;       // uniform
    // local bin index = bin - mB in [0, NB]: bins M jp + q, q < M, hold this thread's complete or lower share, bin
    // M jp + M the upper share of its last interval
#pragma unroll
    for (int q = 0; q <= M; ++q) {
#if FD_PACKED
      const float aq = (sl & 1) ? fd_hi(acc[q][sl >> 1]) : fd_lo(acc[q][sl >> 1]);
#else
      const float aq = acc[q][sl];
#endif
      if (q < M) lo_s[pj * (FD_NB + 1) + M * jp + q] = aq;
      else up_s[pj * (FD_NB + 1) + M * jp + M] = aq;
      if (q > 0 && q < M) up_s[pj * (FD_NB + 1) + M * jp + q] = 0.f;
    }
    __syncthreads();
    // complete bins: local 1 .. NB - 1
    for (int e = tid; e < NPJ * (FD_NB - 1); e += NT) {
      const int q = e / (FD_NB - 1), bl = 1 + e - q * (FD_NB - 1);
      const int b = mB + bl;
      if (q < ck.count && b < prm.B) {
        const int p = sproj[q].p;
        const int64_t orow = prm.n_seg > 1 ? (int64_t)sidx * prm.part_nt + (ck.first + q - prm.part_t0)
                                           : (int64_t)sidx * prm.P + p;
        out[orow * opitch + b] =
            prm.scale * (lo_s[q * (FD_NB + 1) + bl] + up_s[q * (FD_NB + 1) + bl]);
      }
    }
    __syncthreads();
  }
}

// y[s][p][b] = sum_seg part[seg][s][p][b] for the projections of the table (fixed order: deterministic)
__global__ void fd_combine_kernel(float* __restrict__ y, int64_t pitch, const float* __restrict__ part, int64_t part_pitch,
                                  int64_t part_stride, int n_seg, int B, int P, const FdProj* __restrict__ projs, int n_tab,
                                  int64_t n_rows_tab) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t rt = blockIdx.y + (int64_t)blockIdx.z * gridDim.y;
  if (b >= B || rt >= n_rows_tab) return;
  const int64_t sl = rt / n_tab;
  const int64_t row = sl * P + projs[rt - sl * n_tab].p;
  float v = 0.f;
  for (int h = 0; h < n_seg; ++h) v += part[(int64_t)h * part_stride + rt * part_pitch + b];
  y[row * pitch + b] = v;
}

// ---- [S][ny][nx] -> XD, both shears ---------------------------------------------------------------
// XD[layout][g][w][zpad + k]: one float4 (4 slices of group g) per stored position; line w of layout 0
// holds the pixels (j = k, i = w - (nx - 1) + k), of layout 1 the pixels (j = k, i = w - k).  Positions
// that are no pixel (the triangles beside the image, the pads, the spare lines and groups) are zero:
// they are written once per workspace block and never touched by the repack.
__global__ void __launch_bounds__(256) repack_diag_kernel(const float* __restrict__ img, int S, int ny, int nx,
                                                          float4* __restrict__ xd0, float4* __restrict__ xd1,
                                                          int64_t line_f4, int64_t group_f4, int zpad) {
  __shared__ float tile[4][32][32];
  const int g = blockIdx.z;
  const int bx = blockIdx.x * 32, by = blockIdx.y * 32;
  const int x = threadIdx.x;
#pragma unroll
  for (int sl = 0; sl < 4; ++sl) {
    const int sidx = g * 4 + sl;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
      const int i = by + r, j = bx + x;
      tile[sl][r][x] = (sidx < S && i < ny && j < nx) ? img[((int64_t)sidx * ny + i) * nx + j] : 0.f;
    }
  }
  __syncthreads();
  const int j = bx + x;
  if (j >= nx) return;
  float4* o0 = xd0 + (int64_t)g * group_f4 + zpad + j;
  float4* o1 = xd1 + (int64_t)g * group_f4 + zpad + j;
  // diagonals of the tile: d = i_local - j_local in [-31, 31]; anti-diagonals a = i_local + j_local in [0, 62]
  for (int d = (int)threadIdx.y - 31; d <= 31; d += blockDim.y) {
    const int il = x + d;
    if (il >= 0 && il < 32 && by + il < ny) {
      const int w = (by + il) - j + (nx - 1);
      o0[(int64_t)w * line_f4] = make_float4(tile[0][il][x], tile[1][il][x], tile[2][il][x], tile[3][il][x]);
    }
  }
  for (int a = threadIdx.y; a <= 62; a += blockDim.y) {
    const int il = a - x;
    if (il >= 0 && il < 32 && by + il < ny) {
      const int w = (by + il) + j;
      o1[(int64_t)w * line_f4] = make_float4(tile[0][il][x], tile[1][il][x], tile[2][il][x], tile[3][il][x]);
    }
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------
// host: classes, chunks, line ranges and the window width (all in double)
// ------------------------------------------------------------------------------------------
namespace {

struct HostProj {
  FdProj d;
  int layout, sgn, skew;
  double a, b, c;      // t = c + a (j - j0) + b (i - i0)
  double angle;
};

// range of stored lines w on which the band  tlo <= t <= thi  of projection q meets the image
// rectangle (widened by one pixel); empty: lo > hi
void line_range(const HostProj& q, int nx, int ny, double tlo, double thi, double* wlo, double* whi) {
  const double j0 = 0.5 * (nx - 1), i0 = 0.5 * (ny - 1);
  const double xl = -1.0, xh = (double)nx, yl = -1.0, yh = (double)ny;   // widened rectangle
  auto tt = [&](double j, double i) { return q.c + q.a * (j - j0) + q.b * (i - i0); };
  auto ww = [&](double j, double i) { return q.layout == 0 ? i - j + (double)(nx - 1) : i + j; };
  double lo = 1e300, hi = -1e300;
  auto take = [&](double j, double i) {
    const double w = ww(j, i);
    lo = std::min(lo, w);
    hi = std::max(hi, w);
  };
  const double cx[4] = {xl, xh, xh, xl}, cy[4] = {yl, yl, yh, yh};
  for (int v = 0; v < 4; ++v) {
    const double t = tt(cx[v], cy[v]);
    if (t >= tlo && t <= thi) take(cx[v], cy[v]);
  }
  for (int e = 0; e < 4; ++e) {
    const double ax = cx[e], ay = cy[e], bx = cx[(e + 1) & 3], by = cy[(e + 1) & 3];
    const double ta = tt(ax, ay), tb = tt(bx, by);
    for (double tv : {tlo, thi}) {
      if ((ta - tv) * (tb - tv) <= 0.0 && ta != tb) {
        const double u = (tv - ta) / (tb - ta);
        take(ax + u * (bx - ax), ay + u * (by - ay));
      }
    }
  }
  *wlo = lo;
  *whi = hi;
}

}  // namespace

bool build_fd_tables(const pyhst_geom_t* g, FdPlan* plan, std::vector<FdProj>* projs, std::vector<FdChunk>* chunks,
                     std::vector<int32_t>* ranges, std::vector<int32_t>* legacy, int npj) {
  if (npj != 8) npj = FD_NPJ;
  plan->npj = npj;
  const int P = g->n_angles, nx = g->nx, ny = g->ny;
  const double h = g->pixel_size;
  const double j0 = 0.5 * (nx - 1), i0 = 0.5 * (ny - 1);
  projs->clear();
  chunks->clear();
  ranges->clear();
  legacy->clear();
  const int n_bx = (g->n_bins + FD_NB - 2) / (FD_NB - 1);
  const int n_lines = nx + ny - 1;
  std::vector<HostProj> cls[24];    // (two, layout, sgn, skew)
  for (int p = 0; p < P; ++p) {
    HostProj q;
    q.a = h * std::cos(g->angles_rad[p]);
    q.b = h * std::sin(g->angles_rad[p]);
    q.c = g->axis_pos[p];
    q.angle = g->angles_rad[p];
    q.layout = (q.a * q.b >= 0.0) ? 0 : 1;
    const double sigma = q.layout == 0 ? q.a + q.b : q.a - q.b;
    const double as = std::fabs(sigma);
    // at most one pixel per interval and line, with room for the rounding of the boundaries; and a
    // window that fits: FD_NB / |sigma| + divergence + skew residue
    // |sigma| >= 1 + 2^-12: at most one pixel per interval and line, with room for the rounding of the boundaries.
    // 1 - 1e-6 <= |sigma| < 1 + 2^-12 (theta on or next to an image axis at pixel size 1): at most two -- chunks of
    // their own, run by the TWO form of the kernel.  Anything finer goes to the banded kernel.
    if (!(as >= 1.0 - 1e-6) || as > 8.0) {
      legacy->push_back(p);
      continue;
    }
    const int two = as < 1.0 + 1.0 / 4096.0 ? 1 : 0;
    const double T0 = q.layout == 0 ? q.c - q.a * j0 - q.b * ((double)(nx - 1) + i0) : q.c - q.a * j0 - q.b * i0;
    q.sgn = sigma > 0.0 ? 1 : -1;
    q.d.inv = 1.0 / as;
    q.d.K0 = -T0 * q.d.inv;
    q.d.sD = -q.b * q.d.inv;
    q.d.s = (float)q.d.sD;
    q.d.sig = (float)as;
    q.d.p = p;
    q.d.pad_ = 0;
    const double dk = (double)q.sgn * q.d.sD;       // stored positions per line
    q.skew = dk > 0.5 ? 1 : (dk < -0.5 ? -1 : 0);
    cls[two * 12 + (q.layout * 2 + (q.sgn > 0 ? 1 : 0)) * 3 + (q.skew + 1)].push_back(q);
  }
  plan->n_bx = n_bx;
  int w_max = 0;
  // width of the window a set of projections needs for block bx on the band starting at line w0
  auto width_at = [&](const std::vector<HostProj>& v, size_t i0_, size_t i1_, int bx, double w0) {
    const int mB = bx * (FD_NB - 1) - 1;
    double lo = 1e300, hi = -1e300;
    for (size_t i = i0_; i < i1_; ++i) {
      const HostProj& q = v[i];
      for (int mm : {mB, mB + FD_NB})
        for (int r : {0, FD_RB - 1}) {
          const double kpos = (double)q.sgn * (q.d.K0 + (double)mm * q.d.inv + q.d.sD * (w0 + r)) - (double)(q.skew * r);
          lo = std::min(lo, kpos);
          hi = std::max(hi, kpos);
        }
    }
    return (int)(std::ceil(hi) - (std::floor(lo) - 2.0)) + 3;
  };
  plan->n_chunks_one = -1;
  for (int c = 0; c < 24; ++c) {
    if (c == 12) {   // chunks of the TWO form follow
      plan->n_chunks_one = (int32_t)chunks->size();
      plan->n_tab_one = (int32_t)projs->size();
    }
    std::vector<HostProj>& v = cls[c];
    if (v.empty()) continue;
    std::stable_sort(v.begin(), v.end(), [](const HostProj& x, const HostProj& y) { return x.angle < y.angle; });
    size_t i = 0;
    while (i < v.size()) {
      // greedy: add neighbours while the window of every block still fits
      size_t j = i + 1;
      std::vector<int32_t> rg_best;
      int w_best = 0;
      auto eval = [&](size_t i1_, std::vector<int32_t>* rg_out, int* w_out) {
        rg_out->assign((size_t)2 * n_bx, 0);
        int wneed = 0;
        for (int bx = 0; bx < n_bx; ++bx) {
          const int mB = bx * (FD_NB - 1) - 1;
          double lo = 1e300, hi = -1e300;
          for (size_t t = i; t < i1_; ++t) {
            double a_, b_;
            line_range(v[t], nx, ny, (double)mB, (double)(mB + FD_NB), &a_, &b_);
            lo = std::min(lo, a_);
            hi = std::max(hi, b_);
          }
          int wl = 0, wh = 0;
          if (lo <= hi) {
            wl = std::max(0, (int)std::floor(lo) - 1);
            wh = std::min(n_lines, (int)std::ceil(hi) + 2);
            if (wh <= wl) wl = wh = 0;
          }
          (*rg_out)[2 * bx] = wl;
          (*rg_out)[2 * bx + 1] = wh;
          if (wh > wl) {
            const int nb = (wh - wl + FD_RB - 1) / FD_RB;
            wneed = std::max(wneed, width_at(v, i, i1_, bx, (double)wl));
            wneed = std::max(wneed, width_at(v, i, i1_, bx, (double)(wl + (nb - 1) * FD_RB)));
          }
        }
        *w_out = wneed;
      };
      eval(j, &rg_best, &w_best);
      if (w_best > FD_WMAX) {      // one projection alone does not fit: the banded kernel takes it
        legacy->push_back(v[i].d.p);
        ++i;
        continue;
      }
      while (j < v.size() && j - i < (size_t)npj) {
        std::vector<int32_t> rg_try;
        int w_try = 0;
        eval(j + 1, &rg_try, &w_try);
        if (w_try > FD_WMAX) break;
        rg_best.swap(rg_try);
        w_best = w_try;
        ++j;
      }
      FdChunk ck{};
      ck.first = (int32_t)projs->size();
      ck.count = (int32_t)(j - i);
      ck.layout = v[i].layout;
      ck.sgn = v[i].sgn;
      ck.skew = v[i].skew;
      ck.mul16 = 16 * v[i].sgn;
      for (size_t t = i; t < j; ++t) projs->push_back(v[t].d);
      chunks->push_back(ck);
      ranges->insert(ranges->end(), rg_best.begin(), rg_best.end());
      w_max = std::max(w_max, w_best);
      i = j;
    }
  }
  std::sort(legacy->begin(), legacy->end());
  plan->W = std::max(16, (w_max + 3) & ~3);
  plan->n_chunks = (int32_t)chunks->size();
  plan->n_tab = (int32_t)projs->size();
  plan->zpad = FD_WMAX + FD_NB + 2 * FD_RB + 16;
  plan->n_lines_alloc = n_lines + FD_RB;
  return plan->n_chunks > 0 && plan->n_chunks <= 65535;
}

// A stack of n groups (of 4 slices) is covered by launches with 4 groups per block (16 slices per thread: the per-line
// boundary / weight / address logic is shared by twice the FMAs; one block per SM; dense angle lists only), then 2, then 1:
// no block works on a spare group.  Returns the number of launches; ng[i] groups per block, cnt[i] blocks along z.
int fd_group_launches(int n_groups, int npj, int ng[3], int cnt[3]) {
  int n = 0, left = n_groups;
#if FD_NG4
  if (npj != 8 && left >= 4) { ng[n] = 4; cnt[n] = left / 4; left -= 4 * cnt[n]; ++n; }
#endif
  if (left >= 2) { ng[n] = 2; cnt[n] = left / 2; left -= 2 * cnt[n]; ++n; }
  if (left >= 1) { ng[n] = 1; cnt[n] = 1; ++n; }
  return n;
}

void fd_block_shape(int32_t* nb, int32_t* npj) {
  *nb = FD_NB;
  *npj = FD_NPJ;
}

size_t fd_xd_bytes(const FdPlan& plan, const pyhst_geom_t* g, int* n_groups_alloc) {
  const int ng = (g->n_slices + 3) / 4;
  if (n_groups_alloc) *n_groups_alloc = ng;
  const int64_t line_f4 = (int64_t)g->nx + 2 * plan.zpad;
  return (size_t)2 * ng * plan.n_lines_alloc * line_f4 * 16;
}

int launch_forward_project_diag(const float* d_img, float* d_sino, int64_t pitch, const pyhst_geom_t* g,
                                float scale, const FdPlan& plan, cudaStream_t stream) {
  int nga = 0;
  const size_t bytes = fd_xd_bytes(plan, g, &nga);
  const int n_groups = (g->n_slices + 3) / 4;
  const int64_t line_f4 = (int64_t)g->nx + 2 * plan.zpad;
  const int64_t group_f4 = line_f4 * plan.n_lines_alloc;
  void* ws = nullptr;
  PYHST_TRY(get_workspace(WS_XD, bytes, &ws));
  float4* xd0 = static_cast<float4*>(ws);
  float4* xd1 = xd0 + (int64_t)nga * group_f4;
  // zero positions are written once per (block, layout): see repack_diag_kernel.  A stack of FEWER slice groups
  // than the one the block was zeroed for (the last chunk of a host pipeline) is laid out as that larger stack
  // -- the second sheared copy keeps its place -- and finds its zeros in place instead of clearing the block on
  // every call; the kernels read groups < n_groups only.
  struct Key { size_t k[8]; };
  static Key seen_all[PYHST_MAX_DEVICES];
  Key key = {{0, (size_t)g->nx, (size_t)g->ny, (size_t)plan.zpad, (size_t)plan.n_lines_alloc, (size_t)nga,
              (size_t)workspace_generation(WS_XD), (size_t)reinterpret_cast<uintptr_t>(ws)}};
  Key& seen = seen_all[std::max(0, current_device()) % PYHST_MAX_DEVICES];
  const size_t seen_groups = seen.k[5];
  key.k[5] = seen_groups;
  const bool zeros_in_place = std::memcmp(&seen, &key, sizeof(key)) == 0 && seen_groups >= (size_t)nga;
  key.k[5] = (size_t)nga;
  if (zeros_in_place) xd1 = xd0 + (int64_t)seen_groups * group_f4;
  {
    StageScope scope(ST_TRANSPOSE, stream);
    if (!zeros_in_place) {
      PYHST_CUDA_TRY(cudaMemsetAsync(ws, 0, bytes, stream));
      seen = key;
    }
    dim3 block(32, 8, 1);
    dim3 grid((g->nx + 31) / 32, (g->ny + 31) / 32, n_groups);
    if (grid.y > 65535 || grid.z > 65535) return set_error(PYHST_ERR_UNSUPPORTED, "image repack: grid too large");
    scope.kernels();
    repack_diag_kernel<<<grid, block, 0, stream>>>(d_img, g->n_slices, g->ny, g->nx, xd0, xd1, line_f4, group_f4,
                                                   plan.zpad);
    PYHST_CUDA_TRY(cudaGetLastError());
  }
  FdParams prm;
  prm.xd[0] = xd0;
  prm.xd[1] = xd1;
  prm.line_f4 = line_f4;
  prm.group_f4 = group_f4;
  prm.zpad = plan.zpad;
  prm.sino = d_sino;
  prm.pitch = pitch;
  prm.S = g->n_slices;
  prm.P = g->n_angles;
  prm.B = g->n_bins;
  prm.scale = scale;
  prm.projs = plan.d_projs;
  prm.chunks = plan.d_chunks;
  prm.ranges = reinterpret_cast<const int2*>(plan.d_ranges);
  prm.n_bx = plan.n_bx;
  prm.W = plan.W;
  const bool small = plan.npj == 8;     // sparse angle lists: 8 projections per block, 256 threads, bands of 4 lines
  int ngl[3], cntl[3];
  const int n_launch = fd_group_launches(n_groups, plan.npj, ngl, cntl);
  int n_sm = 148;
  require_sm100(&n_sm);
  prm.part = nullptr;
  prm.part_pitch = g->n_bins;
  prm.part_stride = 0;
  static DeviceMask configured[12];
#define FD_LAUNCH(NGV, NPJV, RBV, TWOV)                                                                             \
  do {                                                                                                              \
    if (first)                                                                                                      \
      PYHST_CUDA_TRY(cudaFuncSetAttribute(fp_diag_kernel<NGV, NPJV, RBV, TWOV, (NGV == 4 && FD_M1) ? 1 : ((NGV == 2 && NPJV == 16) ? FD_M2 : FD_M)>,                                     \
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fd_smem(NGV, RBV, NPJV))); \
    StageScope scope(ST_FORWARD, stream);                                                                           \
    scope.kernels();                                                                                                \
    fp_diag_kernel<NGV, NPJV, RBV, TWOV, (NGV == 4 && FD_M1) ? 1 : ((NGV == 2 && NPJV == 16) ? FD_M2 : FD_M)>                                          \
        <<<grid, FD_NB / ((NGV == 4 && FD_M1) ? 1 : ((NGV == 2 && NPJV == 16) ? FD_M2 : FD_M)) * NPJV, fd_smem(NGV, RBV, NPJV), stream>>>(prm);      \
  } while (0)
  const int n_one = plan.n_chunks_one < 0 ? plan.n_chunks : plan.n_chunks_one;
  // two passes: the chunks of the generic projections, then those of the near-axis projections (TWO form).  Each pass
  // splits the line range of its blocks into n_seg segments when its grid would not fill the block slots about four
  // times over (small scans; the one or two near-axis projections of a scan) and adds the partial sums afterwards.
  for (int two = 0; two < 2; ++two) {
    const int n_ck = two ? plan.n_chunks - n_one : n_one;
    if (n_ck <= 0) continue;
    double waves = 0.0;   // of the block slots, over the pass's launches, unsplit
    for (int i = 0; i < n_launch; ++i)
      waves += (double)plan.n_bx * n_ck * cntl[i] / (double)(n_sm * (ngl[i] == 4 ? 1 : (small ? 4 : 2)));
    int n_seg = (int)std::max(1.0, std::min(8.0, std::ceil(4.0 / std::max(waves, 1e-9))));
    n_seg = std::max(1, std::min(n_seg, (g->nx + g->ny) / 256));
    prm.n_seg = n_seg;
    prm.part_t0 = two ? plan.n_tab_one : 0;
    prm.part_nt = two ? plan.n_tab - plan.n_tab_one : plan.n_tab_one;
    prm.part_stride = (int64_t)g->n_slices * prm.part_nt * prm.part_pitch;
    if (n_seg > 1) {
      // (the two passes use the block one after the other on the stream; a regrowth synchronises the device)
      void* wp = nullptr;
      PYHST_TRY(get_workspace(WS_FDP, (size_t)n_seg * prm.part_stride * 4, &wp));
      prm.part = static_cast<float*>(wp);
    }
    prm.chunk_off = two ? n_one : 0;
    int g_off = 0;
    for (int i = 0; i < n_launch; ++i) {
      const int ng = ngl[i];
      prm.g_off = g_off;
      g_off += ng * cntl[i];
#if FD_SWAP
      dim3 grid(n_ck, plan.n_bx, cntl[i] * n_seg);
#else
      dim3 grid(plan.n_bx, n_ck, cntl[i] * n_seg);
#endif
      if (grid.z > 65535) return set_error(PYHST_ERR_UNSUPPORTED, "forward projector: too many slice groups");
      const int vi = ((ng == 4 ? 2 : ng - 1) + (small ? 3 : 0)) * 2 + two;
      const bool first = first_use_on_device(&configured[vi]);
      if (small) {
        if (ng == 2) { if (two) FD_LAUNCH(2, 8, 4, true); else FD_LAUNCH(2, 8, 4, false); }
        else { if (two) FD_LAUNCH(1, 8, 4, true); else FD_LAUNCH(1, 8, 4, false); }
      } else {
        if (ng == 4) { if (two) FD_LAUNCH(4, 16, 8, true); else FD_LAUNCH(4, 16, 8, false); }
        else if (ng == 2) { if (two) FD_LAUNCH(2, 16, 8, true); else FD_LAUNCH(2, 16, 8, false); }
        else { if (two) FD_LAUNCH(1, 16, 8, true); else FD_LAUNCH(1, 16, 8, false); }
      }
      PYHST_CUDA_TRY(cudaGetLastError());
    }
    if (n_seg > 1) {   // the pass's projections: [0, n_tab_one) or [n_tab_one, n_tab) of the table
      const int t0 = prm.part_t0, nt = prm.part_nt;
      const int64_t n_rows_tab = (int64_t)g->n_slices * nt;
      const unsigned gy = (unsigned)std::min<int64_t>(n_rows_tab, 32768);
      dim3 grid_c((g->n_bins + 255) / 256, gy, (unsigned)((n_rows_tab + gy - 1) / gy));
      StageScope scope(ST_FORWARD, stream);
      scope.kernels();
      fd_combine_kernel<<<grid_c, 256, 0, stream>>>(d_sino, pitch, prm.part, prm.part_pitch, prm.part_stride, n_seg,
                                                    g->n_bins, g->n_angles, plan.d_projs + t0, nt, n_rows_tab);
    }
  }
#undef FD_LAUNCH
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

}  // namespace pyhst
