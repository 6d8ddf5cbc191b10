// The two GEMMs of Algorithm 1 (P <- W D and G <- 2 P' D^T, "one single
// matrix-matrix multiplication ... cuBlas") on the 5th-generation tensor cores: the one dense contraction
// of the paper.  C[M x N] = alpha * A[M x K] * B with M ~ 1e5 patches and N, K in {64 .. 256}.
//
// tcgen05.mma kind::tf32 reads FP32 words and uses their upper 19 bits (sign, 8 exponent, 10 mantissa bits),
// which alone gives ~5e-4 relative error -- the parity bar of the gradient is 2e-5.  Hence the 3xTF32
// split: a = a_hi + a_lo with a_hi = the word with its low 13 mantissa bits cleared (what the tensor core
// reads anyway) and a_lo = a - a_hi (exact in FP32); C ~= A_hi B_hi + A_hi B_lo + A_lo B_hi, FP32
// accumulation in tensor memory; the dropped A_lo B_lo term is ~2^-22 relative.
//
// One CTA (128 threads) owns a 128-row tile of A:
//   * B (all of K) is staged once, A in chunks of 32 columns: plain coalesced float4 loads, each 16-byte
//     group stored twice into shared memory -- the raw words (= hi operand) and the lo words -- in the
//     canonical K-major no-swizzle UMMA layout: 8 rows x 16 B core matrices, adjacent in K (LBO = 128 B),
//     8-row groups SBO apart;
//   * thread 0 issues, per 8-column K step, three tcgen05.mma (M = 128, N, K = 8) into one TMEM
//     accumulator (N columns x 128 lanes) and commits the chunk to an mbarrier; the chunk buffer is
//     reused when the barrier flips (two CTAs per SM overlap one another's loads and MMAs);
//   * epilogue: every thread owns TMEM lane = tile row, tcgen05.ld 16 columns at a time, scales by alpha
//     and writes its row with 16-byte stores.
// The FP32 SIMT kernel of patches.cu remains the fall-back for shapes this kernel does not cover
// (K % 32 != 0, N % 16 != 0, N > 256, operands that do not fit in shared memory) and the cross-check.
#include <algorithm>

#include "common.h"

namespace pyhst {

namespace {

constexpr int TC_BM = 128;        // tile rows = UMMA M = TMEM lanes
constexpr int TC_KC = 32;         // K columns per staged chunk of A
constexpr int TC_NT = 128;

__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  // cute::UMMA::SmemDescriptor: start address [0,14), leading byte offset [16,30), stride byte offset
  // [32,46) -- all in 16-byte units --, version [46,48) = 1 (Blackwell), layout type [61,64) = 0 (no swizzle)
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr >> 4) & 0x3FFF);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= (uint64_t)1 << 46;
  return d;
}

__device__ __forceinline__ uint32_t umma_idesc_tf32(int M, int N) {
  // cute::UMMA::InstrDescriptor: c_format [4,6) = 1 (F32), a_format [7,10) = b_format [10,13) = 2 (TF32),
  // a_major [15] = b_major [16] = 0 (K-major), n_dim [17,23) = N >> 3, m_dim [24,29) = M >> 4
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(tmem_d), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}

// 16-byte group -> shared memory twice: raw words (hi operand) and a - hi(a) (lo operand)
__device__ __forceinline__ void store_hi_lo(float* hi, float* lo, float4 v) {
  *reinterpret_cast<float4*>(hi) = v;
  float4 l;
  l.x = v.x - __uint_as_float(__float_as_uint(v.x) & 0xFFFFE000u);
  l.y = v.y - __uint_as_float(__float_as_uint(v.y) & 0xFFFFE000u);
  l.z = v.z - __uint_as_float(__float_as_uint(v.z) & 0xFFFFE000u);
  l.w = v.w - __uint_as_float(__float_as_uint(v.w) & 0xFFFFE000u);
  *reinterpret_cast<float4*>(lo) = l;
}

// canonical K-major interleaved layout: element (r, k) of an [R x Kt] operand at
//   (r / 8) * sbo + (k / 4) * 128 + (r % 8) * 16 + (k % 4) * 4   bytes,  sbo = (Kt / 4) * 128
__device__ __forceinline__ uint32_t core_offset_f(int r, int kc4, int sbo_f) {   // in floats, kc4 = k / 4
  return (uint32_t)((r >> 3) * sbo_f + kc4 * 32 + (r & 7) * 4);
}

// TRANS_B = false: B = Bm[K x N] row-major (element (n, k) = Bm[k * N + n]);  true: Bm[N x K] row-major.
// TMEM_COLS = power of two >= N.
template <bool TRANS_B, int TMEM_COLS>
__global__ void __launch_bounds__(TC_NT)
patch_gemm_tc_kernel(const float* __restrict__ A, const float* __restrict__ Bm, float* __restrict__ C, int64_t M,
                     int N, int K, float alpha, int tiles_per_slice, int64_t n_tiles_total) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  __shared__ uint64_t mma_bar;
  __shared__ uint32_t tmem_base_smem;
  const int tid = threadIdx.x, warp = tid >> 5;
  const float* const A_all = A;
  float* const C_all = C;

  // shared memory: B hi, B lo [N x K]; A chunk hi, lo [128 x 32]
  const int b_floats = N * K;
  float* b_hi = reinterpret_cast<float*>(smem_raw);
  float* b_lo = b_hi + b_floats;
  float* a_hi = b_lo + b_floats;
  float* a_lo = a_hi + TC_BM * TC_KC;
  const int sbo_b_f = (K / 4) * 32;          // floats between 8-row groups of B
  const int sbo_a_f = (TC_KC / 4) * 32;      // ... of an A chunk (= 256 floats = 1024 B)

  if (tid == 0) {
    mbar_init(&mma_bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {   // one warp allocates the accumulator columns
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_smem)),
                 "r"((uint32_t)TMEM_COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  // ---- stage B: 16-byte groups (n, k4); global reads coalesced along the contiguous dimension
  // (consecutive threads take consecutive rows of one 8-row group: their 16-byte stores are contiguous)
  if (TRANS_B) {   // Bm[n][k]: k contiguous
    const int k4n = K / 4;
    for (int e = tid; e < N * k4n; e += TC_NT) {
      const int n = ((e / (8 * k4n)) << 3) | (e & 7), k4 = (e >> 3) % k4n;
      const float4 v = *reinterpret_cast<const float4*>(Bm + (int64_t)n * K + 4 * k4);
      const uint32_t o = core_offset_f(n, k4, sbo_b_f);
      store_hi_lo(b_hi + o, b_lo + o, v);
    }
  } else {         // Bm[k][n]: n contiguous -> gather the four k of a group
    const int k4n = K / 4;
    for (int e = tid; e < N * k4n; e += TC_NT) {
      const int k4 = e / N, n = e - k4 * N;
      float4 v;
      v.x = Bm[(int64_t)(4 * k4 + 0) * N + n];
      v.y = Bm[(int64_t)(4 * k4 + 1) * N + n];
      v.z = Bm[(int64_t)(4 * k4 + 2) * N + n];
      v.w = Bm[(int64_t)(4 * k4 + 3) * N + n];
      const uint32_t o = core_offset_f(n, k4, sbo_b_f);
      store_hi_lo(b_hi + o, b_lo + o, v);
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_d = tmem_base_smem;
  const uint32_t idesc = umma_idesc_tf32(TC_BM, N);
  const uint32_t a_hi_s = smem_u32(a_hi), a_lo_s = smem_u32(a_lo), b_hi_s = smem_u32(b_hi), b_lo_s = smem_u32(b_lo);

  const int n_chunks = K / TC_KC;
  uint32_t phase = 0;
  // persistent CTA: B (hi / lo) is staged once and serves every 128-row tile this CTA takes.  The A chunk that is
  // staged next is always already on its way: its eight 16-byte loads per thread are issued right after the MMAs of
  // the chunk before it (software pipelining through registers), so the global latency overlaps the MMAs, the
  // barrier and the epilogue.
  constexpr int A_PER_THREAD = TC_BM * (TC_KC / 4) / TC_NT;
  float4 av[A_PER_THREAD];
  auto load_chunk = [&](int64_t tl, int c) {   // 128 rows x 8 groups; a warp reads 4 rows x 128 contiguous bytes
    const int zz = (int)(tl / tiles_per_slice);
    const int64_t mm0 = (tl - (int64_t)zz * tiles_per_slice) * TC_BM;
    const float* Az = A_all + (int64_t)zz * M * K;
#pragma unroll
    for (int q = 0; q < A_PER_THREAD; ++q) {
      const int e = tid + q * TC_NT;
      const int r = ((e >> 6) << 3) | (e & 7), k4 = (e >> 3) & 7;   // 8 rows x 4 groups per warp: contiguous stores
      av[q] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (mm0 + r < M) av[q] = __ldg(reinterpret_cast<const float4*>(Az + (mm0 + r) * K + c * TC_KC + 4 * k4));
    }
  };
  if ((int64_t)blockIdx.x < n_tiles_total) load_chunk(blockIdx.x, 0);
  for (int64_t tile = blockIdx.x; tile < n_tiles_total; tile += gridDim.x) {
  const int z = (int)(tile / tiles_per_slice);
  const int64_t m0 = (tile - (int64_t)z * tiles_per_slice) * TC_BM;
  C = C_all + (int64_t)z * M * N;
  for (int c = 0; c < n_chunks; ++c) {
    if (c > 0) {   // the MMAs of the previous chunk have read the A buffers
      mbar_wait(&mma_bar, phase);
      phase ^= 1;
    }
    // ---- stage the A chunk from the registers
#pragma unroll
    for (int q = 0; q < A_PER_THREAD; ++q) {
      const int e = tid + q * TC_NT;
      const int r = ((e >> 6) << 3) | (e & 7), k4 = (e >> 3) & 7;
      const uint32_t o = core_offset_f(r, k4, sbo_a_f);
      store_hi_lo(a_hi + o, a_lo + o, av[q]);
    }
    // generic-proxy writes -> visible to the tensor core (async proxy), then hand over to the issuing thread
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (tid == 0) {
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
      for (int j = 0; j < TC_KC / 8; ++j) {           // K = 8 per instruction = two core matrices = 256 B
        const uint32_t a_off = (uint32_t)j * 256u;
        const uint32_t b_off = (uint32_t)(c * (TC_KC / 4) + 2 * j) * 128u;
        const uint64_t da_hi = umma_desc(a_hi_s + a_off, 128u, (uint32_t)sbo_a_f * 4u);
        const uint64_t da_lo = umma_desc(a_lo_s + a_off, 128u, (uint32_t)sbo_a_f * 4u);
        const uint64_t db_hi = umma_desc(b_hi_s + b_off, 128u, (uint32_t)sbo_b_f * 4u);
        const uint64_t db_lo = umma_desc(b_lo_s + b_off, 128u, (uint32_t)sbo_b_f * 4u);
        umma_tf32(tmem_d, da_lo, db_hi, idesc, (c | j) ? 1u : 0u);   // small terms first; a new tile starts a new sum
        umma_tf32(tmem_d, da_hi, db_lo, idesc, 1u);
        umma_tf32(tmem_d, da_hi, db_hi, idesc, 1u);
      }
      // arrives on the barrier when every MMA issued so far has completed (implies fence::before_thread_sync)
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(
                       smem_u32(&mma_bar))
                   : "memory");
    }
    // the next chunk (of this tile or of the CTA's next tile) goes on its way
    if (c + 1 < n_chunks) load_chunk(tile, c + 1);
    else if (tile + gridDim.x < n_tiles_total) load_chunk(tile + gridDim.x, 0);
  }
  mbar_wait(&mma_bar, phase);
  phase ^= 1;
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

  // ---- epilogue: thread = TMEM lane = tile row
  const int64_t row = m0 + tid;
  const uint32_t lane_addr = tmem_d + ((uint32_t)(warp * 32) << 16);
  for (int n0 = 0; n0 < N; n0 += 16) {
    uint32_t v[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, "
        "[%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(lane_addr + (uint32_t)n0)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    if (row < M) {
      float* dst = C + row * N + n0;
#pragma unroll
      for (int q = 0; q < 4; ++q)
        *reinterpret_cast<float4*>(dst + 4 * q) =
            make_float4(alpha * __uint_as_float(v[4 * q]), alpha * __uint_as_float(v[4 * q + 1]),
                        alpha * __uint_as_float(v[4 * q + 2]), alpha * __uint_as_float(v[4 * q + 3]));
    }
  }
  // the accumulator has been read: the next tile's MMAs may overwrite it
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  }   // tiles
  if (warp == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_d), "r"((uint32_t)TMEM_COLS) : "memory");
}

template <bool TRANS_B>
int launch_tc(const float* A, const float* Bm, float* C, int64_t M, int N, int K, float alpha, int n_slices,
              cudaStream_t stream) {
  const size_t smem = ((size_t)2 * N * K + (size_t)2 * TC_BM * TC_KC) * sizeof(float);
  const int64_t tiles = (M + TC_BM - 1) / TC_BM;
  if (tiles * n_slices > 0x7fffffff) return set_error(PYHST_ERR_UNSUPPORTED, "patch GEMM: too many tiles");
  int n_sm = 148;
  require_sm100(&n_sm);
  // persistent CTAs, two per SM (their loads and MMAs overlap one another); B is staged once per CTA
  const unsigned grid = (unsigned)std::min<int64_t>(tiles * n_slices, (int64_t)2 * n_sm);
#define PYHST_TC_LAUNCH(COLS)                                                                                     \
  do {                                                                                                            \
    static PerDeviceSize configured;                                                                              \
    if (smem > configured.here()) {                                                                               \
      PYHST_CUDA_TRY(cudaFuncSetAttribute(patch_gemm_tc_kernel<TRANS_B, COLS>,                                    \
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));               \
      configured.here() = smem;                                                                                   \
    }                                                                                                             \
    patch_gemm_tc_kernel<TRANS_B, COLS><<<grid, TC_NT, smem, stream>>>(A, Bm, C, M, N, K, alpha, (int)tiles, tiles * n_slices);     \
  } while (0)
  if (N <= 32) PYHST_TC_LAUNCH(32);
  else if (N <= 64) PYHST_TC_LAUNCH(64);
  else if (N <= 128) PYHST_TC_LAUNCH(128);
  else PYHST_TC_LAUNCH(256);
#undef PYHST_TC_LAUNCH
  PYHST_CUDA_TRY(cudaGetLastError());
  return PYHST_OK;
}

}  // namespace

// does the tensor-core kernel cover C[M x N] = A[M x K] B ?
bool patch_gemm_tc_covers(int N, int K) {
  if (N % 16 || N < 16 || N > 256 || K % TC_KC || K < TC_KC) return false;
  const size_t smem = ((size_t)2 * N * K + (size_t)2 * TC_BM * TC_KC) * sizeof(float);
  return smem <= 200 * 1024;
}

int launch_patch_gemm_tc(const float* A, const float* Bm, float* C, int64_t M, int N, int K, float alpha,
                         bool trans_b, int n_slices, cudaStream_t stream) {
  if ((reinterpret_cast<uintptr_t>(A) | reinterpret_cast<uintptr_t>(Bm) | reinterpret_cast<uintptr_t>(C)) & 15)
    return set_error(PYHST_ERR_INVALID_ARG, "patch GEMM: operands must be 16-byte aligned");
  return trans_b ? launch_tc<true>(A, Bm, C, M, N, K, alpha, n_slices, stream)
                 : launch_tc<false>(A, Bm, C, M, N, K, alpha, n_slices, stream);
}

}  // namespace pyhst
