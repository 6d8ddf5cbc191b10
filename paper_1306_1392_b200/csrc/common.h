// Internal helpers of libpyhst_b200 (not part of the C ABI; see include/pyhst.h).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <vector>

#include "../../include/pyhst.h"
#include "../../include/pyhst_test.h"

namespace pyhst {

// ---- thread-local last error ------------------------------------------------------------
char* last_error_buf();
int set_error(int status, const char* fmt, ...);

#define PYHST_CUDA_TRY(expr)                                                                   \
  do {                                                                                         \
    cudaError_t _e = (expr);                                                                   \
    if (_e != cudaSuccess)                                                                     \
      return ::pyhst::set_error(_e == cudaErrorMemoryAllocation ? PYHST_ERR_NOMEM              \
                                                                : PYHST_ERR_CUDA,              \
                                "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e),        \
                                __FILE__, __LINE__);                                           \
  } while (0)

#define PYHST_TRY(expr)            \
  do {                             \
    int _s = (expr);               \
    if (_s != PYHST_OK) return _s; \
  } while (0)

// ---- stage accounting (pyhst_profile_*, include/pyhst.h) ----------------------------------
// Every launcher opens a StageScope: it always counts the library's own kernel launches and the
// cuFFT executions of the stage, and -- only while profiling is enabled -- brackets the stage
// with CUDA events on the launching stream.
enum Stage { ST_FILTER = PYHST_STAGE_FILTER, ST_REPACK = PYHST_STAGE_REPACK,
             ST_BACKPROJECT = PYHST_STAGE_BACKPROJECT, ST_TRANSPOSE = PYHST_STAGE_TRANSPOSE,
             ST_FORWARD = PYHST_STAGE_FORWARD, ST_TV = PYHST_STAGE_TV, ST_COUNT = PYHST_N_STAGES };
struct StageScope {
  StageScope(Stage st, cudaStream_t stream);
  ~StageScope();
  void kernels(int n = 1);   // own kernels launched
  void library(int n = 1);   // cuFFT executions
  Stage st;
  cudaStream_t stream;
  int slot;
};

// sm_100 device present and current?  (no CPU fallback: anything else is UNSUPPORTED)
int require_sm100(int* n_sm);

// ---- per-device state and call serialisation (include/pyhst.h "ONE CALL IN FLIGHT PER DEVICE") ----
// Every public compute entry point opens a CallScope first: it takes the current device's lock for
// the duration of the enqueue (re-entrant: entry points call one another) and, when the outermost
// call runs on another stream than the previous call on this device, makes `stream` wait on the
// device for that call's last kernel.  All caches below (workspace, plans, tables) belong to the
// device of the open scope.
struct DeviceCtx;
struct CallScope {
  explicit CallScope(cudaStream_t stream);
  ~CallScope();
  CallScope(const CallScope&) = delete;
  CallScope& operator=(const CallScope&) = delete;
  int status = PYHST_OK;   // PYHST_ERR_* if the device could not be queried / the wait not enqueued
  DeviceCtx* ctx = nullptr;
  cudaStream_t stream;
};
#define PYHST_CALL_SCOPE(stream)             \
  ::pyhst::CallScope _call_scope(stream);    \
  if (_call_scope.status != PYHST_OK) return _call_scope.status

int current_device();  // cudaGetDevice, -1 on failure
// true exactly once per (mask, device): cudaFuncSetAttribute and friends are per device.  The mask is
// shared by all devices (one bit each, device index < PYHST_MAX_DEVICES), hence atomic: threads working
// on different devices hold different device locks.
constexpr int PYHST_MAX_DEVICES = 64;
using DeviceMask = std::atomic<uint64_t>;
bool first_use_on_device(DeviceMask* mask);
// per-device table of sizes already configured (index = device), for kernels whose dynamic
// shared-memory limit grows with the geometry
struct PerDeviceSize {
  size_t v[PYHST_MAX_DEVICES] = {0};   // one element per device: written under that device's lock only
  size_t& here();
};

// ---- per-projection geometry, built in double on the host (reading R11) -----------------
// t_p(i,j) = c + ch * (j - j0) + sh * (i - i0),  ch = h cos(theta_p), sh = h sin(theta_p)
struct ProjGeom {
  double ch, sh, c;
};

// Per-projection entry of the run backprojector, in processing order (class A first):
//   class A: |sh| <= |ch|, runs along y;  class B: |ch| < |sh|, runs along x.
// ch/sh/c are those of the (possibly reversed) stored row, so that the run step is >= 0.
struct RunProj {
  double ch, sh, c;
  int32_t p;     // row of the interleaved sinogram
  int32_t cls;   // 0 = A, 1 = B
};

struct GeomPlan {
  // key
  int32_t n_angles = 0, n_bins = 0;
  double pixel_size = 0, axis_shift = 0;
  std::vector<double> angles, axis;
  // device table [n_angles]
  ProjGeom* d_proj = nullptr;
  ProjGeom* h_pinned = nullptr;
  // run backprojector: permuted / sign-normalised table and the per-row reversal flags
  RunProj* d_run = nullptr;
  uint8_t* d_flip = nullptr;
  int32_t n_a = 0, n_b = 0;
  uint64_t last_use = 0;
};

// Returns a cached (or new) device geometry table for g (axis shifted by axis_shift bins).
// n_bins = length of the rows the backprojector reads (the filtered length inside pyhst_fbp)
int get_geom_plan(const pyhst_geom_t* g, double axis_shift, int32_t n_bins, cudaStream_t stream,
                  const GeomPlan** out);

// Grow-only device workspace slots owned by the library (freed by pyhst_release_cache).
enum WorkspaceSlot { WS_QI = 0, WS_FFT = 1, WS_WEIGHTS = 2, WS_IMG_T = 3, WS_ROWS = 4,
                     WS_CHUNKS = 5, WS_XI = 6, WS_FISTA = 7, WS_FPL = 8, WS_STITCH = 9, WS_XD = 10, WS_FDP = 11, WS_COUNT = 12 };
int get_workspace(WorkspaceSlot slot, size_t bytes, void** ptr);
// bumped whenever the slot's block is (re)allocated or released: lets a user of the slot remember
// "I initialised this very block" without being fooled by a recycled address
uint64_t workspace_generation(WorkspaceSlot slot);

// ---- interleaved sinogram layout consumed by the tiled backprojector ---------------------
// QI[g][p][zpad + b][sl]: slice group g = s / 4, sl = s % 4, one float4 per (g, p, bin);
// every row carries `zpad` zero bins on both sides so that a tile's detector window is one
// contiguous, 16-byte aligned run of float4 that never leaves the row (reading R6).
struct QiLayout {
  int32_t n_groups, n_angles, n_bins, zpad;
  int64_t row_f4() const { return (int64_t)n_bins + 2 * (int64_t)zpad; }          // float4 per row
  int64_t group_f4() const { return row_f4() * n_angles; }                        // float4 per group
  size_t bytes() const { return (size_t)group_f4() * (size_t)n_groups * 16; }
};

// ---- kernels' host launchers (each validates nothing; api.cu did) -------------------------
struct BpArgs {
  float* d_img;          // [S][ny][nx]
  int32_t n_slices, n_angles, n_bins, nx, ny;
  float scale;
  const ProjGeom* d_proj;
  double pixel_size;
};
int launch_backproject_reference(const float* d_sino, int64_t pitch, const BpArgs& a,
                                 cudaStream_t stream);
// window width (bins) the tiled kernel needs for this pixel size; 0 if unsupported
int backproject_tiled_window(double pixel_size);
int launch_backproject_tiled(const float4* d_qi, const QiLayout& L, const BpArgs& a,
                             cudaStream_t stream);
// [S][P][pitch] -> QI (zero pads and missing slices written as zeros)
int launch_repack_to_qi(const float* d_sino, int64_t pitch, int32_t n_slices, float4* d_qi,
                        const QiLayout& L, const uint8_t* d_flip, cudaStream_t stream);
// run kernel (product path): window width it needs, 0 if the geometry is not covered
int backproject_run_window(double pixel_size);
struct RunProj;
int launch_backproject_run(const float4* d_qi, const QiLayout& L, const BpArgs& a,
                           const RunProj* d_run, int32_t n_a, int32_t n_b, cudaStream_t stream);

// run8 kernel (8 slices per thread, producer warp; backproject_run8.cu)
int backproject_run8_window(double pixel_size);
int launch_backproject_run8(const float4* d_qi, const QiLayout& L, const BpArgs& a,
                            const RunProj* d_run, int32_t n_a, int32_t n_b, cudaStream_t stream);

// run16 kernel (16 slices per thread, stacks of >= 13 slices; backproject_run16.cu)
bool backproject_run16_covers(double pixel_size, int n_groups);
int launch_backproject_run16(const float4* d_qi, const QiLayout& L, const BpArgs& a,
                             const RunProj* d_run, int32_t n_a, int32_t n_b, cudaStream_t stream);
int bp_variant();   // pyhst_set_backproject_variant value

// ---- interleaved, zero-padded image layout consumed by the banded forward projector -------
// XI[g][v][zpad + u][sl]: slice group g = s / 4, one float4 per (g, line v, position u); every
// line carries `zpad` zero float4 on both sides.  Two copies: lines = image rows (u = j, v = i)
// for projections walked along rows, lines = image columns (u = i, v = j) for the others.
struct XiLayout {
  int32_t n_groups, nv, nu, zpad;
  int64_t line_f4() const { return (int64_t)nu + 2 * (int64_t)zpad; }
  int64_t group_f4() const { return line_f4() * nv; }
  size_t bytes() const { return (size_t)group_f4() * (size_t)n_groups * 16; }
};

// Per-projection constants of the banded forward projector (line walk, |cu| >= |cv|):
//   strip centre on line v for bin b:  u*(b, v) = b inv_cu + k0 + sD v   (double, R11)
struct FpProjD {
  double inv_cu, k0, sD;
  float s, hw, cuabs;  // (float)sD, |1/cu| = half-width of the strip in pixels, |cu|
  int32_t p;           // projection index in the caller's order
};
struct FpChunk {
  int32_t first, count;  // range in the permuted FpProjD table
  int32_t cls;           // 0: lines are image rows, 1: lines are image columns
  int32_t pad_;
};
// ---- diagonal-line interval projector (forward_project_diag.cu) ----------------------------------
// Position (in kappa = sgn * stored position k, so that t grows with it) of t = m on stored line w:
//   ks(m, w) = K0 + m inv + sD w      (double, R11)
struct FdProj {
  double K0, inv, sD;
  float s, sig;        // (float)sD, |sigma| = h (|cos| + |sin|) = bins per pixel along the line
  int32_t p, pad_;     // projection index in the caller's order
};
struct FdChunk {
  int32_t first, count;   // range in the permuted FdProj table
  int32_t layout;         // 0: lines are diagonals i - j, 1: anti-diagonals i + j
  int32_t sgn, skew;      // stored position = sgn * kappa; stored positions the strips move per line, rounded
  int32_t mul16;          // 16 * sgn: byte step of the stage per kappa
  int32_t pad_[2];
};
struct FdPlan {
  int32_t n_chunks = 0, n_bx = 0, W = 0, zpad = 0, n_lines_alloc = 0, npj = 16, n_tab = 0, n_chunks_one = 0, n_tab_one = 0;   // npj: projections per chunk at most (16 or 8); n_tab: projections in the table; chunks [n_chunks_one, n_chunks) hold the near-axis projections (two pixels per interval possible)
  FdProj* d_projs = nullptr;
  FdChunk* d_chunks = nullptr;
  int32_t* d_ranges = nullptr;   // [n_chunks][n_bx][2]
};

struct FpPlan {
  // key
  int32_t n_angles = 0, n_bins = 0, nx = 0, ny = 0, n_groups = 0;
  double pixel_size = 0;
  int want_diag = 0;
  // diagonal-line kernel: covers every projection except `n_legacy` ones (too close to an image axis,
  // or a window that does not fit), which the banded tables below then hold alone
  bool diag = false;
  int32_t n_legacy = 0;
  FdPlan fd;
  std::vector<double> angles, axis;
  // product
  int32_t npj = 0, W = 0, nc = 0, n_chunks = 0, n_tab = 0;   // n_tab: projections in the banded tables
  bool any_rows = false, any_cols = false;
  FpProjD* d_projs = nullptr;
  FpChunk* d_chunks = nullptr;
  uint64_t last_use = 0;
};
int get_fp_plan(const pyhst_geom_t* g, cudaStream_t stream, int want_diag, const FpPlan** out);  // api.cu; want_diag: 0 no, 1 automatic, 2 forced
// fills the host tables of a plan (for the projections listed in `subset`, all if null); returns false if
// the banded kernel cannot cover the geometry
bool build_fp_tables(const pyhst_geom_t* g, FpPlan* plan, std::vector<FpProjD>* projs,
                     std::vector<FpChunk>* chunks, const std::vector<int32_t>* subset = nullptr);  // forward_project.cu
// diagonal-line kernel: host tables (projections it does not cover are listed in `legacy`); false if it
// covers none
bool build_fd_tables(const pyhst_geom_t* g, FdPlan* plan, std::vector<FdProj>* projs, std::vector<FdChunk>* chunks,
                     std::vector<int32_t>* ranges, std::vector<int32_t>* legacy, int npj = 16);  // forward_project_diag.cu
size_t fd_xd_bytes(const FdPlan& plan, const pyhst_geom_t* g, int* n_groups_alloc);   // bytes of the WS_XD block
void fd_block_shape(int32_t* nb, int32_t* npj);   // intervals per block, projections per chunk
int launch_forward_project_diag(const float* d_img, float* d_sino, int64_t pitch, const pyhst_geom_t* g,
                                float scale, const FdPlan& plan, cudaStream_t stream);
int launch_forward_project_banded(const float* d_img, float* d_sino, int64_t pitch,
                                  const pyhst_geom_t* g, float scale, const FpPlan& plan,
                                  int interval_groups, cudaStream_t stream);
int forward_project_interval_candidates(double pixel_size);

struct FpArgs {
  const float* d_img;    // [S][ny][nx]
  const float* d_img_t;  // [S][nx][ny] (transposed copy, made by launch_transpose_images)
  float* d_sino;         // [S][P][pitch]
  int64_t pitch;
  int32_t n_slices, n_angles, n_bins, nx, ny;
  float scale;
  const ProjGeom* d_proj;
};
int launch_transpose_images(const float* d_img, float* d_img_t, int32_t n_slices, int32_t ny,
                            int32_t nx, cudaStream_t stream);
int launch_forward_project(const FpArgs& a, cudaStream_t stream);

// Ramp filter of `n_rows` rows.  Exactly one of the two outputs is used:
//   d_out != nullptr : plain rows [n_rows][out_pitch]
//   d_qi  != nullptr : rows are [n_slices_in <= 4][n_angles] of ONE slice group, written
//                      interleaved into d_qi (already offset to that group), pads zeroed.
int launch_ramp_filter(const float* d_in, int64_t in_pitch, int64_t n_rows, int32_t n_bins_in,
                       int32_t n_bins_out, int32_t pad_left, int filter,
                       const float* d_col_weights, float* d_out, int64_t out_pitch,
                       float4* d_qi, const QiLayout* L, int32_t n_slices_in, const uint8_t* d_flip,
                       cudaStream_t stream);
// fused shared-memory FFT filter (filter_fused.cu): same contract as launch_ramp_filter
int ramp_fused_log2m(int32_t n_bins_out);   // 0 if the rows are too long for it
int launch_ramp_filter_fused(const float* d_in, int64_t in_pitch, int64_t n_rows, int32_t n_bins_in,
                             int32_t n_bins_out, int32_t pad_left, int filter, const float* d_col_weights,
                             float* d_out, int64_t out_pitch, float4* d_qi, const QiLayout* L, int32_t n_slices_in,
                             const uint8_t* d_flip, cudaStream_t stream);
// frees the tables of `device` (current, idle, and with its DeviceCtx lock held by the caller)
void release_fused_filter_tables(int device);
int filter_variant();   // 0 automatic, 1 cuFFT path, 2 fused kernel (pyhst_test.h)
// tensor-core GEMM of Algorithm 1 (patch_gemm_tc.cu): C[M x N] = alpha A[M x K] B, per slice of a stack
bool patch_gemm_tc_covers(int N, int K);
int launch_patch_gemm_tc(const float* A, const float* Bm, float* C, int64_t M, int N, int K, float alpha,
                         bool trans_b, int n_slices, cudaStream_t stream);
bool run8_packed();       // run8 backprojector: packed FFMA2 interpolation (test variant 6) instead of scalar FFMA
int patch_gemm_variant();   // 0 automatic, 1 FP32 SIMT kernel, 2 tcgen05 3xTF32 kernel (pyhst_test.h)
int launch_halfacq_weights(float* d_w, int32_t n_bins, double cbar, cudaStream_t stream);
int launch_halfacq_fold(const float* d_rows, float* d_out, int32_t n_slices, int32_t half_angles,
                        int32_t b_out, int32_t b_st, int32_t off, const int* d_two_c, cudaStream_t stream);
// frees the cuFFT plans, spectra and fused-filter tables of `device` (same conditions)
void release_filter_plans(int device);

// ---- device helpers: mbarrier + TMA bulk copy (inline PTX) -----------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}

// (c0, c1) += (a0, a1) * s: one packed FFMA2 (ptxas encodes the broadcast scalar operand directly).  On
// sm_100a an FFMA2 occupies both 16-lane FMA pipes and the dispatch port for two cycles -- the cost of two
// scalar FFMAs; nothing issues in its shadow (profiles/r03_micro.md).
__device__ __forceinline__ void ffma2_bcast(float& c0, float& c1, float a0, float a1, float s) {
  asm("{\n\t.reg .b64 ra, rs, rc;\n\t"
      "mov.b64 ra, {%2, %3};\n\t"
      "mov.b64 rs, {%4, %4};\n\t"
      "mov.b64 rc, {%0, %1};\n\t"
      "fma.rn.f32x2 rc, ra, rs, rc;\n\t"
      "mov.b64 {%0, %1}, rc;\n\t}"
      : "+f"(c0), "+f"(c1)
      : "f"(a0), "f"(a1), "f"(s));
}

#endif  // __CUDACC__

}  // namespace pyhst
