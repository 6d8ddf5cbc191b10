/*
 * pyhst_test.h -- test / bench hooks of libpyhst_b200 (NOT part of the product API of pyhst.h).
 *
 * Process-wide switches that select older or alternative kernels for cross-checks.  They are
 * atomic integers shared by all devices and threads and read at the start of a call: setting
 * one while a call is in flight on another thread is not a data race, but which kernel that call
 * runs is then unspecified -- set them only while no call is in flight.  Every variant computes
 * the operation pyhst.h defines; results agree within FP32 rounding.
 */
#ifndef PYHST_TEST_H_
#define PYHST_TEST_H_

#include "pyhst.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Selects the backprojection kernel: 0 = automatic (default), 1 = reference one-thread-per-
 * pixel kernel (global loads; kept for cross-checks), 2 = tiled shared-memory kernel, 3 = run
 * kernel with 4 slices per thread, 4 = run kernel with 8 slices per thread (what 0 picks for
 * pixel sizes below sqrt(2) bins), 6 = the same with the interpolation written as packed FFMA2 (8 fewer
 * warp instructions per step, same time: an FFMA2 costs two issue slots on sm_100a, profiles/r02_micro.md), 7 = run kernel
 * with 16 slices per thread for stacks of >= 13 slices (runs of 4 pixels, one 512-thread block per SM; 11 % fewer
 * instructions but latency-bound with one run in flight: measured slower, profiles/r02_micro.md sec. C; other stacks
 * as 4).  A variant that does not cover the geometry makes the next
 * call return PYHST_ERR_UNSUPPORTED.  Returns the previous value.  Test/bench hook; results
 * agree within FP32 rounding. */
int pyhst_set_backproject_variant(int variant);

/* PYHST_SCAN_360_HALF only (NEXT row N2): 1 (default) lets pyhst_fbp fold a scan whose projections p
 * and p + P/2 face each other (angles differ by pi to 1e-10, equal axis, 2 x axis integer) into P/2
 * full-width rows, lerp(g_p, t) + lerp(g_{p+P/2}, 2c - t) = lerp(g_p + flip(g_{p+P/2}), t), and
 * backproject half as many projections; 0 always backprojects all P rows.  Scans that do not pair up
 * take the general path either way.  Returns the previous value. */
int pyhst_set_halfacq_stitch(int enable);

/* Selects the forward-projection kernel: 0 = automatic (default: the diagonal-line interval kernel when its
 * blocks are mostly full -- on average at least 0.55 x 16 (dense angle lists) or 0.55 x 8 (sparser ones)
 * neighbouring projections share one staged window -- and the grid has at least one block per SM, else the banded kernel),
 * 1 = generic gather kernel (one thread per bin and slice, global loads; kept for cross-checks and for pixel
 * sizes the shared-memory kernels do not cover), 2 = banded shared-memory kernel, 3 = interval form of the
 * banded kernel (fewer shared-memory loads, more instructions), 4 = interval form with 8 slices per thread
 * (stacks with an even number of slice groups and 16-projection chunks, else as 3), 5 = diagonal-line interval
 * kernel forced (PYHST_ERR_UNSUPPORTED when no projection has >= 1 + 2^-12 bins per pixel along an image
 * diagonal, i.e. pixel sizes below ~0.71 bins; projections it does not cover -- fewer than 1 - 1e-6 bins per pixel
 * along the diagonal, or a window that alone does not fit -- run on the banded kernel).  Returns the previous value. */
int pyhst_set_forward_project_variant(int variant);

/* Which kernel the last pyhst_forward_project of this process ran: 1 generic gather, 2 banded, 3 / 4
 * interval forms, 5 diagonal-line interval kernel (plus the banded kernel for the projections it leaves
 * out), 0 none yet.  For bench labels and tests. */
int pyhst_last_forward_project_kernel(void);

/* Host-only (no device needed): builds the tables of the diagonal-line forward projector for geometry g and reports
 * info[0] = chunks, info[1] = projections left to the banded kernel, info[2] = staged window width (float4 per line),
 * info[3] = detector blocks per chunk, info[4] = intervals per block, info[5] = projections per chunk at most,
 * info[6] = zero pad of a stored line, info[7] = stored lines per slice group.  chunk_of (nullable, [n_angles]) receives
 * the chunk index of every projection, -1 for those left out; ranges (nullable, [chunks][blocks][2]) the lines each block
 * walks.  Returns PYHST_OK, or PYHST_ERR_UNSUPPORTED when the kernel covers no projection of g. */
int pyhst_test_fd_plan(const pyhst_geom_t* g, int32_t* info, int32_t* chunk_of, int32_t* ranges);

/* Selects the ramp-filter implementation: 0 = automatic (default: the fused shared-memory FFT kernel for
 * rows of up to 4096 filtered bins, cuFFT beyond), 1 = the cuFFT path (pad/weight, R2C, x H, C2R, crop:
 * five passes), 2 = the fused kernel (UNSUPPORTED for longer rows).  Returns the previous value. */
int pyhst_set_filter_variant(int variant);

/* Selects the kernel of the two GEMMs of pyhst_patch_gradient / pyhst_patch_fista: 0 = automatic (default: the
 * tcgen05 3xTF32 tensor-core kernel when the shapes allow it -- n_atoms and m*m multiples of 32 resp. 16, at
 * most 256, operands 16-byte aligned -- else the FP32 SIMT kernel), 1 = FP32 SIMT kernel, 2 = tensor-core
 * kernel (UNSUPPORTED for other shapes).  Returns the previous value. */
int pyhst_set_patch_gemm_variant(int variant);

/* Makes every growth of an internal workspace block beyond `max_bytes` fail with PYHST_ERR_NOMEM, as if
 * cudaMalloc had (0 = no limit, the default; blocks that are already large enough are not affected).  Lets a
 * test exercise the out-of-memory paths -- e.g. the forward projector's fall-back from the diagonal-line to the
 * banded kernel -- without exhausting the device.  Returns the previous limit. */
int64_t pyhst_test_set_workspace_limit(int64_t max_bytes);

#ifdef __cplusplus
}
#endif
#endif /* PYHST_TEST_H_ */
