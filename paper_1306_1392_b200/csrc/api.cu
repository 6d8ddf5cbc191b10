// C ABI of libpyhst_b200 (include/pyhst.h): argument validation, plan / workspace caches and the
// sequencing of the kernels.  Every step of the hot path runs on the device; there is no CPU
// fallback (a missing or non-sm_100 device yields PYHST_ERR_UNSUPPORTED).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <list>
#include <map>
#include <memory>
#include <mutex>

#include "common.h"

namespace pyhst {

// ---- errors ------------------------------------------------------------------------------
char* last_error_buf() {
  static thread_local char buf[512] = {0};
  return buf;
}

int set_error(int status, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(last_error_buf(), 512, fmt, ap);
  va_end(ap);
  return status;
}

int require_sm100(int* n_sm) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return set_error(PYHST_ERR_UNSUPPORTED, "no CUDA device (%s); there is no CPU fallback",
                     cudaGetErrorString(e));
  }
  static int cached_dev = -1, cached_major = 0, cached_sms = 0;
  if (dev != cached_dev) {
    int major = 0, sms = 0;
    PYHST_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    PYHST_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    cached_dev = dev;
    cached_major = major;
    cached_sms = sms;
  }
  if (cached_major != 10)
    return set_error(PYHST_ERR_UNSUPPORTED,
                     "device has compute capability %d.x; this library is built for sm_100a only",
                     cached_major);
  if (n_sm) *n_sm = cached_sms;
  return PYHST_OK;
}

// ---- per-device state ----------------------------------------------------------------------
struct Ws { void* p = nullptr; size_t bytes = 0; uint64_t gen = 0; };
struct DeviceCtx {
  int device = 0;
  std::recursive_mutex mu;      // held by the open CallScope(s) of one thread
  int depth = 0;                // nesting of entry points inside the outermost call
  cudaEvent_t last_done = nullptr;
  cudaStream_t last_stream = nullptr;
  bool have_last = false;
  std::list<GeomPlan> geom;
  std::list<FpPlan> fp_plans;
  Ws ws[WS_COUNT];
  cudaStream_t streams[3] = {nullptr, nullptr, nullptr};
  cudaEvent_t events[8] = {nullptr};
  uint64_t tick = 0;
};

namespace {
std::mutex g_map_mu;
std::map<int, std::unique_ptr<DeviceCtx>> g_ctx;
// test / bench hooks of pyhst_test.h: process-wide, read at the start of a call (atomic so that a hook set from one
// thread while another thread is inside a call is a defined, if unspecified, choice -- not a data race)
std::atomic<int> g_bp_variant{0};
std::atomic<int> g_fp_variant{0};
std::atomic<int> g_last_fp_kernel{0};
std::atomic<int> g_halfacq_stitch{1};
std::atomic<int> g_filter_variant{0};
std::atomic<int> g_patch_gemm_variant{0};
std::atomic<int64_t> g_ws_limit{0};   // pyhst_test_set_workspace_limit

DeviceCtx* ctx_of(int dev) {
  std::lock_guard<std::mutex> lock(g_map_mu);
  auto& slot = g_ctx[dev];
  if (!slot) {
    slot.reset(new DeviceCtx());
    slot->device = dev;
  }
  return slot.get();
}
// state of the current device; only called inside an open CallScope (or under its own lock)
DeviceCtx& ctx() { return *ctx_of(std::max(0, current_device())); }
}  // namespace

int filter_variant() { return g_filter_variant; }
int patch_gemm_variant() { return g_patch_gemm_variant; }
bool run8_packed() { return g_bp_variant == 6; }
int bp_variant() { return g_bp_variant; }

int current_device() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  return dev;
}

// (device indices >= PYHST_MAX_DEVICES never get here: CallScope refuses them)
bool first_use_on_device(DeviceMask* mask) {
  const uint64_t bit = (uint64_t)1 << (std::max(0, current_device()) % PYHST_MAX_DEVICES);
  return (mask->fetch_or(bit, std::memory_order_acq_rel) & bit) == 0;
}

size_t& PerDeviceSize::here() { return v[std::max(0, current_device()) % PYHST_MAX_DEVICES]; }

CallScope::CallScope(cudaStream_t stream_) : stream(stream_) {
  const int dev = current_device();
  if (dev < 0) return;   // no device: the entry point's require_sm100() reports it
  if (dev >= PYHST_MAX_DEVICES) {   // the per-device tables (first-use masks, PerDeviceSize) have one entry per index
    status = set_error(PYHST_ERR_UNSUPPORTED, "device index %d: this library keeps state for devices 0..%d only", dev,
                       PYHST_MAX_DEVICES - 1);
    return;
  }
  ctx = ctx_of(dev);
  ctx->mu.lock();
  if (ctx->depth++ == 0 && ctx->have_last && ctx->last_stream != stream) {
    cudaError_t e = cudaStreamWaitEvent(stream, ctx->last_done, 0);
    if (e != cudaSuccess)
      status = set_error(PYHST_ERR_CUDA, "cudaStreamWaitEvent on the previous call failed: %s",
                         cudaGetErrorString(e));
  }
}

CallScope::~CallScope() {
  if (!ctx) return;
  if (--ctx->depth == 0) {
    if (!ctx->last_done) cudaEventCreateWithFlags(&ctx->last_done, cudaEventDisableTiming);
    if (ctx->last_done && cudaEventRecord(ctx->last_done, stream) == cudaSuccess) {
      ctx->last_stream = stream;
      ctx->have_last = true;
    } else {
      cudaGetLastError();
      ctx->have_last = false;
    }
  }
  ctx->mu.unlock();
}

// ---- stage accounting --------------------------------------------------------------------
namespace {
struct StageEvents { Stage st; cudaEvent_t a, b; int dev; };
std::mutex g_prof_mu;
bool g_prof_on = false;
std::vector<StageEvents> g_prof_pending;
std::map<int, std::vector<cudaEvent_t>> g_prof_pool;   // per device: an event can only be recorded on a stream of the device it was created on
double g_prof_ms[ST_COUNT] = {0};
int64_t g_prof_kernels[ST_COUNT] = {0}, g_prof_fft[ST_COUNT] = {0};

cudaEvent_t prof_event(int dev) {
  auto& pool = g_prof_pool[dev];
  if (!pool.empty()) {
    cudaEvent_t e = pool.back();
    pool.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}
}  // namespace

StageScope::StageScope(Stage st_, cudaStream_t stream_) : st(st_), stream(stream_), slot(-1) {
  std::lock_guard<std::mutex> lock(g_prof_mu);
  if (!g_prof_on) return;
  const int dev = current_device();
  if (dev < 0) return;
  StageEvents ev{st, prof_event(dev), prof_event(dev), dev};
  if (!ev.a || !ev.b) return;
  cudaEventRecord(ev.a, stream);
  slot = (int)g_prof_pending.size();
  g_prof_pending.push_back(ev);
}
StageScope::~StageScope() {
  if (slot < 0) return;
  std::lock_guard<std::mutex> lock(g_prof_mu);
  if (slot < (int)g_prof_pending.size()) cudaEventRecord(g_prof_pending[slot].b, stream);
}
void StageScope::kernels(int n) {
  std::lock_guard<std::mutex> lock(g_prof_mu);
  g_prof_kernels[st] += n;
}
void StageScope::library(int n) {
  std::lock_guard<std::mutex> lock(g_prof_mu);
  g_prof_fft[st] += n;
}

int get_geom_plan(const pyhst_geom_t* g, double axis_shift, int32_t n_bins, cudaStream_t stream,
                  const GeomPlan** out) {
  DeviceCtx& c = ctx();
  std::lock_guard<std::recursive_mutex> lock(c.mu);
  auto& g_geom = c.geom;
  uint64_t& g_tick = c.tick;
  const size_t n = (size_t)g->n_angles;
  for (auto& pl : g_geom) {
    if (pl.n_angles == g->n_angles && pl.n_bins == n_bins && pl.pixel_size == g->pixel_size &&
        pl.axis_shift == axis_shift &&
        std::memcmp(pl.angles.data(), g->angles_rad, n * sizeof(double)) == 0 &&
        std::memcmp(pl.axis.data(), g->axis_pos, n * sizeof(double)) == 0) {
      pl.last_use = ++g_tick;
      *out = &pl;
      return PYHST_OK;
    }
  }
  if (g_geom.size() >= 16) {  // evict the least recently used plan
    auto lru = g_geom.begin();
    for (auto it = g_geom.begin(); it != g_geom.end(); ++it)
      if (it->last_use < lru->last_use) lru = it;
    cudaFree(lru->d_proj);  // synchronises: no kernel can still be reading it
    cudaFree(lru->d_run);
    cudaFree(lru->d_flip);
    cudaFreeHost(lru->h_pinned);
    g_geom.erase(lru);
  }
  GeomPlan pl;
  // an early return below (PYHST_CUDA_TRY) must not leak what the plan already owns
  struct GeomGuard {
    GeomPlan* pl;
    bool keep = false;
    ~GeomGuard() {
      if (keep) return;
      cudaFree(pl->d_proj);
      cudaFree(pl->d_run);
      cudaFree(pl->d_flip);
      cudaFreeHost(pl->h_pinned);
    }
  } guard{&pl};
  pl.n_angles = g->n_angles;
  pl.n_bins = n_bins;
  pl.pixel_size = g->pixel_size;
  pl.axis_shift = axis_shift;
  pl.angles.assign(g->angles_rad, g->angles_rad + n);
  pl.axis.assign(g->axis_pos, g->axis_pos + n);
  PYHST_CUDA_TRY(cudaMallocHost(&pl.h_pinned, n * sizeof(ProjGeom)));
  cudaError_t e = cudaMalloc(&pl.d_proj, n * sizeof(ProjGeom));
  if (e != cudaSuccess) {
    return set_error(PYHST_ERR_NOMEM, "cudaMalloc of the geometry table failed: %s",
                     cudaGetErrorString(e));
  }
  for (size_t p = 0; p < n; ++p) {  // cos/sin in double (R11)
    pl.h_pinned[p].ch = g->pixel_size * std::cos(g->angles_rad[p]);
    pl.h_pinned[p].sh = g->pixel_size * std::sin(g->angles_rad[p]);
    pl.h_pinned[p].c = g->axis_pos[p] + axis_shift;
  }
  PYHST_CUDA_TRY(cudaMemcpyAsync(pl.d_proj, pl.h_pinned, n * sizeof(ProjGeom), cudaMemcpyHostToDevice,
                                 stream));
  // run backprojector: class A (|sh| <= |ch|, runs along y) first, then class B (runs along x);
  // a row is stored reversed (t -> n_bins-1-t: ch, sh change sign) when its run step is negative
  {
    std::vector<RunProj> run;
    std::vector<uint8_t> flip(n, 0);
    run.reserve(n);
    for (int cls = 0; cls < 2; ++cls)
      for (size_t p = 0; p < n; ++p) {
        const ProjGeom& pg = pl.h_pinned[p];
        const int c = std::fabs(pg.sh) <= std::fabs(pg.ch) ? 0 : 1;
        if (c != cls) continue;
        const double step = cls ? pg.ch : pg.sh;
        RunProj r{pg.ch, pg.sh, pg.c, (int32_t)p, cls};
        if (step < 0.0) {
          r.ch = -pg.ch;
          r.sh = -pg.sh;
          r.c = (double)(n_bins - 1) - pg.c;
          flip[p] = 1;
        }
        run.push_back(r);
        (cls ? pl.n_b : pl.n_a)++;
      }
    PYHST_CUDA_TRY(cudaMalloc(&pl.d_run, n * sizeof(RunProj)));
    PYHST_CUDA_TRY(cudaMalloc(&pl.d_flip, n));
    // pageable sources: staged before the calls return
    PYHST_CUDA_TRY(cudaMemcpyAsync(pl.d_run, run.data(), n * sizeof(RunProj), cudaMemcpyHostToDevice, stream));
    PYHST_CUDA_TRY(cudaMemcpyAsync(pl.d_flip, flip.data(), n, cudaMemcpyHostToDevice, stream));
  }
  pl.last_use = ++g_tick;
  guard.keep = true;
  g_geom.push_back(std::move(pl));
  *out = &g_geom.back();
  return PYHST_OK;
}

int get_fp_plan(const pyhst_geom_t* g, cudaStream_t stream, int want_diag, const FpPlan** out) {
  DeviceCtx& c = ctx();
  std::lock_guard<std::recursive_mutex> lock(c.mu);
  auto& g_fp_plans = c.fp_plans;
  uint64_t& g_tick = c.tick;
  const size_t n = (size_t)g->n_angles;
  for (auto& pl : g_fp_plans) {
    if (pl.n_angles == g->n_angles && pl.n_bins == g->n_bins && pl.nx == g->nx && pl.ny == g->ny &&
        pl.n_groups == (g->n_slices + 3) / 4 && pl.pixel_size == g->pixel_size && pl.want_diag == want_diag &&
        std::memcmp(pl.angles.data(), g->angles_rad, n * sizeof(double)) == 0 &&
        std::memcmp(pl.axis.data(), g->axis_pos, n * sizeof(double)) == 0) {
      pl.last_use = ++g_tick;
      *out = &pl;
      return PYHST_OK;
    }
  }
  if (g_fp_plans.size() >= 8) {
    auto lru = g_fp_plans.begin();
    for (auto it = g_fp_plans.begin(); it != g_fp_plans.end(); ++it)
      if (it->last_use < lru->last_use) lru = it;
    cudaFree(lru->d_projs);  // synchronises: no kernel can still be reading them
    cudaFree(lru->d_chunks);
    cudaFree(lru->fd.d_projs);
    cudaFree(lru->fd.d_chunks);
    cudaFree(lru->fd.d_ranges);
    g_fp_plans.erase(lru);
  }
  FpPlan pl;
  struct FpGuard {   // frees the device tables of a plan that an early return abandons
    FpPlan* pl;
    bool keep = false;
    ~FpGuard() {
      if (keep) return;
      cudaFree(pl->d_projs);
      cudaFree(pl->d_chunks);
      cudaFree(pl->fd.d_projs);
      cudaFree(pl->fd.d_chunks);
      cudaFree(pl->fd.d_ranges);
    }
  } guard{&pl};
  pl.n_angles = g->n_angles;
  pl.n_bins = g->n_bins;
  pl.nx = g->nx;
  pl.ny = g->ny;
  pl.n_groups = (g->n_slices + 3) / 4;
  pl.pixel_size = g->pixel_size;
  pl.angles.assign(g->angles_rad, g->angles_rad + n);
  pl.axis.assign(g->axis_pos, g->axis_pos + n);
  pl.want_diag = want_diag;
  std::vector<FpProjD> projs;
  std::vector<FpChunk> chunks;
  std::vector<int32_t> legacy;
  bool banded_built = false;   // projs / chunks already hold the banded tables of the `legacy` projections
  if (want_diag) {
    // diagonal-line interval kernel for every projection it covers; the banded tables then hold
    // only the rest (projections within 2^-12 rad of an image axis, windows that do not fit)
    std::vector<FdProj> dprojs;
    std::vector<FdChunk> dchunks;
    std::vector<int32_t> ranges;
    FpPlan probe = pl;
    bool use = build_fd_tables(g, &pl.fd, &dprojs, &dchunks, &ranges, &legacy);
    // sparse angle lists fan out: few projections fit one staged window -- blocks of 8 projections instead of 16
    if (use && (double)dprojs.size() / (double)dchunks.size() < 8.0)
      use = build_fd_tables(g, &pl.fd, &dprojs, &dchunks, &ranges, &legacy, 8);
    if (use && want_diag == 1) {
      // automatic choice: the diagonal-line kernel pays off when its blocks are mostly full (neighbouring
      // projections share a window) and fill the GPU; very sparse lists and small scans stay on the banded kernel
      const double per_chunk = (double)dprojs.size() / (double)dchunks.size();
      const int64_t blocks = (int64_t)pl.fd.n_bx * pl.fd.n_chunks * std::max(1, (pl.n_groups + 1) / 2);
      int n_sm = 148;
      require_sm100(&n_sm);
      // (grids of fewer blocks than 4 per SM are split along the lines by the launcher; below one block per SM the
      // banded kernel's smaller blocks win)
      use = per_chunk >= 0.55 * pl.fd.npj && blocks >= (int64_t)n_sm;
    }
    if (use && !legacy.empty()) banded_built = build_fp_tables(g, &probe, &projs, &chunks, &legacy);
    if (use && (legacy.empty() || banded_built)) {
      pl.diag = true;
      if (banded_built) {   // keep the probe's tables: the banded part of the plan is exactly what it built
        pl.nc = probe.nc; pl.W = probe.W; pl.npj = probe.npj; pl.n_chunks = probe.n_chunks; pl.n_tab = probe.n_tab;
        pl.any_rows = probe.any_rows; pl.any_cols = probe.any_cols;
      }
      pl.n_legacy = (int32_t)legacy.size();
      PYHST_CUDA_TRY(cudaMalloc(&pl.fd.d_projs, dprojs.size() * sizeof(FdProj)));
      PYHST_CUDA_TRY(cudaMalloc(&pl.fd.d_chunks, dchunks.size() * sizeof(FdChunk)));
      PYHST_CUDA_TRY(cudaMalloc(&pl.fd.d_ranges, ranges.size() * sizeof(int32_t)));
      PYHST_CUDA_TRY(cudaMemcpyAsync(pl.fd.d_projs, dprojs.data(), dprojs.size() * sizeof(FdProj),
                                     cudaMemcpyHostToDevice, stream));
      PYHST_CUDA_TRY(cudaMemcpyAsync(pl.fd.d_chunks, dchunks.data(), dchunks.size() * sizeof(FdChunk),
                                     cudaMemcpyHostToDevice, stream));
      PYHST_CUDA_TRY(cudaMemcpyAsync(pl.fd.d_ranges, ranges.data(), ranges.size() * sizeof(int32_t),
                                     cudaMemcpyHostToDevice, stream));
      if (std::getenv("PYHST_DEBUG"))
        fprintf(stderr, "[pyhst] fp diag plan: P=%d B=%d %dx%d h=%g -> W=%d chunks=%d n_bx=%d legacy=%d\n",
                g->n_angles, g->n_bins, g->nx, g->ny, g->pixel_size, pl.fd.W, pl.fd.n_chunks, pl.fd.n_bx,
                pl.n_legacy);
    }
    banded_built = banded_built && pl.diag;
    if (!banded_built) {
      projs.clear();
      chunks.clear();
    }
  }
  if (pl.diag && legacy.empty()) {
    pl.n_chunks = 0;
  } else if (banded_built || build_fp_tables(g, &pl, &projs, &chunks, pl.diag ? &legacy : nullptr)) {
    PYHST_CUDA_TRY(cudaMalloc(&pl.d_projs, projs.size() * sizeof(FpProjD)));
    PYHST_CUDA_TRY(cudaMalloc(&pl.d_chunks, chunks.size() * sizeof(FpChunk)));
    // pageable sources: the copies are complete (staged) when the calls return
    PYHST_CUDA_TRY(cudaMemcpyAsync(pl.d_projs, projs.data(), projs.size() * sizeof(FpProjD),
                                   cudaMemcpyHostToDevice, stream));
    PYHST_CUDA_TRY(cudaMemcpyAsync(pl.d_chunks, chunks.data(), chunks.size() * sizeof(FpChunk),
                                   cudaMemcpyHostToDevice, stream));
    if (std::getenv("PYHST_DEBUG"))
      fprintf(stderr, "[pyhst] fp plan: P=%d B=%d %dx%d h=%g -> W=%d nc=%d chunks=%d (rows %d cols %d)\n",
              g->n_angles, g->n_bins, g->nx, g->ny, g->pixel_size, pl.W, pl.nc, pl.n_chunks,
              (int)pl.any_rows, (int)pl.any_cols);
  } else {
    pl.n_chunks = 0;  // geometry not covered by the banded kernel: the generic gather kernel runs
  }
  pl.last_use = ++g_tick;
  guard.keep = true;
  g_fp_plans.push_back(std::move(pl));
  *out = &g_fp_plans.back();
  return PYHST_OK;
}

int get_workspace(WorkspaceSlot slot, size_t bytes, void** ptr) {
  DeviceCtx& c = ctx();
  std::lock_guard<std::recursive_mutex> lock(c.mu);
  Ws& w = c.ws[slot];
  if (w.bytes < bytes) {
    if (w.p) {
      cudaFree(w.p);  // synchronises the device: nothing can still be using the old block
      w.p = nullptr;
      w.bytes = 0;
    }
    ++w.gen;
    const int64_t limit = g_ws_limit.load();
    if (limit > 0 && bytes > (size_t)limit)
      return set_error(PYHST_ERR_NOMEM, "workspace allocation of %zu bytes refused (test limit %lld)", bytes,
                       (long long)limit);
    cudaError_t e = cudaMalloc(&w.p, bytes);
    if (e != cudaSuccess) {
      cudaGetLastError();
      w.p = nullptr;
      return set_error(PYHST_ERR_NOMEM, "workspace allocation of %zu bytes failed: %s", bytes,
                       cudaGetErrorString(e));
    }
    w.bytes = bytes;
  }
  *ptr = w.p;
  return PYHST_OK;
}

uint64_t workspace_generation(WorkspaceSlot slot) {
  DeviceCtx& c = ctx();
  std::lock_guard<std::recursive_mutex> lock(c.mu);
  return c.ws[slot].gen;
}

// ---- validation --------------------------------------------------------------------------
static int check_geom(const pyhst_geom_t* g, int64_t* pitch) {
  if (!g) return set_error(PYHST_ERR_INVALID_ARG, "geometry is NULL");
  if (g->n_slices <= 0 || g->n_angles <= 0 || g->n_bins <= 0 || g->nx <= 0 || g->ny <= 0)
    return set_error(PYHST_ERR_INVALID_ARG, "sizes must be positive (S=%d P=%d B=%d nx=%d ny=%d)",
                     g->n_slices, g->n_angles, g->n_bins, g->nx, g->ny);
  if (!g->angles_rad || !g->axis_pos)
    return set_error(PYHST_ERR_INVALID_ARG, "angles_rad / axis_pos is NULL");
  if (!(g->pixel_size > 0.0) || !std::isfinite(g->pixel_size))
    return set_error(PYHST_ERR_INVALID_ARG, "pixel_size must be positive and finite");
  if (g->sino_pitch != 0 && g->sino_pitch < g->n_bins)
    return set_error(PYHST_ERR_INVALID_ARG, "sino_pitch %lld < n_bins %d", (long long)g->sino_pitch,
                     g->n_bins);
  for (int32_t p = 0; p < g->n_angles; ++p)
    if (!std::isfinite(g->angles_rad[p]) || !std::isfinite(g->axis_pos[p]))
      return set_error(PYHST_ERR_INVALID_ARG, "angle / axis position %d is not finite", p);
  if (g->n_angles > 65535)
    return set_error(PYHST_ERR_UNSUPPORTED, "more than 65535 projections");
  *pitch = g->sino_pitch ? g->sino_pitch : g->n_bins;
  return PYHST_OK;
}

static int check_ptr(const void* p, const char* name) {
  if (!p) return set_error(PYHST_ERR_INVALID_ARG, "%s is NULL", name);
  if (reinterpret_cast<uintptr_t>(p) & 3)
    return set_error(PYHST_ERR_INVALID_ARG, "%s is not 4-byte aligned", name);
  return PYHST_OK;
}

static QiLayout qi_layout(int32_t n_slices, int32_t n_angles, int32_t n_bins, double pixel_size) {
  QiLayout L;
  L.n_groups = (n_slices + 3) / 4;
  L.n_angles = n_angles;
  L.n_bins = n_bins;
  const int W = backproject_tiled_window(pixel_size);
  L.zpad = W > 0 ? W + 4 : 16;
  return L;
}

// 1 = reference, 2 = tiled, 3 = run (4 slices per thread), 4 = run8 (8 slices per thread, the
// product path); -1 = the requested variant does not cover the geometry
static int pick_bp_kernel(double pixel_size, int32_t n_slices) {
  const bool tiled_ok = backproject_tiled_window(pixel_size) > 0;
  const bool run_ok = backproject_run_window(pixel_size) > 0;
  const bool run8_ok = run_ok && backproject_run8_window(pixel_size) > 0;
  switch (g_bp_variant) {
    case 1: return 1;
    case 2: return tiled_ok ? 2 : -1;
    case 3: return run_ok ? 3 : -1;
    case 4: return run8_ok ? 4 : -1;
    case 6: return run8_ok ? 4 : -1;   // run8 with packed FFMA2 interpolation (measured alternative)
    case 7: return run8_ok ? 4 : -1;   // run16 forced where it covers the stack (else run8)
    // one slice group (<= 4 slices): the 8-slice kernel would spend half of its FMAs on a duplicate
    default: return (run8_ok && n_slices > 4) ? 4 : (run_ok ? 3 : (tiled_ok ? 2 : 1));
  }
}

// run8 takes the slice groups in pairs; a stack with an odd number (>= 3) of groups would pay a whole duplicate group
// for the last one: the pairs go to run8, the last group to the 4-slice run kernel (12 slices: 0.96 -> 0.78 ms)
static int launch_bp_run8_auto(const float4* qi, const QiLayout& L, const BpArgs& a, const GeomPlan* plan,
                               cudaStream_t stream) {
  if (g_bp_variant == 0 && L.n_groups >= 3 && (L.n_groups & 1) && backproject_run_window(a.pixel_size) > 0) {
    QiLayout L2 = L;
    L2.n_groups = L.n_groups - 1;
    BpArgs a2 = a;
    a2.n_slices = 4 * L2.n_groups;
    PYHST_TRY(launch_backproject_run8(qi, L2, a2, plan->d_run, plan->n_a, plan->n_b, stream));
    QiLayout L1 = L;
    L1.n_groups = 1;
    BpArgs a1 = a;
    a1.n_slices = a.n_slices - a2.n_slices;
    a1.d_img = a.d_img + (int64_t)a2.n_slices * a.nx * a.ny;
    return launch_backproject_run(qi + (int64_t)L2.n_groups * L.group_f4(), L1, a1, plan->d_run, plan->n_a, plan->n_b,
                                  stream);
  }
  return launch_backproject_run8(qi, L, a, plan->d_run, plan->n_a, plan->n_b, stream);
}

}  // namespace pyhst

using namespace pyhst;

extern "C" {

const char* pyhst_last_error(void) { return last_error_buf(); }

int pyhst_profile_enable(int enable) {
  std::lock_guard<std::mutex> lock(g_prof_mu);
  const int prev = g_prof_on ? 1 : 0;
  g_prof_on = enable != 0;
  return prev;
}

int pyhst_profile_read(double* ms, int64_t* kernels, int64_t* fft_execs, int32_t reset) {
  std::lock_guard<std::mutex> lock(g_prof_mu);
  for (auto& ev : g_prof_pending) {
    PYHST_CUDA_TRY(cudaEventSynchronize(ev.b));
    float t = 0.f;
    PYHST_CUDA_TRY(cudaEventElapsedTime(&t, ev.a, ev.b));
    g_prof_ms[ev.st] += (double)t;
    g_prof_pool[ev.dev].push_back(ev.a);
    g_prof_pool[ev.dev].push_back(ev.b);
  }
  g_prof_pending.clear();
  for (int i = 0; i < ST_COUNT; ++i) {
    if (ms) ms[i] = g_prof_ms[i];
    if (kernels) kernels[i] = g_prof_kernels[i];
    if (fft_execs) fft_execs[i] = g_prof_fft[i];
    if (reset) { g_prof_ms[i] = 0; g_prof_kernels[i] = 0; g_prof_fft[i] = 0; }
  }
  return PYHST_OK;
}

int pyhst_set_backproject_variant(int variant) {
  const int prev = g_bp_variant;
  if (variant >= 0 && variant <= 7 && variant != 5) g_bp_variant = variant;
  return prev;
}

int64_t pyhst_test_set_workspace_limit(int64_t max_bytes) { return g_ws_limit.exchange(max_bytes < 0 ? 0 : max_bytes); }

int pyhst_set_halfacq_stitch(int enable) {
  const int prev = g_halfacq_stitch;
  if (enable == 0 || enable == 1) g_halfacq_stitch = enable;
  return prev;
}

int pyhst_set_patch_gemm_variant(int variant) {
  const int prev = g_patch_gemm_variant;
  if (variant >= 0 && variant <= 2) g_patch_gemm_variant = variant;
  return prev;
}

int pyhst_set_filter_variant(int variant) {
  const int prev = g_filter_variant;
  if (variant >= 0 && variant <= 2) g_filter_variant = variant;
  return prev;
}

int pyhst_set_forward_project_variant(int variant) {
  const int prev = g_fp_variant;
  if (variant >= 0 && variant <= 5) g_fp_variant = variant;
  return prev;
}

int pyhst_last_forward_project_kernel(void) { return g_last_fp_kernel; }

int pyhst_test_fd_plan(const pyhst_geom_t* g, int32_t* info, int32_t* chunk_of, int32_t* ranges) {
  int64_t pitch = 0;
  PYHST_TRY(check_geom(g, &pitch));
  if (!info) return set_error(PYHST_ERR_INVALID_ARG, "info is NULL");
  FdPlan pl;
  std::vector<FdProj> projs;
  std::vector<FdChunk> chunks;
  std::vector<int32_t> rg, legacy;
  const bool ok = build_fd_tables(g, &pl, &projs, &chunks, &rg, &legacy);
  int32_t nb = 0, npj = 0;
  fd_block_shape(&nb, &npj);
  info[0] = ok ? pl.n_chunks : 0;
  info[1] = (int32_t)legacy.size();
  info[2] = pl.W;
  info[3] = pl.n_bx;
  info[4] = nb;
  info[5] = npj;
  info[6] = pl.zpad;
  info[7] = pl.n_lines_alloc;
  if (chunk_of) {
    for (int p = 0; p < g->n_angles; ++p) chunk_of[p] = -1;
    for (size_t c = 0; c < chunks.size(); ++c)
      for (int q = 0; q < chunks[c].count; ++q) chunk_of[projs[chunks[c].first + q].p] = (int32_t)c;
  }
  if (ranges && ok) std::memcpy(ranges, rg.data(), rg.size() * sizeof(int32_t));
  if (!ok) return set_error(PYHST_ERR_UNSUPPORTED, "diagonal-line forward projector covers no projection of this geometry");
  return PYHST_OK;
}

void pyhst_release_cache(void) {
  int prev = current_device();
  std::vector<DeviceCtx*> all;
  {
    std::lock_guard<std::mutex> lock(g_map_mu);
    for (auto& kv : g_ctx) all.push_back(kv.second.get());
  }
  for (DeviceCtx* c : all) {
    std::lock_guard<std::recursive_mutex> lock(c->mu);
    if (cudaSetDevice(c->device) != cudaSuccess) { cudaGetLastError(); continue; }
    cudaDeviceSynchronize();
    for (auto& pl : c->fp_plans) {
      cudaFree(pl.d_projs);
      cudaFree(pl.d_chunks);
      cudaFree(pl.fd.d_projs);
      cudaFree(pl.fd.d_chunks);
      cudaFree(pl.fd.d_ranges);
    }
    c->fp_plans.clear();
    for (auto& pl : c->geom) {
      cudaFree(pl.d_proj);
      cudaFree(pl.d_run);
      cudaFree(pl.d_flip);
      cudaFreeHost(pl.h_pinned);
    }
    c->geom.clear();
    for (int i = 0; i < WS_COUNT; ++i) {
      if (c->ws[i].p) cudaFree(c->ws[i].p);
      c->ws[i].p = nullptr;
      c->ws[i].bytes = 0;
      ++c->ws[i].gen;
    }
    for (auto& st : c->streams) if (st) { cudaStreamDestroy(st); st = nullptr; }
    for (auto& e : c->events) if (e) { cudaEventDestroy(e); e = nullptr; }
    if (c->last_done) { cudaEventDestroy(c->last_done); c->last_done = nullptr; }
    c->have_last = false;
    // while c->mu is still held: a call in flight on another thread may have copied a table pointer or a
    // cuFFT handle out of the maps and be about to launch with it
    release_filter_plans(c->device);
  }
  if (prev >= 0) cudaSetDevice(prev);
  cudaGetLastError();
}

int pyhst_halfacq_extent(int32_t n_bins, double cbar, int32_t* n_bins_ext, int32_t* pad_left) {
  if (n_bins <= 0 || !n_bins_ext || !pad_left || !std::isfinite(cbar))
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_halfacq_extent: bad argument");
  // R10: the virtual detector is symmetric about the mean axis and reaches as far as
  // the longer physical side does.  Distances from the axis to the two detector edges:
  const double to_first_bin = cbar, to_last_bin = (double)(n_bins - 1) - cbar;
  const bool long_side_is_left = to_first_bin >= to_last_bin;   // i.e. the axis sits right of centre
  const double reach = std::fmax(to_first_bin, to_last_bin);
  // bins -reach .. +reach about the axis, never shorter than the physical row; rounded up to whole
  // 64-bin units so that the extended rows stay 16-byte aligned for the bulk copies
  int64_t n_virtual = (int64_t)std::ceil(reach + reach) + 1;
  n_virtual = std::max<int64_t>(n_virtual, n_bins);
  const int64_t n_units = (n_virtual + 63) >> 6;
  if (n_units > (1 << 14)) return set_error(PYHST_ERR_INVALID_ARG, "axis too far off the detector");
  *n_bins_ext = (int32_t)(n_units << 6);
  // the physical row keeps its place when the missing half lies to its right (long side left),
  // and is pushed to the far end of the extended row when the missing half lies to its left
  *pad_left = long_side_is_left ? 0 : *n_bins_ext - n_bins;
  return PYHST_OK;
}

int pyhst_ramp_filter(const float* d_in, float* d_out, int64_t n_rows, int32_t n_bins_in,
                      int32_t n_bins_out, int32_t pad_left, int64_t out_pitch, pyhst_filter_t f,
                      const float* d_col_weights, void* stream) {
  if (n_rows == 0 && n_bins_in > 0 && n_bins_out >= n_bins_in + pad_left && pad_left >= 0)
    return PYHST_OK;  // empty stack: nothing to read or write (pointers may be NULL)
  PYHST_TRY(check_ptr(d_in, "d_in"));
  PYHST_TRY(check_ptr(d_out, "d_out"));
  if (d_col_weights) PYHST_TRY(check_ptr(d_col_weights, "d_col_weights"));
  if (n_rows < 0 || n_bins_in <= 0 || n_bins_out <= 0 || pad_left < 0)
    return set_error(PYHST_ERR_INVALID_ARG, "pyhst_ramp_filter: sizes must be positive");
  if (n_bins_out < n_bins_in + pad_left)
    return set_error(PYHST_ERR_INVALID_ARG, "n_bins_out %d < n_bins_in %d + pad_left %d", n_bins_out,
                     n_bins_in, pad_left);
  if (out_pitch == 0) out_pitch = n_bins_out;
  if (out_pitch < n_bins_out)
    return set_error(PYHST_ERR_INVALID_ARG, "out_pitch %lld < n_bins_out %d", (long long)out_pitch,
                     n_bins_out);
  if ((int)f < PYHST_FILTER_RAMLAK || (int)f > PYHST_FILTER_COSINE)
    return set_error(PYHST_ERR_INVALID_ARG, "unknown filter %d", (int)f);
  if ((int64_t)n_bins_in + n_bins_out > 16384)
    return set_error(PYHST_ERR_UNSUPPORTED, "n_bins_in + n_bins_out > 16384");
  PYHST_TRY(require_sm100(nullptr));
  PYHST_CALL_SCOPE(static_cast<cudaStream_t>(stream));
  return launch_ramp_filter(d_in, n_bins_in, n_rows, n_bins_in, n_bins_out, pad_left, (int)f,
                            d_col_weights, d_out, out_pitch, nullptr, nullptr, 0, nullptr,
                            static_cast<cudaStream_t>(stream));
}

int pyhst_backproject(const float* d_sino, float* d_img, const pyhst_geom_t* g, float scale,
                      void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  int64_t pitch = 0;
  PYHST_TRY(check_ptr(d_sino, "d_sino"));
  PYHST_TRY(check_ptr(d_img, "d_img"));
  PYHST_TRY(check_geom(g, &pitch));
  PYHST_TRY(require_sm100(nullptr));
  PYHST_CALL_SCOPE(stream);
  const GeomPlan* plan = nullptr;
  PYHST_TRY(get_geom_plan(g, 0.0, g->n_bins, stream, &plan));
  BpArgs a{d_img, g->n_slices, g->n_angles, g->n_bins, g->nx, g->ny, scale, plan->d_proj,
           g->pixel_size};
  const int kern = pick_bp_kernel(g->pixel_size, g->n_slices);
  if (kern < 0)
    return set_error(PYHST_ERR_UNSUPPORTED, "backprojector variant %d does not cover pixel_size %g",
                     g_bp_variant.load(), g->pixel_size);
  if (kern == 1) return launch_backproject_reference(d_sino, pitch, a, stream);
  const QiLayout L = qi_layout(g->n_slices, g->n_angles, g->n_bins, g->pixel_size);
  void* qi = nullptr;
  PYHST_TRY(get_workspace(WS_QI, L.bytes(), &qi));
  PYHST_TRY(launch_repack_to_qi(d_sino, pitch, g->n_slices, static_cast<float4*>(qi), L,
                                kern >= 3 ? plan->d_flip : nullptr, stream));
  if (kern == 4) return launch_bp_run8_auto(static_cast<const float4*>(qi), L, a, plan, stream);
  if (kern == 3)
    return launch_backproject_run(static_cast<const float4*>(qi), L, a, plan->d_run, plan->n_a, plan->n_b,
                                  stream);
  return launch_backproject_tiled(static_cast<const float4*>(qi), L, a, stream);
}

int pyhst_forward_project(const float* d_img, float* d_sino, const pyhst_geom_t* g, float scale,
                          void* stream_) {
  cudaStream_t stream = static_cast<cudaStream_t>(stream_);
  int64_t pitch = 0;
  PYHST_TRY(check_ptr(d_img, "d_img"));
  PYHST_TRY(check_ptr(d_sino, "d_sino"));
  PYHST_TRY(check_geom(g, &pitch));
  PYHST_TRY(require_sm100(nullptr));
  PYHST_CALL_SCOPE(stream);
  const int fp_variant = g_fp_variant.load();   // one choice per call
  const GeomPlan* plan = nullptr;
  PYHST_TRY(get_geom_plan(g, 0.0, g->n_bins, stream, &plan));
  if (fp_variant != 1) {
    const FpPlan* fplan = nullptr;
    PYHST_TRY(get_fp_plan(g, stream, fp_variant == 5 ? 2 : (fp_variant == 0 ? 1 : 0), &fplan));
    if (fplan->diag && fp_variant == 0) {
      // automatic choice: the diagonal-line kernel needs two sheared copies of the stack (about 4.6x its size,
      // see pyhst.h).  If that block cannot be had, the banded kernel (about 2x) still can run: take its plan.
      void* xd = nullptr;
      if (get_workspace(WS_XD, fd_xd_bytes(fplan->fd, g, nullptr), &xd) == PYHST_ERR_NOMEM)
        PYHST_TRY(get_fp_plan(g, stream, 0, &fplan));
    }
    if (fplan->diag) {
      g_last_fp_kernel = 5;
      PYHST_TRY(launch_forward_project_diag(d_img, d_sino, pitch, g, scale, fplan->fd, stream));
      if (fplan->n_chunks > 0)
        return launch_forward_project_banded(d_img, d_sino, pitch, g, scale, *fplan, 0, stream);
      return PYHST_OK;
    }
    if (fp_variant == 5)
      return set_error(PYHST_ERR_UNSUPPORTED, "diagonal-line forward projector does not cover this geometry");
    if (fplan->n_chunks > 0) {
      g_last_fp_kernel = fp_variant == 3 || fp_variant == 4 ? fp_variant : 2;
      return launch_forward_project_banded(d_img, d_sino, pitch, g, scale, *fplan, fp_variant == 3 ? 1 : (fp_variant == 4 ? 2 : 0), stream);
    }
    if (fp_variant == 2)
      return set_error(PYHST_ERR_UNSUPPORTED, "banded forward projector does not cover pixel_size %g",
                       g->pixel_size);
  }
  g_last_fp_kernel = 1;
  void* img_t = nullptr;
  PYHST_TRY(get_workspace(WS_IMG_T, (size_t)g->n_slices * g->nx * g->ny * 4, &img_t));
  PYHST_TRY(launch_transpose_images(d_img, static_cast<float*>(img_t), g->n_slices, g->ny, g->nx,
                                    stream));
  FpArgs a{d_img, static_cast<const float*>(img_t), d_sino, pitch, g->n_slices, g->n_angles,
           g->n_bins, g->nx, g->ny, scale, plan->d_proj};
  return launch_forward_project(a, stream);
}

// FBP of slices [s0, s0 + ns) of a device stack; d_img points at slice s0's image.
static int fbp_device(const float* d_sino_raw, int64_t pitch, float* d_img, const pyhst_geom_t* g,
                      int32_t ns, pyhst_filter_t f, pyhst_scan_t mode, cudaStream_t stream) {
  const double PI = 3.14159265358979323846264338327950288;
  int32_t b_out = g->n_bins, pad_left = 0;
  const float* d_w = nullptr;
  double scale = PI / (double)g->n_angles;
  if (mode == PYHST_SCAN_360_HALF) {
    double cbar = 0.0;
    for (int32_t p = 0; p < g->n_angles; ++p) cbar += g->axis_pos[p];
    cbar /= (double)g->n_angles;
    const double mid = 0.5 * (double)(g->n_bins - 1);
    const double omega = cbar >= mid ? (double)(g->n_bins - 1) - cbar : cbar;
    if (!(omega > 0.0))
      return set_error(PYHST_ERR_INVALID_ARG, "half acquisition: mean axis %g is off the detector", cbar);
    PYHST_TRY(pyhst_halfacq_extent(g->n_bins, cbar, &b_out, &pad_left));
    void* w = nullptr;
    PYHST_TRY(get_workspace(WS_WEIGHTS, (size_t)g->n_bins * 4, &w));
    PYHST_TRY(launch_halfacq_weights(static_cast<float*>(w), g->n_bins, cbar, stream));
    d_w = static_cast<const float*>(w);
    scale = 2.0 * PI / (double)g->n_angles;
  }
  if ((int64_t)g->n_bins + b_out > 16384)
    return set_error(PYHST_ERR_UNSUPPORTED, "n_bins + filtered row length > 16384");
  if (mode == PYHST_SCAN_360_HALF && g_halfacq_stitch && g_bp_variant != 1) {
    // N2: projections p and p + P/2 face each other (angles differ by pi, same axis, 2c integer):
    // fold the scan into P/2 full-width rows and backproject half as many projections (filter.cu)
    const int32_t P2 = g->n_angles / 2;
    bool ok = g->n_angles % 2 == 0 && P2 > 0;
    std::vector<int> two_c((size_t)std::max(P2, 1));
    int lo = 0, hi = b_out - 1;  // range of bins the folded rows must hold
    for (int32_t p = 0; ok && p < P2; ++p) {
      const double c2 = 2.0 * (g->axis_pos[p] + (double)pad_left);
      ok = std::fabs(g->angles_rad[p + P2] - g->angles_rad[p] - PI) <= 1e-10 &&
           g->axis_pos[p + P2] == g->axis_pos[p] && std::fabs(c2 - std::nearbyint(c2)) <= 1e-9 &&
           std::fabs(c2) < 1e6;
      if (!ok) break;
      two_c[p] = (int)std::nearbyint(c2);
      lo = std::min(lo, two_c[p] - (b_out - 1));
      hi = std::max(hi, two_c[p]);
    }
    const int32_t off = -lo, b_st = hi - lo + 1;
    if (ok && b_st <= 16384) {
      const int64_t P = g->n_angles;
      void *r1 = nullptr, *r2 = nullptr;
      const size_t r2_bytes = (((size_t)ns * P2 * b_st * 4) + 255) & ~(size_t)255;
      PYHST_TRY(get_workspace(WS_ROWS, (size_t)ns * P * b_out * 4, &r1));
      PYHST_TRY(get_workspace(WS_STITCH, r2_bytes + (size_t)P2 * sizeof(int), &r2));
      int* d_two_c = reinterpret_cast<int*>(static_cast<char*>(r2) + r2_bytes);
      PYHST_CUDA_TRY(cudaMemcpyAsync(d_two_c, two_c.data(), (size_t)P2 * sizeof(int), cudaMemcpyHostToDevice,
                                     stream));
      // rows of the whole stack are equally pitched: one call filters all ns * P of them
      PYHST_TRY(launch_ramp_filter(d_sino_raw, pitch, (int64_t)ns * P, g->n_bins, b_out, pad_left, (int)f, d_w,
                                   static_cast<float*>(r1), b_out, nullptr, nullptr, 0, nullptr, stream));
      PYHST_TRY(launch_halfacq_fold(static_cast<const float*>(r1), static_cast<float*>(r2), ns, P2, b_out,
                                    b_st, off, d_two_c, stream));
      std::vector<double> axis2((size_t)P2);
      for (int32_t p = 0; p < P2; ++p) axis2[p] = g->axis_pos[p] + (double)pad_left + (double)off;
      pyhst_geom_t g2 = *g;
      g2.n_slices = ns;
      g2.n_angles = P2;
      g2.n_bins = b_st;
      g2.sino_pitch = 0;
      g2.axis_pos = axis2.data();
      return pyhst_backproject(static_cast<const float*>(r2), d_img, &g2, (float)scale, stream);
    }
  }
  const GeomPlan* plan = nullptr;
  PYHST_TRY(get_geom_plan(g, (double)pad_left, b_out, stream, &plan));
  BpArgs a{d_img, ns, g->n_angles, b_out, g->nx, g->ny, (float)scale, plan->d_proj, g->pixel_size};
  const int64_t P = g->n_angles;
  const int kern = pick_bp_kernel(g->pixel_size, ns);
  if (kern < 0)
    return set_error(PYHST_ERR_UNSUPPORTED, "backprojector variant %d does not cover pixel_size %g",
                     g_bp_variant.load(), g->pixel_size);
  if (kern == 1) {
    void* rows = nullptr;
    PYHST_TRY(get_workspace(WS_ROWS, (size_t)ns * P * b_out * 4, &rows));
    PYHST_TRY(launch_ramp_filter(d_sino_raw, pitch, (int64_t)ns * P, g->n_bins, b_out, pad_left, (int)f, d_w,
                                 static_cast<float*>(rows), b_out, nullptr, nullptr, 0, nullptr, stream));
    return launch_backproject_reference(static_cast<const float*>(rows), b_out, a, stream);
  }
  const QiLayout L = qi_layout(ns, g->n_angles, b_out, g->pixel_size);
  void* qi = nullptr;
  PYHST_TRY(get_workspace(WS_QI, L.bytes(), &qi));
  if (filter_variant() != 1 && ramp_fused_log2m(b_out)) {
    // fused filter: every slice group in one launch, written straight into the interleaved layout
    PYHST_TRY(launch_ramp_filter_fused(d_sino_raw, pitch, (int64_t)ns * P, g->n_bins, b_out, pad_left, (int)f, d_w,
                                       nullptr, 0, static_cast<float4*>(qi), &L, ns,
                                       kern >= 3 ? plan->d_flip : nullptr, stream));
  } else {
    for (int32_t grp = 0; grp < L.n_groups; ++grp) {
      const int32_t n_in = std::min(4, ns - grp * 4);
      PYHST_TRY(launch_ramp_filter(d_sino_raw + (int64_t)grp * 4 * P * pitch, pitch, (int64_t)n_in * P,
                                   g->n_bins, b_out, pad_left, (int)f, d_w, nullptr, 0,
                                   static_cast<float4*>(qi) + (int64_t)grp * L.group_f4(), &L, n_in,
                                   kern >= 3 ? plan->d_flip : nullptr, stream));
    }
  }
  if (kern == 4) return launch_bp_run8_auto(static_cast<const float4*>(qi), L, a, plan, stream);
  if (kern == 3)
    return launch_backproject_run(static_cast<const float4*>(qi), L, a, plan->d_run, plan->n_a, plan->n_b,
                                  stream);
  return launch_backproject_tiled(static_cast<const float4*>(qi), L, a, stream);
}

static int check_fbp(const pyhst_geom_t* g, pyhst_filter_t f, pyhst_scan_t mode, int64_t* pitch) {
  PYHST_TRY(check_geom(g, pitch));
  if ((int)f < PYHST_FILTER_RAMLAK || (int)f > PYHST_FILTER_COSINE)
    return set_error(PYHST_ERR_INVALID_ARG, "unknown filter %d", (int)f);
  if (mode != PYHST_SCAN_180 && mode != PYHST_SCAN_360 && mode != PYHST_SCAN_360_HALF)
    return set_error(PYHST_ERR_INVALID_ARG, "unknown scan mode %d", (int)mode);
  return require_sm100(nullptr);
}

int pyhst_fbp(const float* d_sino_raw, float* d_img, const pyhst_geom_t* g, pyhst_filter_t f,
              pyhst_scan_t mode, void* stream) {
  int64_t pitch = 0;
  PYHST_TRY(check_ptr(d_sino_raw, "d_sino_raw"));
  PYHST_TRY(check_ptr(d_img, "d_img"));
  PYHST_TRY(check_fbp(g, f, mode, &pitch));
  PYHST_CALL_SCOPE(static_cast<cudaStream_t>(stream));
  return fbp_device(d_sino_raw, pitch, d_img, g, g->n_slices, f, mode, static_cast<cudaStream_t>(stream));
}

}  // extern "C"

// Host-buffer pipeline shared by the *_host entry points: the stack is cut into chunks of
// `chunk` slices; H2D of chunk n+1 and D2H of chunk n-1 overlap the kernels of chunk n
// (three internal streams ordered after `user`, double-buffered device blocks).
template <class Body>
static int host_pipeline(const float* h_in, size_t in_floats_per_slice, float* h_out,
                         size_t out_floats_per_slice, int32_t n_slices, int32_t chunk,
                         cudaStream_t user, Body body) {
  PYHST_CALL_SCOPE(user);   // the device's lock is held until the pipeline has drained
  DeviceCtx& c = *_call_scope.ctx;
  const size_t in_bytes = (size_t)chunk * in_floats_per_slice * 4;
  const size_t out_bytes = (size_t)chunk * out_floats_per_slice * 4;
  for (int i = 0; i < 3; ++i)
    if (!c.streams[i]) PYHST_CUDA_TRY(cudaStreamCreateWithFlags(&c.streams[i], cudaStreamNonBlocking));
  for (int i = 0; i < 8; ++i)
    if (!c.events[i]) PYHST_CUDA_TRY(cudaEventCreateWithFlags(&c.events[i], cudaEventDisableTiming));
  cudaStream_t s_in = c.streams[0], s_k = c.streams[1], s_out = c.streams[2];
  void *d_in[2], *d_out[2];
  void* blk = nullptr;
  PYHST_TRY(get_workspace(WS_CHUNKS, 2 * in_bytes + 2 * out_bytes, &blk));
  d_in[0] = blk;
  d_in[1] = static_cast<char*>(blk) + in_bytes;
  d_out[0] = static_cast<char*>(blk) + 2 * in_bytes;
  d_out[1] = static_cast<char*>(blk) + 2 * in_bytes + out_bytes;
  cudaEvent_t ev_start = c.events[0];
  cudaEvent_t ev_in[2] = {c.events[1], c.events[2]}, ev_k[2] = {c.events[3], c.events[4]},
              ev_out[2] = {c.events[5], c.events[6]};
  // the enqueue loop; whatever it returns, the copies it has started are drained below, so that no
  // DMA touches the caller's host buffers after the call has returned (also on error)
  auto enqueue = [&]() -> int {
    PYHST_CUDA_TRY(cudaEventRecord(ev_start, user));
    for (int i = 0; i < 3; ++i) PYHST_CUDA_TRY(cudaStreamWaitEvent(c.streams[i], ev_start, 0));
    int n = 0;
    for (int32_t s0 = 0; s0 < n_slices; s0 += chunk, ++n) {
      const int32_t ns = std::min(chunk, n_slices - s0);
      const int b = n & 1;
      if (n >= 2) PYHST_CUDA_TRY(cudaStreamWaitEvent(s_in, ev_k[b], 0));   // kernels of chunk n-2 read d_in[b]
      PYHST_CUDA_TRY(cudaMemcpyAsync(d_in[b], h_in + (size_t)s0 * in_floats_per_slice,
                                     (size_t)ns * in_floats_per_slice * 4, cudaMemcpyHostToDevice, s_in));
      PYHST_CUDA_TRY(cudaEventRecord(ev_in[b], s_in));
      PYHST_CUDA_TRY(cudaStreamWaitEvent(s_k, ev_in[b], 0));
      if (n >= 2) PYHST_CUDA_TRY(cudaStreamWaitEvent(s_k, ev_out[b], 0));  // D2H of chunk n-2 reads d_out[b]
      PYHST_TRY(body(static_cast<const float*>(d_in[b]), static_cast<float*>(d_out[b]), ns, s_k));
      PYHST_CUDA_TRY(cudaEventRecord(ev_k[b], s_k));
      PYHST_CUDA_TRY(cudaStreamWaitEvent(s_out, ev_k[b], 0));
      PYHST_CUDA_TRY(cudaMemcpyAsync(h_out + (size_t)s0 * out_floats_per_slice, d_out[b],
                                     (size_t)ns * out_floats_per_slice * 4, cudaMemcpyDeviceToHost, s_out));
      PYHST_CUDA_TRY(cudaEventRecord(ev_out[b], s_out));
    }
    return PYHST_OK;
  };
  const int rc = enqueue();
  cudaError_t drain = cudaSuccess;
  for (int i = 0; i < 3; ++i) {
    cudaError_t e = cudaStreamSynchronize(c.streams[i]);
    if (e != cudaSuccess && drain == cudaSuccess) drain = e;
  }
  {
    cudaError_t e = cudaStreamSynchronize(user);
    if (e != cudaSuccess && drain == cudaSuccess) drain = e;
  }
  if (rc != PYHST_OK) return rc;
  if (drain != cudaSuccess)
    return set_error(PYHST_ERR_CUDA, "host pipeline: %s while draining the copies", cudaGetErrorString(drain));
  return PYHST_OK;
}

// chunk = a multiple of 4 slices (one slice group of the interleaved layout)
static int32_t host_chunk(int32_t requested, int32_t n_slices) {
  int32_t chunk = requested > 0 ? requested : 8;
  chunk = std::max(4, (chunk / 4) * 4);
  return std::min(chunk, ((n_slices + 3) / 4) * 4);
}

extern "C" {

int pyhst_fbp_host(const float* h_sino_raw, float* h_img, const pyhst_geom_t* g, pyhst_filter_t f,
                   pyhst_scan_t mode, int32_t max_slices_per_chunk, void* stream_) {
  int64_t pitch = 0;
  PYHST_TRY(check_ptr(h_sino_raw, "h_sino_raw"));
  PYHST_TRY(check_ptr(h_img, "h_img"));
  PYHST_TRY(check_fbp(g, f, mode, &pitch));
  return host_pipeline(
      h_sino_raw, (size_t)g->n_angles * pitch, h_img, (size_t)g->nx * g->ny, g->n_slices,
      host_chunk(max_slices_per_chunk, g->n_slices), static_cast<cudaStream_t>(stream_),
      [&](const float* d_in, float* d_out, int32_t ns, cudaStream_t s) {
        pyhst_geom_t gc = *g;
        gc.n_slices = ns;
        return fbp_device(d_in, pitch, d_out, &gc, ns, f, mode, s);
      });
}

int pyhst_backproject_host(const float* h_sino, float* h_img, const pyhst_geom_t* g, float scale,
                           int32_t max_slices_per_chunk, void* stream_) {
  int64_t pitch = 0;
  PYHST_TRY(check_ptr(h_sino, "h_sino"));
  PYHST_TRY(check_ptr(h_img, "h_img"));
  PYHST_TRY(check_geom(g, &pitch));
  PYHST_TRY(require_sm100(nullptr));
  return host_pipeline(
      h_sino, (size_t)g->n_angles * pitch, h_img, (size_t)g->nx * g->ny, g->n_slices,
      host_chunk(max_slices_per_chunk, g->n_slices), static_cast<cudaStream_t>(stream_),
      [&](const float* d_in, float* d_out, int32_t ns, cudaStream_t s) {
        pyhst_geom_t gc = *g;
        gc.n_slices = ns;
        return pyhst_backproject(d_in, d_out, &gc, scale, s);
      });
}

int pyhst_forward_project_host(const float* h_img, float* h_sino, const pyhst_geom_t* g, float scale,
                               int32_t max_slices_per_chunk, void* stream_) {
  int64_t pitch = 0;
  PYHST_TRY(check_ptr(h_img, "h_img"));
  PYHST_TRY(check_ptr(h_sino, "h_sino"));
  PYHST_TRY(check_geom(g, &pitch));
  PYHST_TRY(require_sm100(nullptr));
  return host_pipeline(
      h_img, (size_t)g->nx * g->ny, h_sino, (size_t)g->n_angles * pitch, g->n_slices,
      host_chunk(max_slices_per_chunk, g->n_slices), static_cast<cudaStream_t>(stream_),
      [&](const float* d_in, float* d_out, int32_t ns, cudaStream_t s) {
        pyhst_geom_t gc = *g;
        gc.n_slices = ns;
        return pyhst_forward_project(d_in, d_out, &gc, scale, s);
      });
}

}  // extern "C"
